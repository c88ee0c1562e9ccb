// kx_contract.cu -- the exact streaming path as ONE fused kernel per operator evaluation, and the small kernels around it.
//
//   k_stream   a4-a5 (contract_group: one exp per entry and member in LOG mode) -> grid barrier -> a6-a8 (finish_member)
//   k_moments  a9  moments                                                         eq. B.2
//   k_adapt_*  accept / reject and the step-size controller of kx_evolve_adaptive  Sec. 4.2
//   k_delta_source  monoenergetic source deposition
//
// The device code of the contraction and of the finishing phase lives in kx_device.cuh (shared with the tensor-core
// kernel, whose exact fallback and finishing phase are the same code).
//
// Compiled with --fmad=false; every fused multiply-add is an explicit fma().
#include "kx_device.cuh"
#include <stdlib.h>

namespace {

using namespace kxd;

// barrier and finishing phase, NQ = ceil(N / 256) rows per thread
template <int NQ>
__device__ __forceinline__ void stream_tail(const KxDev& d, const double* __restrict__ f, int B, const KxStage& st,
                                            unsigned char* smem_raw, double* s_red)
{
    const unsigned cta = blockIdx.y * gridDim.x + blockIdx.x, nctas = gridDim.x * gridDim.y;
    FinishPre<NQ> pre;
    if ((int)cta < B) finish_preload<NQ>(d, f, (int)cta, pre);    // static inputs of the finishing phase: before the barrier
    grid_barrier_count(st.bar + 3, st.bar_target);
    if (threadIdx.x == 0) stamp(st.trace, 2);
    for (int b = (int)cta; b < B; b += (int)nctas)
        finish_member<NQ>(d, f, B, st, nullptr, false, b, reinterpret_cast<double*>(smem_raw), s_red, b == (int)cta ? &pre : nullptr);
}

// grid (gx, gy): CTA (x, y) takes the member groups y, y + gy, ... and of each the tasks x, x + gx, ...; after the grid
// barrier CTA c = y gx + x finishes the members c, c + gx gy, ...
template <int BT, int MODE, int QS>
__global__ void __launch_bounds__(KX_CTA, 2)
k_stream(KxDev d, const double* __restrict__ f, const double2* __restrict__ yd, int B, KxStage st)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_red[8 * 8];
    if (threadIdx.x == 0) stamp(st.trace, 0);
    const int groups = (B + BT - 1) / BT;
    for (int g = blockIdx.y; g < groups; g += gridDim.y)
        contract_any<BT, MODE, QS>(d, f, yd, st.part, B, g * BT, blockIdx.x, gridDim.x, smem_raw);
    if (threadIdx.x == 0) stamp(st.trace, 1);
    if (d.N <= KX_CTA) stream_tail<1>(d, f, B, st, smem_raw, s_red);
    else if (d.N <= 2 * KX_CTA) stream_tail<2>(d, f, B, st, smem_raw, s_red);
    else stream_tail<4>(d, f, B, st, smem_raw, s_red);
    if (threadIdx.x == 0) stamp(st.trace, 3);
}

// ---------------------------------------------------------------- a whole fixed-step integration in ONE launch
// Small problems (configs 1 and 2: a stage is a few microseconds of work) are bound by the kernel launch and its grid
// barrier when every Runge-Kutta stage is its own launch.  k_stream_run keeps the grid resident for all S steps of
// kx_evolve (static mass, no per-step diagnostics): per stage, contraction -> grid barrier -> finishing phase (which writes
// the next stage input and its y) -> grid barrier.  The step data (tau, rate, source amplitudes) is read from device
// arrays; the barriers use the growing counter, one target per barrier.
struct KxRun {
    int method, S;            // KX_EULER | KX_HEUN | KX_RK4, number of steps
    const double* tau;        // device [S+1]
    const double* rate;       // device [2S+1] or null
    const double* amp;        // device [nsrc, S] or null
};

template <int BT, int MODE, int QS, int NQ>
__device__ __forceinline__ void stream_run(const KxDev& d, double* __restrict__ f, int B, const KxStage& st0, const KxRun& run,
                                           unsigned char* smem_raw, double* s_red)
{
    const unsigned cta = blockIdx.y * gridDim.x + blockIdx.x, nctas = gridDim.x * gridDim.y;
    const int groups = (B + BT - 1) / BT;
    const int nstage = run.method == KX_EULER ? 1 : (run.method == KX_HEUN ? 2 : 4);
    KxStage st = st0;
    unsigned target = st0.bar_target;                 // value of the counter after the first barrier of this launch
    bool have_yd = false;
    for (int k = 0; k < run.S; ++k) {
        const double t0 = run.tau[k], t1 = run.tau[k + 1];
        st.dt = t1 - t0;
        for (int q = 0; q < st.nsrc; ++q) st.amp[q] = run.amp[(size_t)q * run.S + k];
        for (int stg = 0; stg < nstage; ++stg) {
            int pos;                                  // node (0), midpoint (1) or end (2) of the step for this stage
            if (run.method == KX_EULER) pos = 0;
            else if (run.method == KX_HEUN) pos = stg == 0 ? 0 : 2;
            else pos = stg == 0 ? 0 : (stg == 3 ? 2 : 1);
            st.rate = run.rate ? run.rate[2 * k + pos] : 1.0;
            st.rk_stage = stg;
            const double* fin = stg == 0 ? f : st.fstage;
            const double2* yd = have_yd ? reinterpret_cast<const double2*>(st.ydnext) : nullptr;
            for (int g = blockIdx.y; g < groups; g += gridDim.y)
                contract_any<BT, MODE, QS>(d, fin, yd, st.part, B, g * BT, blockIdx.x, gridDim.x, smem_raw, !have_yd);
            grid_barrier_count(st.bar + 3, target);
            target += nctas;
            // (the finishing phase's scratch, N doubles at the head of the shared memory, lies inside the per-stage y rows: the
            // tables behind them survive)
            for (int b = (int)cta; b < B; b += (int)nctas)
                finish_member<NQ>(d, fin, B, st, nullptr, false, b, reinterpret_cast<double*>(smem_raw), s_red, nullptr);
            grid_barrier_count(st.bar + 3, target);
            target += nctas;
            have_yd = true;
        }
    }
}

template <int BT, int MODE, int QS>
__global__ void __launch_bounds__(KX_CTA, 2)
k_stream_run(KxDev d, double* __restrict__ f, int B, KxStage st, KxRun run)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    __shared__ double s_red[8 * 8];
    if (d.N <= KX_CTA) stream_run<BT, MODE, QS, 1>(d, f, B, st, run, smem_raw, s_red);
    else if (d.N <= 2 * KX_CTA) stream_run<BT, MODE, QS, 2>(d, f, B, st, run, smem_raw, s_red);
    else stream_run<BT, MODE, QS, 4>(d, f, B, st, run, smem_raw, s_red);
}

// ---------------------------------------------------------------- adaptive Heun: accept / reject, controller update
// k_adapt_accept: one CTA per member; every CTA reads the same error norm and takes the same decision.
__global__ void __launch_bounds__(KX_CTA) k_adapt_accept(int N, double* __restrict__ f, const double* __restrict__ fnew,
                                                         const KxAdapt* __restrict__ ad, int* __restrict__ flag)
{
    if (ad->done) return;
    const long long k = ad->errkey;
    const double err = __longlong_as_double(k >= 0 ? k : (k ^ 0x7fffffffffffffffLL));
    if (!(err <= 1.0)) return;                                   // rejected (also when err is inf / nan)
    bool bad = false;
    for (int i = threadIdx.x; i < N; i += KX_CTA) {
        const double v = fnew[(size_t)blockIdx.x * N + i];
        f[(size_t)blockIdx.x * N + i] = v;
        if (!isfinite(v)) bad = true;
    }
    if (bad) atomicOr(flag, 1);
}

// k_adapt_ctrl: one thread.  du <- du clamp(safety / sqrt(err), 0.2, 5); accepted: u <- u + du_old, du <= u1 - u.
__global__ void k_adapt_ctrl(KxAdapt* ad, double u1, double safety)
{
    if (ad->done) return;
    const long long k = ad->errkey;
    const double err = __longlong_as_double(k >= 0 ? k : (k ^ 0x7fffffffffffffffLL));
    const bool ok = err <= 1.0;
    double fac = safety / sqrt(fmax(err, 1e-10));
    if (!(fac == fac)) fac = 0.2;                                // nan error: shrink
    fac = fmin(fmax(fac, 0.2), 5.0);
    double u = ad->u, du = ad->du;
    if (ok) { u += du; ad->accepted += 1; } else { ad->rejected += 1; }
    du *= fac;
    if (u1 - u <= 1e-14 * fmax(fabs(u1), 1.0)) { ad->done = 1; u = u1; }
    else if (du > u1 - u) du = u1 - u;
    ad->u = u; ad->du = du;
    ad->errkey = kx_dkey(0.0);
}

// ---------------------------------------------------------------- m(u) of the adaptive integrator, on the device
// comoving momenta q = a p: the kinematics of a stage at u see the mass m a, m(u) = mass0 e^{slope (u - u0)}
__global__ void k_adapt_mass(const KxAdapt* ad, int stage, double u0, double mass0, double slope, double* m_dev)
{
    const double us = stage ? ad->u + ad->du : ad->u;
    *m_dev = mass0 * exp(slope * (us - u0));
}

// ---------------------------------------------------------------- regime 1 of Sec. 4.2
// k_regime1_monitor (one CTA): Gamma_2->2 / H = kappa_b R(u) sum_i h_i loss_i / sum_i h_i f_i per member (reading D16; `loss`
// is the loss term of the operator evaluated on f with the kinematics of m(u)), the largest member decides: above eps_switch
// the batch switches to regime 2 at this u; else, at u1, the run is done; else the step that follows is taken.
__global__ void __launch_bounds__(KX_CTA)
k_regime1_monitor(KxDev d, const double* __restrict__ f, const double* __restrict__ loss, int B, const double* __restrict__ kappa,
                  KxAdapt* ad, double u0, double u1, double eps_switch, double rate0, double rate_slope)
{
    __shared__ double s_red[8 * 8];
    if (ad->switched || ad->done) return;
    const int N = d.N;
    const double u = ad->u;
    const double R = rate0 * exp(rate_slope * (u - u0));
    double ratio = 0.0;
    for (int b = 0; b < B; ++b) {
        double v[2] = {0.0, 0.0};
        for (int i = threadIdx.x; i < N; i += KX_CTA) {
            v[0] += d.h[i] * loss[(size_t)b * N + i];
            v[1] += d.h[i] * f[(size_t)b * N + i];
        }
        block_sum<2>(v, s_red);
        const double r = v[1] > 0.0 ? (kappa ? kappa[b] : 1.0) * R * (v[0] / v[1]) : 0.0;
        if (r > ratio) ratio = r;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        ad->ratio = ratio;
        if (!(eps_switch > 0.0) || ratio > eps_switch) { ad->switched = 1; ad->u_switch = u; }
        else if (u1 - u <= 1e-14 * fmax(fabs(u1), 1.0)) { ad->done = 1; ad->u = u1; }
    }
}

// k_regime1_step (one CTA per member): "we set the self-collisions to zero ... and evolve the distribution with a fourth-order
// Runge-Kutta method on fixed intervals in u": the source rates are constant in u, so the four slopes are the same vector
// k = sum_s amp_s G_s and the RK4 update is f + du k, du = min(du_fixed, u1 - u).  k_regime1_advance then moves u.
__global__ void __launch_bounds__(KX_CTA)
k_regime1_step(int N, double* __restrict__ f, int nsrc, const double* __restrict__ G, const double* __restrict__ amp,
               const KxAdapt* __restrict__ ad, double u1, double du_fixed)
{
    if (ad->switched || ad->done) return;
    const double rem = u1 - ad->u, du = du_fixed < rem ? du_fixed : rem;
    for (int i = threadIdx.x; i < N; i += KX_CTA) {
        double k = 0.0;
        for (int q = 0; q < nsrc; ++q) k += amp[q] * G[(size_t)q * N + i];
        f[(size_t)blockIdx.x * N + i] += du * k;
    }
}

__global__ void k_regime1_advance(KxAdapt* ad, double u1, double du_fixed)
{
    if (ad->switched || ad->done) return;
    const double rem = u1 - ad->u, du = du_fixed < rem ? du_fixed : rem;
    ad->u += du;
    ad->fixed_steps += 1;
}

// ---------------------------------------------------------------- monoenergetic source deposition
__global__ void __launch_bounds__(KX_CTA) k_delta_source(KxDev d, double p0, double* __restrict__ G)
{
    __shared__ int s_L;
    const int N = d.N;
    if (threadIdx.x == 0) {            // largest L <= N-2 with p_L <= p0
        int lo = 0, hi = N - 2;
        while (lo < hi) {
            int mid = (lo + hi + 1) >> 1;
            if (d.p[mid] <= p0) lo = mid; else hi = mid - 1;
        }
        s_L = lo;
    }
    __syncthreads();
    const int L = s_L;
    const double E0 = sqrt(p0 * p0 + d.m * d.m);
    const double aR = (E0 - d.E[L]) / (d.E[L + 1] - d.E[L]);      // energy-linear deposition fractions
    for (int i = threadIdx.x; i < N; i += KX_CTA)
        G[i] = i == L ? (1.0 - aR) / d.h[L] : (i == L + 1 ? aR / d.h[L + 1] : 0.0);
}

// ---------------------------------------------------------------- a9: moments, eq. B.2
__global__ void __launch_bounds__(KX_CTA)
k_moments(KxDev d, const double* __restrict__ f, double* n, double* rho, double* p1, double* p2, int stride)
{
    __shared__ double s_red[8 * 8];
    const int N = d.N, b = blockIdx.x;
    double v[4] = {0.0, 0.0, 0.0, 0.0};
    for (int i = threadIdx.x; i < N; i += KX_CTA) {
        const double hf = d.h[i] * f[(size_t)b * N + i];
        const double p = d.p[i];
        v[0] += hf;
        v[1] += hf * d.E[i];
        v[2] += hf * p;
        v[3] += hf * p * p;
    }
    block_sum<4>(v, s_red);
    if (threadIdx.x == 0) {
        const double fac = d.g_chi / (2.0 * 3.14159265358979323846 * 3.14159265358979323846);
        if (n) n[(size_t)b * stride] = fac * v[0];
        if (rho) rho[(size_t)b * stride] = fac * v[1];
        if (p1) p1[(size_t)b * stride] = v[0] != 0.0 ? v[2] / v[0] : 0.0;
        if (p2) p2[(size_t)b * stride] = v[0] != 0.0 ? v[3] / v[0] : 0.0;
    }
}

// ---------------------------------------------------------------- launchers
// Per instantiation: the dynamic shared memory limit is raised once (kx_stream_configure) and the number of CTAs that fit
// an SM at the grid's N is cached, so that a launch does no host work beyond cudaLaunchKernelEx.
struct StreamCfg { bool ready; int occ_N; int occ; };

template <int BT, int MODE, int QS>
StreamCfg& stream_cfg() { static StreamCfg c = {false, 0, 0}; return c; }

template <int BT, int MODE, int QS>
cudaError_t launch_stream_t(const KxDev& d, int sm_count, const double* f, const double* yd, int B, KxStage& st,
                            unsigned* bar_total, cudaStream_t s, const KxRun* run = nullptr)
{
    const int N = d.N;
    size_t smem = contract_smem<BT, MODE, QS>(N);
    const size_t fin = finish_scratch_bytes(N, 0, 0, 0, 0);
    if (smem < fin) smem = fin;
    StreamCfg& c = stream_cfg<BT, MODE, QS>();
    cudaError_t e;
    if (!c.ready) {
        e = cudaFuncSetAttribute(k_stream<BT, MODE, QS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024);
        if (e != cudaSuccess) return e;
        e = cudaFuncSetAttribute(k_stream_run<BT, MODE, QS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024);
        if (e != cudaSuccess) return e;
        c.ready = true;
    }
    if (c.occ_N != N) {
        int occ = 0;
        e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_stream<BT, MODE, QS>, KX_CTA, smem);
        if (e != cudaSuccess) return e;
        c.occ = occ < 1 ? 1 : occ; c.occ_N = N;
    }
    // all CTAs must be resident (grid barrier): at most occ per SM.  Small problems take fewer CTAs than that: one per
    // task is enough, and the barrier is cheaper.
    const int cap = sm_count * c.occ;
    const int groups = (B + BT - 1) / BT;
    const int gy = groups < cap ? groups : cap;
    int gx = cap / gy;
    const long long tasks_bound = (long long)N + (long long)N * ((long long)N * (N + 1) / 2) / (d.chunk > 0 ? d.chunk : 1024);
    if ((long long)gx > tasks_bound) gx = (int)tasks_bound;
    if (gx < 1) gx = 1;
    st.bar_target = *bar_total + (unsigned)(gx * gy);
    if (run) {          // the whole integration in one launch: two barriers per stage
        const unsigned nstage = run->method == KX_EULER ? 1u : (run->method == KX_HEUN ? 2u : 4u);
        const unsigned nbar = 2u * nstage * (unsigned)run->S;
        e = kx_launch_coop(k_stream_run<BT, MODE, QS>, dim3(gx, gy), dim3(KX_CTA), smem, s, d, const_cast<double*>(f), B, st, *run);
        if (e == cudaSuccess) *bar_total += nbar * (unsigned)(gx * gy);
        return e;
    }
    e = kx_launch_coop(k_stream<BT, MODE, QS>, dim3(gx, gy), dim3(KX_CTA), smem, s, d, f,
                       reinterpret_cast<const double2*>(yd), B, st);
    if (e == cudaSuccess) *bar_total = st.bar_target;
    return e;
}

template <int BT>
cudaError_t launch_stream_m(const KxDev& d, int sm_count, const double* f, const double* yd, int B, KxStage& st,
                            unsigned* bar_total, cudaStream_t s, const KxRun* run)
{
    if (d.prec == KX_FP32) {      // optional single-precision contraction (classical statistics only, checked in kx_build)
        if (d.interp == KX_INTERP_LINEAR) return launch_stream_t<BT, MODE_LINEAR_F32, 0>(d, sm_count, f, yd, B, st, bar_total, s, run);
        return launch_stream_t<BT, MODE_LOG_F32, 0>(d, sm_count, f, yd, B, st, bar_total, s, run);
    }
    if (d.eta) {         // quantum statistics: LOG interpolation only (checked in kx_build)
        if (d.exp_impl == KX_EXP_LIBM) return launch_stream_t<BT, MODE_LOG_LIBM, 1>(d, sm_count, f, yd, B, st, bar_total, s, run);
        return launch_stream_t<BT, MODE_LOG_TAB, 1>(d, sm_count, f, yd, B, st, bar_total, s, run);
    }
    if (d.interp == KX_INTERP_LINEAR) return launch_stream_t<BT, MODE_LINEAR, 0>(d, sm_count, f, yd, B, st, bar_total, s, run);
    if (d.exp_impl == KX_EXP_LIBM) return launch_stream_t<BT, MODE_LOG_LIBM, 0>(d, sm_count, f, yd, B, st, bar_total, s, run);
    return launch_stream_t<BT, MODE_LOG_TAB, 0>(d, sm_count, f, yd, B, st, bar_total, s, run);
}

}  // namespace

int kx_pick_bt(int N, int B)
{
    int cap = N > 512 ? 4 : 8;
    int bt = 1;
    while (bt < B && bt < cap) bt <<= 1;
    return bt;
}

int kx_pick_chunk(long long nnz_est, int N, int B, int sm_count)
{
    const int bt = kx_pick_bt(N, B);
    const long long groups = (B + bt - 1) / bt;
    long long c = nnz_est * groups / ((long long)sm_count * 12);
    c = (c / KX_CTA) * KX_CTA;
    if (c < 1024) c = 1024;
    if (c > 8192) c = 8192;
    return (int)c;
}

cudaError_t kx_launch_stream(const KxDev& d, int sm_count, const double* f, const double* yd, int B,
                             KxStage st, unsigned* bar_total, cudaStream_t s)
{
    switch (kx_pick_bt(d.N, B)) {
        case 1: return launch_stream_m<1>(d, sm_count, f, yd, B, st, bar_total, s, nullptr);
        case 2: return launch_stream_m<2>(d, sm_count, f, yd, B, st, bar_total, s, nullptr);
        case 4: return launch_stream_m<4>(d, sm_count, f, yd, B, st, bar_total, s, nullptr);
        default: return launch_stream_m<8>(d, sm_count, f, yd, B, st, bar_total, s, nullptr);
    }
}

cudaError_t kx_launch_stream_run(const KxDev& d, int sm_count, double* f, int B, KxStage st, int method, int S,
                                 const double* tau_dev, const double* rate_dev, const double* amp_dev,
                                 unsigned* bar_total, cudaStream_t s)
{
    KxRun run = {method, S, tau_dev, rate_dev, amp_dev};
    switch (kx_pick_bt(d.N, B)) {
        case 1: return launch_stream_m<1>(d, sm_count, f, nullptr, B, st, bar_total, s, &run);
        case 2: return launch_stream_m<2>(d, sm_count, f, nullptr, B, st, bar_total, s, &run);
        case 4: return launch_stream_m<4>(d, sm_count, f, nullptr, B, st, bar_total, s, &run);
        default: return launch_stream_m<8>(d, sm_count, f, nullptr, B, st, bar_total, s, &run);
    }
}

cudaError_t kx_launch_adapt_step(const KxDev& d, double* f, const double* fnew, int B, KxAdapt* ad, double u1, double safety,
                                 int* flag, cudaStream_t s)
{
    k_adapt_accept<<<B, KX_CTA, 0, s>>>(d.N, f, fnew, ad, flag);
    k_adapt_ctrl<<<1, 1, 0, s>>>(ad, u1, safety);
    return cudaGetLastError();
}

cudaError_t kx_launch_adapt_mass(KxAdapt* ad, int stage, double u0, double mass0, double slope, double* m_dev, cudaStream_t s)
{
    k_adapt_mass<<<1, 1, 0, s>>>(ad, stage, u0, mass0, slope, m_dev);
    return cudaGetLastError();
}

cudaError_t kx_launch_regime1_step(const KxDev& d, double* f, const double* loss, int B, const double* kappa, int nsrc,
                                   const double* G, const double* amp_dev, KxAdapt* ad, double u0, double u1, double du_fixed,
                                   double eps_switch, double rate0, double rate_slope, cudaStream_t s)
{
    k_regime1_monitor<<<1, KX_CTA, 0, s>>>(d, f, loss, B, kappa, ad, u0, u1, eps_switch, rate0, rate_slope);
    k_regime1_step<<<B, KX_CTA, 0, s>>>(d.N, f, nsrc, G, amp_dev, ad, u1, du_fixed);
    k_regime1_advance<<<1, 1, 0, s>>>(ad, u1, du_fixed);
    return cudaGetLastError();
}

cudaError_t kx_launch_delta_source(const KxDev& d, double p0, double* G, cudaStream_t s)
{
    k_delta_source<<<1, KX_CTA, 0, s>>>(d, p0, G);
    return cudaGetLastError();
}

cudaError_t kx_launch_moments(const KxDev& d, const double* f, int B, double* n, double* rho,
                              double* p1, double* p2, int stride, cudaStream_t s)
{
    k_moments<<<B, KX_CTA, 0, s>>>(d, f, n, rho, p1, p2, stride);
    return cudaGetLastError();
}
