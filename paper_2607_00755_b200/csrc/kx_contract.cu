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
        case 1: return kx_launch_stream_bt1(d, sm_count, f, yd, B, st, bar_total, s, nullptr);
        case 2: return kx_launch_stream_bt2(d, sm_count, f, yd, B, st, bar_total, s, nullptr);
        case 4: return kx_launch_stream_bt4(d, sm_count, f, yd, B, st, bar_total, s, nullptr);
        default: return kx_launch_stream_bt8(d, sm_count, f, yd, B, st, bar_total, s, nullptr);
    }
}

bool kx_stream_run_supported(const KxDev& d)
{
    return d.prec == KX_FP64 && d.eta == 0 && (d.interp == KX_INTERP_LINEAR || d.exp_impl == KX_EXP_TABLE);
}

cudaError_t kx_launch_stream_run(const KxDev& d, int sm_count, double* f, int B, KxStage st, int method, int S,
                                 const double* tau_dev, const double* rate_dev, const double* amp_dev,
                                 unsigned* bar_total, cudaStream_t s)
{
    KxRun run = {method, S, tau_dev, rate_dev, amp_dev};
    switch (kx_pick_bt(d.N, B)) {
        case 1: return kx_launch_stream_bt1(d, sm_count, f, nullptr, B, st, bar_total, s, &run);
        case 2: return kx_launch_stream_bt2(d, sm_count, f, nullptr, B, st, bar_total, s, &run);
        case 4: return kx_launch_stream_bt4(d, sm_count, f, nullptr, B, st, bar_total, s, &run);
        default: return kx_launch_stream_bt8(d, sm_count, f, nullptr, B, st, bar_total, s, &run);
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
