// kx_stream.cuh -- the fused kernels of the exact streaming path and their launcher, included by the translation units
// kx_stream_bt{1,2,4,8}.cu, each of which instantiates them for one member-group size BT (the instantiations take minutes
// to compile in one file; four files compile in parallel).  Kernel descriptions: kx_contract.cu / kx_device.cuh.
#pragma once
#include "kx_device.cuh"

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
template <int BT, int MODE, int QS>
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
            for (int b = (int)cta; b < B; b += (int)nctas) {
                double* scr = reinterpret_cast<double*>(smem_raw);
                if (d.N <= KX_CTA) finish_member<1>(d, fin, B, st, nullptr, false, b, scr, s_red, nullptr);
                else if (d.N <= 2 * KX_CTA) finish_member<2>(d, fin, B, st, nullptr, false, b, scr, s_red, nullptr);
                else finish_member<4>(d, fin, B, st, nullptr, false, b, scr, s_red, nullptr);
            }
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
    stream_run<BT, MODE, QS>(d, f, B, st, run, smem_raw, s_red);
}

// The one-launch integrator is built for the two default fp64 paths only (LOG with the table exp2, LINEAR; classical
// statistics): every other combination takes one launch per stage (kx_stream_run_supported).  Keeps the build short.
template <int MODE, int QS> constexpr bool run_built() { return QS == 0 && (MODE == MODE_LOG_TAB || MODE == MODE_LINEAR); }

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
        if constexpr (run_built<MODE, QS>()) {
            e = cudaFuncSetAttribute(k_stream_run<BT, MODE, QS>, cudaFuncAttributeMaxDynamicSharedMemorySize, 226 * 1024);
            if (e != cudaSuccess) return e;
        }
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
        if constexpr (run_built<MODE, QS>()) {
            e = kx_launch_coop(k_stream_run<BT, MODE, QS>, dim3(gx, gy), dim3(KX_CTA), smem, s, d, const_cast<double*>(f), B, st, *run);
            if (e == cudaSuccess) *bar_total += nbar * (unsigned)(gx * gy);
            return e;
        } else {
            return cudaErrorNotSupported;
        }
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
