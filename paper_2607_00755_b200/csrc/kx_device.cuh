// kx_device.cuh -- device code shared by the two fused evaluation kernels of libkx: k_stream (kx_contract.cu, the exact
// streaming path) and k_dmma (kx_tiled.cu, the tensor-core path).  One operator evaluation is ONE cooperative kernel:
//
//   contraction phase  (a4-a5; streaming tasks or the DMMA roles)  ->  per-CTA partials in global memory
//   grid barrier
//   [tensor-core path only, when a member is flagged: exact streaming contraction of the flagged member groups by the
//    whole grid, second grid barrier]
//   finishing phase    (a6-a8: one CTA per member adds the partials in a fixed order, raw operator, projection of
//                       App. C, diagnostics, the fused Runge-Kutta stage update)
//
// A kernel launch costs about 4 us on B200 and a grid barrier 1.8 us (measured, profiles/r02_*): fusing the four kernels
// of round 1 into one removes three launches from the step.  No atomics on data: results are bit-reproducible.
//
// Compiled with --fmad=false; every fused multiply-add below is an explicit fma().
#pragma once
#include "kx_internal.cuh"

namespace kxd {

constexpr int kDmmaWarps = 8;                      // warps per CTA of k_dmma (gain workers per CTA)
constexpr int kMaxPerThread = KX_MAX_N / KX_CTA;   // rows per thread of the finishing phase: 4

// ---------------------------------------------------------------- clock stamps (measurement aid, kx_trace)
__device__ __forceinline__ unsigned long long gtime()
{
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
__device__ __forceinline__ void stamp(unsigned long long* trace, int slot)
{
    if (trace) {
        const unsigned cta = blockIdx.y * gridDim.x + blockIdx.x;
        if (cta < KX_TRACE_CTAS) trace[cta * KX_TRACE_SLOTS + slot] = gtime();
    }
}

// ---------------------------------------------------------------- grid barrier (cooperative launch: all CTAs resident)
// bar[0] counts arrivals and is reset by the last arriver; bar[1] holds the epoch released last.  Every barrier of every
// launch has its own epoch (kx_handle_s::epoch), different from its predecessor's.
__device__ __forceinline__ unsigned ld_acquire(const unsigned* p)
{
    unsigned v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void grid_barrier(unsigned* bar, unsigned epoch)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned nctas = gridDim.x * gridDim.y;
        __threadfence();
        const unsigned old = atomicAdd(&bar[0], 1u);
        if (old == nctas - 1u) {
            bar[0] = 0u;
            __threadfence();
            atomicExch(&bar[1], epoch);
        } else {
            while (ld_acquire(&bar[1]) != epoch) { }
        }
        __threadfence();
    }
    __syncthreads();
}

// The first barrier of a launch, cheaper: a counter that only grows (bar[3]); the host knows how many CTAs every launch
// adds and hands each launch its target.  Everybody polls the counter itself: one L2 round trip less than the epoch form.
__device__ __forceinline__ void grid_barrier_count(unsigned* ctr, unsigned target)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        __threadfence();
        atomicAdd(ctr, 1u);
        while ((int)(ld_acquire(ctr) - target) < 0) { }
        __threadfence();
    }
    __syncthreads();
}

// statistics written by other CTAs of the same launch: read through L2, one 16-byte load
__device__ __forceinline__ bool member_flagged(const long long* mstat, int b)
{
    const longlong2 v = __ldcg(reinterpret_cast<const longlong2*>(mstat) + b);
    const double fm = __longlong_as_double(v.y);
    if (!isfinite(fm)) return true;                        // Inf / NaN in f: the exact path treats them entry by entry
    const long long k = v.x;
    if (k == KX_MSTAT_NONE) return false;
    const double lb = __longlong_as_double(k >= 0 ? k : (k ^ 0x7fffffffffffffffLL));
    // log2(fm) >= its unbiased exponent: far below the threshold (the usual case) without evaluating the logarithm
    const int ex = (int)((v.y >> 52) & 0x7ff) - 1023;
    if (v.y != 0 && lb - (double)ex <= -49.82892142331043) return false;
    return lb - log2(fm) > -49.82892142331043;             // log2(1e-15)
}

// ---------------------------------------------------------------- y of eq. B.20 in base 2
// log2(f / (1 + eta f)), f floored (reading D8); LINEAR interpolation works on f itself
__device__ __forceinline__ double yval(double f, int interp, double f_floor, int eta)
{
    if (interp != KX_INTERP_LOG) return f;
    const double ff = fmax(f, f_floor);
    return eta == 0 ? log2(ff) : log2(ff / (1.0 + (double)eta * ff));
}

// ---------------------------------------------------------------- exact streaming contraction (a4-a5)
//   gain_i = sum_{n<=m} Wsym[i,nm] f_n f_m                              eq. 4.6 with 2.6
//   nu_i   = sum_{n<=m} Wsym[i,nm] f_j~,  loss_i = f_i nu_i
//       LOG:    f_j~ = 2^(y_L + omega_R (y_R - y_L)),  y = log2 max(f, f_floor)   eq. B.20 at eta=0, D7/D8
//       LINEAR: f_j~ = f_L + omega_R (f_R - f_L)                                  eq. B.19
// QS = 1: quantum statistics (eq. 4.3).  With x = f_j~ = e^y / (1 - eta e^y) four sums per (row, member) are kept,
//   G1 = sum W f_n f_m,  L1 = sum W x,  G2 = sum W f_n f_m x,  L2 = sum W x (f_n + f_m),
// from which  gain = (1 + eta f_i)(G1 + eta G2),  loss = f_i (L1 + eta L2 + G2)   (eta^2 = 1; finishing phase).
//
// Row i of the row-compressed tensor is cut into tasks of `chunk` entries (taskptr); the CTA takes the tasks task0,
// task0 + tstride, ...; each thread owns entries e0+tid, e0+tid+256, ... and keeps BT accumulators per sum (one per member
// of the group b0 .. b0+BT-1) in registers; a fixed-order shuffle / shared-memory reduction writes one partial per
// (task, member).
enum { MODE_LOG_TAB = 0, MODE_LOG_LIBM = 1, MODE_LINEAR = 2, MODE_LOG_F32 = 3, MODE_LINEAR_F32 = 4 };

template <int BT, int MODE, int QS>
__host__ __device__ constexpr size_t contract_smem(int N)
{
    if (MODE >= MODE_LOG_F32)       // fp32 mode: float2 y rows, float f rows, double partials of the warps, task table
        return (size_t)BT * N * 12 + (size_t)(KX_CTA / 32) * 2 * BT * 8 + 16 + (((size_t)(N + 1) * 4 + 15) & ~(size_t)15);
    return (size_t)BT * N * 24 + (size_t)(KX_CTA / 32) * (QS ? 4 : 2) * BT * 8
         + (MODE == MODE_LOG_TAB ? (size_t)(KX_EXP_REP << KX_EXP_BITS) * 8 : 0) + (((size_t)(N + 1) * 4 + 15) & ~(size_t)15);
}

template <int BT, int MODE, int QS>
__device__ __forceinline__ void contract_group(const KxDev& d, const double* __restrict__ f, const double2* __restrict__ yd,
                                               double* __restrict__ part, int B, int b0, unsigned task0, unsigned tstride,
                                               unsigned char* smem_raw, bool load_static = true)
{
    const int N = d.N;
    double2* s_yd = reinterpret_cast<double2*>(smem_raw);                 // [BT][N]
    double* s_f = reinterpret_cast<double*>(s_yd + (size_t)BT * N);       // [BT][N]
    constexpr int NV = QS ? 4 : 2;                                         // sums per (row, member)
    double* s_red = s_f + (size_t)BT * N;                                 // [8][NV*BT]
    double* s_tab = s_red + (KX_CTA / 32) * NV * BT;                       // [256][16] (MODE_LOG_TAB)
    unsigned* s_tp = reinterpret_cast<unsigned*>(s_tab + (MODE == MODE_LOG_TAB ? (KX_EXP_REP << KX_EXP_BITS) : 0)); // [N+1]

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nb = min(BT, B - b0);
    for (int k = tid; k < BT * N; k += KX_CTA) {
        int b = k / N, j = k - b * N;
        if (b < nb) {
            // (read through L2: inside the one-launch integrator these were written by other CTAs a grid barrier ago)
            const double fv = __ldcg(f + (size_t)(b0 + b) * N + j);
            if (yd) s_yd[k] = __ldcg(yd + (size_t)(b0 + b) * N + j);
            else {        // no prepared y: computed here
                const double y0 = yval(fv, d.interp, d.f_floor, d.eta);
                const double y1 = j + 1 < N ? yval(__ldcg(f + (size_t)(b0 + b) * N + j + 1), d.interp, d.f_floor, d.eta) : y0;
                s_yd[k] = make_double2(y0, y1 - y0);
            }
            s_f[k] = fv;
        } else {                                  // ragged last group: harmless values, results discarded
            s_yd[k] = make_double2(0.0, 0.0);
            s_f[k] = 0.0;
        }
    }
    if (load_static) {        // the exp2 table and the task table do not change between the stages of a one-launch integration
        if (MODE == MODE_LOG_TAB)
            for (int k = tid; k < (KX_EXP_REP << KX_EXP_BITS); k += KX_CTA) s_tab[k] = d.exptab[k / KX_EXP_REP];
        for (int k = tid; k <= N; k += KX_CTA) s_tp[k] = d.taskptr[k];
    }
    __syncthreads();

    const unsigned ntasks = s_tp[N];
    const double* tab_lane = s_tab + (lane & (KX_EXP_REP - 1));
    const unsigned chunk = (unsigned)d.chunk;

    for (unsigned task = task0; task < ntasks; task += tstride) {
        // row of this task: largest i with taskptr[i] <= task
        int lo = 0, hi = N - 1;
        while (lo < hi) {
            int mid = (lo + hi + 1) >> 1;
            if (s_tp[mid] <= task) lo = mid; else hi = mid - 1;
        }
        const int i = lo;
        const unsigned r0 = d.rowptr[i], r1 = d.rowptr[i + 1];
        const unsigned e0 = r0 + (task - s_tp[i]) * chunk;
        const unsigned e1 = min(e0 + chunk, r1);

        double g[BT], l[BT], g2[QS ? BT : 1], l2[QS ? BT : 1];
#pragma unroll
        for (int b = 0; b < BT; ++b) { g[b] = 0.0; l[b] = 0.0; if (QS) { g2[b] = 0.0; l2[b] = 0.0; } }
        const double eta = (double)d.eta;

        unsigned e = e0 + tid;
        double W = 0.0, om = 0.0;
        unsigned pk = 0;
        if (e < e1) { W = d.W[e]; om = d.omega[e]; pk = d.nmj[e]; }
        while (e < e1) {
            const double Wc = W, omc = om;
            const unsigned pkc = pk;
            e += KX_CTA;
            if (e < e1) { W = d.W[e]; om = d.omega[e]; pk = d.nmj[e]; }   // prefetch the next entry
            const int n = pkc & 1023, m = (pkc >> 10) & 1023, j = pkc >> 20;
#pragma unroll
            for (int b = 0; b < BT; ++b) {
                const double fn = s_f[b * N + n], fm = s_f[b * N + m];
                const double pn = fn * fm;
                g[b] = fma(Wc, pn, g[b]);
                const double2 y = s_yd[b * N + j];
                const double t = fma(omc, y.y, y.x);
                double x;
                if (MODE == MODE_LOG_TAB) x = kx_exp2_tab<KX_EXP_REP>(t, tab_lane);
                else if (MODE == MODE_LOG_LIBM) x = exp2(t);
                else x = t;
                if (QS) {
                    // W f_j~, eq. B.20: x / (1 - eta x) with the reciprocal from the hardware estimate (2^-23) and two
                    // Newton steps (2^-46, 2^-92: full double precision) instead of the IEEE division sequence
                    const double dn = fma(-eta, x, 1.0);
                    double rc;
                    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(rc) : "d"(dn));
                    double er = fma(-dn, rc, 1.0);
                    rc = fma(rc, er, rc);
                    er = fma(-dn, rc, 1.0);
                    rc = fma(rc, er, rc);
                    const double wf = Wc * (x * rc);
                    l[b] += wf;
                    g2[b] = fma(wf, pn, g2[b]);
                    l2[b] = fma(wf, fn + fm, l2[b]);
                } else {
                    l[b] = fma(Wc, x, l[b]);
                }
            }
        }
        // fixed-order reduction: xor butterfly inside the warp, then warps 0..7 in order
#pragma unroll
        for (int b = 0; b < BT; ++b) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                g[b] += __shfl_xor_sync(0xffffffffu, g[b], o);
                l[b] += __shfl_xor_sync(0xffffffffu, l[b], o);
                if (QS) {
                    g2[b] += __shfl_xor_sync(0xffffffffu, g2[b], o);
                    l2[b] += __shfl_xor_sync(0xffffffffu, l2[b], o);
                }
            }
        }
        if (lane == 0) {
#pragma unroll
            for (int b = 0; b < BT; ++b) {
                s_red[warp * NV * BT + NV * b] = g[b];
                s_red[warp * NV * BT + NV * b + 1] = l[b];
                if (QS) { s_red[warp * NV * BT + NV * b + 2] = g2[b]; s_red[warp * NV * BT + NV * b + 3] = l2[b]; }
            }
        }
        __syncthreads();
        if (tid < NV * BT) {
            double acc = 0.0;
#pragma unroll
            for (int w = 0; w < KX_CTA / 32; ++w) acc += s_red[w * NV * BT + tid];
            const int b = tid / NV;
            if (b < nb) part[((size_t)task * B + (b0 + b)) * NV + (tid % NV)] = acc;
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- the same contraction in fp32 (KX_FP32, optional mode)
// The paper times its GPU path in single precision (Fig. 3); BASELINE.json asks for <= 1e-4 of max |gain|.
// W, omega are read as stored (fp64) and rounded; f, y = log2 max(f, 1e-37), the products and the per-thread sums are
// float (exp2f: ex2.approx), the reduction over threads and everything after it (finishing phase) is fp64.
template <int BT, int LIN>
__device__ __forceinline__ void contract_group_f32(const KxDev& d, const double* __restrict__ f, double* __restrict__ part, int B,
                                                   int b0, unsigned task0, unsigned tstride, unsigned char* smem_raw,
                                                   bool load_static = true)
{
    const int N = d.N;
    float2* s_yd = reinterpret_cast<float2*>(smem_raw);                    // [BT][N]
    float* s_f = reinterpret_cast<float*>(s_yd + (size_t)BT * N);          // [BT][N]
    double* s_red = reinterpret_cast<double*>(smem_raw + (((size_t)BT * N * 12 + 15) & ~(size_t)15));    // [8][2*BT]
    unsigned* s_tp = reinterpret_cast<unsigned*>(s_red + (KX_CTA / 32) * 2 * BT);                         // [N+1]
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nb = min(BT, B - b0);
    const float floor32 = fmaxf((float)d.f_floor, 1e-37f);
    for (int k = tid; k < BT * N; k += KX_CTA) {
        const int b = k / N, j = k - b * N;
        float fv = 0.f, y0 = 0.f, y1 = 0.f;
        if (b < nb) {
            fv = (float)__ldcg(f + (size_t)(b0 + b) * N + j);
            const float fn = j + 1 < N ? (float)__ldcg(f + (size_t)(b0 + b) * N + j + 1) : fv;
            y0 = LIN ? fv : log2f(fmaxf(fv, floor32));
            y1 = LIN ? fn : log2f(fmaxf(fn, floor32));
        }
        s_yd[k] = make_float2(y0, y1 - y0);
        s_f[k] = fv;
    }
    if (load_static) for (int k = tid; k <= N; k += KX_CTA) s_tp[k] = d.taskptr[k];
    __syncthreads();
    const unsigned ntasks = s_tp[N];
    const unsigned chunk = (unsigned)d.chunk;
    for (unsigned task = task0; task < ntasks; task += tstride) {
        int lo = 0, hi = N - 1;
        while (lo < hi) {
            int mid = (lo + hi + 1) >> 1;
            if (s_tp[mid] <= task) lo = mid; else hi = mid - 1;
        }
        const int i = lo;
        const unsigned r0 = d.rowptr[i], r1 = d.rowptr[i + 1];
        const unsigned e0 = r0 + (task - s_tp[i]) * chunk;
        const unsigned e1 = min(e0 + chunk, r1);
        float g[BT], l[BT];
#pragma unroll
        for (int b = 0; b < BT; ++b) { g[b] = 0.f; l[b] = 0.f; }
        unsigned e = e0 + tid;
        double W = 0.0, om = 0.0;
        unsigned pk = 0;
        if (e < e1) { W = d.W[e]; om = d.omega[e]; pk = d.nmj[e]; }
        while (e < e1) {
            const float Wc = (float)W, omc = (float)om;
            const unsigned pkc = pk;
            e += KX_CTA;
            if (e < e1) { W = d.W[e]; om = d.omega[e]; pk = d.nmj[e]; }
            const int n = pkc & 1023, m = (pkc >> 10) & 1023, j = pkc >> 20;
#pragma unroll
            for (int b = 0; b < BT; ++b) {
                const float pn = s_f[b * N + n] * s_f[b * N + m];
                g[b] = fmaf(Wc, pn, g[b]);
                const float2 y = s_yd[b * N + j];
                const float t = fmaf(omc, y.y, y.x);
                l[b] = fmaf(Wc, LIN ? t : exp2f(t), l[b]);
            }
        }
        double gd[BT], ld[BT];
#pragma unroll
        for (int b = 0; b < BT; ++b) {
            gd[b] = (double)g[b]; ld[b] = (double)l[b];
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                gd[b] += __shfl_xor_sync(0xffffffffu, gd[b], o);
                ld[b] += __shfl_xor_sync(0xffffffffu, ld[b], o);
            }
        }
        if (lane == 0) {
#pragma unroll
            for (int b = 0; b < BT; ++b) { s_red[warp * 2 * BT + 2 * b] = gd[b]; s_red[warp * 2 * BT + 2 * b + 1] = ld[b]; }
        }
        __syncthreads();
        if (tid < 2 * BT) {
            double acc = 0.0;
#pragma unroll
            for (int w = 0; w < KX_CTA / 32; ++w) acc += s_red[w * 2 * BT + tid];
            const int b = tid / 2;
            if (b < nb) part[((size_t)task * B + (b0 + b)) * 2 + (tid % 2)] = acc;
        }
        __syncthreads();
    }
}

// one dispatch point for the kernels: fp64 (MODE 0-2) or fp32 (MODE 3-4) contraction of a member group
template <int BT, int MODE, int QS>
__device__ __forceinline__ void contract_any(const KxDev& d, const double* __restrict__ f, const double2* __restrict__ yd,
                                             double* __restrict__ part, int B, int b0, unsigned task0, unsigned tstride,
                                             unsigned char* smem_raw, bool load_static = true)
{
    if (MODE >= MODE_LOG_F32) contract_group_f32<BT, MODE == MODE_LINEAR_F32>(d, f, part, B, b0, task0, tstride, smem_raw, load_static);
    else contract_group<BT, (MODE >= MODE_LOG_F32 ? MODE_LOG_TAB : MODE), QS>(d, f, yd, part, B, b0, task0, tstride, smem_raw, load_static);
}

// ---------------------------------------------------------------- block reductions (256 threads, fixed order)
template <int NV>
__device__ __forceinline__ void block_sum(double (&v)[NV], double* s_red /* [NV*8] */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NV; ++k)
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v[k] += __shfl_xor_sync(0xffffffffu, v[k], o);
    __syncthreads();
    if (lane == 0)
#pragma unroll
        for (int k = 0; k < NV; ++k) s_red[k * 8 + warp] = v[k];
    __syncthreads();
#pragma unroll
    for (int k = 0; k < NV; ++k) {
        double a = 0.0;
#pragma unroll
        for (int w = 0; w < 8; ++w) a += s_red[k * 8 + w];
        v[k] = a;
    }
}

__device__ __forceinline__ double block_max(double v, double* s_red)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    __syncthreads();
    if (lane == 0) s_red[warp] = v;
    __syncthreads();
    double a = s_red[0];
#pragma unroll
    for (int w = 1; w < 8; ++w) a = fmax(a, s_red[w]);
    return a;
}

// ---------------------------------------------------------------- bulk copies (TMA, 1-D) and their mbarrier
__device__ __forceinline__ unsigned smem_addr(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned long long* bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" :: "r"(smem_addr(bar)), "r"(count) : "memory");
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(unsigned long long* bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" :: "r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(unsigned long long* bar, unsigned parity)
{
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "WAIT_%=:\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
        "@p bra DONE_%=;\n\t"
        "bra WAIT_%=;\n\t"
        "DONE_%=:\n\t}" :: "r"(smem_addr(bar)), "r"(parity) : "memory");
}
// global -> shared, `bytes` a multiple of 16, both addresses 16-byte aligned; completion is signalled on `bar`
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, unsigned bytes, unsigned long long* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
                 :: "r"(smem_addr(dst)), "l"(src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}
// orders earlier generic-proxy accesses (other CTAs' stores made visible by the grid barrier, this CTA's own shared-memory
// traffic) before the async-proxy copies that follow
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// ---------------------------------------------------------------- partials of the DMMA phase -> (gain, nu)[b, i]
// gain: tile = i/16; the warps [wstart[tile], wstart[tile+1]) of the plan worked on it, i.e. the CTAs c0 = wstart[tile]/8
// ... c1 = (wstart[tile+1]-1)/8, each of which wrote one partial into slot c + tile.  loss: supertile = i/256, chunk units
// [sp LC, (sp+1) LC) of the RS LC units were taken by the loss CTAs ld0[sp]..ld1[sp], slot = c + sp.
// The partials are stored member-major (gpart [member][slot][16], lpart [member][slot][256]), so the member's slice of all
// gain slots is one contiguous piece and that of all loss slots another: two bulk copies (TMA) fetch them into shared
// memory (164 small copies of 128 B / 2 KiB took 2 us: the copy engine handles them one after the other); a thread then
// adds the partials of its row in slot order: a fixed order, bit-reproducible.
//   scratch: s_y [Npad] | s_gp [GG + NT][16] | s_lp [sum_sp (ld1 - ld0 + 1)][256]
__host__ __device__ inline size_t finish_scratch_bytes(int N, int GG, int GL, int NT, int RS)
{
    return (size_t)((N + 3) & ~3) * 8 + (size_t)(GG + NT) * 128 + (size_t)(GL + RS) * 2048;
}

__device__ __forceinline__ void gather_partials(int N, const KxStage& st, const KxPlan& plan, int b, double* scratch,
                                                unsigned long long* mbar)
{
    // member-major partials: all gain slots of member b are one contiguous piece, all loss slots another: two bulk copies
    const int Npad = (N + 3) & ~3;
    double* s_gp = scratch + Npad;
    const int ng = plan.GG + st.NT;
    double* s_lp = s_gp + (size_t)ng * 16;
    const unsigned l0 = plan.ld0[0];
    const unsigned nl = plan.ld1[st.RS - 1] + (unsigned)(st.RS - 1) - l0 + 1u;       // slots l0 .. ld1[RS-1] + RS - 1
    fence_proxy_async();
    if (threadIdx.x == 0) {
        mbar_expect_tx(mbar, (unsigned)ng * 128u + nl * 2048u);
        bulk_g2s(s_gp, st.gpart + (size_t)b * st.gslots * 16, (unsigned)ng * 128u, mbar);
        bulk_g2s(s_lp, st.lpart + ((size_t)b * st.lslots + l0) * 256, nl * 2048u, mbar);
    }
}

// ---------------------------------------------------------------- finishing phase: one CTA (256 threads) per member b
//   a6  C_raw = gain - f_i nu_i
//   a7  projection C.2-C.8 in the basis {1, K_i} (D3: same span as {1, E_i}, well conditioned), diag C.1, C.9
//   a8  Runge-Kutta stage update                                                  eq. 4.9
// from_dmma: the member's (gain, nu) come from the partials of the DMMA phase (plan != null), else from the partials
// `st.part` of the exact streaming contraction.  scratch: finish_scratch_bytes() of shared memory (streaming path: the s_y part only).
template <int NQ> struct FinishPre { double fi[NQ], h[NQ], E[NQ], K[NQ]; };      // NQ = ceil(N / 256) rows per thread

// the member's stage input and the kinematics: nothing a kernel of this launch writes, so a finishing CTA may fetch them
// before the grid barrier
template <int NQ>
__device__ __forceinline__ void finish_preload(const KxDev& d, const double* __restrict__ fin, int b, FinishPre<NQ>& pre)
{
    const int N = d.N, tid = threadIdx.x;
    const double* fb = fin + (size_t)b * N;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int i = tid + q * KX_CTA;
        pre.fi[q] = 0.0; pre.h[q] = 0.0; pre.E[q] = 0.0; pre.K[q] = 0.0;
        if (i < N) { pre.fi[q] = fb[i]; pre.h[q] = d.h[i]; pre.E[q] = d.E[i]; pre.K[q] = d.K[i]; }
    }
}

// (gain, nu) of row i from the gathered slots: four interleaved sums each (slot = first + k mod 4), added as
// (s0 + s1) + (s2 + s3): short dependency chains, a fixed order
__device__ __forceinline__ void sum_partials_row(int N, const KxStage& st, const KxPlan& plan, const double* scratch, int i,
                                                 double& g, double& nu)
{
    const double* s_gp = scratch + ((N + 3) & ~3);
    const double* s_lp = s_gp + (size_t)(plan.GG + st.NT) * 16;
    const int tile = i >> 4, sp = i >> 8;
    double a[4] = {0.0, 0.0, 0.0, 0.0}, l[4] = {0.0, 0.0, 0.0, 0.0};
    const unsigned w0 = plan.wstart[tile], w1 = plan.wstart[tile + 1];
    if (w1 > w0) {
        const unsigned c0 = w0 / kDmmaWarps, ng = (w1 - 1u) / kDmmaWarps - c0 + 1u;
        const double* pg = s_gp + (size_t)(c0 + tile) * 16 + (i & 15);
        unsigned c = 0;
        for (; c + 4 <= ng; c += 4) {
#pragma unroll
            for (int k = 0; k < 4; ++k) a[k] += pg[(size_t)(c + k) * 16];
        }
        for (int k = 0; c < ng; ++c, ++k) a[k] += pg[(size_t)c * 16];
    }
    const unsigned lo = plan.ld0[sp] + (unsigned)sp - plan.ld0[0];     // the slots of supertile sp start at CTA ld0[sp] + sp
    const unsigned nls = plan.ld1[sp] - plan.ld0[sp] + 1u;
    const double* pl = s_lp + (size_t)lo * 256 + (i & 255);
    unsigned c = 0;
    for (; c + 4 <= nls; c += 4) {
#pragma unroll
        for (int k = 0; k < 4; ++k) l[k] += pl[(size_t)(c + k) * 256];
    }
    for (int k = 0; c < nls; ++c, ++k) l[k] += pl[(size_t)c * 256];
    g = (a[0] + a[1]) + (a[2] + a[3]);
    nu = (l[0] + l[1]) + (l[2] + l[3]);
}

// ---------------------------------------------------------------- finishing phase, the plain case of the tensor-core path
// C_raw = gain - f_i nu_i only (a6): no projection, no diagnostics, no Runge-Kutta stage, no separate gain / loss outputs.
// Kept apart from finish_member and as short as possible: this code runs once per launch, so what it costs is mostly the
// instruction fetch (after an L2 flush the fetch comes from HBM).
template <int NQ>
__device__ __forceinline__ void finish_raw(int N, const KxStage& st, const KxPlan& plan, int b, const double* scratch,
                                           const FinishPre<NQ>& pre, unsigned long long* mbar, unsigned parity)
{
    const int tid = threadIdx.x;
    mbar_wait(mbar, parity);
    if (tid == 0) stamp(st.trace, 7);
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int i = tid + q * KX_CTA;
        if (i < N) {
            double g, nu;
            sum_partials_row(N, st, plan, scratch, i, g, nu);
            st.C[(size_t)b * N + i] = fma(-pre.fi[q], nu, g);
        }
    }
    __syncthreads();       // the scratch may be reused by the next member of this CTA
}

// from_dmma: the member's partials of the DMMA phase are on their way into the scratch (gather_partials(b) was issued by
// the caller; `mbar` flips to `parity` when they have landed)
template <int NQ>
__device__ __forceinline__ void finish_member(const KxDev& d, const double* __restrict__ fin, int B, const KxStage& st,
                                              const KxPlan* plan, bool from_dmma, int b, double* scratch, double* s_red /* [64] */,
                                              const FinishPre<NQ>* pre = nullptr, unsigned long long* mbar = nullptr,
                                              unsigned parity = 0)
{
    const int N = d.N, tid = threadIdx.x;
    const double* fb = fin + (size_t)b * N;
    const int Npad = (N + 3) & ~3;
    double* s_y = scratch;                         // [Npad]
    double C[NQ], fi[NQ], hi_[NQ], Ei[NQ], Ki[NQ];
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int i = tid + q * KX_CTA;
        C[q] = 0.0; fi[q] = 0.0; hi_[q] = 0.0; Ei[q] = 0.0; Ki[q] = 0.0;
        if (pre) { fi[q] = pre->fi[q]; hi_[q] = pre->h[q]; Ei[q] = pre->E[q]; Ki[q] = pre->K[q]; }
        else if (i < N) { fi[q] = fb[i]; hi_[q] = d.h[i]; Ei[q] = d.E[i]; Ki[q] = d.K[i]; }
    }
    if (from_dmma) mbar_wait(mbar, parity);

#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int i = tid + q * KX_CTA;
        if (i < N) {
            double g = 0.0, nu = 0.0, gq2 = 0.0, lq2 = 0.0;
            if (from_dmma) {
                sum_partials_row(N, st, *plan, scratch, i, g, nu);
            } else {
                const unsigned t0 = d.taskptr[i], t1 = d.taskptr[i + 1];
                const int nv = d.eta ? 4 : 2;
                for (unsigned t = t0; t < t1; ++t) {
                    const double* pp = st.part + ((size_t)t * B + b) * nv;
                    if (d.eta) {
                        const double2 a = __ldcg(reinterpret_cast<const double2*>(pp)), c2 = __ldcg(reinterpret_cast<const double2*>(pp) + 1);
                        g += a.x; nu += a.y; gq2 += c2.x; lq2 += c2.y;
                    } else {
                        const double2 a = __ldcg(reinterpret_cast<const double2*>(pp));
                        g += a.x; nu += a.y;
                    }
                }
            }
            if (d.eta) {                                          // eq. 4.3 from the four sums (see contract_group)
                const double eta = (double)d.eta;
                g = (1.0 + eta * fi[q]) * (g + eta * gq2);
                nu = nu + eta * lq2 + gq2;
            }
            C[q] = fma(-fi[q], nu, g);                            // a6
            if (st.gain) st.gain[(size_t)b * N + i] = g;
            if (st.loss) st.loss[(size_t)b * N + i] = fi[q] * nu;
        }
    }

    const bool project = (st.flags & KX_PROJECT) != 0;
    if (project || st.diag) {
        // C.2 and the denominators of C.1 / C.9
        double v[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
        double fm = 0.0;
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const double hc = hi_[q] * C[q];
            v[0] += hc;                       // R0 = sum h C
            v[1] += hc * Ki[q];               // RK = sum h K C
            v[2] += hc * Ei[q];               // R1 = sum h E C
            v[3] += fabs(hc);                 // S0
            v[4] += fabs(hc) * Ei[q];         // S1
            fm = fmax(fm, fabs(fi[q]));
        }
        block_sum<5>(v, s_red);
        const double fmax_ = block_max(fm, s_red);
        const double R0 = v[0], RK = v[1], R1 = v[2], S0 = v[3], S1 = v[4];
        double alpha = 0.0, beta = 0.0, D0 = 0.0, D1 = 0.0;
        if (project) {
            double xi[NQ];
            double a[3] = {0.0, 0.0, 0.0};
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const double r = fmax_ > 0.0 ? fabs(fi[q]) / fmax_ : 0.0;     // C.4
                xi[q] = r > d.eps_supp ? r : 0.0;
                const double hx = hi_[q] * xi[q];
                a[0] += hx;                   // A00
                a[1] += hx * Ki[q];           // A0K
                a[2] += hx * Ki[q] * Ki[q];   // AKK
            }
            block_sum<3>(a, s_red);
            const double A00 = a[0], A0K = a[1], AKK = a[2];
            if (fmax_ > 0.0 && A00 > 0.0) {
                const double det = A00 * AKK - A0K * A0K;                    // C.8
                if (det <= 1e-14 * A00 * AKK) { alpha = R0 / A00; beta = 0.0; }   // D9
                else { alpha = (R0 * AKK - RK * A0K) / det; beta = (RK * A00 - R0 * A0K) / det; }
            }
            double dsum[2] = {0.0, 0.0};
#pragma unroll
            for (int q = 0; q < NQ; ++q) {
                const double corr = xi[q] * (alpha + beta * Ki[q]);
                C[q] = C[q] - corr;                                          // C.3
                dsum[0] += hi_[q] * fabs(corr);
                dsum[1] += hi_[q] * Ei[q] * fabs(corr);
            }
            if (st.diag) { block_sum<2>(dsum, s_red); D0 = dsum[0]; D1 = dsum[1]; }
        }
        if (st.diag && tid == 0) {
            double* dg = st.diag + (size_t)b * st.diag_stride;
            dg[0] = S0 > 0.0 ? R0 / S0 : 0.0;       // eps_N, C.1
            dg[1] = S1 > 0.0 ? R1 / S1 : 0.0;       // eps_E
            dg[2] = S0 > 0.0 ? D0 / S0 : 0.0;       // R_N, C.9
            dg[3] = S1 > 0.0 ? D1 / S1 : 0.0;       // R_E
        }
    }

    if (st.C) {
#pragma unroll
        for (int q = 0; q < NQ; ++q) {
            const int i = tid + q * KX_CTA;
            if (i < N) st.C[(size_t)b * N + i] = C[q];
        }
    }
    if (!st.evolve) { __syncthreads(); return; }

    // ---- a8: k = kappa_b R C + sum_s amp_s G_s, then the Runge-Kutta bookkeeping of this stage
    double rate = st.rate, dt = st.dt;
    if (st.rk_method == KX_HEUN_ADAPT) {      // step and rate from the device controller (kx_evolve_adaptive)
        const double u = st.ad->u;
        dt = st.ad->du;
        rate = st.ad_rate0 * exp(st.ad_slope * ((st.rk_stage == 0 ? u : u + dt) - st.ad_u0));
    }
    const double kR = (st.kappa ? st.kappa[b] : 1.0) * rate;
    bool bad = false;
    double errmax = 0.0;
#pragma unroll
    for (int q = 0; q < NQ; ++q) {
        const int i = tid + q * KX_CTA;
        if (i >= N) continue;
        const size_t o = (size_t)b * N + i;
        double s = 0.0;
        for (int r = 0; r < st.nsrc; ++r) s += st.amp[r] * st.G[(size_t)r * N + i];
        const double k = kR * C[q] + s;
        const double f0 = st.f[o];
        double next;      // input of the next operator evaluation
        if (st.rk_method == KX_EULER) {
            next = f0 + dt * k;
            st.f[o] = next;
        } else if (st.rk_method == KX_HEUN) {
            if (st.rk_stage == 0) { st.k1[o] = k; next = f0 + dt * k; st.fstage[o] = next; }
            else { next = f0 + 0.5 * dt * (st.k1[o] + k); st.f[o] = next; }
        } else if (st.rk_method == KX_HEUN_ADAPT) {
            if (st.rk_stage == 0) { st.k1[o] = k; next = f0 + dt * k; st.fstage[o] = next; }      // Euler predictor
            else {                                                                                  // Heun corrector, kept aside
                next = f0 + 0.5 * dt * (st.k1[o] + k);
                st.k2[o] = next;
                const double e = fabs(next - st.fstage[o]) / (st.ad_atol + st.ad_rtol * fmax(fabs(f0), fabs(next)));
                errmax = isfinite(e) ? fmax(errmax, e) : INFINITY;
            }
        } else {
            if (st.rk_stage == 0) { st.k1[o] = k; next = f0 + 0.5 * dt * k; st.fstage[o] = next; }
            else if (st.rk_stage == 1) { st.k2[o] = k; next = f0 + 0.5 * dt * k; st.fstage[o] = next; }
            else if (st.rk_stage == 2) { st.k3[o] = k; next = f0 + dt * k; st.fstage[o] = next; }
            else { next = f0 + (dt / 6.0) * (st.k1[o] + 2.0 * st.k2[o] + 2.0 * st.k3[o] + k); st.f[o] = next; }
        }
        if (!isfinite(next)) bad = true;
        s_y[i] = yval(next, d.interp, d.f_floor, d.eta);
    }
    if (bad && st.rk_method != KX_HEUN_ADAPT) atomicOr(st.flag, 1);      // a rejected attempt may overflow harmlessly
    if (st.rk_method == KX_HEUN_ADAPT && st.rk_stage == 1) {
        const double e = block_max(errmax, s_red);                         // order independent: deterministic
        if (tid == 0) atomicMax(&st.ad->errkey, kx_dkey(e));
    }
    __syncthreads();
    if (st.ydnext) {
        double2* ydn = reinterpret_cast<double2*>(st.ydnext) + (size_t)b * N;
        for (int i = tid; i < N; i += KX_CTA) {
            const double y0 = s_y[i], y1 = (i + 1 < N) ? s_y[i + 1] : y0;
            ydn[i] = make_double2(y0, y1 - y0);
        }
    }
    __syncthreads();       // the scratch may be reused by the next member of this CTA
}

}  // namespace kxd
