// kx_tiled.cu -- one operator evaluation on the tensor-core path (KX_STORE_TILED) as ONE cooperative kernel:
//
//   DMMA phase       gain[b,i] = sum_{n<=m} (W_inm + W_imn) f_n f_m                 eq. 4.6 with 2.6
//                    nu[b,i]   = sum_j sum_{c<Q} M_c(i,j) a_c(b,j)  (loss_i = f_i nu_i)   eq. B.19-B.20,
//                    see kx_tiled_build.cu for the Chebyshev-moment form of the interpolated loss term and its error bound
//   grid barrier
//   [exact fallback  members whose interpolation error bound is not negligible are evaluated by the streaming contraction
//                    (kxd::contract_group), spread over the whole grid; second grid barrier.  Normally skipped.]
//   finishing phase  a6-a8 (kxd::finish_member): CTA b adds the partials of member b in a fixed order, raw operator,
//                    projection, diagnostics, fused Runge-Kutta stage
//
// Both contractions are out[b,i] += sum_k X[b,k] A[k,i] with A streamed once from HBM/L2 (cp.async) and X built in shared
// memory from the caller's f: X = f_n f_m for the gain, X = a_c(b,j) for the loss.  The products run on the FP64 tensor
// pipe: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4), M = 8 members, N = 8 rows, K = 4.  The CTAs (one per SM) are split between
// the two terms in proportion to their work (kx_dmma_plan).  No atomics on data: bit-reproducible.
//
// Compiled with --fmad=false; fused multiply-adds are explicit.
#include "kx_device.cuh"

#include <vector>

namespace {

using namespace kxd;

// cost of one loss DMMA relative to one gain DMMA in the CTA split (the loss CTAs also compute their Chebyshev
// coefficients first; calibrated with the clock-stamp trace on cfg3 so that both roles reach the barrier together)
constexpr double kLossCost = 1.26;
// cost of one run (tile, n) of the gain stream in units of one group (see kx_dmma_plan)
constexpr double kRunCost = 0.09;
// loss role in the plan's time model (units of one gain group of a warp): DMMA cost of a chunk relative to the same DMMA count of
// the gain stream, and what the loss prologue (operand X: log2, exp2 at the nodes) takes longer than staging f
constexpr double kLossChunk = 1.05, kLossPrologue = 3.9;

// D[8 members x 8 rows] += X[8 members x 4 k] * A[4 k x 8 rows]
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPEND>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(NPEND) : "memory"); }

constexpr int WARPS = kDmmaWarps;
constexpr int NTHR = WARPS * 32;
static_assert(NTHR == KX_CTA, "the finishing phase and the exact fallback run with 256 threads");
constexpr int kStageBytes = KX_GROUP_DBL * 8 + 16;     // gain ring stage: 2 KiB of A + 4 descriptors
// ring stages of a loss warp (4 KiB each).  (6 stages for small batches, where the kernel streams from HBM, were measured:
// the X window no longer fits in one piece and every further window repeats the prologue: slower)
__host__ __device__ constexpr int loss_stages(int nbt) { return 3; }
constexpr int kLossABytes = 32 * 1024;                 // loss stage: 16 k x 256 rows of AL

// ---------------------------------------------------------------- gain role
// The rows f[b, :] of the pass's 8 NBT members sit in shared memory (row stride = 4 mod 16 doubles when N = 0 mod 16: the
// 8 members x 4 k fragment reads of a quad are bank-conflict free), copied straight from the caller's f.  Every warp is
// an independent worker: it streams its own contiguous share of ONE tile's groups (plan.wstart) through a private
// cp.async ring and holds a 16-row x 8 NBT-member accumulator (2 NBT DMMA per quad and fragment pair).  The DMMAs of a
// run (fixed n) take X = f_m and accumulate into T; f_n multiplies T once, when the run ends.  When all warps are done
// they leave their accumulators in shared memory and the CTA adds those of the same tile in warp order: one partial per
// (CTA, tile), slot = CTA + tile.
template <int NBT, int STAGES, int LDNC>
__device__ __forceinline__ void gain_role(const KxTiled& t, const KxPlan& plan, int N, int B, int bcol0,
                                          const double* __restrict__ f, int gslots, double* __restrict__ gpart,
                                          unsigned char* smem, int* s_wtile, unsigned long long* trace,
                                          unsigned long long* mbar, unsigned& mpar)
{
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int krow = lane & 3, lr = lane >> 2;
    // row stride of s_f: >= N + 4, = 0 mod 4; N = 0 mod 16 gives 4 mod 16.  LDNC != 0: a compile-time stride (260 for N <= 256),
    // so that the eight member-tile rows of a fragment load sit at immediate offsets (28 address adds less per group)
    const int LDN = LDNC ? LDNC : ((N + 7) & ~3);
    double* s_f = reinterpret_cast<double*>(smem);                                    // [8 NBT][LDN]
    unsigned char* ring = smem + (size_t)(NBT * 8) * LDN * 8 + (size_t)warp * STAGES * kStageBytes;

    // this warp's tile and its share of the tile's groups
    const unsigned wk = blockIdx.x * WARPS + warp;
    int tile = -1;
    unsigned g0 = 0, n = 0;
    if (wk < plan.wstart[t.NT]) {
        int lo = 0, hi = t.NT - 1;
        while (lo < hi) {
            const int mid = (lo + hi + 1) >> 1;
            if (plan.wstart[mid] <= wk) lo = mid; else hi = mid - 1;
        }
        tile = lo;
        const unsigned w0 = plan.wstart[tile], wt = plan.wstart[tile + 1] - w0, r = wk - w0;
        const unsigned a0 = plan.vt[tile], gt = plan.vt[tile + 1] - a0;
        g0 = a0 + (unsigned)((unsigned long long)r * gt / wt);
        n = a0 + (unsigned)((unsigned long long)(r + 1) * gt / wt) - g0;
    }
    auto issue = [&](unsigned gi) {
        const double* src = t.A + (size_t)(g0 + gi) * KX_GROUP_DBL;
        unsigned char* dst = ring + (size_t)(gi % STAGES) * kStageBytes;
#pragma unroll
        for (int k = 0; k < 4; ++k) cp_async16(dst + (k * 32 + lane) * 16, src + (k * 32 + lane) * 2);
        if (lane == 0) cp_async16(dst + KX_GROUP_DBL * 8, t.desc + (size_t)(g0 + gi) * 4);
    };
    // the tensor stream starts first; f arrives while it is in flight
#pragma unroll
    for (int s = 0; s < STAGES - 1; ++s) {
        if ((unsigned)s < n) issue(s);
        cp_async_commit();
    }
    // s_f[b][n] = f[bcol0 + b][n], n < N; s_f[b][N] = 1 (the scale of padding quads), s_f[b][N+1..] = 0.  The rows of
    // f are copied as they are (16-byte cp.async when N is even); members beyond B are zero.  Every CTA starts its
    // walk somewhere else so that the CTAs do not all ask the same L2 lines at once.
    // N even: one bulk copy (TMA) per row, completion on the CTA's mbarrier; else element by element.
    {
        const bool bulk = (N & 1) == 0;
        const int nrows = min(NBT * 8, B - bcol0);
        if (bulk) {
            if (tid == 0) mbar_expect_tx(mbar, (unsigned)nrows * (unsigned)N * 8u);
            const int rot = (int)(blockIdx.x % (unsigned)nrows);     // every CTA starts its walk somewhere else
            for (int k = tid; k < nrows; k += NTHR) {
                int bb = k + rot;
                if (bb >= nrows) bb -= nrows;
                bulk_g2s(s_f + (size_t)bb * LDN, f + (size_t)(bcol0 + bb) * N, (unsigned)N * 8u, mbar);
            }
        } else {
            for (int k = tid; k < nrows * N; k += NTHR) {
                const int bb = k / N, nn = k - bb * N;
                s_f[(size_t)bb * LDN + nn] = __ldcg(f + (size_t)(bcol0 + bb) * N + nn);
            }
        }
        for (int k = tid; k < (NBT * 8 - nrows) * N; k += NTHR) {          // members beyond B: zero
            const int bb = nrows + k / N, nn = k % N;
            s_f[(size_t)bb * LDN + nn] = 0.0;
        }
        for (int k = tid; k < NBT * 8 * (LDN - N); k += NTHR) {
            const int bb = k / (LDN - N), cc = k - bb * (LDN - N);
            s_f[(size_t)bb * LDN + N + cc] = cc == 0 ? 1.0 : 0.0;
        }
        cp_async_wait<0>();
        if (bulk) mbar_wait(mbar, mpar);
        mpar ^= bulk ? 1u : 0u;
    }
    __syncthreads();
    if (tid == 0) stamp(trace, 1);

    // acc: the tile's partial.  T: sum over the m of the current run (fixed n) of f_m A[(n,m), i]; when the run ends,
    // acc += f_n T.  Lane holds out[b = 8 bt + lane/4][i = 8 rb + 2 (lane%4) + {0,1}], the same member b as its
    // fragment of X, so f_n[b] scales its own accumulators.
    double acc[NBT][2][2];
#pragma unroll
    for (int bt = 0; bt < NBT; ++bt)
#pragma unroll
        for (int rb = 0; rb < 2; ++rb) acc[bt][rb][0] = acc[bt][rb][1] = 0.0;
    const long long ck0_ = clock64();
    unsigned nfold_ = 0;

    if (n > 0) {
        const double* xb = s_f + (size_t)lr * LDN + krow;    // + 8 bt LDN + column: the lane's member row of tile bt
        const int LD8 = 8 * LDN;
        double T[NBT][2][2], sn[NBT];
#pragma unroll
        for (int bt = 0; bt < NBT; ++bt)
#pragma unroll
            for (int rb = 0; rb < 2; ++rb) T[bt][rb][0] = T[bt][rb][1] = 0.0;
        auto fold = [&]() {
#pragma unroll
            for (int bt = 0; bt < NBT; ++bt)
#pragma unroll
                for (int rb = 0; rb < 2; ++rb) {
                    acc[bt][rb][0] = fma(sn[bt], T[bt][rb][0], acc[bt][rb][0]);
                    acc[bt][rb][1] = fma(sn[bt], T[bt][rb][1], acc[bt][rb][1]);
                    T[bt][rb][0] = T[bt][rb][1] = 0.0;
                }
        };
        // descriptors of the current group (dc) and the next one (dn) stay in registers: the f_m rows of a quad are
        // requested a whole quad before they are used
        uint4 dc = *reinterpret_cast<const uint4*>(ring + KX_GROUP_DBL * 8);
        unsigned srow_cur = dc.x >> 20;
        double xv[NBT];
        {
            const double* xr = xb + (dc.x & 0xFFFFFu);
            const double* sr = xb + srow_cur - krow;
#pragma unroll
            for (int bt = 0; bt < NBT; ++bt) { sn[bt] = sr[bt * LD8]; xv[bt] = xr[bt * LD8]; }
        }

        for (unsigned gi = 0; gi < n; ++gi) {
            // refill the slot freed by group gi-1, then make sure groups gi and gi+1 are in shared memory
            if (gi + STAGES - 1 < n) issue(gi + STAGES - 1);
            cp_async_commit();
            cp_async_wait<STAGES - 2>();
            __syncwarp();
            const unsigned char* stg = ring + (size_t)(gi % STAGES) * kStageBytes;
            const double* wd = reinterpret_cast<const double*>(stg) + lane;
            const bool last_group = gi + 1 >= n;
            uint4 dn = dc;
            if (!last_group) dn = *reinterpret_cast<const uint4*>(ring + (size_t)((gi + 1) % STAGES) * kStageBytes + KX_GROUP_DBL * 8);
#pragma unroll
            for (int q = 0; q < 4; ++q) {
                const unsigned dsc = q == 0 ? dc.y : (q == 1 ? dc.z : (q == 2 ? dc.w : dn.x));    // next quad
                const bool more = (q < 3) || !last_group;
                double xn[NBT];
                {
                    const double* xr = xb + (dsc & 0xFFFFFu);
#pragma unroll
                    for (int bt = 0; bt < NBT; ++bt) xn[bt] = xr[bt * LD8];
                }
                const double w0 = wd[q * 64], w1 = wd[q * 64 + 32];
#pragma unroll
                for (int bt = 0; bt < NBT; ++bt) {
                    dmma884(T[bt][0][0], T[bt][0][1], xv[bt], w0);
                    dmma884(T[bt][1][0], T[bt][1][1], xv[bt], w1);
                }
                const unsigned srow = dsc >> 20;
                if (__builtin_expect(more && srow != srow_cur, 0)) {              // the run (n) ends with this quad
                    fold(); ++nfold_;
                    srow_cur = srow;
                    const double* sr = xb + srow - krow;
#pragma unroll
                    for (int bt = 0; bt < NBT; ++bt) sn[bt] = sr[bt * LD8];
                }
#pragma unroll
                for (int bt = 0; bt < NBT; ++bt) xv[bt] = xn[bt];
            }
            dc = dn;
            __syncwarp();     // every lane is done with this stage before it is refilled
        }
        fold();
        cp_async_wait<0>();
        __syncwarp();
        // the warp's accumulators -> its own (drained) ring: [8 NBT members][16 rows]
        double* mine = reinterpret_cast<double*>(ring);
#pragma unroll
        for (int bt = 0; bt < NBT; ++bt)
#pragma unroll
            for (int rb = 0; rb < 2; ++rb)
                *reinterpret_cast<double2*>(mine + (8 * bt + lr) * 16 + 8 * rb + 2 * krow) = make_double2(acc[bt][rb][0], acc[bt][rb][1]);
    }
    if (lane == 0) {
        s_wtile[warp] = n > 0 ? tile : -1;
        if (trace) {
            const unsigned cta = blockIdx.x;
            if (cta < KX_TRACE_CTAS) { trace[cta * KX_TRACE_SLOTS + 8 + warp] = gtime(); trace[cta * KX_TRACE_SLOTS + 24 + warp] = ((unsigned long long)(clock64() - ck0_) << 24) | ((unsigned long long)nfold_ << 12) | n; }
        }
    }
    __syncthreads();
    // one partial per (CTA, tile): the accumulators of the warps that worked on the same tile, added in warp order
    const unsigned char* ring0 = smem + (size_t)(NBT * 8) * LDN * 8;
    for (int wa = 0; wa < WARPS;) {
        const int tl = s_wtile[wa];
        int wb = wa + 1;
        while (wb < WARPS && s_wtile[wb] == tl) ++wb;
        if (tl >= 0) {
            // member-major: member b's slots are contiguous, so the finishing phase fetches them with one bulk copy
            double* dst = gpart + ((size_t)bcol0 * gslots + (blockIdx.x + tl)) * 16;
            for (int o = tid; o < NBT * 128; o += NTHR) {
                double s = 0.0;
                for (int w = wa; w < wb; ++w) s += reinterpret_cast<const double*>(ring0 + (size_t)w * STAGES * kStageBytes)[o];
                dst[(size_t)(o >> 4) * gslots * 16 + (o & 15)] = s;
            }
        }
        wa = wb;
    }
}

// ---------------------------------------------------------------- loss role
// A dense GEMM.  The CTA first computes the Chebyshev coefficients a_c(b,j) of its own share of k = (j,c) rows straight
// into shared memory (window by window if the share does not fit): exp2 at the Chebyshev nodes, then the discrete
// Chebyshev transform on the tensor pipe; it also accumulates the per-member statistics that route a member to the exact
// fallback.  Then warp w streams its rows [32 w, 32 w + 32) of AL through a private 3-stage cp.async ring (4 KiB per chunk
// of 16 k) and multiplies them with the resident coefficients (4 NBT DMMA per quad).  A range that crosses a supertile
// (256 rows) boundary produces one partial per piece, slot = loss CTA + supertile.
template <int NBT>
__device__ __forceinline__ void loss_role(const KxDev& dk, const KxTiled& t, const KxPlan& plan, int N, int B, int bcol0,
                                          const double* __restrict__ f, long long* __restrict__ mstat, int lslots,
                                          double* __restrict__ lpart, unsigned char* smem, unsigned long long* trace)
{
    constexpr int LD = NBT * 8 + 4;
    constexpr int kLossStages = loss_stages(NBT);
    constexpr int R8 = 32 / WARPS;            // 8-row blocks per warp: the CTA covers a 256-row supertile
    static_assert(WARPS == 8, "loss role: 8 warps");
    constexpr int MB = NBT * 8;               // members of this CTA
    constexpr int PARTS = NTHR / MB;          // threads per member in the coefficient pass: each takes every PARTS-th node
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int krow = lane & 3, lr = lane >> 2;
    const int N_ = N, Q = t.Q, WC = plan.WC, GG = plan.GG, GL = plan.GL;
    const bool logm = dk.interp == KX_INTERP_LOG, tab = dk.exp_impl == KX_EXP_TABLE;
    // shared memory: [A stages | scratch of the coefficient pass] [X window] [nodes, exp2 table]
    unsigned char* sStage = smem;
    double* sXw = reinterpret_cast<double*>(smem + (size_t)kLossStages * kLossABytes);          // [WC*16][LD]
    double* s_node = sXw + (size_t)WC * 16 * LD;                                                // [QMAX]
    double* s_tab = s_node + KX_QMAX;                                                           // [256]
    long long* s_stat = reinterpret_cast<long long*>(s_tab + (1 << KX_EXP_BITS));               // [2][64] member statistics of this CTA
    double* s_y = reinterpret_cast<double*>(smem);                                              // [brackets + 1][MB] (aliases the stages)
    if (logm) {
        if (tid < Q) s_node[tid] = t.nodes[tid];
        for (int k = tid; k < (1 << KX_EXP_BITS); k += NTHR) s_tab[k] = dk.exptab[k];
    }
    int npass_ = 0;

    // The operand X of the window's rows k = (j, q), k in [K0, K0 + 16 wn), straight into shared memory.
    // LOG: X = g(omega_q) = 2^(y_j + omega_q (y_(j+1) - y_j)), the interpolated occupation at the Q Chebyshev nodes (the
    // tensor holds the bucket moments in the Lagrange basis of these nodes, kx_tiled_build.cu), y = log2 max(f, f_floor);
    // LINEAR: the two exact coefficients a_0 = (f_j + f_(j+1))/2, a_1 = (f_(j+1) - f_j)/2.  Also the member statistics
    // (flags) of kx_internal.cuh.
    auto build_window = [&](unsigned K0, unsigned wn) {
        const unsigned K1 = K0 + 16u * wn;
        const int jlo = (int)(K0 / (unsigned)Q);
        const int jhi = min((int)((K1 - 1u) / (unsigned)Q), N_ - 2);
        // rows beyond the last bracket are padding: zero
        {
            const unsigned kpad = (unsigned)(N_ - 1) * (unsigned)Q;
            for (unsigned k = max(K0, kpad) + (unsigned)warp; k < K1; k += WARPS)
                for (int c2 = lane; c2 < LD; c2 += 32) sXw[(size_t)(k - K0) * LD + c2] = 0.0;
        }
        if (!logm) {          // LINEAR: two exact coefficients per bracket, no transform: one flat loop
            const int total = (jhi - jlo + 1) * MB;
            for (int i0 = tid; i0 < total; i0 += 8 * NTHR) {          // 16 independent loads in flight per thread
                double v0[8], v1[8];
#pragma unroll
                for (int u2 = 0; u2 < 8; ++u2) {
                    const int idx = i0 + u2 * NTHR, j = jlo + idx / MB, bm = idx % MB, b = bcol0 + bm;
                    const bool ok = idx < total && b < B;
                    v0[u2] = ok ? __ldcg(f + (size_t)b * N_ + j) : 0.0;
                    v1[u2] = ok ? __ldcg(f + (size_t)b * N_ + j + 1) : 0.0;
                }
#pragma unroll
                for (int u2 = 0; u2 < 8; ++u2) {
                    const int idx = i0 + u2 * NTHR, j = jlo + idx / MB, bm = idx % MB;
                    if (idx < total) {
                        const unsigned k = (unsigned)j * 2u;
                        if (k >= K0 && k < K1) sXw[(size_t)(k - K0) * LD + bm] = 0.5 * (v0[u2] + v1[u2]);
                        if (k + 1 >= K0 && k + 1 < K1) sXw[(size_t)(k + 1 - K0) * LD + bm] = 0.5 * (v1[u2] - v0[u2]);
                    }
                }
            }
            __syncthreads();
            return;
        }
        // step 1: y_j = log2 max(f_j, f_floor) of the brackets' end points j = jlo .. jhi + 1, and max |f|.  The member
        // statistics are reduced inside the CTA first (shared-memory atomics) and sent with ONE global atomic per member:
        // 39 CTAs x 600 same-address atomics each were queueing in L2 and throttling the loads behind them
        const int nj = jhi - jlo + 1;
        if (tid < 2 * 64) s_stat[tid] = tid < 64 ? KX_MSTAT_NONE : 0;
        __syncthreads();
        {
            // consecutive threads read consecutive j of one member: nj + 1 doubles of a row are 2-3 sectors, not nj + 1
            const int nj1 = nj + 1, total = nj1 * MB;
            for (int i0 = tid; i0 < total; i0 += 4 * NTHR) {
                double v[4];
#pragma unroll
                for (int u2 = 0; u2 < 4; ++u2) {
                    const int idx = i0 + u2 * NTHR, b = bcol0 + idx / nj1;
                    v[u2] = (idx < total && b < B) ? __ldcg(f + (size_t)b * N_ + jlo + idx % nj1) : 0.0;
                }
#pragma unroll
                for (int u2 = 0; u2 < 4; ++u2) {
                    const int idx = i0 + u2 * NTHR, bm = idx / nj1, b = bcol0 + bm;
                    if (idx < total) {
                        if (b < B) atomicMax(s_stat + 64 + bm, __double_as_longlong(fabs(v[u2])));
                        s_y[(idx % nj1) * MB + bm] = log2(fmax(v[u2], dk.f_floor));
                    }
                }
            }
        }
        __syncthreads();
        if (tid == 0 && npass_ < 2) stamp(trace, 17 + 2 * npass_);
        // step 2: thread (member bl, part) takes the nodes q = part, part + PARTS, ... of every bracket
        {
            const int bl = tid % MB, part = tid / MB;
            const int b = bcol0 + bl;
            constexpr int QP = (KX_QMAX + PARTS - 1) / PARTS;       // nodes per thread and bracket, at most
#pragma unroll(QP >= 4 ? 1 : 4)
            for (int jj = 0; jj < nj; ++jj) {
                const double y0 = s_y[jj * MB + bl], y1 = s_y[(jj + 1) * MB + bl], dy = y1 - y0;
                if (part == (jj & (PARTS - 1)) && b < B) {
                    // log2 of the bracket's error bound (log2 max_i f_i is subtracted by the consumers); the atomics return
                    // nothing, so nobody waits for them
                    const double cabs = 0.6931471805599453 * fabs(dy);
                    if (cabs > 0.0)
                        atomicMax(s_stat + bl, kx_dkey(fmax(y0, y1) + (double)Q * (log2(cabs) - 2.0) + t.flag_log2));
                }
                if (tid == 0 && npass_ == 0 && (jj == 1 || jj == 2 || jj == 5)) stamp(trace, jj == 1 ? 19 : (jj == 2 ? 20 : 21));
                const unsigned kb = (unsigned)(jlo + jj) * (unsigned)Q;
                double e[QP];
#pragma unroll
                for (int u2 = 0; u2 < QP; ++u2) {
                    // branch-free (nodes beyond Q are clamped and their value dropped below): the QP chains interleave
                    const int q = min(part + u2 * PARTS, Q - 1);
                    const double arg = fma(s_node[q], dy, y0);
                    e[u2] = kx_exp2_tab<1>(arg, s_tab);
                }
                if (!tab) {
#pragma unroll 1
                    for (int u2 = 0; u2 < QP; ++u2) e[u2] = exp2(fma(s_node[min(part + u2 * PARTS, Q - 1)], dy, y0));
                }
#pragma unroll
                for (int u2 = 0; u2 < QP; ++u2) {
                    const int q = part + u2 * PARTS;
                    const unsigned k = kb + (unsigned)q;
                    if (q < Q && k >= K0 && k < K1) sXw[(size_t)(k - K0) * LD + bl] = e[u2];
                }
            }
        }
        __syncthreads();
        if (tid < MB && bcol0 + tid < B) {
            if (s_stat[tid] != KX_MSTAT_NONE) atomicMax(mstat + 2 * (bcol0 + tid), s_stat[tid]);
            atomicMax(mstat + 2 * (bcol0 + tid) + 1, s_stat[64 + tid]);
        }
        if (tid == 0 && npass_ < 2) stamp(trace, 18 + 2 * npass_);
        ++npass_;
    };

    const unsigned cl = blockIdx.x - GG;
    const unsigned LC = (unsigned)t.LC;
    const unsigned U = (unsigned)t.RS * LC;
    const unsigned u0 = (unsigned)((unsigned long long)cl * U / (unsigned)GL);
    const unsigned u1 = (unsigned)((unsigned long long)(cl + 1) * U / (unsigned)GL);
    unsigned u = u0;
    bool first = true;
    while (u < u1) {
        const unsigned sp = u / LC;                                  // supertile
        const unsigned ue = min(u1, (sp + 1) * LC);
        const unsigned ka = u - sp * LC, n = ue - u;
        const int nb = min(32, t.NR8 - 32 * (int)sp);                // 8-row blocks of this supertile
        const int nbw = min(R8, max(0, nb - R8 * warp));             // ... of this warp

        // every warp streams its own rows of the tensor (4 KiB per chunk: 4 eight-row blocks) through a private
        // cp.async ring: no CTA-wide barrier inside a window
        unsigned char* wring = sStage + (size_t)warp * (kLossStages * kLossABytes / WARPS);
        constexpr int kWStage = kLossABytes / WARPS;                  // 4 KiB
        auto issue = [&](unsigned kc, int slot) {
            if (nbw > 0) {
                const double* srcA = t.AL + ((size_t)kc * t.NR8 + 32 * sp + R8 * warp) * 128;
                unsigned char* dstA = wring + (size_t)slot * kWStage;
                for (int k = lane; k < nbw * 64; k += 32) cp_async16(dstA + (size_t)k * 16, srcA + (size_t)k * 2);
            }
        };

        double acc[R8][NBT][2];
#pragma unroll
        for (int r = 0; r < R8; ++r)
#pragma unroll
            for (int bt = 0; bt < NBT; ++bt) acc[r][bt][0] = acc[r][bt][1] = 0.0;

        for (unsigned w0 = 0; w0 < n; w0 += (unsigned)WC) {
            const unsigned wn = min((unsigned)WC, n - w0), kw = ka + w0;
            build_window(16u * kw, wn);          // ends with a barrier: the scratch (= the rings) is free again
            if (first && tid == 0) stamp(trace, 1);
            first = false;
#pragma unroll
            for (int s2 = 0; s2 < kLossStages - 1; ++s2) {
                if ((unsigned)s2 < wn) issue(kw + s2, s2);
                cp_async_commit();
            }
            for (unsigned it = 0; it < wn; ++it) {
                if (it + kLossStages - 1 < wn) issue(kw + it + kLossStages - 1, (int)((it + kLossStages - 1) % kLossStages));
                cp_async_commit();
                cp_async_wait<kLossStages - 1>();        // chunk `it` of this warp has landed
                __syncwarp();
                if (nbw > 0) {
                    const double* sA = reinterpret_cast<const double*>(wring + (size_t)(it % kLossStages) * kWStage) + lane;
                    const double* sX = sXw + (size_t)(16 * it + krow) * LD + lr;
#pragma unroll
                    for (int q = 0; q < 4; ++q) {
                        double xv[NBT];
#pragma unroll
                        for (int bt = 0; bt < NBT; ++bt) xv[bt] = sX[(size_t)(4 * q) * LD + 8 * bt];
#pragma unroll
                        for (int r = 0; r < R8; ++r) {
                            const double w = sA[(r * 4 + q) * 32];
#pragma unroll
                            for (int bt = 0; bt < NBT; ++bt) dmma884(acc[r][bt][0], acc[r][bt][1], xv[bt], w);
                        }
                    }
                }
                __syncwarp();                            // the stage is refilled two iterations from now
            }
            cp_async_wait<0>();
            __syncthreads();              // the rings are free again (next window's scratch, next piece)
        }

        double* dst = lpart + ((size_t)bcol0 * lslots + (cl + sp)) * 256 + 8 * R8 * warp + 2 * krow;
#pragma unroll
        for (int r = 0; r < R8; ++r)
            if (r < nbw)
#pragma unroll
                for (int bt = 0; bt < NBT; ++bt)
                    *reinterpret_cast<double2*>(dst + (size_t)(8 * bt + lr) * lslots * 256 + 8 * r) = make_double2(acc[r][bt][0], acc[r][bt][1]);
        u = ue;
    }
}

// ---------------------------------------------------------------- what follows the DMMA phase (NQ = rows per thread)
// The code after the grid barrier runs once per launch, so what it costs is mostly instruction fetch (about 0.3 us per
// jump into code that is not in the instruction cache, measured as stall_no_instruction with ncu).  The plain case
// (finish_raw) is kept short and inline; everything else is called out of line so that the kernel body stays compact.
template <int NQ>
__device__ __noinline__ void finish_member_cold(const KxDev& d, const double* __restrict__ fin, int B, const KxStage& st,
                                                const KxPlan* plan, bool from_dmma, int b, double* scratch, double* s_red,
                                                const FinishPre<NQ>* pre, unsigned long long* mbar, unsigned parity)
{
    finish_member<NQ>(d, fin, B, st, plan, from_dmma, b, scratch, s_red, pre, mbar, parity);
}

__device__ __noinline__ void fallback_cold(const KxDev& dk, const double* __restrict__ f, double* __restrict__ part, int B, int g0,
                                           unsigned char* smem)
{
    if (dk.exp_impl == KX_EXP_LIBM) contract_group<KX_FB_BT, MODE_LOG_LIBM, 0>(dk, f, nullptr, part, B, g0, blockIdx.x, gridDim.x, smem);
    else contract_group<KX_FB_BT, MODE_LOG_TAB, 0>(dk, f, nullptr, part, B, g0, blockIdx.x, gridDim.x, smem);
}

template <int NQ>
__device__ __forceinline__ void dmma_tail(const KxDev& dk, const KxPlan& plan, int B, const double* __restrict__ f,
                                          const KxStage& st, unsigned char* smem, double* s_red, int& s_myflag,
                                          unsigned long long* mbar, unsigned parity)
{
    const int tid = threadIdx.x, N = dk.N;
    const bool mine = (int)blockIdx.x < B;          // this CTA finishes member blockIdx.x (and blockIdx.x + gridDim.x, ...)
    FinishPre<NQ> pre;
    if (mine) finish_preload(dk, f, blockIdx.x, pre);              // static inputs of the finishing phase: before the barrier
    if (tid == 0) s_myflag = 0;
    grid_barrier_count(st.bar + 3, st.bar_target);
    if (tid == 0) stamp(st.trace, 3);

    // The statistics of all members (one 16-byte load per thread) and the partials of this CTA's own member are requested
    // together: one L2 round trip.  Members whose interpolation error bound is not negligible (rare) take the exact
    // streaming contraction: their groups of KX_FB_BT members, the tasks dealt to all CTAs; every CTA takes the same
    // decisions from the same statistics.
    bool any = false;
    {
        // (the gather first: its proxy fence would otherwise wait for the statistics load)
        if (mine) gather_partials(N, st, plan, blockIdx.x, reinterpret_cast<double*>(smem), mbar);
        const bool fl0 = st.mstat && tid < B && member_flagged(st.mstat, tid);
        if (fl0 && tid == (int)blockIdx.x) s_myflag = 1;
        any = __syncthreads_or(fl0) != 0;
        if (st.mstat) {
#pragma unroll 1
            for (int b0 = NTHR; b0 < B; b0 += NTHR) {
                const bool fl = b0 + tid < B && member_flagged(st.mstat, b0 + tid);
                if (fl && b0 + tid == (int)blockIdx.x) s_myflag = 1;
                any |= __syncthreads_or(fl) != 0;
            }
        }
    }
    bool gathered = mine;
    if (any) {
        if (gathered) { mbar_wait(mbar, parity); parity ^= 1u; gathered = false; }      // the contraction reuses the scratch
        __syncthreads();
        for (int g0 = 0; g0 < B; g0 += KX_FB_BT) {
            const int hit = __syncthreads_or(tid < KX_FB_BT && g0 + tid < B && member_flagged(st.mstat, g0 + tid));
            if (!hit) continue;
            fallback_cold(dk, f, st.part, B, g0, smem);
        }
        grid_barrier(st.bar, st.epoch);
    }
    if (tid == 0) stamp(st.trace, 4);

    if (st.mstat_next && blockIdx.x == gridDim.x - 1)          // clean statistics for the next launch (the other buffer)
        for (int k = tid; k < st.mstat_cap; k += NTHR) { st.mstat_next[2 * k] = KX_MSTAT_NONE; st.mstat_next[2 * k + 1] = 0; }
    const bool plain = st.C && !st.gain && !st.loss && !st.diag && !st.evolve && !(st.flags & KX_PROJECT);
    for (int b = blockIdx.x; b < B; b += gridDim.x) {
        const bool first = b == (int)blockIdx.x;
        const bool flagged = st.mstat && (first ? s_myflag != 0 : member_flagged(st.mstat, b));
        if (flagged && tid == 0 && st.fb_count) atomicAdd(st.fb_count, 1u);
        // (a flagged member implies `any`, so a gather still in flight belongs to an unflagged first member)
        if (!flagged && !(first && gathered)) gather_partials(N, st, plan, b, reinterpret_cast<double*>(smem), mbar);
        if (plain && !flagged) {
            if (!first) finish_preload(dk, f, b, pre);
            finish_raw<NQ>(N, st, plan, b, reinterpret_cast<const double*>(smem), pre, mbar, parity);
        } else {
            finish_member_cold<NQ>(dk, f, B, st, &plan, !flagged, b, reinterpret_cast<double*>(smem), s_red, first ? &pre : nullptr,
                                   mbar, parity);
        }
        if (!flagged) parity ^= 1u;
    }
}

// ---------------------------------------------------------------- the fused kernel: one CTA per SM, cooperative
// Clock stamps (st.trace, per CTA): 0 entry, 1 prologue done (f staged / first coefficient window built), 2 partials
// written, 3 first barrier passed, 4 fallback done, 5 finishing phase done; 8..15 end of each gain warp's stream.
template <int NBT, int STAGES, int LDNC>
__global__ void __launch_bounds__(NTHR, 1)
k_dmma(const __grid_constant__ KxDev dk, const __grid_constant__ KxTiled t, const __grid_constant__ KxPlan plan, int B,
       const double* __restrict__ f, const __grid_constant__ KxStage st)
{
    extern __shared__ __align__(16) unsigned char smem[];
    __shared__ double s_red[8 * 8];
    __shared__ int s_wtile[WARPS];
    __shared__ int s_myflag;
    __shared__ __align__(8) unsigned long long s_mbar;      // completion of the bulk copies of the finishing phase
    const int tid = threadIdx.x, N = dk.N;
    if (tid == 0) { stamp(st.trace, 0); mbar_init(&s_mbar, 1u); if (st.trace && blockIdx.x < KX_TRACE_CTAS) st.trace[blockIdx.x * KX_TRACE_SLOTS + 22] = clock64(); }

    const int ny = (B + NBT * 8 - 1) / (NBT * 8);
    unsigned mpar = 0;                              // phase of s_mbar
    __syncthreads();                                // the barrier is initialised
    for (int by = 0; by < ny; ++by) {          // member groups of 8 NBT: one pass each (more than one for B > 64 only)
        const int bcol0 = by * NBT * 8;
        if ((int)blockIdx.x < plan.GG) gain_role<NBT, STAGES, LDNC>(t, plan, N, B, bcol0, f, st.gslots, st.gpart, smem, s_wtile, st.trace, &s_mbar, mpar);
        else loss_role<NBT>(dk, t, plan, N, B, bcol0, f, st.mstat, st.lslots, st.lpart, smem, st.trace);
        __syncthreads();
    }
    if (tid == 0) stamp(st.trace, 2);
    if (N <= KX_CTA) dmma_tail<1>(dk, plan, B, f, st, smem, s_red, s_myflag, &s_mbar, mpar);
    else if (N <= 2 * KX_CTA) dmma_tail<2>(dk, plan, B, f, st, smem, s_red, s_myflag, &s_mbar, mpar);
    else dmma_tail<4>(dk, plan, B, f, st, smem, s_red, s_myflag, &s_mbar, mpar);
    if (tid == 0) { stamp(st.trace, 5); if (st.trace && blockIdx.x < KX_TRACE_CTAS) st.trace[blockIdx.x * KX_TRACE_SLOTS + 23] = clock64(); }
}

constexpr size_t loss_fixed_bytes(int nbt) { return (size_t)loss_stages(nbt) * kLossABytes + (KX_QMAX + (1 << KX_EXP_BITS) + 2 * 64) * 8; }
constexpr size_t kSmemMax = 226u * 1024u;       // dynamic shared memory: 227 KiB per CTA minus the kernel's static 544 bytes

// chunks of 16 k whose Chebyshev coefficients a loss CTA keeps in shared memory at a time: its whole share if it fits
int loss_window(const KxTiled& t, int GL, int nbt)
{
    const long long U = (long long)t.RS * t.LC;
    const long long share = (U + GL - 1) / GL + 1;
    const long long fit = (long long)((kSmemMax - loss_fixed_bytes(nbt)) / ((size_t)16 * (nbt * 8 + 4) * 8));
    long long wc = share < fit ? share : fit;
    return (int)(wc < 1 ? 1 : wc);
}

// row stride of the staged f in the gain role (see gain_role): a constant 260 for the 8-tile kernel on grids up to 256
int gain_ldn(int nbt, int N) { return (nbt == 8 && N <= 256) ? 260 : ((N + 7) & ~3); }

int dmma_stages(int nbt) { return nbt <= 2 ? 8 : (nbt == 8 ? 5 : 4); }

size_t dmma_smem(int nbt, int N, const KxTiled& t, const KxPlan& plan)
{
    const int WC = plan.WC;
    const size_t gain = (size_t)(nbt * 8) * gain_ldn(nbt, N) * 8 + (size_t)WARPS * dmma_stages(nbt) * kStageBytes;
    const size_t loss = loss_fixed_bytes(nbt) + (size_t)WC * 16 * (nbt * 8 + 4) * 8;
    const size_t fb = contract_smem<KX_FB_BT, MODE_LOG_TAB, 0>(N);
    const size_t fin = finish_scratch_bytes(N, plan.GG, plan.GL, t.NT, t.RS);
    size_t m = gain > loss ? gain : loss;
    if (fb > m) m = fb;
    if (fin > m) m = fin;
    return m;
}

// member tiles (of 8) per pass: limited by the batch and by the shared memory the rows of f need in the gain role
int dmma_nbt(int N, int B)
{
    int nbt = B <= 8 ? 1 : (B <= 16 ? 2 : (B <= 32 ? 4 : 8));
    auto need = [&](int k) { return (size_t)(k * 8) * gain_ldn(k, N) * 8 + (size_t)WARPS * dmma_stages(k) * kStageBytes + 512; };
    while (nbt > 1 && need(nbt) > kSmemMax) nbt >>= 1;
    return nbt;
}

template <int NBT, int STAGES, int LDNC>
cudaError_t launch_dmma_t(const KxDev& d, const KxTiled& t, const KxPlan& plan, const double* f, int B, KxStage& st,
                          unsigned* bar_total, cudaStream_t s)
{
    const size_t smem = dmma_smem(NBT, d.N, t, plan);
    st.bar_target = *bar_total + (unsigned)(plan.GG + plan.GL);
    const cudaError_t e = kx_launch_coop(k_dmma<NBT, STAGES, LDNC>, dim3(plan.GG + plan.GL), dim3(NTHR), smem, s, d, t, plan, B, f, st);
    if (e == cudaSuccess) *bar_total = st.bar_target;
    return e;
}

}  // namespace

// columns of the partials for a batch of B members: whole 8-member MMA tiles, whole passes
int kx_xstride(int B)
{
    if (B <= 8) return 8;
    if (B <= 16) return 16;
    if (B <= 32) return 32;
    return ((B + 63) / 64) * 64;
}

cudaError_t kx_dmma_configure()
{
    static bool done = false;
    if (done) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(k_dmma<1, 8, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dmma<2, 8, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dmma<4, 4, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dmma<8, 5, 0>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_dmma<8, 5, 260>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)kSmemMax);
    done = e == cudaSuccess;
    return e;
}

// The plan of one launch.  Work in units of one gain group (8 DMMA per member tile): gain = groups, loss = LC NR8 / 2
// (weighted by kLossCost).  Every CTA must be resident (grid barrier): at most one per SM.  The gain warps are dealt to the
// tiles in proportion to the tiles' groups (largest remainder), at least one and at most one per group.
void kx_dmma_plan(const KxDev& d, const KxTiled& t, int sm_count, const unsigned* vt_host, int B, KxPlan* plan)
{
    const int nbt = dmma_nbt(d.N, B);
    const int NT = t.NT;
    const unsigned Gtot = vt_host[NT];
    const double wg = (double)(Gtot > 0 ? Gtot : 1);
    const double wl = 0.5 * (double)t.LC * (double)t.NR8 * kLossCost;
    long long G = (long long)((wg + wl) / 8.0);
    if (G > sm_count) G = sm_count;
    if (G < 2) G = 2;
    const long long U = (long long)t.RS * t.LC;

    // cost of a tile in units of one group: its groups plus kRunCost per run (one run per n: the fold at the end of a run and
    // the short runs of the high tiles cost DMMA issue slots; measured with the clock-stamp trace: 0.83 of the DMMA peak on
    // tile 0, 0.76 on the last tile of cfg3)
    std::vector<unsigned> g(NT, 0u);
    std::vector<double> c(NT, 0.0);
    double Ctot = 0.0;
    for (int k = 0; k < NT; ++k) {
        g[k] = vt_host[k + 1] - vt_host[k];
        c[k] = g[k] ? (double)g[k] + (nbt <= 2 ? 0.0 : kRunCost) * (double)d.N : 0.0;     // small batches: bytes, not issue slots
        Ctot += c[k];
    }
    // the gain warps of GG CTAs dealt to the tiles in proportion to the tiles' costs (largest remainder), at least one and at
    // most one per group; returns the load of the busiest warp in group units
    auto deal = [&](int GG, std::vector<unsigned>& w) -> double {
        const unsigned NW = (unsigned)GG * WARPS;
        w.assign(NT, 0u);
        unsigned used = 0;
        for (int k = 0; k < NT; ++k) {
            if (g[k]) {
                unsigned v = (unsigned)((double)NW * c[k] / Ctot);
                if (v < 1) v = 1;
                if (v > g[k]) v = g[k];
                w[k] = v; used += v;
            }
        }
        while (used > NW) {            // the minimum of one warp per tile overshot: take from the lightest-loaded warps
            int best = -1;
            for (int k = 0; k < NT; ++k)
                if (w[k] > 1 && (best < 0 || c[k] * w[best] < c[best] * w[k])) best = k;
            if (best < 0) break;
            --w[best]; --used;
        }
        while (used < NW) {            // left-over warps go where a warp has the most work
            int best = -1;
            for (int k = 0; k < NT; ++k)
                if (w[k] < g[k] && (best < 0 || c[k] * w[best] > c[best] * w[k])) best = k;
            if (best < 0) break;
            ++w[best]; ++used;
        }
        // whole groups per warp: move warps from the tile that can best spare one to the tile with the busiest warp while
        // that lowers the maximum
        auto load_of = [&](int k, unsigned wk) { return (double)((g[k] + wk - 1) / wk) * (c[k] / (double)g[k]); };
        for (int it = 0; it < 4 * NT; ++it) {
            int kmax = -1, kmin = -1;
            double lmax = 0.0, lmin = 1e300;
            for (int k = 0; k < NT; ++k)
                if (w[k]) { const double l = load_of(k, w[k]); if (l > lmax) { lmax = l; kmax = k; } }
            for (int k = 0; k < NT; ++k)
                if (w[k] > 1 && k != kmax) { const double l = load_of(k, w[k] - 1); if (l < lmin) { lmin = l; kmin = k; } }
            if (kmax < 0 || kmin < 0 || w[kmax] >= g[kmax] || !(lmin < lmax)) break;
            ++w[kmax]; --w[kmin];
        }
        double load = 0.0;
        for (int k = 0; k < NT; ++k)
            if (w[k]) { const double l = load_of(k, w[k]); if (l > load) load = l; }
        return load;
    };

    // Role split.  First guess: in proportion to the DMMA counts.  Both roles are quantised (whole groups per gain warp,
    // whole chunks of 16 k per loss CTA: 10 or 11 chunks at cfg3 is a 10 % step), so the neighbours of the guess are tried
    // and the split with the earliest barrier wins: gain = load of the busiest warp; loss = chunks of the busiest CTA, one
    // chunk of a full supertile being two groups' worth of DMMA per warp, plus the longer prologue of the loss role
    // (kLossPrologue groups, from the clock-stamp trace).
    // the finishing phase gathers one 2 KiB slice per loss slot and one 128-byte slice per gain slot into shared memory: that
    // bounds the number of loss CTAs (found by tests/test_plan_cpu.py on profiles with hardly any gain work)
    const long long gl_cap = ((long long)kSmemMax - (long long)((d.N + 3) & ~3) * 8 - (G + NT) * 128) / 2048 - t.RS;
    int gl_max = (int)G - 1;
    if (gl_max > U) gl_max = (int)U;
    if (gl_max > gl_cap) gl_max = (int)gl_cap;
    if (gl_max < 1) gl_max = 1;
    int gl0 = (int)((double)G * wl / (wg + wl) + 0.5);
    if (gl0 < 1) gl0 = 1;
    if (gl0 > gl_max) gl0 = gl_max;
    // small batches stream from HBM: a loss warp has 8 KiB in flight (2 of its 3 ring stages), a gain warp 14 KiB (7 of 8), and
    // the loss chunk costs 2.7 instead of 2.1 groups (measured on cfg4: 0.78 us per chunk, 0.29 us per group)
    const double chunk_w = nbt <= 2 ? 1.35 : kLossChunk, prologue_w = nbt <= 2 ? 13.0 : kLossPrologue;
    const double chunk_groups = 2.0 * (double)(t.NR8 < 32 * t.RS ? t.NR8 : 32 * t.RS) / (32.0 * t.RS) * chunk_w;
    int gl = gl0;
    double best_t = 1e300;
    std::vector<unsigned> w, wtry;
    for (int cand = gl0 - 4; cand <= gl0 + 12; ++cand) {
        if (cand < 1 || cand > gl_max) continue;
        const double tg = deal((int)G - cand, wtry);
        const double tl = (double)((U + cand - 1) / cand) * chunk_groups + prologue_w;
        const double tt = tg > tl ? tg : tl;
        if (tt < best_t - 1e-9) { best_t = tt; gl = cand; }
    }
    if (gl > gl_max) gl = gl_max;                  // every loss CTA has at least one chunk, the finishing scratch fits
    plan->nbt = nbt;
    plan->GL = gl;
    plan->GG = (int)G - gl;
    plan->WC = loss_window(t, gl, nbt);
    deal(plan->GG, w);

    unsigned run = 0;
    for (int k = 0; k < NT; ++k) { plan->wstart[k] = run; plan->vt[k] = vt_host[k]; run += w[k]; }
    plan->wstart[NT] = run; plan->vt[NT] = vt_host[NT];
    for (int sp = 0; sp < 4; ++sp) {
        const unsigned long long l0 = (unsigned long long)sp * t.LC, l1 = l0 + t.LC;
        plan->ld0[sp] = sp < t.RS ? (unsigned)(((l0 + 1ull) * (unsigned)gl - 1ull) / (unsigned long long)U) : 1u;
        plan->ld1[sp] = sp < t.RS ? (unsigned)((l1 * (unsigned)gl - 1ull) / (unsigned long long)U) : 0u;
    }
    for (int k = NT + 1; k <= KX_MAX_NT; ++k) { plan->wstart[k] = run; plan->vt[k] = vt_host[NT]; }
}

cudaError_t kx_launch_dmma(const KxDev& d, const KxTiled& t, const KxPlan& plan, const double* f, int B,
                           KxStage st, unsigned* bar_total, cudaStream_t s)
{
    switch (plan.nbt) {
        case 1: return launch_dmma_t<1, 8, 0>(d, t, plan, f, B, st, bar_total, s);
        case 2: return launch_dmma_t<2, 8, 0>(d, t, plan, f, B, st, bar_total, s);
        case 4: return launch_dmma_t<4, 4, 0>(d, t, plan, f, B, st, bar_total, s);
        default:
            if (d.N <= 256) return launch_dmma_t<8, 5, 260>(d, t, plan, f, B, st, bar_total, s);
            return launch_dmma_t<8, 5, 0>(d, t, plan, f, B, st, bar_total, s);
    }
}

// Host-only view of the launch plan (no device needed): used by the CPU tests of the planner's invariants.
extern "C" kx_status_t kx_plan_probe(int32_t N, int32_t B, int32_t Q, int32_t sm_count, const uint32_t* groups_per_tile,
                                     int32_t* head, uint32_t* wstart, uint32_t* ld)
{
    if (N < 4 || N > KX_MAX_N || B < 1 || sm_count < 2 || !groups_per_tile || !head || !wstart || !ld) return KX_ERR_INVALID_ARG;
    if (Q != 2 && Q != 8 && Q != 16 && Q != 24 && Q != 32) return KX_ERR_INVALID_ARG;
    KxDev d = {};
    d.N = N;
    KxTiled t = {};
    t.NT = (N + KX_TI - 1) / KX_TI;
    t.Q = Q;
    t.LC = ((N - 1) * Q + 15) / 16;
    t.NR8 = (N + 7) / 8;
    t.RS = (N + 255) / 256;
    std::vector<unsigned> vt((size_t)t.NT + 1, 0u);
    for (int k = 0; k < t.NT; ++k) vt[k + 1] = vt[k] + groups_per_tile[k];
    KxPlan plan = {};
    kx_dmma_plan(d, t, sm_count, vt.data(), B, &plan);
    head[0] = plan.GG; head[1] = plan.GL; head[2] = plan.nbt; head[3] = plan.WC; head[4] = t.NT; head[5] = t.RS; head[6] = t.LC;
    head[7] = (int32_t)dmma_smem(plan.nbt, N, t, plan);
    for (int k = 0; k <= t.NT; ++k) wstart[k] = plan.wstart[k];
    for (int k = 0; k < 4; ++k) { ld[k] = plan.ld0[k]; ld[4 + k] = plan.ld1[k]; }
    return KX_OK;
}
