// kx_tiled.cu -- steps a4-a5 as one FP64 tensor-core contraction over the tiled storage (KX_STORE_TILED).
//
//   gain[b,i] = sum_{n<=m} (W_inm + W_imn) f_n f_m                        eq. 4.6 with 2.6
//   nu[b,i]   = sum_j sum_{c<Q} M_c(i,j) a_c(b,j)   (loss_i = f_i nu_i)   eq. B.19-B.20, see
//               kx_tiled_build.cu for the Chebyshev-moment form of the interpolated loss term and its error bound
//
// Both are out[b,i] += sum_k X[b,k] A[k,i] with A streamed once from HBM/L2 (cp.async) and X built from the small
// operand array XT: X = f_n f_m for the gain, X = a_c(b,j) for the loss.  The products run on the FP64 tensor
// pipe: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4), M = 8 members, N = 8 rows, K = 4.  The CTAs of one launch are split
// between the two terms in proportion to their work (see k_dmma); the finishing kernel (kx_contract.cu) adds the
// partials: no atomics, bit-reproducible.
//
// Compiled with --fmad=false; fused multiply-adds are explicit.
#include "kx_internal.cuh"


namespace {

// cost of one loss DMMA relative to one gain DMMA in the CTA split of k_dmma (measured on cfg3: the split that
// makes both roles finish together)
constexpr double kLossCost = 1.0;

// D[8 members x 8 rows] += X[8 members x 4 k] * A[4 k x 8 rows]
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
        : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

// ---------------------------------------------------------------- operand rows XT[row, b]
//   rows loss_row0 + jQ + c    a_c(b,j), c < Q, j < N-1      (loss; the gain role of k_dmma reads f itself)
// LOG:    g(omega_q) = 2^(y_j + omega_q (y_{j+1}-y_j)), y = log2 max(f, f_floor), at the Q Chebyshev nodes of [0,1];
//         a_c = (2-delta_c0)/Q sum_q g(omega_q) cos(c theta_q)            (discrete Chebyshev transform)
//         A member is flagged for the exact streaming path when, for some bracket,
//             2 (|ln(f_{j+1}/f_j)|/4)^Q / Q! * max(f_j, f_{j+1}) > 1e-15 max_i f_i    (interpolation error bound);
//         this kernel accumulates the two maxima per member (mstat, kx_internal.cuh), the consumers compare them.
// LINEAR: a_0 = (f_j + f_{j+1})/2, a_1 = (f_{j+1} - f_j)/2 (exact).
// Also writes yd[b,j] = (y_j, y_{j+1}-y_j) for the streaming kernel.
// grid.x = N (row j), 256 threads = 64 members x 4 coefficient phases.
__global__ void __launch_bounds__(256) k_xt(KxDev d, KxTiled t, const double* __restrict__ f, double2* __restrict__ yd,
                                            double* __restrict__ XT, int xstride, long long* __restrict__ mstat, int B)
{
    __shared__ double s_node[KX_QMAX];
    __shared__ double s_G[KX_QMAX][68];        // row stride 4 mod 16: the 4 x 8 fragment reads below are conflict free
    __shared__ double s_y[2][64];
    __shared__ double s_tab[1 << KX_EXP_BITS];
    const int N = d.N, Q = t.Q, j = blockIdx.x;
    const bool tab = d.exp_impl == KX_EXP_TABLE;
    const int bl = threadIdx.x & 63, ph = threadIdx.x >> 6;
    const bool logm = d.interp == KX_INTERP_LOG;
    kx_pdl_trigger();       // first kernel of the call (ordinary launch): the contraction kernel may start right away
    // the transform runs on the tensor pipe: a_c[b] = sum_q dct[c,q] G[q,b] is a (Q x Q) x (Q x 64) product, warp w takes
    // members 8w..8w+7; its fragments of dct (lane: dct[8 ct + lane/4][4 ks + lane%4]) stay in registers
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    double afr[KX_QMAX / 8][KX_QMAX / 4];
    if (logm) {
#pragma unroll
        for (int ct = 0; ct < KX_QMAX / 8; ++ct)
#pragma unroll
            for (int ks = 0; ks < KX_QMAX / 4; ++ks)
                afr[ct][ks] = (8 * ct < Q && 4 * ks < Q) ? t.dct[(8 * ct + (lane >> 2)) * Q + 4 * ks + (lane & 3)] : 0.0;
        if (threadIdx.x < Q) s_node[threadIdx.x] = t.nodes[threadIdx.x];
        if (tab) s_tab[threadIdx.x] = d.exptab[threadIdx.x];          // 256 threads, 2^KX_EXP_BITS = 256 entries
    }
    __syncthreads();
    for (int b0 = 0; b0 < B; b0 += 64) {
        const int b = b0 + bl;
        const bool act = b < B;
        double fj = 0.0, fj1 = 0.0;
        if (act) {
            fj = f[(size_t)b * N + j];
            fj1 = j + 1 < N ? f[(size_t)b * N + j + 1] : fj;
        }
        if (act && ph == 0) {
            const long long fk = __double_as_longlong(fabs(fj));
            if (fk > mstat[2 * b + 1]) atomicMax(mstat + 2 * b + 1, fk);
        }
        if (!logm) {
            if (act && ph == 0) {
                yd[(size_t)b * N + j] = make_double2(fj, fj1 - fj);
                if (j < N - 1) {
                    double* row = XT + (size_t)(t.loss_row0 + 2 * j) * xstride + b;
                    row[0] = 0.5 * (fj + fj1);
                    row[xstride] = 0.5 * (fj1 - fj);
                }
            }
            continue;
        }
        // one logarithm per thread: phase 0 takes f_j, phase 1 takes f_(j+1)
        if (ph < 2) s_y[ph][bl] = log2(fmax(ph == 0 ? fj : fj1, d.f_floor));
        __syncthreads();
        const double y0 = s_y[0][bl];
        const double y1 = j + 1 < N ? s_y[1][bl] : y0;
        const double dy = y1 - y0;
        if (act && ph == 0) {
            yd[(size_t)b * N + j] = make_double2(y0, dy);
            const double c = 0.6931471805599453 * fabs(dy);
            if (j < N - 1 && c > 0.0) {
                // log2 of the bracket's error bound (log2 max_i f_i is subtracted by the consumers)
                const long long lk = kx_dkey(fmax(y0, y1) + (double)Q * (log2(c) - 2.0) + t.flag_log2);
                if (lk > mstat[2 * b]) atomicMax(mstat + 2 * b, lk);
            }
        }
        if (j >= N - 1) { __syncthreads(); continue; }       // uniform over the CTA
        if (tab) for (int q = ph; q < Q; q += 4) s_G[q][bl] = kx_exp2_tab<1>(fma(s_node[q], dy, y0), s_tab);
        else for (int q = ph; q < Q; q += 4) s_G[q][bl] = exp2(fma(s_node[q], dy, y0));
        __syncthreads();
        {
            double D[KX_QMAX / 8][2];
#pragma unroll
            for (int ct = 0; ct < KX_QMAX / 8; ++ct) D[ct][0] = D[ct][1] = 0.0;
#pragma unroll
            for (int ks = 0; ks < KX_QMAX / 4; ++ks) {
                if (4 * ks < Q) {                                        // uniform
                    const double g = s_G[4 * ks + (lane & 3)][8 * warp + (lane >> 2)];
#pragma unroll
                    for (int ct = 0; ct < KX_QMAX / 8; ++ct)
                        if (8 * ct < Q) dmma884(D[ct][0], D[ct][1], afr[ct][ks], g);
                }
            }
            const int bw = b0 + 8 * warp + 2 * (lane & 3);                // lane holds a_c[bw], a_c[bw+1], c = 8 ct + lane/4
#pragma unroll
            for (int ct = 0; ct < KX_QMAX / 8; ++ct) {
                if (8 * ct < Q) {
                    double* dst = XT + (size_t)(t.loss_row0 + j * Q + 8 * ct + (lane >> 2)) * xstride + bw;
                    if (bw + 1 < B) *reinterpret_cast<double2*>(dst) = make_double2(D[ct][0], D[ct][1]);
                    else if (bw < B) dst[0] = D[ct][0];
                }
            }
        }
        __syncthreads();
    }
}

// ---------------------------------------------------------------- the contraction
__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc)
{
    const unsigned sa = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" :: "r"(sa), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int NPEND>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" :: "n"(NPEND) : "memory"); }

constexpr int kStageBytes = KX_GROUP_DBL * 8 + 16;     // gain ring stage: 2 KiB of A + 4 descriptors
constexpr int kLossStages = 3;
constexpr int kLossABytes = 32 * 1024;                 // loss stage: 16 k x 256 rows of AL ...
__host__ __device__ constexpr int loss_stage_bytes(int NBT) { return kLossABytes + 16 * (NBT * 8 + 4) * 8; }   // ... + 16 k x members of X

// One CTA per SM.  CTAs [0, GG) take equal ranges of gain groups, CTAs [GG, GG+GL) equal ranges of loss chunks.
//
// gain role: the rows f[b, :] of the CTA's 8 NBT members sit in shared memory (row stride = 4 mod 16 doubles when
//   N = 0 mod 16: the 8 members x 4 k fragment reads of a quad are bank-conflict free), copied straight from the
//   caller's f; every warp streams its own share of the groups through a private
//   cp.async ring and holds a 16-row x 8 NBT-member accumulator (2 NBT DMMA per quad and fragment pair).
//   The DMMAs of a run (fixed n) take X = f_m and accumulate into T; f_n multiplies T once, when the run ends.
//   The ring keeps flowing across tile boundaries.
// loss role: a dense GEMM.  The CTA stages chunks of 16 k (32 KiB of AL for 256 rows + the matching 16 rows of
//   Chebyshev coefficients) through a 3-stage cp.async pipeline shared by all warps; warp w owns rows
//   [32 w, 32 w + 32) x 8 NBT members (4 NBT DMMA per quad).
// A range that crosses a tile (supertile) boundary produces one partial per piece, slot = worker + tile (a gain
// worker is a warp, a loss worker a CTA); the finishing kernel adds the partials of a row in slot order: no
// atomics, bit-reproducible.
template <int NBT, int WARPS, int STAGES>
__global__ void __launch_bounds__(WARPS * 32, 1)
k_dmma(KxTiled t, int N, int B, unsigned Gtot, const double* __restrict__ f, const double* __restrict__ XT, int xstride,
       double* __restrict__ gpart, double* __restrict__ lpart, int GG, int GL)
{
    extern __shared__ __align__(16) unsigned char smem[];
    constexpr int LD = NBT * 8 + 4;
    constexpr int NTHR = WARPS * 32;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int krow = lane & 3, lr = lane >> 2;
    const int bcol0 = blockIdx.y * (NBT * 8);
    kx_pdl_trigger();

    if ((int)blockIdx.x < GG) {
        // ------------------------------------------------------------ gain role: every warp is an independent worker
        unsigned* s_vt = reinterpret_cast<unsigned*>(smem);                               // [NT + 1]
        const int vtbytes = ((t.NT + 1) * 4 + 15) & ~15;
        const int LDN = (N + 7) & ~3;             // row stride of s_f: >= N + 4, = 0 mod 4; N = 0 mod 16 gives 4 mod 16
        double* s_f = reinterpret_cast<double*>(smem + vtbytes);                          // [8 NBT][LDN]
        unsigned char* ring = smem + vtbytes + (size_t)(NBT * 8) * LDN * 8 + (size_t)warp * STAGES * kStageBytes;

        const unsigned NW = (unsigned)GG * WARPS, wk = blockIdx.x * WARPS + warp;
        const unsigned g0 = (unsigned)((unsigned long long)wk * Gtot / NW);
        const unsigned g1 = (unsigned)((unsigned long long)(wk + 1) * Gtot / NW);
        const unsigned n = g1 - g0;
        auto issue = [&](unsigned gi) {
            const double* src = t.A + (size_t)(g0 + gi) * KX_GROUP_DBL;
            unsigned char* dst = ring + (size_t)(gi % STAGES) * kStageBytes;
#pragma unroll
            for (int k = 0; k < 4; ++k) cp_async16(dst + (k * 32 + lane) * 16, src + (k * 32 + lane) * 2);
            if (lane == 0) cp_async16(dst + KX_GROUP_DBL * 8, t.desc + (size_t)(g0 + gi) * 4);
        };
        // The gain role reads only the caller's f and the tensor, nothing an earlier kernel of this call writes: under
        // programmatic dependent launch it runs while the operand-preparation kernel is still at work.
        // The tensor stream starts first; f^T and the tile table arrive while it is in flight.
#pragma unroll
        for (int s = 0; s < STAGES - 1; ++s) {
            if ((unsigned)s < n) issue(s);
            cp_async_commit();
        }
        // s_f[b][n] = f[bcol0 + b][n], n < N; s_f[b][N] = 1 (the scale of padding quads), s_f[b][N+1..] = 0.  The rows of
        // f are copied as they are (16-byte cp.async when N is even); members beyond B are zero.  Every CTA starts its
        // walk somewhere else so that the CTAs do not all ask the same L2 lines at once.
        {
            const int chunks = (N & 1) ? 0 : N >> 1;                   // 16-byte chunks per row
            const int total = NBT * 8 * chunks;
            const int rot = total ? (int)((blockIdx.x * 977u) % (unsigned)total) : 0;
            for (int k0 = tid; k0 < total; k0 += NTHR) {
                int k = k0 + rot;
                if (k >= total) k -= total;
                const int bb = k / chunks, cc = k - bb * chunks;
                if (bcol0 + bb < B) cp_async16(s_f + (size_t)bb * LDN + 2 * cc, f + (size_t)(bcol0 + bb) * N + 2 * cc);
                else *reinterpret_cast<double2*>(s_f + (size_t)bb * LDN + 2 * cc) = make_double2(0.0, 0.0);
            }
            if (!chunks)
                for (int k = tid; k < NBT * 8 * N; k += NTHR) {
                    const int bb = k / N, nn = k - bb * N;
                    s_f[(size_t)bb * LDN + nn] = bcol0 + bb < B ? __ldcg(f + (size_t)(bcol0 + bb) * N + nn) : 0.0;
                }
            for (int k = tid; k < NBT * 8 * (LDN - N); k += NTHR) {
                const int bb = k / (LDN - N), cc = k - bb * (LDN - N);
                s_f[(size_t)bb * LDN + N + cc] = cc == 0 ? 1.0 : 0.0;
            }
        }
        cp_async_commit();
        for (int k = tid; k <= t.NT; k += NTHR) s_vt[k] = t.vtptr[k];
        cp_async_wait<0>();
        __syncthreads();
        if (n == 0) { kx_pdl_wait(); return; }

        const double* xb = s_f + (size_t)lr * LDN + krow;    // + 8 bt LDN + column: the lane's member row of tile bt
        const int LD8 = 8 * LDN;
        int vt = 0;
        while (s_vt[vt + 1] <= g0) ++vt;
        unsigned bnd = s_vt[vt + 1] - g0;                    // first group (relative) of the next tile

        // acc: the tile's partial.  T: sum over the m of the current run (fixed n) of f_m A[(n,m), i]; when the run ends,
        // acc += f_n T.  Lane holds out[b = 8 bt + lane/4][i = 8 rb + 2 (lane%4) + {0,1}], the same member b as its
        // fragment of X, so f_n[b] scales its own accumulators.
        double acc[NBT][2][2], T[NBT][2][2], sn[NBT];
#pragma unroll
        for (int bt = 0; bt < NBT; ++bt)
#pragma unroll
            for (int rb = 0; rb < 2; ++rb) { acc[bt][rb][0] = acc[bt][rb][1] = 0.0; T[bt][rb][0] = T[bt][rb][1] = 0.0; }
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
        // one partial per (worker, tile), slot = worker + tile
        auto flush = [&](int tile) {
            double* dst = gpart + ((size_t)(wk + tile) * xstride + bcol0 + lr) * 16 + 2 * krow;
#pragma unroll
            for (int bt = 0; bt < NBT; ++bt)
#pragma unroll
                for (int rb = 0; rb < 2; ++rb) {
                    *reinterpret_cast<double2*>(dst + (size_t)bt * 128 + rb * 8) = make_double2(acc[bt][rb][0], acc[bt][rb][1]);
                    acc[bt][rb][0] = acc[bt][rb][1] = 0.0;
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
            if (gi == bnd) {                                 // the range crosses into the next tile
                fold();
                flush(vt);
                do { ++vt; } while (s_vt[vt + 1] - g0 <= gi);
                bnd = s_vt[vt + 1] - g0;
            }
            // refill the slot freed by group gi-1, then make sure groups gi and gi+1 are in shared memory
            if (gi + STAGES - 1 < n) issue(gi + STAGES - 1);
            cp_async_commit();
            cp_async_wait<STAGES - 2>();
            __syncwarp();
            const unsigned char* st = ring + (size_t)(gi % STAGES) * kStageBytes;
            const double* wd = reinterpret_cast<const double*>(st) + lane;
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
                if (more && srow != srow_cur) {              // the run (n) ends with this quad
                    fold();
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
        flush(vt);
        kx_pdl_wait();        // the grid must not complete before the kernels it follows have
        return;
    }

    // ---------------------------------------------------------------- loss role
    {
        constexpr int SB = loss_stage_bytes(NBT);
        constexpr int R8 = 32 / WARPS;            // 8-row blocks per warp: the CTA covers a 256-row supertile
        static_assert(WARPS == 8 || WARPS == 16, "loss role: 8 or 16 warps");
        bool waited = false;  // the Chebyshev coefficients in XT come from k_xt: griddepcontrol.wait before the first X copy
        const unsigned cl = blockIdx.x - GG;
        const unsigned LC = (unsigned)t.LC;
        const unsigned U = (unsigned)t.RS * LC;
        const unsigned u0 = (unsigned)((unsigned long long)cl * U / (unsigned)GL);
        const unsigned u1 = (unsigned)((unsigned long long)(cl + 1) * U / (unsigned)GL);
        unsigned u = u0;
        while (u < u1) {
            const unsigned sp = u / LC;                                  // supertile
            const unsigned ue = min(u1, (sp + 1) * LC);
            const unsigned ka = u - sp * LC, n = ue - u;
            const int nb = min(32, t.NR8 - 32 * (int)sp);                // 8-row blocks of this supertile
            const int nbw = min(R8, max(0, nb - R8 * warp));             // ... of this warp

            auto issueA = [&](unsigned kc, int slot) {          // the tensor: does not depend on any kernel of this call
                unsigned char* dstA = smem + (size_t)slot * SB;
                const double* srcA = t.AL + ((size_t)kc * t.NR8 + 32 * sp) * 128;
                for (int k = tid; k < nb * 64; k += NTHR) cp_async16(dstA + (size_t)k * 16, srcA + (size_t)k * 2);
            };
            auto issueX = [&](unsigned kc, int slot) {          // the coefficients written by k_xt
                double* dstX = reinterpret_cast<double*>(smem + (size_t)slot * SB + kLossABytes);
                const double* srcX = XT + (size_t)(t.loss_row0 + 16 * kc) * xstride + bcol0;
                for (int k = tid; k < 16 * NBT * 4; k += NTHR) {
                    const int r = k / (NBT * 4), cc = k - r * (NBT * 4);
                    cp_async16(dstX + (size_t)r * LD + 2 * cc, srcX + (size_t)r * xstride + 2 * cc);
                }
            };
            auto issue = [&](unsigned kc, int slot) { issueA(kc, slot); issueX(kc, slot); };

            double acc[R8][NBT][2];
#pragma unroll
            for (int r = 0; r < R8; ++r)
#pragma unroll
                for (int bt = 0; bt < NBT; ++bt) acc[r][bt][0] = acc[r][bt][1] = 0.0;

            // prologue: the tensor chunks are requested before the wait on the operand-preparation kernel
#pragma unroll
            for (int s = 0; s < kLossStages - 1; ++s)
                if ((unsigned)s < n) issueA(ka + s, s);
            if (!waited) { kx_pdl_wait(); waited = true; }
#pragma unroll
            for (int s = 0; s < kLossStages - 1; ++s) {
                if ((unsigned)s < n) issueX(ka + s, s);
                cp_async_commit();
            }
            for (unsigned it = 0; it < n; ++it) {
                cp_async_wait<kLossStages - 2>();        // this thread's copies of chunk `it` have landed
                __syncthreads();                         // everyone's have; everyone is done with chunk it-1
                if (it + kLossStages - 1 < n) issue(ka + it + kLossStages - 1, (int)((it + kLossStages - 1) % kLossStages));
                cp_async_commit();
                if (nbw > 0) {
                    const double* sA = reinterpret_cast<const double*>(smem + (size_t)(it % kLossStages) * SB) + (size_t)warp * (R8 * 128) + lane;
                    const double* sX = reinterpret_cast<const double*>(smem + (size_t)(it % kLossStages) * SB + kLossABytes) + (size_t)krow * LD + lr;
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
            }
            cp_async_wait<0>();
            __syncthreads();              // the stages are free again for the next piece

            double* dst = lpart + ((size_t)(cl + sp) * xstride + bcol0) * 256 + 8 * R8 * warp + 2 * krow;
#pragma unroll
            for (int r = 0; r < R8; ++r)
                if (r < nbw)
#pragma unroll
                    for (int bt = 0; bt < NBT; ++bt)
                        *reinterpret_cast<double2*>(dst + (size_t)(8 * bt + lr) * 256 + 8 * r) = make_double2(acc[r][bt][0], acc[r][bt][1]);
            u = ue;
        }
        if (!waited) kx_pdl_wait();
    }
}

template <int NBT, int WARPS, int STAGES>
size_t dmma_smem(const KxTiled& t, int N)
{
    const size_t gain = (size_t)(((t.NT + 1) * 4 + 15) & ~15) + (size_t)(NBT * 8) * ((N + 7) & ~3) * 8 + (size_t)WARPS * STAGES * kStageBytes;
    const size_t loss = (size_t)kLossStages * loss_stage_bytes(NBT);
    return gain > loss ? gain : loss;
}

template <int NBT, int WARPS, int STAGES>
cudaError_t launch_dmma_t(const KxTiled& t, int N, unsigned Gtot, int GG, int GL, const double* f, const double* XT, int xstride,
                          double* gpart, double* lpart, int B, cudaStream_t s)
{
    const size_t smem = dmma_smem<NBT, WARPS, STAGES>(t, N);
    cudaError_t e = cudaFuncSetAttribute(k_dmma<NBT, WARPS, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(GG + GL, (B + NBT * 8 - 1) / (NBT * 8));
    return kx_launch(k_dmma<NBT, WARPS, STAGES>, grid, dim3(WARPS * 32), smem, s, true, t, N, B, Gtot, f, XT, xstride, gpart, lpart, GG, GL);
}

// member tiles (of 8) per CTA: limited by the batch and by the shared memory f^T of the gain role needs
int kx_dmma_warps(int nbt) { (void)nbt; return 8; }
int dmma_nbt(int N, int B)
{
    int nbt = B <= 8 ? 1 : (B <= 16 ? 2 : (B <= 32 ? 4 : 8));
    auto need = [&](int k) { return (size_t)(k * 8) * ((N + 7) & ~3) * 8 + (size_t)kx_dmma_warps(k) * (k <= 2 ? 8 : 4) * kStageBytes + 512; };
    while (nbt > 1 && need(nbt) > 227u * 1024u) nbt >>= 1;
    return nbt;
}

}  // namespace

int kx_dmma_workers(int N, int B) { return kx_dmma_warps(dmma_nbt(N, B)); }

// columns of XT / the partials for a batch of B members: whole 8-member MMA tiles, whole CTA column groups
int kx_xstride(int B)
{
    if (B <= 8) return 8;
    if (B <= 16) return 16;
    if (B <= 32) return 32;
    return ((B + 63) / 64) * 64;
}

// CTAs per role.  Work in units of one gain group (8 DMMA per member tile): gain = groups, loss = LC * NR8 / 2.
void kx_dmma_split(const KxDev& d, const KxTiled& t, int sm_count, long long groups, int B, int* GG, int* GL)
{
    const int nbt = dmma_nbt(d.N, B);
    const int ny = (B + nbt * 8 - 1) / (nbt * 8);
    const double wg = (double)(groups > 0 ? groups : 1);
    const double wl = 0.5 * (double)t.LC * (double)t.NR8 * kLossCost;
    long long G = (long long)((wg + wl) / 8.0);
    const long long cap = sm_count / ny > 2 ? sm_count / ny : 2;
    if (G > cap) G = cap;
    if (G < 2) G = 2;
    int gl = (int)((double)G * wl / (wg + wl) + 0.5);
    if (gl < 1) gl = 1;
    if (gl > (int)G - 1) gl = (int)G - 1;
    *GL = gl;
    *GG = (int)G - gl;
}

cudaError_t kx_launch_xt(const KxDev& d, const KxTiled& t, const double* f, double* yd, double* XT, int xstride,
                         long long* mstat, int B, cudaStream_t s)
{
    // first kernel of the call: ordinary launch
    return kx_launch(k_xt, dim3(d.N), dim3(256), 0, s, false, d, t, f, reinterpret_cast<double2*>(yd), XT, xstride, mstat, B);
}

cudaError_t kx_launch_dmma(const KxDev& d, const KxTiled& t, long long groups, int GG, int GL, const double* f,
                           const double* XT, int xstride, double* gpart, double* lpart, int B, cudaStream_t s)
{
    switch (dmma_nbt(d.N, B)) {
        case 1: return launch_dmma_t<1, 8, 8>(t, d.N, (unsigned)groups, GG, GL, f, XT, xstride, gpart, lpart, B, s);
        case 2: return launch_dmma_t<2, 8, 8>(t, d.N, (unsigned)groups, GG, GL, f, XT, xstride, gpart, lpart, B, s);
        case 4: return launch_dmma_t<4, 8, 4>(t, d.N, (unsigned)groups, GG, GL, f, XT, xstride, gpart, lpart, B, s);
        default: return launch_dmma_t<8, 8, 4>(t, d.N, (unsigned)groups, GG, GL, f, XT, xstride, gpart, lpart, B, s);
    }
}
