// kx_tiled.cu -- steps a4-a5 as one FP64 tensor-core contraction over the tiled storage (KX_STORE_TILED).
//
//   gain[b,i] = sum_{n<=m} (W_inm + W_imn) f_n f_m                        eq. 4.6 with 2.6
//   nu[b,i]   = sum_j sum_{c<Q} M_c(i,j) a_c(b,j)   (loss_i = f_i nu_i)   eq. B.19-B.20, see
//               kx_tiled_build.cu for the Chebyshev-moment form of the interpolated loss term and its error bound
//
// Both are out[b,i] += sum_k X[b,k] A[k,i] with A streamed once from HBM/L2 (cp.async ring per warp) and X read
// from the small operand array XT (L1/L2 resident): X = f_n f_m for gain quads, X = a_c(b,j) for loss quads.
// The products run on the FP64 tensor pipe: mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4), M = 8 members, N = 8 rows,
// K = 4.  Work is cut into equal ranges of groups (4 quads = 2 KiB of A) per CTA; a range that crosses a
// virtual-tile boundary produces one partial per piece, slot = CTA + virtual tile, and the finishing kernel
// (kx_contract.cu) adds the partials of a tile in slot order: no atomics, bit-reproducible.
//
// Compiled with --fmad=false; fused multiply-adds are explicit.
#include "kx_internal.cuh"

namespace {

// ---------------------------------------------------------------- per-member maximum, flag reset
__global__ void __launch_bounds__(256) k_fmax(int N, const double* __restrict__ f, double* __restrict__ fmx,
                                              int* __restrict__ mflag)
{
    __shared__ double s_red[8];
    const int b = blockIdx.x;
    double v = 0.0;
    for (int i = threadIdx.x; i < N; i += 256) v = fmax(v, fabs(f[(size_t)b * N + i]));
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
    if ((threadIdx.x & 31) == 0) s_red[threadIdx.x >> 5] = v;
    __syncthreads();
    if (threadIdx.x == 0) {
        double a = s_red[0];
#pragma unroll
        for (int w = 1; w < 8; ++w) a = fmax(a, s_red[w]);
        fmx[b] = a;
        mflag[b] = 0;
    }
}

// ---------------------------------------------------------------- operand rows XT[row, b]
//   rows 0..N-1        f^T                                   (gain: X = f_n f_m)
//   row  N             1                                     (scale row of the loss quads)
//   rows N+1+jQ+c      a_c(b,j), c < Q, j < N-1              (loss)
// LOG:    g(omega_q) = 2^(y_j + omega_q (y_{j+1}-y_j)), y = log2 max(f, f_floor), at the Q Chebyshev nodes of [0,1];
//         a_c = (2-delta_c0)/Q sum_q g(omega_q) cos(c theta_q)            (discrete Chebyshev transform)
//         A member is flagged for the exact streaming path when, for some bracket,
//             2 (|ln(f_{j+1}/f_j)|/4)^Q / Q! * max(f_j, f_{j+1}) > 1e-15 max_i f_i    (interpolation error bound)
// LINEAR: a_0 = (f_j + f_{j+1})/2, a_1 = (f_{j+1} - f_j)/2 (exact).
// Also writes yd[b,j] = (y_j, y_{j+1}-y_j) for the streaming kernel.
// grid.x = N+1 (row j), 256 threads = 64 members x 4 coefficient phases.
__global__ void __launch_bounds__(256) k_xt(KxDev d, KxTiled t, const double* __restrict__ f, double2* __restrict__ yd,
                                            double* __restrict__ XT, int xstride, const double* __restrict__ fmx,
                                            int* __restrict__ mflag, int B)
{
    __shared__ double s_dct[KX_QMAX * KX_QMAX];
    __shared__ double s_node[KX_QMAX];
    __shared__ double s_G[KX_QMAX][64];
    const int N = d.N, Q = t.Q, j = blockIdx.x;
    const int bl = threadIdx.x & 63, ph = threadIdx.x >> 6;
    const bool logm = d.interp == KX_INTERP_LOG;
    if (logm) {
        for (int k = threadIdx.x; k < Q * Q; k += 256) s_dct[k] = t.dct[k];
        if (threadIdx.x < Q) s_node[threadIdx.x] = t.nodes[threadIdx.x];
    }
    __syncthreads();
    for (int b0 = 0; b0 < B; b0 += 64) {
        const int b = b0 + bl;
        const bool act = b < B;
        if (j == N) {
            if (act && ph == 0) XT[(size_t)t.ones_row * xstride + b] = 1.0;
            continue;
        }
        double fj = 0.0, fj1 = 0.0;
        if (act) {
            fj = f[(size_t)b * N + j];
            fj1 = j + 1 < N ? f[(size_t)b * N + j + 1] : fj;
        }
        if (act && ph == 0) XT[(size_t)j * xstride + b] = fj;
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
        const double y0 = log2(fmax(fj, d.f_floor));
        const double y1 = log2(fmax(fj1, d.f_floor));
        const double dy = y1 - y0;
        if (act && ph == 0) {
            yd[(size_t)b * N + j] = make_double2(y0, dy);
            const double c = 0.6931471805599453 * fabs(dy);
            if (j < N - 1 && c > 0.0) {
                // log2 of the bound relative to max f, against log2(1e-15)
                const double lb = fmax(y0, y1) - log2(fmx[b]) + (double)Q * (log2(c) - 2.0) + t.flag_log2;
                if (lb > -49.82892142331043) mflag[b] = 1;
            }
        }
        if (j >= N - 1) continue;       // uniform over the CTA
        for (int q = ph; q < Q; q += 4) s_G[q][bl] = exp2(fma(s_node[q], dy, y0));
        __syncthreads();
        if (act) {
            for (int c = ph; c < Q; c += 4) {
                double a = 0.0;
                for (int q = 0; q < Q; ++q) a = fma(s_dct[c * Q + q], s_G[q][bl], a);
                XT[(size_t)(t.loss_row0 + j * Q + c) * xstride + b] = a;
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

// D[8 members x 8 rows] += X[8 members x 4 k] * A[4 k x 8 rows]
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

constexpr int kStageBytes = KX_GROUP_DBL * 8 + 16;     // 2 KiB of A + 4 descriptors

template <int NBT, int WARPS, int STAGES>
__global__ void __launch_bounds__(WARPS * 32, 1)
k_dmma(KxTiled t, const double* __restrict__ XT, int xstride, double* __restrict__ part)
{
    extern __shared__ __align__(16) unsigned char smem[];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    unsigned char* ring = smem + (size_t)warp * STAGES * kStageBytes;
    double* slab = reinterpret_cast<double*>(smem + (size_t)WARPS * STAGES * kStageBytes);   // [WARPS][NBT*8][16]

    const unsigned Gtot = t.vtptr[2 * t.NT];
    const unsigned nC = gridDim.x, c = blockIdx.x;
    const unsigned g0 = (unsigned)((unsigned long long)c * Gtot / nC);
    const unsigned g1 = (unsigned)((unsigned long long)(c + 1) * Gtot / nC);
    const int bcol0 = blockIdx.y * (NBT * 8);
    const double* __restrict__ xcol = XT + bcol0 + (lane >> 2);   // + row * xstride + 8 bt
    const int krow = lane & 3;

    int vt = 0;
    unsigned g = g0;
    while (g < g1) {
        while (t.vtptr[vt + 1] <= g) ++vt;
        const unsigned pe = min(g1, t.vtptr[vt + 1]);
        const unsigned len = pe - g, per = (len + WARPS - 1) / WARPS;
        const unsigned wg0 = min(g + warp * per, pe), wg1 = min(wg0 + per, pe);
        const unsigned n = wg1 - wg0;

        double acc[NBT][2][2];
#pragma unroll
        for (int bt = 0; bt < NBT; ++bt) { acc[bt][0][0] = acc[bt][0][1] = acc[bt][1][0] = acc[bt][1][1] = 0.0; }

        if (n > 0) {
            auto issue = [&](unsigned grp) {
                const double* src = t.A + (size_t)grp * KX_GROUP_DBL;
                unsigned char* dst = ring + (size_t)((grp - wg0) % STAGES) * kStageBytes;
#pragma unroll
                for (int k = 0; k < 4; ++k) cp_async16(dst + (k * 32 + lane) * 16, src + (k * 32 + lane) * 2);
                if (lane == 0) cp_async16(dst + KX_GROUP_DBL * 8, t.desc + (size_t)grp * 4);
            };
#pragma unroll
            for (int s = 0; s < STAGES - 1; ++s) {
                if ((unsigned)s < n) issue(wg0 + s);
                cp_async_commit();
            }
            // groups 0 and 1 must have landed before the first quad (X of quad q+1 is fetched during quad q)
            cp_async_wait<STAGES - 3>();
            __syncwarp();

            double xn[NBT], sn[NBT];
            unsigned srow_cur;
            {
                const unsigned dsc = *reinterpret_cast<const unsigned*>(ring + KX_GROUP_DBL * 8);
                const unsigned xrow = dsc & 0xFFFFFu;
                srow_cur = dsc >> 20;
                const double* xr = xcol + (size_t)(xrow + krow) * xstride;
                const double* sr = xcol + (size_t)srow_cur * xstride;
#pragma unroll
                for (int bt = 0; bt < NBT; ++bt) { xn[bt] = xr[8 * bt]; sn[bt] = sr[8 * bt]; }
            }
            double sc[NBT];
#pragma unroll
            for (int bt = 0; bt < NBT; ++bt) sc[bt] = sn[bt];

            for (unsigned gi = 0; gi < n; ++gi) {
                // refill the slot freed by group gi-1, then make sure groups gi and gi+1 are in shared memory
                if (gi + STAGES - 1 < n) issue(wg0 + gi + STAGES - 1);
                cp_async_commit();
                cp_async_wait<STAGES - 2>();
                __syncwarp();
                const unsigned char* st = ring + (size_t)(gi % STAGES) * kStageBytes;
                const double* wd = reinterpret_cast<const double*>(st);
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    double xv[NBT];
#pragma unroll
                    for (int bt = 0; bt < NBT; ++bt) xv[bt] = xn[bt] * sc[bt];
                    // prefetch X (and the scale row when it changes) of the next quad
                    const bool more = (q < 3) || (gi + 1 < n);
                    if (more) {
                        const unsigned char* stn = (q < 3) ? st : ring + (size_t)((gi + 1) % STAGES) * kStageBytes;
                        const unsigned dsc = *reinterpret_cast<const unsigned*>(stn + KX_GROUP_DBL * 8 + 4 * ((q + 1) & 3));
                        const unsigned xrow = dsc & 0xFFFFFu, srow = dsc >> 20;
                        const double* xr = xcol + (size_t)(xrow + krow) * xstride;
#pragma unroll
                        for (int bt = 0; bt < NBT; ++bt) xn[bt] = xr[8 * bt];
                        if (srow != srow_cur) {
                            srow_cur = srow;
                            const double* sr = xcol + (size_t)srow * xstride;
#pragma unroll
                            for (int bt = 0; bt < NBT; ++bt) sn[bt] = sr[8 * bt];
                        }
                    }
                    const double w0 = wd[q * 64 + lane], w1 = wd[q * 64 + 32 + lane];
#pragma unroll
                    for (int bt = 0; bt < NBT; ++bt) {
                        dmma884(acc[bt][0][0], acc[bt][0][1], xv[bt], w0);
                        dmma884(acc[bt][1][0], acc[bt][1][1], xv[bt], w1);
                    }
#pragma unroll
                    for (int bt = 0; bt < NBT; ++bt) sc[bt] = sn[bt];
                }
                __syncwarp();     // every lane is done with this stage before it is refilled
            }
            cp_async_wait<0>();
        }

        // fixed-order reduction over the CTA's warps: lane holds out[b = 8 bt + lane/4][i = 8 rb + 2 (lane%4) + {0,1}]
#pragma unroll
        for (int bt = 0; bt < NBT; ++bt)
#pragma unroll
            for (int rb = 0; rb < 2; ++rb)
                *reinterpret_cast<double2*>(&slab[((size_t)warp * NBT * 8 + bt * 8 + (lane >> 2)) * 16 + rb * 8 + 2 * (lane & 3)]) =
                    make_double2(acc[bt][rb][0], acc[bt][rb][1]);
        __syncthreads();
        double* dst = part + ((size_t)(c + vt) * xstride + bcol0) * 16;
        for (int e = tid; e < NBT * 128; e += WARPS * 32) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < WARPS; ++w) s += slab[(size_t)w * NBT * 128 + e];
            dst[e] = s;
        }
        __syncthreads();
        g = pe;
    }
}

template <int NBT, int WARPS, int STAGES>
cudaError_t launch_dmma_t(const KxTiled& t, int G, const double* XT, int xstride, double* tpart, int B, cudaStream_t s)
{
    const size_t smem = (size_t)WARPS * STAGES * kStageBytes + (size_t)WARPS * NBT * 128 * 8;
    cudaError_t e = cudaFuncSetAttribute(k_dmma<NBT, WARPS, STAGES>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    dim3 grid(G, (B + NBT * 8 - 1) / (NBT * 8));
    k_dmma<NBT, WARPS, STAGES><<<grid, WARPS * 32, smem, s>>>(t, XT, xstride, tpart);
    return cudaGetLastError();
}

}  // namespace

// columns of XT / tpart for a batch of B members: whole 8-member MMA tiles, whole CTA column groups
int kx_xstride(int B)
{
    if (B <= 8) return 8;
    if (B <= 16) return 16;
    if (B <= 32) return 32;
    return ((B + 63) / 64) * 64;
}

int kx_dmma_ctas(int sm_count, long long groups)
{
    long long g = groups / 8;
    if (g < 1) g = 1;
    return (int)(g < sm_count ? g : sm_count);
}

cudaError_t kx_launch_xt(const KxDev& d, const KxTiled& t, const double* f, double* yd, double* XT, int xstride,
                         double* fmax, int* mflag, int B, cudaStream_t s)
{
    k_fmax<<<B, 256, 0, s>>>(d.N, f, fmax, mflag);
    k_xt<<<d.N + 1, 256, 0, s>>>(d, t, f, reinterpret_cast<double2*>(yd), XT, xstride, fmax, mflag, B);
    return cudaGetLastError();
}

cudaError_t kx_launch_dmma(const KxDev& d, const KxTiled& t, int G, const double* XT, int xstride,
                           double* tpart, int B, cudaStream_t s)
{
    (void)d;
    if (B <= 8) return launch_dmma_t<1, 8, 8>(t, G, XT, xstride, tpart, B, s);
    if (B <= 16) return launch_dmma_t<2, 8, 8>(t, G, XT, xstride, tpart, B, s);
    if (B <= 32) return launch_dmma_t<4, 8, 4>(t, G, XT, xstride, tpart, B, s);
    return launch_dmma_t<8, 8, 4>(t, G, XT, xstride, tpart, B, s);
}
