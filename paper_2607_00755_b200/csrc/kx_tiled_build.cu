// kx_tiled_build.cu -- steps a2-a3 written in the layout the DMMA contraction kernel consumes (KX_STORE_TILED).
//
// The entries are the SAME W_inm, j_L, omega_R as in kx_build.cu (they come from the same device functions of
// kx_entry.cuh and from the same run table), regrouped in two ways:
//
//   gain operand  A[k=(n,m), i] = W_inm + W_imn for 16-row tiles, runs (tile, n) -> interval of m     eq. 4.6/4.7
//   loss operand  M_c(i,j) = sum over the bucket {(n<=m): j_L(i,n,m) = j} of Wsym T_c(2 omega_R - 1), c < Q, stored for
//                 LOG interpolation in the Lagrange basis of the Chebyshev nodes (see k_cheb_moments)
//
// Why Chebyshev moments: inside bracket j the interpolated occupation of eq. B.20 (eta = 0) is the smooth function
// g(omega) = f_j^(1-omega) f_(j+1)^omega, omega in [0,1] (eq. B.19).  Its degree-(Q-1) interpolant at the Q
// Chebyshev nodes of [0,1], p(omega) = sum_c a_c T_c(2 omega - 1), differs from g by at most
//     2 (|ln(f_(j+1)/f_j)| / 4)^Q / Q! * max(f_j, f_(j+1))
// so sum_e W_e g(omega_e) = sum_c a_c M_c(i,j) up to that bound: N^3 B exponentials become an N^2 Q B contraction.
// Brackets whose bound is not negligible are evaluated exactly by the streaming kernel (kx_contract.cu); the
// decision is taken per member from the statistics the loss role of k_dmma accumulates (kx_tiled.cu).  LINEAR
// interpolation is the exact case Q = 2.
//
// Compiled with --fmad=false; fused multiply-adds are explicit.
#include "kx_internal.cuh"
#include "kx_entry.cuh"

namespace {

using namespace kxe;

// ---------------------------------------------------------------- runs of the gain operand
// one thread per (tile, n): union over the tile's rows of the kept m intervals (n <= m)
__global__ void k_tile_runs(KxDev d, KxTiled t)
{
    const int n = blockIdx.x * blockDim.x + threadIdx.x;
    const int tile = blockIdx.y;
    const int N = d.N;
    if (n >= N) return;
    int lo = N, hi = -1;
    const int i1 = min(N, (tile + 1) * KX_TI);
    for (int i = tile * KX_TI; i < i1; ++i) {
        const int len = d.run_len[i * N + n];
        if (len <= 0) continue;
        const int a = d.run_mlo[i * N + n];
        lo = min(lo, a);
        hi = max(hi, a + len);
    }
    t.trun_mlo[tile * N + n] = hi > lo ? lo : 0;
    t.trun_q[tile * N + n] = hi > lo ? (unsigned)((hi - lo + 3) >> 2) : 0u;
}

// exclusive scan of trun_q inside each tile (one CTA of 1024 threads per tile, N <= 1024)
__global__ void __launch_bounds__(1024) k_tile_scan(KxDev d, KxTiled t)
{
    __shared__ unsigned s_warp[32];
    const int tid = threadIdx.x, tile = blockIdx.x, N = d.N;
    const unsigned cnt = tid < N ? t.trun_q[tile * N + tid] : 0u;
    unsigned v = cnt;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned u = __shfl_up_sync(0xffffffffu, v, o);
        if ((tid & 31) >= o) v += u;
    }
    if ((tid & 31) == 31) s_warp[tid >> 5] = v;
    __syncthreads();
    if (tid < 32) {
        unsigned w = s_warp[tid];
        for (int o = 1; o < 32; o <<= 1) {
            unsigned u = __shfl_up_sync(0xffffffffu, w, o);
            if (tid >= o) w += u;
        }
        s_warp[tid] = w;
    }
    __syncthreads();
    const unsigned excl = v - cnt + ((tid >> 5) ? s_warp[(tid >> 5) - 1] : 0u);
    if (tid < N) t.trun_off[tile * (N + 1) + tid] = excl;
    if (tid == N - 1) t.trun_off[tile * (N + 1) + N] = excl + cnt;
}

// gain groups per tile -> vtptr
__global__ void k_vt_scan(KxDev d, KxTiled t)
{
    if (threadIdx.x || blockIdx.x) return;
    unsigned run = 0;
    for (int tile = 0; tile < t.NT; ++tile) {
        t.vtptr[tile] = run;
        run += (t.trun_off[tile * (d.N + 1) + d.N] + 3u) >> 2;
    }
    t.vtptr[t.NT] = run;
}

// ---------------------------------------------------------------- gain operand
// one warp per (quad, row block) of a tile: lane -> (row i = 16 tile + 8 rb + lane/4, m = m0 + lane%4)
__global__ void __launch_bounds__(256) k_pack_gain(KxDev d, KxTiled t)
{
    const int N = d.N, tile = blockIdx.y;
    const int lane = threadIdx.x & 31;
    const unsigned* __restrict__ off = t.trun_off + (size_t)tile * (N + 1);
    const unsigned tq = off[N];                       // quads of this tile
    const unsigned nq = ((tq + 3u) >> 2) << 2;        // padded to whole groups
    const size_t qbase = (size_t)t.vtptr[tile] * 4;
    const double* __restrict__ K = d.K;
    const double* __restrict__ P = d.p;
    const double K0 = K[0], KN1 = K[N - 1];
    const unsigned nwork = nq * 2;
    for (unsigned w = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); w < nwork; w += gridDim.x * (blockDim.x >> 5)) {
        const unsigned q = w >> 1;
        const int rb = (int)(w & 1u);
        double W = 0.0;
        unsigned desc = (unsigned)N << 20;            // padding quad: f_m columns 0..3 scaled by the ones column N, A = 0
        if (q < tq) {
            int lo = 0, hi = N - 1;                   // the run: off[n] <= q < off[n+1]
            while (lo < hi) {
                int mid = (lo + hi + 1) >> 1;
                if (off[mid] <= q) lo = mid; else hi = mid - 1;
            }
            const int n = lo;
            const int m0 = t.trun_mlo[tile * N + n] + 4 * (int)(q - off[n]);
            desc = (unsigned)m0 | ((unsigned)n << 20);
            const int i = tile * KX_TI + rb * 8 + (lane >> 2);
            const int m = m0 + (lane & 3);
            if (i < N && m < N) {
                const int len = d.run_len[i * N + n];
                const int a = d.run_mlo[i * N + n];
                if (len > 0 && m >= a && m < a + len) {
                    const double Ki = K[i], Kn = K[n], Km = K[m];
                    const double Kt = kx_Kt(Kn, Km, Ki, K0, KN1);
                    W = kx_Wsym(d, P, n, m, P[i], P[n], Ki, Kn, Km, Kt, d.arow[i] * d.ccol[n]);
                }
            }
        }
        t.A[(qbase + q) * 64 + rb * 32 + lane] = W;
        if (rb == 0 && lane == 0) t.desc[qbase + q] = desc;
    }
}

// ---------------------------------------------------------------- loss operand: Chebyshev moments of the buckets
// one thread per bucket (i, j).  For every n the kept m of row i with j_L = j form an interval of the run (i,n)
// (K~ is monotone in m); it is found with the SAME comparisons as kx_bracket: j_L >= j <=> K~ >= K_j.
template <int Q>
__global__ void __launch_bounds__(128) k_cheb_moments(KxDev d, KxTiled t)
{
    // LOG: the moments are stored in the Lagrange basis of the Chebyshev nodes, L_q(omega) = sum_c D[c][q] T_c(2 omega - 1)
    // with D = t.dct (the discrete Chebyshev transform, a_c = sum_q D[c][q] g(omega_q)):
    //     sum_c a_c M_c = sum_q g(omega_q) ML_q,   ML_q = sum_c D[c][q] M_c,
    // so that the operand X of the contraction is the interpolated occupation at the nodes itself and k_dmma needs no
    // transform.  LINEAR (Q = 2) keeps the two exact Chebyshev coefficients.
    __shared__ double s_D[Q > 2 ? Q * Q : 1];
    if (Q > 2) {
        for (int k = threadIdx.x; k < Q * Q; k += blockDim.x) s_D[k] = t.dct[k];
        __syncthreads();
    }
    const int N = d.N;
    const int i = blockIdx.x;
    const int rb8 = i >> 3, ir = i & 7;
    const double* __restrict__ K = d.K;
    const double* __restrict__ P = d.p;
    const double K0 = K[0], KN1 = K[N - 1], Ki = K[i], pi_ = P[i];
    for (int j = threadIdx.x; j < N - 1; j += blockDim.x) {
        const double Kj = K[j], Kj1 = K[j + 1];
        const double inv = Kj1 - Kj;
        const bool last = (j == N - 2);
        double M[Q];
#pragma unroll
        for (int c = 0; c < Q; ++c) M[c] = 0.0;
        for (int n = 0; n < N; ++n) {
            const int len = d.run_len[i * N + n];
            if (len <= 0) continue;
            const int a = d.run_mlo[i * N + n], b = a + len;
            const double Kn = K[n];
            if (kx_Kt(Kn, K[b - 1], Ki, K0, KN1) < Kj) continue;                // whole run below the bracket
            if (!last && !(kx_Kt(Kn, K[a], Ki, K0, KN1) < Kj1)) continue;        // whole run above it
            int lo = a, hi = b;                                                  // first m with K~ >= K_j
            while (lo < hi) {
                int mid = (lo + hi) >> 1;
                if (kx_Kt(Kn, K[mid], Ki, K0, KN1) >= Kj) hi = mid; else lo = mid + 1;
            }
            const int ma = lo;
            int mb = b;
            if (!last) {                                                         // first m with K~ >= K_{j+1}
                lo = ma; hi = b;
                while (lo < hi) {
                    int mid = (lo + hi) >> 1;
                    if (kx_Kt(Kn, K[mid], Ki, K0, KN1) >= Kj1) hi = mid; else lo = mid + 1;
                }
                mb = lo;
            }
            const double pn = P[n];
            const double pref_in = d.arow[i] * d.ccol[n];
            for (int m = ma; m < mb; ++m) {
                const double Km = K[m];
                const double Kt = kx_Kt(Kn, Km, Ki, K0, KN1);
                const double W = kx_Wsym(d, P, n, m, pi_, pn, Ki, Kn, Km, Kt, pref_in);
                const double om = (Kt - Kj) / inv;                               // eq. B.19
                const double x = 2.0 * om - 1.0, x2 = 2.0 * x;
                double T0 = 1.0, T1 = x;
                M[0] += W;
                if (Q > 1) M[1] = fma(W, x, M[1]);
#pragma unroll
                for (int c = 2; c < Q; ++c) {
                    const double T2 = fma(x2, T1, -T0);
                    M[c] = fma(W, T2, M[c]);
                    T0 = T1; T1 = T2;
                }
            }
        }
#pragma unroll 1
        for (int q = 0; q < Q; ++q) {
            double v;
            if (Q > 2) {
                v = 0.0;
#pragma unroll
                for (int c = 0; c < Q; ++c) v = fma(s_D[c * Q + q], M[c], v);
            } else {
                v = q == 0 ? M[0] : M[Q > 1 ? 1 : 0];
            }
            const int k = j * Q + q;
            t.AL[(((size_t)(k >> 4) * t.NR8 + rb8) * 4 + ((k >> 2) & 3)) * 32 + ir * 4 + (k & 3)] = v;
        }
    }
}

}  // namespace

cudaError_t kx_launch_tile_runs(const KxDev& d, const KxTiled& t, cudaStream_t s)
{
    dim3 grid((d.N + 127) / 128, t.NT);
    k_tile_runs<<<grid, 128, 0, s>>>(d, t);
    k_tile_scan<<<t.NT, 1024, 0, s>>>(d, t);
    k_vt_scan<<<1, 32, 0, s>>>(d, t);
    return cudaGetLastError();
}

cudaError_t kx_launch_tile_fill(const KxDev& d, const KxTiled& t, cudaStream_t s)
{
    int per_tile = (148 * 8 + t.NT - 1) / t.NT;
    dim3 gg(per_tile, t.NT);
    k_pack_gain<<<gg, 256, 0, s>>>(d, t);
    switch (t.Q) {
        case 2:  k_cheb_moments<2><<<d.N, 128, 0, s>>>(d, t); break;
        case 8:  k_cheb_moments<8><<<d.N, 128, 0, s>>>(d, t); break;
        case 16: k_cheb_moments<16><<<d.N, 128, 0, s>>>(d, t); break;
        case 24: k_cheb_moments<24><<<d.N, 128, 0, s>>>(d, t); break;
        case 32: k_cheb_moments<32><<<d.N, 128, 0, s>>>(d, t); break;
        default: return cudaErrorInvalidValue;
    }
    return cudaGetLastError();
}
