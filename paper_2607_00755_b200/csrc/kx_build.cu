// kx_build.cu -- steps a1-a3 on the device: kinematics, energy-conserving index map, kernel tensor.
//
//   a1  E_i = sqrt(p_i^2+m^2), K_i = p_i^2/(E_i+m) (= E_i-m without cancellation, reading D3),
//       h_i = p_i^2 dp_i                                                   eq. B.1
//   a2  K~ = (K_n+K_m)-K_i  (eq. 4.4: E_j~ = E_n+E_m-E_i); kept iff K_0 <= K~ <= K_{N-1}
//       after snapping ties at the domain edge (reading D4); bracket j_L and
//       omega_R = (K~-K_jL)/(K_{jL+1}-K_jL)                                  eq. B.19
//   a3  W_inm = dp_n dp_m/(2 E_i g_chi) * 1/(64 pi^3 p_i) * p_n p_m/(E_n E_m) * J_inm
//       J = |M|^2 [Q+ - Q-]_+ (contact, eq. B.15-B.17) or int_{Q-}^{Q+} |M|^2(Q) dQ (D5)
//
// Storage (KX_STORE_SYM_ROWS): gain and f_j~ are symmetric under n<->m, so only n<=m is kept with
// W_inm+W_imn; structural zeros (dropped triples) are not stored.  For fixed (i,n) the kept m form ONE
// interval because K~ is monotone in m, so a run table (i,n)->(m_lo,len) plus an exclusive scan gives
// every entry a deterministic slot: row i, then n ascending, then m ascending.
//
// Compiled with --fmad=false: validity decisions and omega must not depend on FMA contraction.
#include "kx_internal.cuh"
#include "kx_entry.cuh"

namespace {

using namespace kxe;

__global__ void k_kinematics(KxDev d, double m)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.N) return;
    if (d.m_dev) m = __ldg(d.m_dev);
    double p = d.p[i], dp = d.dp[i], E, K;
    kin_point(p, m, E, K);
    d.E[i] = E;
    d.K[i] = K;
    d.h[i] = (p * p) * dp;
    d.arow[i] = 1.0 / ((2.0 * E * d.g_chi) * (64.0 * (kPi * kPi * kPi) * p));
    d.ccol[i] = dp * p / E;
    if (i + 1 < d.N) {
        double E1, K1;
        kin_point(d.p[i + 1], m, E1, K1);
        d.invdK[i] = 1.0 / (K1 - K);
    } else {
        d.invdK[i] = 0.0;
    }
}

// bracket look-up table (kx_entry.cuh): one CTA; thread per key
__global__ void __launch_bounds__(1024) k_bracket_lut(KxDev d)
{
    const int N = d.N;
    const double* __restrict__ K = d.K;
    const unsigned key0 = kx_key17(K[0]), key1 = kx_key17(K[N - 1]);
    const unsigned size = key1 - key0 + 1u;
    if (!(K[0] > 0.0) || size > KX_BLUT_MAX) {          // no table: k_fill falls back to the binary search
        if (threadIdx.x == 0) { d.blut[0] = 0u; d.blut[1] = 0u; }
        return;
    }
    if (threadIdx.x == 0) { d.blut[0] = key0; d.blut[1] = size; }
    for (unsigned k = threadIdx.x; k < size; k += blockDim.x) {
        // number of j with key(K_j) < key0 + k, minus one (clamped to 0): binary search on the monotone keys
        int lo = 0, hi = N;
        while (lo < hi) {
            const int mid = (lo + hi) >> 1;
            if (kx_key17(K[mid]) < key0 + k) lo = mid + 1; else hi = mid;
        }
        const int j = lo - 1;
        d.blut[2 + k] = (unsigned)(j < 0 ? 0 : (j > N - 2 ? N - 2 : j));
    }
}

// one thread per (i,n): the interval of kept m in [n, N)
__global__ void k_runs(KxDev d)
{
    int n = blockIdx.x * blockDim.x + threadIdx.x;
    int i = blockIdx.y;
    int N = d.N;
    if (n >= N) return;
    const double* __restrict__ K = d.K;
    double Ki = K[i], Kn = K[n], K0 = K[0], KN1 = K[N - 1];
    // first m >= n passing the lower test (monotone in m)
    int lo = n, hi = N;
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (keep_lo(Kn, K[mid], Ki, K0)) hi = mid; else lo = mid + 1;
    }
    int mlo = lo;
    // first m >= n failing the upper test
    lo = n; hi = N;
    while (lo < hi) {
        int mid = (lo + hi) >> 1;
        if (keep_hi(Kn, K[mid], Ki, KN1)) lo = mid + 1; else hi = mid;
    }
    int mend = lo;
    int len = mend - mlo;
    d.run_mlo[i * N + n] = mlo;
    d.run_len[i * N + n] = len > 0 ? len : 0;
}

// exclusive scan of run_len[N*N] in two coalesced passes, one CTA of 1024 threads per row i (N <= 1024):
//   k_scan_rows: run_off[i,n] = sum_{n'<n} run_len[i,n'], row total -> taskptr[i] (scratch: k_tasks rebuilds taskptr later)
//   k_scan_base: base_i = sum_{i'<i} total_i'; run_off[i,n] += base_i; rowptr[i] = base_i; run_off[N*N] = rowptr[N] = nnz
__device__ __forceinline__ unsigned block_scan_1024(unsigned v, unsigned* s_warp, unsigned* total)
{
    const int t = threadIdx.x;
    const unsigned own = v;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned u = __shfl_up_sync(0xffffffffu, v, o);
        if ((t & 31) >= o) v += u;
    }
    if ((t & 31) == 31) s_warp[t >> 5] = v;
    __syncthreads();
    if (t < 32) {
        unsigned w = s_warp[t];
        for (int o = 1; o < 32; o <<= 1) {
            unsigned u = __shfl_up_sync(0xffffffffu, w, o);
            if (t >= o) w += u;
        }
        s_warp[t] = w;
    }
    __syncthreads();
    *total = s_warp[31];
    return v - own + ((t >> 5) ? s_warp[(t >> 5) - 1] : 0u);     // exclusive
}

__global__ void __launch_bounds__(1024) k_scan_rows(KxDev d)
{
    __shared__ unsigned s_warp[32];
    const int i = blockIdx.x, t = threadIdx.x, N = d.N;
    const unsigned len = t < N ? (unsigned)d.run_len[i * N + t] : 0u;
    unsigned total;
    const unsigned excl = block_scan_1024(len, s_warp, &total);
    if (t < N) d.run_off[i * N + t] = excl;
    if (t == 0) d.taskptr[i] = total;
}

__global__ void __launch_bounds__(1024) k_scan_base(KxDev d)
{
    __shared__ unsigned s_warp[32];
    const int i = blockIdx.x, t = threadIdx.x, N = d.N;
    const unsigned tot = t < N ? d.taskptr[t] : 0u;
    unsigned all;
    const unsigned excl = block_scan_1024(tot, s_warp, &all);      // thread t holds base_t
    __shared__ unsigned s_base;
    if (t == i) s_base = excl;
    __syncthreads();
    const unsigned base = s_base;
    if (t < N) d.run_off[i * N + t] += base;
    if (t == 0) d.rowptr[i] = base;
    if (i == N - 1 && t == 0) { d.rowptr[N] = all; d.run_off[N * N] = all; }
}

// one warp per run (i,n); lanes over m.  Writes W (symmetrised), omega_R and n|m<<10|jL<<20.
__global__ void __launch_bounds__(256, 4) k_fill(KxDev d)
{
    const int N = d.N;
    const int lane = threadIdx.x & 31;
    const int warps_per_cta = blockDim.x >> 5;
    const int nruns = N * N;
    const double* __restrict__ K = d.K;
    const double* __restrict__ P = d.p;
    const double K0 = K[0], KN1 = K[N - 1];
    for (int r = blockIdx.x * warps_per_cta + (threadIdx.x >> 5); r < nruns; r += gridDim.x * warps_per_cta) {
        const int len = d.run_len[r];
        if (len <= 0) continue;
        const int i = r / N, n = r - i * N;
        const int mlo = d.run_mlo[r];
        const unsigned off = d.run_off[r];
        const double Ki = K[i], Kn = K[n], pi_ = P[i], pn = P[n];
        const double pref_in = d.arow[i] * d.ccol[n];
        for (int k = lane; k < len; k += 32) {
            const int m = mlo + k;
            const double Km = K[m];
            const double Kt = kx_Kt(Kn, Km, Ki, K0, KN1);       // D4: the kept triple's K~ snapped into the domain
            const double W = kx_Wsym(d, P, n, m, pi_, pn, Ki, Kn, Km, Kt, pref_in);
            const int lo = kx_bracket_lut(K, N, Kt, d.blut);
            const double om = (Kt - K[lo]) / (K[lo + 1] - K[lo]);   // eq. B.19
            const size_t e = (size_t)off + k;
            d.W[e] = W;
            d.omega[e] = om;
            d.nmj[e] = (unsigned)n | ((unsigned)m << 10) | ((unsigned)lo << 20);
        }
    }
}

// taskptr[i] = exclusive scan of ceil(len_i / chunk); one CTA, N <= 1024 threads used
__global__ void __launch_bounds__(1024) k_tasks(KxDev d, int chunk)
{
    __shared__ unsigned s_warp[32];
    const int t = threadIdx.x;
    unsigned cnt = 0;
    if (t < d.N) {
        unsigned len = d.rowptr[t + 1] - d.rowptr[t];
        cnt = (len + (unsigned)chunk - 1u) / (unsigned)chunk;
    }
    unsigned v = cnt;
    for (int o = 1; o < 32; o <<= 1) {
        unsigned u = __shfl_up_sync(0xffffffffu, v, o);
        if ((t & 31) >= o) v += u;
    }
    if ((t & 31) == 31) s_warp[t >> 5] = v;
    __syncthreads();
    if (t < 32) {
        unsigned w = s_warp[t];
        for (int o = 1; o < 32; o <<= 1) {
            unsigned u = __shfl_up_sync(0xffffffffu, w, o);
            if (t >= o) w += u;
        }
        s_warp[t] = w;
    }
    __syncthreads();
    unsigned excl = v - cnt + ((t >> 5) ? s_warp[(t >> 5) - 1] : 0u);
    if (t < d.N) d.taskptr[t] = excl;
    if (t == d.N - 1) d.taskptr[d.N] = excl + cnt;
}

}  // namespace

cudaError_t kx_launch_kinematics(const KxDev& d, double m, cudaStream_t s)
{
    k_kinematics<<<(d.N + 255) / 256, 256, 0, s>>>(d, m);
    return cudaGetLastError();
}

cudaError_t kx_launch_runs(const KxDev& d, cudaStream_t s)
{
    dim3 grid((d.N + 127) / 128, d.N);
    k_bracket_lut<<<1, 1024, 0, s>>>(d);
    k_runs<<<grid, 128, 0, s>>>(d);
    k_scan_rows<<<d.N, 1024, 0, s>>>(d);
    k_scan_base<<<d.N, 1024, 0, s>>>(d);
    return cudaGetLastError();
}

cudaError_t kx_launch_fill(const KxDev& d, cudaStream_t s)
{
    int ctas = (d.N * d.N + 7) / 8;
    if (ctas > 148 * 16) ctas = 148 * 16;
    k_fill<<<ctas, 256, 0, s>>>(d);
    return cudaGetLastError();
}

cudaError_t kx_launch_tasks(const KxDev& d, int chunk, cudaStream_t s)
{
    k_tasks<<<1, 1024, 0, s>>>(d, chunk);
    return cudaGetLastError();
}
