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
#include <float.h>

namespace {

constexpr double kPi = 3.14159265358979323846;

// ---------------------------------------------------------------- a1
__device__ __forceinline__ void kin_point(double p, double m, double& E, double& K)
{
    E = sqrt(p * p + m * m);
    K = (p * p) / (E + m);
}

__global__ void k_kinematics(KxDev d, double m)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= d.N) return;
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

// ---------------------------------------------------------------- a2: validity (reading D4)
// tau = 32 eps (K_n+K_m+K_i); a triple is kept iff K_0 - tau <= K~ <= K_{N-1} + tau, and K~ is then
// clamped into [K_0, K_{N-1}].
__device__ __forceinline__ bool keep_lo(double Kn, double Km, double Ki, double K0)
{
    double S = Kn + Km, Kt = S - Ki, tau = (32.0 * DBL_EPSILON) * (S + Ki);
    return Kt >= K0 - tau;
}
__device__ __forceinline__ bool keep_hi(double Kn, double Km, double Ki, double KN1)
{
    double S = Kn + Km, Kt = S - Ki, tau = (32.0 * DBL_EPSILON) * (S + Ki);
    return Kt <= KN1 + tau;
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

// exclusive scan of run_len[N*N] by ONE CTA of 1024 threads (N*N <= 2^20), then rowptr
__global__ void __launch_bounds__(1024) k_scan_runs(KxDev d)
{
    __shared__ unsigned s_warp[32];
    const int total = d.N * d.N;
    const int per = (total + 1023) / 1024;
    const int t = threadIdx.x;
    const int b0 = t * per, b1 = min(b0 + per, total);
    unsigned sum = 0;
    for (int k = b0; k < b1; ++k) sum += (unsigned)d.run_len[k];
    // block exclusive scan of `sum`
    unsigned v = sum;
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
    unsigned excl = v - sum + ((t >> 5) ? s_warp[(t >> 5) - 1] : 0u);
    unsigned run = excl;
    for (int k = b0; k < b1; ++k) {
        d.run_off[k] = run;
        run += (unsigned)d.run_len[k];
    }
    if (t == 1023) d.run_off[total] = s_warp[31];
    __syncthreads();   // global writes of this CTA are visible to the CTA after the barrier
    for (int i = t; i <= d.N; i += 1024) d.rowptr[i] = d.run_off[i * d.N];
}

// ---------------------------------------------------------------- a3: J = int_{Q-}^{Q+} |M|^2 dQ
// contact: M2_0 (Q+ - Q-)                                                eq. B.17
// mediator (reading D5): M2_0 m_med^4 int dQ/(Q^2+c2)^2, c2 = m_med^2 - (K_i-K_n)^2.  The difference of
// the antiderivative Q/(2c2(Q^2+c2)) + atan(Q/c)/(2c^3) between a=Q- and b=Q+ is combined analytically
// (no subtraction of two large terms); a series in c2 covers |c2| << a^2.
__device__ double kx_J(double a, double b, double dK, double M2_0, double m_med)
{
    if (!(b > a)) return 0.0;
    double d = b - a;
    if (m_med <= 0.0) return M2_0 * d;
    double mm = m_med * m_med;
    double c2 = mm - dK * dK;
    double ab = a * b;
    double val;
    if (fabs(c2) <= 0.05 * (a * a)) {
        // 1/(Q^2+c2)^2 = sum_k (k+1) (-c2)^k Q^(-2k-4);  |c2|/a^2 <= 0.05: 14 terms reach 1e-17
        double u = 1.0 / (a * a), v = 1.0 / (b * b);
        double ta = u / a, tb = v / b, pw = 1.0;
        val = 0.0;
#pragma unroll 1
        for (int k = 0; k < 14; ++k) {
            val += pw * (double)(k + 1) * (ta - tb) / (double)(2 * k + 3);
            pw *= -c2; ta *= u; tb *= v;
        }
    } else if (c2 > 0.0) {
        double c = sqrt(c2);
        val = d * (c2 - ab) / (2.0 * c2 * (a * a + c2) * (b * b + c2))
            + atan2(c * d, c2 + ab) / (2.0 * c2 * c);
    } else {
        double k2 = -c2, k = sqrt(k2);
        val = d * (ab + k2) / (2.0 * k2 * ((a - k) * (a + k)) * ((b - k) * (b + k)))
            + log1p(-2.0 * k * d / ((b - k) * (a + k))) / (4.0 * k2 * k);
    }
    return M2_0 * (mm * mm) * val;
}

// one warp per run (i,n); lanes over m.  Writes W (symmetrised), omega_R and n|m<<10|jL<<20.
__global__ void __launch_bounds__(256) k_fill(KxDev d)
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
            const double Km = K[m], pm = P[m];
            double Kt = (Kn + Km) - Ki;
            Kt = fmin(fmax(Kt, K0), KN1);                 // D4: the kept triple's K~ snapped into the domain
            const double pj = sqrt(Kt * (Kt + 2.0 * d.m)); // eq. 4.4
            // eq. B.15-B.16
            double J = kx_J(fmax(fabs(pi_ - pn), fabs(pm - pj)), fmin(pi_ + pn, pm + pj), Ki - Kn, d.M2_0, d.m_med);
            if (m != n)   // the (i,m,n) ordering: second half of the symmetrised entry
                J += kx_J(fmax(fabs(pi_ - pm), fabs(pn - pj)), fmin(pi_ + pm, pn + pj), Ki - Km, d.M2_0, d.m_med);
            const double W = pref_in * d.ccol[m] * J;
            // bracket: largest j in [0, N-2] with K_j <= K~
            int lo = 0, hi = N - 2;
            while (lo < hi) {
                int mid = (lo + hi + 1) >> 1;
                if (K[mid] <= Kt) lo = mid; else hi = mid - 1;
            }
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
    k_runs<<<grid, 128, 0, s>>>(d);
    k_scan_runs<<<1, 1024, 0, s>>>(d);
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
