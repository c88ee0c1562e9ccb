// kx_entry.cuh -- device functions that evaluate ONE entry of the kernel tensor (steps a2-a3), shared by
// every builder kernel of libkx so that all storage layouts take bit-identical decisions and values.
// NOT shared with oracle/.  Compiled with --fmad=false.
#pragma once
#include "kx_internal.cuh"
#include <float.h>

namespace kxe {

constexpr double kPi = 3.14159265358979323846;

// kinematic mass of this build: a host value, or read from the device (adaptive integration with m(u))
__device__ __forceinline__ double kx_mass(const KxDev& d) { return d.m_dev ? __ldg(d.m_dev) : d.m; }

// ---------------------------------------------------------------- a1
__device__ __forceinline__ void kin_point(double p, double m, double& E, double& K)
{
    E = sqrt(p * p + m * m);
    K = (p * p) / (E + m);
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

// ---------------------------------------------------------------- a3: J = int_{Q-}^{Q+} |M|^2 dQ
// contact: M2_0 (Q+ - Q-)                                                eq. B.17
// mediator (reading D5): M2_0 m_med^4 int dQ/(Q^2+c2)^2, c2 = m_med^2 - (K_i-K_n)^2.  The difference of
// the antiderivative Q/(2c2(Q^2+c2)) + atan(Q/c)/(2c^3) between a=Q- and b=Q+ is combined analytically
// (no subtraction of two large terms); a series in c2 covers |c2| << a^2.
static __device__ double kx_J(double a, double b, double dK, double M2_0, double m_med)
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


// Numerical reduced kernel F(p_i, p_n, p_m) of eq. B.4-B.12: Gauss-Legendre quadrature over
// mu = cos(p_i, p_n); for every node the nu-integral is analytic (B.11) between the roots of the quadratic B.8-B.10
// clipped to [-1,1]; |M|^2 is evaluated at t(mu) = 2 m^2 - 2 E_i E_n + 2 p_i p_n mu (reading D5).
static __device__ double kx_F_quad(const KxDev& d, double pi_, double pn, double pm)
{
    const double m = kx_mass(d);
    const double Ei = sqrt(pi_ * pi_ + m * m), En = sqrt(pn * pn + m * m), Em = sqrt(pm * pm + m * m);
    double acc = 0.0;
    for (int q = 0; q < d.n_mu; ++q) {
        const double u = d.gl_mu[q];
        const double A0 = m * m + En * Em - En * Ei - Em * Ei + pi_ * pn * u;      // B.5
        const double A1 = pi_ * pm - pn * pm * u;                                    // B.6
        const double K2 = pn * pn * pm * pm * (1.0 - u * u);                         // B.7
        const double a = -(K2 + A1 * A1), b = -2.0 * A0 * A1, c = K2 - A0 * A0;      // B.8
        const double disc = b * b - 4.0 * a * c;
        if (!(disc > 0.0) || !(a < 0.0)) continue;
        const double sq = sqrt(disc);
        const double r1 = (-b + sq) / (2.0 * a), r2 = (-b - sq) / (2.0 * a);         // B.10
        const double lo = fmin(r1, r2), hi = fmax(r1, r2);
        if (hi <= -1.0 || lo >= 1.0) continue;
        const double vm = fmax(lo, -1.0), vp = fmin(hi, 1.0);
        const double am = fmax(-1.0, fmin(1.0, (2.0 * a * vm + b) / sq));
        const double ap = fmax(-1.0, fmin(1.0, (2.0 * a * vp + b) / sq));
        const double I = (asin(am) - asin(ap)) / sqrt(-a);                           // B.11
        double M2 = d.M2_0;
        if (d.m_med > 0.0) {
            const double t = 2.0 * m * m - 2.0 * Ei * En + 2.0 * pi_ * pn * u;
            const double dd = 1.0 + (-t) / (d.m_med * d.m_med);
            M2 = d.M2_0 / (dd * dd);
        }
        acc += d.gl_w[q] * I * M2;
    }
    const double twopi = 2.0 * kPi;
    const double pref = 1.0 / (4.0 * (twopi * twopi) * (twopi * twopi)) * (pn * pm) * (pn * pm) / (En * Em);   // B.12
    return pref * acc;
}

// K~ of a KEPT triple, snapped into the domain (reading D4)                       eq. 4.4
__device__ __forceinline__ double kx_Kt(double Kn, double Km, double Ki, double K0, double KN1)
{
    double Kt = (Kn + Km) - Ki;
    return fmin(fmax(Kt, K0), KN1);
}

// symmetrised kernel-tensor entry W_inm + W_imn (n < m) or W_inn for a kept triple     eq. 4.7 + B.15-B.17
__device__ __forceinline__ double kx_Wsym(const KxDev& d, const double* __restrict__ P, int n, int m,
                                          double pi_, double pn, double Ki, double Kn, double Km, double Kt,
                                          double pref_in)
{
    const double pm = P[m];
    if (d.n_mu > 0) {      // numerical angular kernel: W = dp_n dp_m F_inm / (2 E_i g_chi), both orderings       eq. 4.7
        const double mq = kx_mass(d);
        const double Ei = sqrt(pi_ * pi_ + mq * mq);
        double F = kx_F_quad(d, pi_, pn, pm);
        if (m != n) F += kx_F_quad(d, pi_, pm, pn);
        return d.dp[n] * d.dp[m] / (2.0 * Ei * d.g_chi) * F;
    }
    const double pj = sqrt(Kt * (Kt + 2.0 * kx_mass(d)));   // eq. 4.4
    // eq. B.15-B.16
    double J = kx_J(fmax(fabs(pi_ - pn), fabs(pm - pj)), fmin(pi_ + pn, pm + pj), Ki - Kn, d.M2_0, d.m_med);
    if (m != n)   // the (i,m,n) ordering: second half of the symmetrised entry
        J += kx_J(fmax(fabs(pi_ - pm), fabs(pn - pj)), fmin(pi_ + pm, pn + pj), Ki - Km, d.M2_0, d.m_med);
    return pref_in * d.ccol[m] * J;
}

// The same bracket through a look-up table: key(x) = the 18 leading bits of a positive double (exponent and 6 mantissa bits,
// monotone in x); lut[key - key0] = the largest j whose key is BELOW that key (so K_j <= any value with the key), a lower
// bound from which a short linear scan reaches the bracket: one table load and one or two comparisons instead of a binary
// search of log2 N dependent loads.  The result is the same j by construction.  size 0 = no table (K spans too many binades).
__device__ __forceinline__ unsigned kx_key17(double x) { return (unsigned)(__double_as_longlong(x) >> 46); }
__device__ __forceinline__ int kx_bracket(const double* __restrict__ K, int N, double Kt);
__device__ __forceinline__ int kx_bracket_lut(const double* __restrict__ K, int N, double Kt, const unsigned* __restrict__ lut)
{
    const unsigned key0 = __ldg(lut), size = __ldg(lut + 1);
    if (size == 0) return kx_bracket(K, N, Kt);
    const unsigned k = kx_key17(Kt);
    int j = k <= key0 ? 0 : (int)__ldg(lut + 2 + min(k - key0, size - 1u));
    while (j < N - 2 && K[j + 1] <= Kt) ++j;
    return j;
}

// bracket: largest j in [0, N-2] with K_j <= K~                                   eq. B.19
__device__ __forceinline__ int kx_bracket(const double* __restrict__ K, int N, double Kt)
{
    int lo = 0, hi = N - 2;
    while (lo < hi) {
        int mid = (lo + hi + 1) >> 1;
        if (K[mid] <= Kt) lo = mid; else hi = mid - 1;
    }
    return lo;
}

}  // namespace kxe
