/*
 * kx_oracle.c -- plain, slow, obviously-correct CPU oracle for the discretized 2->2 elastic
 * self-collision operator of KineticXGPU (arxiv/paper_2607_00755).
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may call it.  It shares no code, header,
 * table or constant with paper_2607_00755_b200/csrc (the CUDA path) and neither includes the other.
 *
 * The method is a discretization, so the oracle follows the paper's algorithm step by step in the
 * paper's notation; citations are PAPER.md line numbers.
 *   build   : literal quadruple loop (i, n, m, j)          -- eq. 4.4, 4.7, B.15-B.19
 *   evaluate: literal triple loop over dense W[i][n][m]     -- eq. 4.6 with 2.6, B.18, B.20
 *   project : App. C, eq. C.2-C.8 ; diagnostics C.1, C.9
 *   moments : eq. B.1-B.2
 *   evolve  : fixed-step Euler / Heun / RK4 on eq. 4.9
 * No symmetry reduction, no sparsity tricks, no blocking, no fusion.  Sums use long double
 * accumulators (x87 80-bit on x86-64).  Compile with -O2 -ffp-contract=off.
 *
 * Readings of the paper (D1-D13) are listed in DESIGN.md.  Pins: tests/test_oracle_pins.py
 * (P1-P10).  Functions with no pin outside themselves: none on the hot path; the paper's
 * Fig. 2 / Table 1 / Figs. 4-8, 12-13 comparisons are "parity unpinned" (need BEST and SM tables).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define OKX_PI 3.14159265358979323846264338327950288L

/* ---- O1: kinematics.  E_i = sqrt(p_i^2+m^2); K_i = E_i - m written as
 * p_i^2/(E_i+m) (reading D3: same number, no cancellation); h_i = p_i^2 dp_i (eq. B.1). */
void okx_kinematics(int N, const double *p, const double *dp, double m,
                    double *E, double *K, double *h)
{
    for (int i = 0; i < N; ++i) {
        E[i] = sqrt(p[i] * p[i] + m * m);
        K[i] = (p[i] * p[i]) / (E[i] + m);
        h[i] = (p[i] * p[i]) * dp[i];
    }
}

/* Antiderivative of 1/(Q^2+c2)^2 (reading D5), long double.  c2 may have either sign; Q^2+c2>0. */
static long double okx_anti(long double Q, long double c2)
{
    if (c2 > 0.0L) {
        long double c = sqrtl(c2);
        return Q / (2.0L * c2 * (Q * Q + c2)) + atanl(Q / c) / (2.0L * c2 * c);
    } else {
        long double k2 = -c2, k = sqrtl(k2);
        return -Q / (2.0L * k2 * (Q * Q - k2)) + logl((Q + k) / (Q - k)) / (4.0L * k2 * k);
    }
}

/* J = int_{Q-}^{Q+} |M|^2(Q) dQ.  Contact: |M|^2 = M2_0 (eq. B.17).
 * Mediator (reading D5): |M|^2 = M2_0/(1+(-t)/m_med^2)^2 with -t = Q^2-(E_i-E_n)^2, so
 * J = M2_0 m_med^4 int dQ/(Q^2+c2)^2, c2 = m_med^2-(E_i-E_n)^2 = m_med^2-(K_i-K_n)^2. */
static double okx_J(double Qm, double Qp, double M2_0, double m_med, double Ki, double Kn)
{
    if (!(Qp > Qm)) return 0.0;
    if (m_med <= 0.0) return M2_0 * (Qp - Qm);
    long double dK = (long double)Ki - (long double)Kn;
    long double mm = (long double)m_med * (long double)m_med;
    long double c2 = mm - dK * dK;
    long double a = Qm, b = Qp, val;
    if (fabsl(c2) < 1e-6L * a * b) {
        /* series in c2: 1/(Q^2+c2)^2 = sum_k (k+1)(-c2)^k Q^(-2k-4) */
        val = 0.0L;
        long double pw = 1.0L;
        for (int k = 0; k < 8; ++k) {
            long double e = (long double)(2 * k + 3);
            val += pw * (long double)(k + 1) * (powl(a, -e) - powl(b, -e)) / e;
            pw *= -c2;
        }
    } else {
        val = okx_anti(b, c2) - okx_anti(a, c2);
    }
    return (double)((long double)M2_0 * mm * mm * val);
}

/* ---- O2-O7 for ONE ordered triple (i,n,m): W_inm, bracket jL (-1 = dropped) and omega_R; the fourth loop is
 * the bracket scan over j.  Returns 1 if the triple is kept. */
static int okx_triple(int N, const double *p, const double *dp, const double *E, const double *K,
                      double m, double g_chi, double M2_0, double m_med, int i, int n, int mm,
                      double *W, int32_t *jL, double *wR)
{
    const double pi3 = (double)(OKX_PI * OKX_PI * OKX_PI);
    *W = 0.0; *jL = -1; *wR = 0.0;
    /* O2: energy conservation, eq. 4.4: E_j = E_n+E_m-E_i  <=>  K~ = K_n+K_m-K_i */
    double Kt = (K[n] + K[mm]) - K[i];
    /* D4: snap ties at the domain edge */
    double tau = 32.0 * 2.220446049250313e-16 * (K[n] + K[mm] + K[i]);
    if (Kt < K[0] && Kt >= K[0] - tau) Kt = K[0];
    if (Kt > K[N - 1] && Kt <= K[N - 1] + tau) Kt = K[N - 1];
    /* O3: keep iff E_j >= m and q_min <= q_j <= q_max <=> K_0 <= K~ <= K_{N-1} */
    if (!(Kt >= K[0] && Kt <= K[N - 1])) return 0;
    /* O4 */
    double pj = sqrt(Kt * (Kt + 2.0 * m));
    /* O5: eq. B.15-B.16 */
    double Qm = fmax(fabs(p[i] - p[n]), fabs(p[mm] - pj));
    double Qp = fmin(p[i] + p[n], p[mm] + pj);
    double J = okx_J(Qm, Qp, M2_0, m_med, K[i], K[n]);
    /* O6: eq. 4.7 with F of eq. B.17 */
    double w = dp[n] * dp[mm] / (2.0 * E[i] * g_chi);
    w = w * (1.0 / (64.0 * pi3 * p[i]));
    w = w * (p[n] * p[mm] / (E[n] * E[mm]));
    w = w * J;
    /* O7: bracket scan, largest j with K_j <= K~ <= K_{j+1}; eq. B.19 */
    int jb = -1;
    for (int j = 0; j <= N - 2; ++j)
        if (K[j] <= Kt && Kt <= K[j + 1]) jb = j;
    if (jb < 0) return 0; /* cannot happen after O3 */
    *W = w;
    *jL = jb;
    *wR = (Kt - K[jb]) / (K[jb + 1] - K[jb]);
    return 1;
}

/* ---- O2-O7: build W_inm, jL(i,n,m), omega_R(i,n,m) for every ORDERED triple (literal quadruple loop).
 * jL = -1 marks a dropped triple (W = 0).  Returns the number of kept triples. */
long okx_build(int N, const double *p, const double *dp, double m, double g_chi,
               double M2_0, double m_med, double *W, int32_t *jL, double *wR)
{
    double *E = malloc(sizeof(double) * N), *K = malloc(sizeof(double) * N), *h = malloc(sizeof(double) * N);
    okx_kinematics(N, p, dp, m, E, K, h);
    long kept = 0;
#pragma omp parallel for schedule(dynamic) reduction(+ : kept)
    for (int i = 0; i < N; ++i)
        for (int n = 0; n < N; ++n)
            for (int mm = 0; mm < N; ++mm) {
                size_t idx = ((size_t)i * N + n) * N + mm;
                kept += okx_triple(N, p, dp, E, K, m, g_chi, M2_0, m_med, i, n, mm, &W[idx], &jL[idx], &wR[idx]);
            }
    free(E); free(K); free(h);
    return kept;
}

/* ---- O8-O9: evaluate.  interp 0 = LOG (eq. B.20 at eta=0; reading D7),
 * 1 = LINEAR.  gain_i = sum_nm W f_n f_m ; loss_i = f_i sum_nm W f_j~ ; C_raw = gain - loss
 * (eq. 4.6 with the dilute factor of eq. 2.6). f is [B,N] row-major. */
void okx_collide(int N, int B, const double *f, const double *W, const int32_t *jL, const double *wR,
                 int interp, double f_floor, double *gain, double *loss, double *C)
{
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int b = 0; b < B; ++b)
        for (int i = 0; i < N; ++i) {
            const double *fb = f + (size_t)b * N;
            long double g = 0.0L, l = 0.0L;
            for (int n = 0; n < N; ++n)
                for (int mm = 0; mm < N; ++mm) {
                    size_t idx = ((size_t)i * N + n) * N + mm;
                    int j = jL[idx];
                    if (j < 0) continue;
                    double w = W[idx];
                    double oR = wR[idx], oL = 1.0 - oR;
                    double fj;
                    if (interp == 0) {
                        /* D8: y = ln(max(f, f_floor)) */
                        double yL = log(fmax(fb[j], f_floor)), yR = log(fmax(fb[j + 1], f_floor));
                        fj = exp(oL * yL + oR * yR);
                    } else {
                        fj = oL * fb[j] + oR * fb[j + 1];
                    }
                    g += (long double)w * (long double)fb[n] * (long double)fb[mm];
                    l += (long double)w * (long double)fj;
                }
            double gi = (double)g, li = (double)((long double)fb[i] * l);
            if (gain) gain[(size_t)b * N + i] = gi;
            if (loss) loss[(size_t)b * N + i] = li;
            if (C) C[(size_t)b * N + i] = (double)(g - (long double)fb[i] * l);
        }
}

/* ---- Quantum-statistics operator: the full Lambda_inm of eq. 4.3,
 *     Lambda = f_n f_m (1 + eta f_i)(1 + eta f_j~) - f_i f_j~ (1 + eta f_n)(1 + eta f_m),
 * eta = +1 (Bose-Einstein), -1 (Fermi-Dirac); one species, so eta_i = eta_n = eta_m = eta_j~ = eta.
 * Off-grid occupation by eq. B.20: y_k = ln(f_k / (1 + eta f_k)), y_j~ = w_L y_L + w_R y_R,
 * f_j~ = e^y / (1 - eta e^y); f_k is floored at f_floor inside the logarithm (reading D8).
 * gain_i = sum W f_n f_m (1+eta f_i)(1+eta f_j~), loss_i = f_i sum W f_j~ (1+eta f_n)(1+eta f_m), C = gain - loss. */
void okx_collide_q(int N, int B, const double *f, const double *W, const int32_t *jL, const double *wR,
                   int eta, double f_floor, double *gain, double *loss, double *C)
{
#pragma omp parallel for collapse(2) schedule(dynamic)
    for (int b = 0; b < B; ++b)
        for (int i = 0; i < N; ++i) {
            const double *fb = f + (size_t)b * N;
            const long double e = (long double)eta, fi = fb[i];
            long double g = 0.0L, l = 0.0L;
            for (int n = 0; n < N; ++n)
                for (int mm = 0; mm < N; ++mm) {
                    size_t idx = ((size_t)i * N + n) * N + mm;
                    int j = jL[idx];
                    if (j < 0) continue;
                    double oR = wR[idx], oL = 1.0 - oR;
                    double fL = fmax(fb[j], f_floor), fR = fmax(fb[j + 1], f_floor);
                    double yL = log(fL / (1.0 + eta * fL)), yR = log(fR / (1.0 + eta * fR));
                    double ey = exp(oL * yL + oR * yR);
                    long double fj = (long double)ey / (1.0L - e * (long double)ey);
                    long double fn = fb[n], fm = fb[mm], w = W[idx];
                    g += w * fn * fm * (1.0L + e * fi) * (1.0L + e * fj);
                    l += w * fi * fj * (1.0L + e * fn) * (1.0L + e * fm);
                }
            if (gain) gain[(size_t)b * N + i] = (double)g;
            if (loss) loss[(size_t)b * N + i] = (double)l;
            if (C) C[(size_t)b * N + i] = (double)(g - l);
        }
}

/* ---- O2-O9 for SELECTED rows i only, without storing the tables: the same per-triple code (okx_triple) and the
 * same accumulation as okx_collide, used to sample the operator at sizes where the dense N^3 tables are too
 * slow to build (N = 512).  rows[nrows]; outputs are [B, nrows]. */
void okx_collide_rows(int N, int B, const double *p, const double *dp, double m, double g_chi,
                      double M2_0, double m_med, const double *f, int nrows, const int32_t *rows,
                      int interp, double f_floor, double *gain, double *loss, double *C)
{
    double *E = malloc(sizeof(double) * N), *K = malloc(sizeof(double) * N), *h = malloc(sizeof(double) * N);
    okx_kinematics(N, p, dp, m, E, K, h);
#pragma omp parallel for schedule(dynamic)
    for (int r = 0; r < nrows; ++r) {
        int i = rows[r];
        long double *g = calloc(B, sizeof(long double)), *l = calloc(B, sizeof(long double));
        for (int n = 0; n < N; ++n)
            for (int mm = 0; mm < N; ++mm) {
                double w, oR; int32_t j;
                if (!okx_triple(N, p, dp, E, K, m, g_chi, M2_0, m_med, i, n, mm, &w, &j, &oR)) continue;
                double oL = 1.0 - oR;
                for (int b = 0; b < B; ++b) {
                    const double *fb = f + (size_t)b * N;
                    double fj;
                    if (interp == 0) {
                        double yL = log(fmax(fb[j], f_floor)), yR = log(fmax(fb[j + 1], f_floor));
                        fj = exp(oL * yL + oR * yR);
                    } else {
                        fj = oL * fb[j] + oR * fb[j + 1];
                    }
                    g[b] += (long double)w * (long double)fb[n] * (long double)fb[mm];
                    l[b] += (long double)w * (long double)fj;
                }
            }
        for (int b = 0; b < B; ++b) {
            long double fi = f[(size_t)b * N + i];
            if (gain) gain[(size_t)b * nrows + r] = (double)g[b];
            if (loss) loss[(size_t)b * nrows + r] = (double)(fi * l[b]);
            if (C) C[(size_t)b * nrows + r] = (double)(g[b] - fi * l[b]);
        }
        free(g); free(l);
    }
    free(E); free(K); free(h);
}

/* ---- O10: two-moment projection, App. C eq. C.2-C.8, support mask C.4 with
 * f_max = max_i |f_i|; degenerate cases per reading D9.  diag (may be NULL) receives
 * eps_N, eps_E (C.1, raw), R_N, R_E (C.9).  One distribution.
 *
 * Reading D3 applied to App. C: the correction xi_i (alpha + beta E_i) lives in span{1, E_i} =
 * span{1, K_i} (E_i = m + K_i), and the two conditions (C.5) "sum h C = 0, sum h E C = 0" are
 * equivalent to "sum h C = 0, sum h K C = 0".  The 2x2 system (C.7) is therefore solved in the
 * basis {1, K_i}: alpha' + beta K_i with alpha' = alpha + beta m.  Same projection, but the
 * determinant A00*A11 - A01^2 no longer cancels catastrophically when K << m (with the literal
 * E-basis even long double loses the result at m/T = 1e3: 1e-10 of max gain, measured against
 * exact rational arithmetic; pin tests/test_oracle_pins.py::test_P6_projection_exact_rational). */
void okx_project(int N, const double *f, const double *Craw, const double *h, const double *E,
                 const double *K, double eps_supp, double *Cproj, double *diag)
{
    long double R0 = 0, R1 = 0, RK = 0, S0 = 0, S1 = 0;
    double fmax = 0.0;
    for (int i = 0; i < N; ++i) {
        R0 += (long double)h[i] * Craw[i];                    /* C.2 */
        R1 += (long double)h[i] * E[i] * Craw[i];
        RK += (long double)h[i] * K[i] * Craw[i];             /* = R1 - m R0 */
        S0 += (long double)h[i] * fabs(Craw[i]);
        S1 += (long double)h[i] * E[i] * fabs(Craw[i]);
        if (fabs(f[i]) > fmax) fmax = fabs(f[i]);
    }
    long double A00 = 0, A0K = 0, AKK = 0;
    double *xi = malloc(sizeof(double) * N);
    for (int i = 0; i < N; ++i) {
        double r = (fmax > 0.0) ? fabs(f[i]) / fmax : 0.0;    /* C.4 */
        xi[i] = (r > eps_supp) ? r : 0.0;
        A00 += (long double)h[i] * xi[i];                     /* C.6 in the {1,K} basis */
        A0K += (long double)h[i] * K[i] * xi[i];
        AKK += (long double)h[i] * K[i] * K[i] * xi[i];
    }
    long double alpha = 0, beta = 0;                          /* correction = xi (alpha + beta K) */
    if (fmax > 0.0 && A00 > 0.0L) {
        long double det = A00 * AKK - A0K * A0K;              /* C.8 */
        if (det <= 1e-14L * A00 * AKK) { alpha = R0 / A00; beta = 0; }   /* D9: number only */
        else { alpha = (R0 * AKK - RK * A0K) / det; beta = (RK * A00 - R0 * A0K) / det; }
    }
    long double D0 = 0, D1 = 0;
    for (int i = 0; i < N; ++i) {
        double corr = (double)((long double)xi[i] * (alpha + beta * (long double)K[i]));
        Cproj[i] = Craw[i] - corr;                            /* C.3 */
        D0 += (long double)h[i] * fabs(corr);
        D1 += (long double)h[i] * E[i] * fabs(corr);
    }
    if (diag) {
        diag[0] = (S0 > 0) ? (double)(R0 / S0) : 0.0;         /* C.1 */
        diag[1] = (S1 > 0) ? (double)(R1 / S1) : 0.0;
        diag[2] = (S0 > 0) ? (double)(D0 / S0) : 0.0;         /* C.9 */
        diag[3] = (S1 > 0) ? (double)(D1 / S1) : 0.0;
    }
    free(xi);
}

/* ---- O11: moments, eq. B.2 with the factor g_chi/(2 pi^2);
 * <p^k> = sum h p^k f / sum h f.  out = n, rho, <p>, <p^2>. */
void okx_moments(int N, const double *f, const double *p, const double *h, const double *E,
                 double g_chi, double *out)
{
    long double s0 = 0, s1 = 0, sp = 0, sp2 = 0;
    for (int i = 0; i < N; ++i) {
        s0 += (long double)h[i] * f[i];
        s1 += (long double)h[i] * E[i] * f[i];
        sp += (long double)h[i] * p[i] * f[i];
        sp2 += (long double)h[i] * p[i] * p[i] * f[i];
    }
    long double fac = (long double)g_chi / (2.0L * OKX_PI * OKX_PI);
    out[0] = (double)(fac * s0);
    out[1] = (double)(fac * s1);
    out[2] = (s0 != 0) ? (double)(sp / s0) : 0.0;
    out[3] = (s0 != 0) ? (double)(sp2 / s0) : 0.0;
}

/* ---- O12: fixed-step integrators on  df/dtau = kappa_b R(tau) C[f; m(tau)] + sum_s amp_s(step) G_s
 * (eq. 4.9; regime description PAPER.md:225-227; reading D11/D12: source amplitude is
 * constant over a step, expansion enters through rate[] and mass[]).
 * method 0 Euler, 1 Heun, 2 RK4.  rate/mass are [2S+1] (nodes and midpoints) or NULL.  When mass is
 * given the tables are rebuilt (O1-O7) at every stage.  project != 0 applies O10.
 * diag: NULL or [S,B,6] = eps_N, eps_E, R_N, R_E (of the step's first stage), n, rho (after the step). */
typedef struct {
    int N; const double *p, *dp; double m, g_chi, M2_0, m_med; int interp; double f_floor, eps_supp;
    double *W; int32_t *jL; double *wR; double *E, *K, *h; double cur_m; int eta;
} okx_ctx;

static void okx_rhs(okx_ctx *c, const double *f, double mass, int use_mass, double kR, int project,
                    int nsrc, const double *G, const double *ampk, double *k, double *diag4)
{
    int N = c->N;
    if (use_mass && mass != c->cur_m) {
        okx_build(N, c->p, c->dp, mass, c->g_chi, c->M2_0, c->m_med, c->W, c->jL, c->wR);
        okx_kinematics(N, c->p, c->dp, mass, c->E, c->K, c->h);
        c->cur_m = mass;
    }
    double *Craw = malloc(sizeof(double) * N), *Cp = malloc(sizeof(double) * N);
    if (c->eta) okx_collide_q(N, 1, f, c->W, c->jL, c->wR, c->eta, c->f_floor, NULL, NULL, Craw);
    else okx_collide(N, 1, f, c->W, c->jL, c->wR, c->interp, c->f_floor, NULL, NULL, Craw);
    if (project) okx_project(N, f, Craw, c->h, c->E, c->K, c->eps_supp, Cp, diag4);
    else { memcpy(Cp, Craw, sizeof(double) * N); if (diag4) okx_project(N, f, Craw, c->h, c->E, c->K, c->eps_supp, Craw, diag4); }
    for (int i = 0; i < N; ++i) {
        double s = 0.0;
        for (int q = 0; q < nsrc; ++q) s += ampk[q] * G[(size_t)q * N + i];
        k[i] = kR * Cp[i] + s;
    }
    free(Craw); free(Cp);
}

static int okx_evolve_impl(int eta, int N, int B, const double *p, const double *dp, double m, double g_chi,
               double M2_0, double m_med, int interp, double f_floor, double eps_supp,
               double *f, int method, int S, const double *tau, const double *rate,
               const double *mass, const double *kappa, int project,
               int nsrc, const double *G, const double *amp, double *diag)
{
    size_t N3 = (size_t)N * N * N;
    okx_ctx c = { N, p, dp, m, g_chi, M2_0, m_med, interp, f_floor, eps_supp,
                  malloc(sizeof(double) * N3), malloc(sizeof(int32_t) * N3), malloc(sizeof(double) * N3),
                  malloc(sizeof(double) * N), malloc(sizeof(double) * N), malloc(sizeof(double) * N), m };
    c.eta = eta;
    okx_build(N, p, dp, m, g_chi, M2_0, m_med, c.W, c.jL, c.wR);
    okx_kinematics(N, p, dp, m, c.E, c.K, c.h);
    double *k1 = malloc(sizeof(double) * N), *k2 = malloc(sizeof(double) * N), *k3 = malloc(sizeof(double) * N),
           *k4 = malloc(sizeof(double) * N), *ft = malloc(sizeof(double) * N), *ampk = malloc(sizeof(double) * (nsrc > 0 ? nsrc : 1));
    int use_mass = mass != NULL;
    /* the step loop is outermost so that a time-dependent mass needs one rebuild per stage, shared by all b */
    for (int s = 0; s < S; ++s) {
        double dt = tau[s + 1] - tau[s];
        double R0 = rate ? rate[2 * s] : 1.0, Rh = rate ? rate[2 * s + 1] : 1.0, R1 = rate ? rate[2 * s + 2] : 1.0;
        double m0 = use_mass ? mass[2 * s] : m, mh = use_mass ? mass[2 * s + 1] : m, m1 = use_mass ? mass[2 * s + 2] : m;
        for (int q = 0; q < nsrc; ++q) ampk[q] = amp[(size_t)q * S + s];
        /* stage-major over b so each rebuild is reused by every member */
        if (method == 0) {
            for (int b = 0; b < B; ++b) {
                double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N;
                okx_rhs(&c, fb, m0, use_mass, kb * R0, project, nsrc, G, ampk, k1, diag ? diag + ((size_t)s * B + b) * 6 : NULL);
                for (int i = 0; i < N; ++i) fb[i] = fb[i] + dt * k1[i];
            }
        } else if (method == 1) {
            double *K1 = malloc(sizeof(double) * N * B);
            for (int b = 0; b < B; ++b) {
                double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N;
                okx_rhs(&c, fb, m0, use_mass, kb * R0, project, nsrc, G, ampk, K1 + (size_t)b * N, diag ? diag + ((size_t)s * B + b) * 6 : NULL);
            }
            for (int b = 0; b < B; ++b) {
                double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N, *kk = K1 + (size_t)b * N;
                for (int i = 0; i < N; ++i) ft[i] = fb[i] + dt * kk[i];
                okx_rhs(&c, ft, m1, use_mass, kb * R1, project, nsrc, G, ampk, k2, NULL);
                for (int i = 0; i < N; ++i) fb[i] = fb[i] + 0.5 * dt * (kk[i] + k2[i]);
            }
            free(K1);
        } else {
            double *K1 = malloc(sizeof(double) * N * B), *K2 = malloc(sizeof(double) * N * B), *K3 = malloc(sizeof(double) * N * B);
            for (int b = 0; b < B; ++b) {
                double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N;
                okx_rhs(&c, fb, m0, use_mass, kb * R0, project, nsrc, G, ampk, K1 + (size_t)b * N, diag ? diag + ((size_t)s * B + b) * 6 : NULL);
            }
            for (int b = 0; b < B; ++b) {
                double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N;
                for (int i = 0; i < N; ++i) ft[i] = fb[i] + 0.5 * dt * K1[(size_t)b * N + i];
                okx_rhs(&c, ft, mh, use_mass, kb * Rh, project, nsrc, G, ampk, K2 + (size_t)b * N, NULL);
            }
            for (int b = 0; b < B; ++b) {
                double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N;
                for (int i = 0; i < N; ++i) ft[i] = fb[i] + 0.5 * dt * K2[(size_t)b * N + i];
                okx_rhs(&c, ft, mh, use_mass, kb * Rh, project, nsrc, G, ampk, K3 + (size_t)b * N, NULL);
            }
            for (int b = 0; b < B; ++b) {
                double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N;
                for (int i = 0; i < N; ++i) ft[i] = fb[i] + dt * K3[(size_t)b * N + i];
                okx_rhs(&c, ft, m1, use_mass, kb * R1, project, nsrc, G, ampk, k4, NULL);
                for (int i = 0; i < N; ++i)
                    fb[i] = fb[i] + (dt / 6.0) * (K1[(size_t)b * N + i] + 2.0 * K2[(size_t)b * N + i] + 2.0 * K3[(size_t)b * N + i] + k4[i]);
            }
            free(K1); free(K2); free(K3);
        }
        if (diag) {
            double mend = use_mass ? m1 : m;
            if (use_mass && mend != c.cur_m) { okx_kinematics(N, p, dp, mend, c.E, c.K, c.h); }
            for (int b = 0; b < B; ++b) {
                double mo[4];
                okx_moments(N, f + (size_t)b * N, p, c.h, c.E, g_chi, mo);
                diag[((size_t)s * B + b) * 6 + 4] = mo[0];
                diag[((size_t)s * B + b) * 6 + 5] = mo[1];
            }
            if (use_mass && mend != c.cur_m) { okx_kinematics(N, p, dp, c.cur_m, c.E, c.K, c.h); }
        }
    }
    free(k1); free(k2); free(k3); free(k4); free(ft); free(ampk);
    free(c.W); free(c.jL); free(c.wR); free(c.E); free(c.K); free(c.h);
    return 0;
}

int okx_evolve(int N, int B, const double *p, const double *dp, double m, double g_chi,
               double M2_0, double m_med, int interp, double f_floor, double eps_supp,
               double *f, int method, int S, const double *tau, const double *rate,
               const double *mass, const double *kappa, int project,
               int nsrc, const double *G, const double *amp, double *diag)
{
    return okx_evolve_impl(0, N, B, p, dp, m, g_chi, M2_0, m_med, interp, f_floor, eps_supp, f, method, S, tau, rate,
                           mass, kappa, project, nsrc, G, amp, diag);
}

/* the same integrators with the quantum-statistics operator okx_collide_q (eta = +1 / -1) */
int okx_evolve_q(int eta, int N, int B, const double *p, const double *dp, double m, double g_chi,
                 double M2_0, double m_med, double f_floor, double eps_supp,
                 double *f, int method, int S, const double *tau, const double *rate,
                 const double *mass, const double *kappa, int project,
                 int nsrc, const double *G, const double *amp, double *diag)
{
    return okx_evolve_impl(eta, N, B, p, dp, m, g_chi, M2_0, m_med, 0, f_floor, eps_supp, f, method, S, tau, rate,
                           mass, kappa, project, nsrc, G, amp, diag);
}

/* ---- Monoenergetic source (eq. 3.7) deposited on the grid: "split between the two
 * neighboring grid points q_L < q_0 < q_R using the energy-linear deposition fractions alpha_R = (E_0 - E_L)/(E_R - E_L)
 * and alpha_L = 1 - alpha_R ... normalized so that the discrete zeroth and energy moments reproduce exactly the injected
 * particle-number and energy rates": G_L = alpha_L/h_L, G_R = alpha_R/h_R, so sum h G = 1 and sum h E G = E_0. */
int okx_delta_source(int N, const double *p, const double *dp, double m, double p0, double *G)
{
    if (!(p0 >= p[0] && p0 <= p[N - 1])) return 1;
    int L = 0;
    for (int j = 0; j <= N - 2; ++j) if (p[j] <= p0) L = j;        /* largest L <= N-2 with p_L <= p0 */
    double EL = sqrt(p[L] * p[L] + m * m), ER = sqrt(p[L + 1] * p[L + 1] + m * m), E0 = sqrt(p0 * p0 + m * m);
    double aR = (E0 - EL) / (ER - EL);
    for (int i = 0; i < N; ++i) G[i] = 0.0;
    G[L] = (1.0 - aR) / (p[L] * p[L] * dp[L]);
    G[L + 1] = aR / (p[L + 1] * p[L + 1] * dp[L + 1]);
    return 0;
}

/* ---- Adaptive Heun in u = ln a (Sec. 4.2: "first computes an Euler predictor and then corrects it
 * using the average of the slopes at the beginning and end of the step. The difference between the predictor and
 * corrected value provides a local error estimate used to adjust the step size"; settings rtol, atol, du0, safety of
 * PAPER.md:474).  df/du = kappa_b R(u) C[f; m(u)] + sum_s amp_s G_s, R(u) = rate0 exp(slope (u - u0)),
 * m(u) = mass0 exp(mass_slope (u - u0)) (comoving momenta q = a p: the kinematics of eq. 4.4/B.17 see the mass m a,
 * PAPER.md:166; mass_slope = 0: static mass).
 * Controller (the paper does not print it; reading D15): err = max_{b,i} |f_H - f_P| / (atol + rtol
 * max(|f|, |f_H|)) over the whole batch; accept iff err <= 1; du <- du clamp(safety / sqrt(max(err, 1e-10)), 0.2, 5);
 * du <= u1 - u; stop when u1 - u <= 1e-14 max(|u1|, 1).  The loop runs from ustart (>= u0) with first step du_first. */
static void okx_adaptive_core(okx_ctx *c, int B, double *f, double u0, double ustart, double u1, double du_first,
                              double rtol, double atol, double safety, double rate0, double slope,
                              double mass0, double mass_slope, const double *kappa, int project,
                              int nsrc, const double *G, const double *amp, int max_steps,
                              double *u_out, double *du_out, long *acc_out, long *rej_out, int *done_out)
{
    int N = c->N;
    int use_mass = mass_slope != 0.0;
    double *K1 = malloc(sizeof(double) * (size_t)B * N), *k2 = malloc(sizeof(double) * N);
    double *fP = malloc(sizeof(double) * (size_t)B * N), *fH = malloc(sizeof(double) * (size_t)B * N);
    double u = ustart, du = du_first < u1 - ustart ? du_first : u1 - ustart;
    long acc = 0, rej = 0;
    int done = u1 - u <= 1e-14 * fmax(fabs(u1), 1.0);
    for (int step = 0; step < max_steps && !done; ++step) {
        double err = 0.0;
        double ma = use_mass ? mass0 * exp(mass_slope * (u - u0)) : mass0;
        double mb = use_mass ? mass0 * exp(mass_slope * (u + du - u0)) : mass0;
        /* stage-major over the members, so that a time-dependent mass needs one rebuild per stage */
        for (int b = 0; b < B; ++b) {
            double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N;
            okx_rhs(c, fb, ma, use_mass, kb * rate0 * exp(slope * (u - u0)), project, nsrc, G, amp, K1 + (size_t)b * N, NULL);
            for (int i = 0; i < N; ++i) fP[(size_t)b * N + i] = fb[i] + du * K1[(size_t)b * N + i];   /* Euler predictor */
        }
        for (int b = 0; b < B; ++b) {
            double kb = kappa ? kappa[b] : 1.0, *fb = f + (size_t)b * N;
            okx_rhs(c, fP + (size_t)b * N, mb, use_mass, kb * rate0 * exp(slope * (u + du - u0)), project, nsrc, G, amp, k2, NULL);
            for (int i = 0; i < N; ++i) {
                double fh = fb[i] + 0.5 * du * (K1[(size_t)b * N + i] + k2[i]);                       /* Heun corrector */
                fH[(size_t)b * N + i] = fh;
                double e = fabs(fh - fP[(size_t)b * N + i]) / (atol + rtol * fmax(fabs(fb[i]), fabs(fh)));
                if (!(e <= err)) err = isfinite(e) ? e : INFINITY;
            }
        }
        int ok = err <= 1.0;
        double fac = safety / sqrt(fmax(err, 1e-10));
        if (!(fac == fac)) fac = 0.2;
        fac = fmin(fmax(fac, 0.2), 5.0);
        if (ok) { memcpy(f, fH, sizeof(double) * (size_t)B * N); u += du; ++acc; } else ++rej;
        du *= fac;
        if (u1 - u <= 1e-14 * fmax(fabs(u1), 1.0)) { done = 1; u = u1; }
        else if (du > u1 - u) du = u1 - u;
    }
    *u_out = u; *du_out = du; *acc_out = acc; *rej_out = rej; *done_out = done;
    free(K1); free(k2); free(fP); free(fH);
}

static okx_ctx okx_ctx_new(int eta, int N, const double *p, const double *dp, double m, double g_chi, double M2_0,
                           double m_med, double f_floor, double eps_supp)
{
    size_t N3 = (size_t)N * N * N;
    okx_ctx c = { N, p, dp, m, g_chi, M2_0, m_med, 0, f_floor, eps_supp,
                  malloc(sizeof(double) * N3), malloc(sizeof(int32_t) * N3), malloc(sizeof(double) * N3),
                  malloc(sizeof(double) * N), malloc(sizeof(double) * N), malloc(sizeof(double) * N), m };
    c.eta = eta;
    okx_build(N, p, dp, m, g_chi, M2_0, m_med, c.W, c.jL, c.wR);
    okx_kinematics(N, p, dp, m, c.E, c.K, c.h);
    return c;
}
static void okx_ctx_free(okx_ctx *c) { free(c->W); free(c->jL); free(c->wR); free(c->E); free(c->K); free(c->h); }

/* out = {u, du, accepted, rejected, done} */
int okx_evolve_adaptive(int eta, int N, int B, const double *p, const double *dp, double m, double g_chi,
                        double M2_0, double m_med, double f_floor, double eps_supp, double *f,
                        double u0, double u1, double du0, double rtol, double atol, double safety,
                        double rate0, double slope, double mass_slope, const double *kappa, int project,
                        int nsrc, const double *G, const double *amp, int max_steps, double *out)
{
    okx_ctx c = okx_ctx_new(eta, N, p, dp, m, g_chi, M2_0, m_med, f_floor, eps_supp);
    double u, du; long acc, rej; int done;
    okx_adaptive_core(&c, B, f, u0, u0, u1, du0, rtol, atol, safety, rate0, slope, m, mass_slope, kappa, project,
                      nsrc, G, amp, max_steps, &u, &du, &acc, &rej, &done);
    out[0] = u; out[1] = du; out[2] = (double)acc; out[3] = (double)rej; out[4] = (double)done;
    okx_ctx_free(&c);
    return 0;
}

/* ---- The two regimes of Sec. 4.2.
 * Regime 1, "the self-scattering rate is negligible compared with the Hubble rate, and the evolution is driven only by
 * the freeze-in source terms.  In this regime, we set the self-collisions to zero, C_el[f] = 0, and evolve the
 * distribution with a fourth-order Runge-Kutta method on fixed intervals in u": steps of du_fixed (the last one cut at
 * u1).  The source rates amp_s are constant in u here, so all four Runge-Kutta slopes are the same vector
 * k = sum_s amp_s G_s and the RK4 update f + (du/6)(k + 2k + 2k + k) is f + du k: that is what is evaluated.
 * "The code also monitors the effective self-scattering rate, Gamma_2->2 = n_chi <sigma v>, and compares it with the
 * Hubble rate.  Once Gamma_2->2 / H > eps_switch = 1e-2, the elastic self-collision operator is included."  Reading D16
 * (the paper gives only the definition): the discretized n_chi <sigma v> seen by a particle of bin i is the loss
 * frequency nu_i = loss_i / f_i = sum_nm W_inm f_j~ of eq. 4.6, its average over the population is
 * nu_bar = sum_i h_i loss_i / sum_i h_i f_i, and with the time variable u of eq. 4.9 the ratio is
 *     Gamma_2->2 / H = kappa_b R(u) nu_bar[f(u); m(u)]          (0 when sum h f = 0).
 * It is evaluated at u0 and after every fixed step; the whole batch switches at the first such point where the LARGEST
 * member ratio exceeds eps_switch (eps_switch <= 0: regime 2 from the start).
 * Regime 2: adaptive Heun (okx_adaptive_core) from the switch point to u1 with first step du0.
 * out = {u, du, accepted, rejected, done, u_switch, fixed_steps, ratio_at_switch}; max_steps bounds the attempted Heun
 * steps; u_switch = u1 and ratio = the last monitored value if the switch never happens. */
int okx_evolve_regimes(int N, int B, const double *p, const double *dp, double m, double g_chi,
                       double M2_0, double m_med, double f_floor, double eps_supp, double *f,
                       double u0, double u1, double du_fixed, double eps_switch,
                       double du0, double rtol, double atol, double safety,
                       double rate0, double slope, double mass_slope, const double *kappa, int project,
                       int nsrc, const double *G, const double *amp, int max_steps, double *out)
{
    okx_ctx c = okx_ctx_new(0, N, p, dp, m, g_chi, M2_0, m_med, f_floor, eps_supp);
    int use_mass = mass_slope != 0.0;
    double *loss = malloc(sizeof(double) * N);
    double u = u0, ratio = 0.0;
    long fixed = 0;
    int switched = 0, done = 0;
    for (;;) {
        /* monitor at u */
        double mu_ = use_mass ? m * exp(mass_slope * (u - u0)) : m;
        if (use_mass && mu_ != c.cur_m) {
            okx_build(N, p, dp, mu_, g_chi, M2_0, m_med, c.W, c.jL, c.wR);
            okx_kinematics(N, p, dp, mu_, c.E, c.K, c.h);
            c.cur_m = mu_;
        }
        ratio = 0.0;
        for (int b = 0; b < B; ++b) {
            const double *fb = f + (size_t)b * N;
            okx_collide(N, 1, fb, c.W, c.jL, c.wR, 0, f_floor, NULL, loss, NULL);
            long double sl = 0.0L, sf = 0.0L;
            for (int i = 0; i < N; ++i) { sl += (long double)c.h[i] * loss[i]; sf += (long double)c.h[i] * fb[i]; }
            double r = sf > 0.0L ? (kappa ? kappa[b] : 1.0) * rate0 * exp(slope * (u - u0)) * (double)(sl / sf) : 0.0;
            if (r > ratio) ratio = r;
        }
        if (!(eps_switch > 0.0) || ratio > eps_switch) { switched = 1; break; }
        if (u1 - u <= 1e-14 * fmax(fabs(u1), 1.0)) { done = 1; u = u1; break; }
        /* one fixed step with C_el = 0 */
        double du = du_fixed < u1 - u ? du_fixed : u1 - u;
        for (int b = 0; b < B; ++b)
            for (int i = 0; i < N; ++i) {
                double k = 0.0;
                for (int q = 0; q < nsrc; ++q) k += amp[q] * G[(size_t)q * N + i];
                f[(size_t)b * N + i] += du * k;
            }
        u += du;
        ++fixed;
    }
    double usw = switched ? u : u1, du_next = du0;
    long acc = 0, rej = 0;
    if (switched)
        okx_adaptive_core(&c, B, f, u0, u, u1, du0, rtol, atol, safety, rate0, slope, m, mass_slope, kappa, project,
                          nsrc, G, amp, max_steps, &u, &du_next, &acc, &rej, &done);
    out[0] = u; out[1] = du_next; out[2] = (double)acc; out[3] = (double)rej; out[4] = (double)done;
    out[5] = usw; out[6] = (double)fixed; out[7] = ratio;
    free(loss);
    okx_ctx_free(&c);
    return 0;
}

/* ---- Pin helper (P9), NOT on the evaluate path: the reduced kernel F(p_i,p_n,p_m) by the
 * mu-quadrature of eq. B.5-B.12, nodes/weights supplied by the caller.
 * If m_med > 0 the integrand carries |M|^2(t(mu)), t = 2m^2-2E_iE_n+2p_ip_n mu (reading D5). */
double okx_F_quadrature(double pi_, double pn, double pm, double m, double M2_0, double m_med,
                        int nmu, const double *mu, const double *wmu)
{
    double Ei = sqrt(pi_ * pi_ + m * m), En = sqrt(pn * pn + m * m), Em = sqrt(pm * pm + m * m);
    long double acc = 0.0L;
    for (int q = 0; q < nmu; ++q) {
        double u = mu[q];
        double A0 = m * m + En * Em - En * Ei - Em * Ei + pi_ * pn * u;   /* B.5 */
        double A1 = pi_ * pm - pn * pm * u;                                 /* B.6 */
        double K2 = pn * pn * pm * pm * (1.0 - u * u);                      /* B.7 */
        double a = -(K2 + A1 * A1), b = -2.0 * A0 * A1, c = K2 - A0 * A0;   /* B.8 */
        double disc = b * b - 4.0 * a * c;
        if (!(disc > 0.0) || !(a < 0.0)) continue;
        double sq = sqrt(disc);
        double r1 = (-b + sq) / (2.0 * a), r2 = (-b - sq) / (2.0 * a);      /* B.10 */
        double lo = fmin(r1, r2), hi = fmax(r1, r2);
        if (hi <= -1.0 || lo >= 1.0) continue;
        double vm = fmax(lo, -1.0), vp = fmin(hi, 1.0);
        double am = fmax(-1.0, fmin(1.0, (2.0 * a * vm + b) / sq));
        double ap = fmax(-1.0, fmin(1.0, (2.0 * a * vp + b) / sq));
        double I = (asin(am) - asin(ap)) / sqrt(-a);                        /* B.11 */
        double M2 = M2_0;
        if (m_med > 0.0) {
            double t = 2.0 * m * m - 2.0 * Ei * En + 2.0 * pi_ * pn * u;
            double d = 1.0 + (-t) / (m_med * m_med);
            M2 = M2_0 / (d * d);
        }
        acc += (long double)wmu[q] * I * M2;
    }
    double pref = 1.0 / (4.0 * pow(2.0 * (double)OKX_PI, 4)) * (pn * pm) * (pn * pm) / (En * Em); /* B.12 */
    return pref * (double)acc;
}

/* The closed-form F used inside okx_build for one triple (exposed for the P9 pin): eq. B.17 / D5. */
double okx_F_closed(double pi_, double pn, double pm, double m, double M2_0, double m_med)
{
    double Ei = sqrt(pi_ * pi_ + m * m), En = sqrt(pn * pn + m * m), Em = sqrt(pm * pm + m * m);
    double Ki = pi_ * pi_ / (Ei + m), Kn = pn * pn / (En + m), Km = pm * pm / (Em + m);
    double Kt = (Kn + Km) - Ki;
    if (Kt < 0.0) return 0.0;
    double pj = sqrt(Kt * (Kt + 2.0 * m));
    double Qm = fmax(fabs(pi_ - pn), fabs(pm - pj)), Qp = fmin(pi_ + pn, pm + pj);
    double J = okx_J(Qm, Qp, M2_0, m_med, Ki, Kn);
    const double pi3 = (double)(OKX_PI * OKX_PI * OKX_PI);
    return (1.0 / (64.0 * pi3 * pi_)) * (pn * pm / (En * Em)) * J;
}

/* ---- Numerical angular kernel: replace the analytic F of every KEPT triple by the
 * mu-quadrature of eq. B.5-B.12 (okx_F_quadrature above): W_inm = dp_n dp_m F_inm / (2 E_i g_chi), eq. 4.7.  The index
 * map (jL, omega_R) is untouched: it is fixed by energy conservation alone. */
void okx_requadrature(int N, const double *p, const double *dp, double m, double g_chi, double M2_0, double m_med,
                      int nmu, const double *mu, const double *wmu, double *W, const int32_t *jL)
{
#pragma omp parallel for schedule(dynamic)
    for (int i = 0; i < N; ++i) {
        double Ei = sqrt(p[i] * p[i] + m * m);
        for (int n = 0; n < N; ++n)
            for (int mm = 0; mm < N; ++mm) {
                size_t idx = ((size_t)i * N + n) * N + mm;
                if (jL[idx] < 0) continue;
                W[idx] = dp[n] * dp[mm] / (2.0 * Ei * g_chi) * okx_F_quadrature(p[i], p[n], p[mm], m, M2_0, m_med, nmu, mu, wmu);
            }
    }
}
