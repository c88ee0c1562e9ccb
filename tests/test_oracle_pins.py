"""Pins of the CPU oracle against what the paper and the mathematics fix.

None of these retype the oracle's formulas: they are closed forms, invariants, special cases and a
brute-force angular quadrature chosen so that a dropped term, wrong sign/index or transposed operand
in `oracle/kx_oracle.c` fails at least one of them.  CPU only.
"""
import itertools
import math
import os

import numpy as np
import pytest
from scipy.integrate import quad

import kx_inputs as kin

HERE = os.path.dirname(os.path.abspath(__file__))


# ------------------------------------------------------------------ P1: W_inm = W_imn (B.17 symmetric)
@pytest.mark.parametrize("cfg", [1, 3])
def test_P1_W_symmetric(oracle, cfg):
    c = kin.config(cfg, N=48 if cfg == 3 else None)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    if c["m_med"] <= 0:     # contact: B.17 is symmetric in n<->m.  A t-channel |M|^2(t), t=(p_i-p_n)^2, is not (D5)
        assert np.abs(T.W - T.W.transpose(0, 2, 1)).max() <= 1e-11 * np.abs(T.W).max()
    assert (T.jL == T.jL.transpose(0, 2, 1)).all()          # the index map always is
    assert (T.W >= 0).all() and T.kept == int((T.jL >= 0).sum())


# ------------------------------------------------------------------ P2: overlap invariance, massless = 2 min(p)
def test_P2_massless_overlap_is_twice_min(oracle):
    rng = np.random.default_rng(7)
    for _ in range(200):
        pi, pn, pm = rng.uniform(0.05, 5.0, size=3)
        pj = pn + pm - pi
        F = oracle.F_closed(pi, pn, pm, 0.0, 1.0, 0.0)
        if pj <= 0:
            assert F == 0.0
            continue
        expect = 2.0 * min(pi, pn, pm, pj) / (64.0 * math.pi ** 3 * pi)       # p/E = 1 at m = 0
        assert F == pytest.approx(expect, rel=1e-12, abs=1e-18)


def test_P2_permutation_invariance_massive(oracle):
    """[min(a+b,c+d)-max(|a-b|,|c-d|)]_+ is invariant under all 24 permutations of (p_i,p_n,p_m,p_j):
    exchanging the roles (i<->n) and (i,n)<->(m,j) must leave p_i*E_n*E_m*F/(p_n p_m) unchanged."""
    rng = np.random.default_rng(8)
    m = 1.0
    E = lambda p: math.sqrt(p * p + m * m)
    for _ in range(100):
        pi, pn, pm = rng.uniform(0.05, 4.0, size=3)
        Ej = E(pn) + E(pm) - E(pi)
        if Ej <= m * (1 + 1e-9):
            continue
        pj = math.sqrt(Ej * Ej - m * m)
        ov = lambda a, b, c: oracle.F_closed(a, b, c, m, 1.0, 0.0) * a * E(b) * E(c) / (b * c)
        base = ov(pi, pn, pm)
        # (i,n,m,j) -> (n,i,j,m): chi_n chi_i <- chi_j chi_m has the same overlap
        assert ov(pn, pi, pj) == pytest.approx(base, rel=1e-9, abs=1e-15)
        assert ov(pi, pm, pn) == pytest.approx(base, rel=1e-9, abs=1e-15)
        assert ov(pj, pm, pn) == pytest.approx(base, rel=1e-9, abs=1e-15)


# ------------------------------------------------------------------ P3: zeros of W only from the validity test
def test_P3_zeros_only_from_validity(oracle):
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    kept = T.jL >= 0
    # interior kept triples (strictly inside the K range) have a strictly positive overlap
    Kt = T.K[None, :, None] + T.K[None, None, :] - T.K[:, None, None]
    interior = kept & (Kt > T.K[0] * (1 + 1e-9)) & (Kt < T.K[-1] * (1 - 1e-9))
    assert (T.W[interior] > 0).all()
    assert (T.W[~kept] == 0).all()
    # validity is exactly E_j >= m, q_min <= q_j <= q_max away from ties
    far = np.abs(Kt - T.K[0]) > 1e-9
    far &= np.abs(Kt - T.K[-1]) > 1e-9
    assert (kept[far] == ((Kt >= T.K[0]) & (Kt <= T.K[-1]))[far]).all()


# ------------------------------------------------------------------ P4: exact conservation special case
@pytest.mark.parametrize("interp", [0, 1])
def test_P4_exact_conservation_massless_uniform(oracle, interp):
    N, D = 40, 0.25
    p = D * np.arange(1, N + 1)
    dp = np.full(N, D)
    T = oracle.Tables(p, dp, 0.0)
    assert np.all((T.wR[T.jL >= 0] < 1e-12) | (T.wR[T.jL >= 0] > 1 - 1e-12))   # every j~ on-grid
    f = kin.bimodal(p, (2.0, 6.0), (0.5, 1.0))[None, :]
    g, l, C = oracle.collide(T, f, interp)
    h, E = T.h, T.E
    epsN = (h * C[0]).sum() / (h * np.abs(C[0])).sum()
    epsE = (h * E * C[0]).sum() / (h * E * np.abs(C[0])).sum()
    assert abs(epsN) <= 1e-14 and abs(epsE) <= 1e-14
    # total gain = total loss, and energy-weighted too (number / energy conservation, eq. 2.7 / 4.8)
    assert (h * g[0]).sum() == pytest.approx((h * l[0]).sum(), rel=1e-13)


def test_P4_exchange_symmetry_of_W(oracle):
    """Detailed-balance structure: h_i W_inm = h_n W_{n,i,j} on the exact grid (exchange (i,j)<->(n,m))."""
    N, D = 24, 0.5
    p = D * np.arange(1, N + 1)
    T = oracle.Tables(p, np.full(N, D), 0.0)
    checked = 0
    for i, n, m in itertools.product(range(N), repeat=3):
        j = n + m - i                                    # p_j = p_n + p_m - p_i  ->  index n+m-i+... (p_k=(k+1)D)
        jj = (n + 1) + (m + 1) - (i + 1) - 1
        if 0 <= jj < N and T.jL[i, n, m] >= 0:
            lhs = T.h[i] * T.W[i, n, m]
            rhs = T.h[n] * T.W[n, i, jj]
            assert lhs == pytest.approx(rhs, rel=1e-12, abs=1e-300)
            checked += 1
    assert checked > 1000


# ------------------------------------------------------------------ P5: thermal fixed point under LOG
@pytest.mark.parametrize("cfg,Tchi", [(1, 1.3), (3, 0.7)])
def test_P5_thermal_fixed_point(oracle, cfg, Tchi):
    c = kin.config(cfg, N=64 if cfg == 3 else None)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    f = (0.37 * np.exp(-T.E / Tchi))[None, :]
    g, l, C = oracle.collide(T, f, 0)
    assert np.abs(C).max() <= 1e-13 * np.abs(g).max()
    # LINEAR does not have this property: O(Delta^2) residual (P8)
    g1, l1, C1 = oracle.collide(T, f, 1)
    assert np.abs(C1).max() > 1e-8 * np.abs(g1).max()


# ------------------------------------------------------------------ P6: projection conserves both moments
def test_P6_projection_and_steps_conserve(oracle):
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    g, l, C = oracle.collide(T, c["f"], 0)
    Cp, diag = oracle.project(T, c["f"], C)
    sc = (T.h * np.abs(C[0])).sum()
    assert abs((T.h * Cp[0]).sum()) <= 1e-14 * sc
    assert abs((T.h * T.E * Cp[0]).sum()) <= 1e-14 * (T.h * T.E * np.abs(C[0])).sum()
    # diag = eps_N, eps_E (C.1) and R_N, R_E (C.9), recomputed here from their definitions
    assert diag[0, 0] == pytest.approx((T.h * C[0]).sum() / sc, rel=1e-10)
    assert diag[0, 2] == pytest.approx((T.h * np.abs(Cp[0] - C[0])).sum() / sc, rel=1e-10)
    # 50 RK4 steps: number and energy drift <= 1e-12 relative per step
    nu_max = (l[0] / c["f"][0]).max()
    S = 50
    tau = np.arange(S + 1) * (0.2 / nu_max)
    f1 = oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=oracle.RK4, tau=tau)
    n0, n1 = oracle.moments(T, c["f"])[0], oracle.moments(T, f1)[0]
    assert abs(n1[0] / n0[0] - 1) <= 1e-12 * S and abs(n1[1] / n0[1] - 1) <= 1e-12 * S
    assert np.abs(f1 - c["f"]).max() > 1e-3 * c["f"].max()          # it did move


@pytest.mark.parametrize("m", [1.0, 30.0, 1000.0])
def test_P6_projection_exact_rational(oracle, m):
    """App. C solved LITERALLY (eq. C.2-C.8, basis {1, E_i}) in exact rational arithmetic on the same doubles.
    The oracle solves the same system in the basis {1, K_i} (reading D3); the projections must coincide, also at
    m/T = 1e3 where the E-basis determinant cancels to 4e-10 of its terms.  The energies of the exact solve are
    E_i = m + K_i taken exactly (the stable kinetic energies of O1 define the grid; the rounded double
    sqrt(p^2+m^2) differs from m + K_i by up to 1e-10 K_i at this mass, which alone moves the result by 3e-13)."""
    from fractions import Fraction as Fr
    N = 48
    p = kin.log_grid(N, 1e-3, 100.0)
    T = oracle.Tables(p, kin.trapezoid_widths(p), m)
    f = kin.bimodal(p, (3.0, 8.0), (1.0, 2.0))[None, :]
    g, l, C = oracle.collide(T, f, 0)
    Cp, _ = oracle.project(T, f, C, eps_supp=1e-12)
    h, E, c = [Fr(x) for x in T.h], [Fr(m) + Fr(x) for x in T.K], [Fr(x) for x in C[0]]
    fmax = float(np.abs(f[0]).max())
    xi = [Fr(abs(float(x)) / fmax) if abs(float(x)) / fmax > 1e-12 else Fr(0) for x in f[0]]     # C.4
    R0 = sum(a * b for a, b in zip(h, c))                                                           # C.2
    R1 = sum(a * e * b for a, e, b in zip(h, E, c))
    A00 = sum(a * x for a, x in zip(h, xi))                                                         # C.6
    A01 = sum(a * e * x for a, e, x in zip(h, E, xi))
    A11 = sum(a * e * e * x for a, e, x in zip(h, E, xi))
    det = A00 * A11 - A01 * A01                                                                     # C.8
    al, be = (R0 * A11 - R1 * A01) / det, (R1 * A00 - R0 * A01) / det
    exact = np.array([float(ci - x * (al + be * e)) for ci, x, e in zip(c, xi, E)])                 # C.3
    assert np.abs(Cp[0] - exact).max() <= 1e-15 * np.abs(g).max()
    assert np.abs(exact - C[0]).max() > 1e-4 * np.abs(g).max()          # the correction is not trivially zero


def test_P6_relaxes_towards_maxwell_boltzmann(oracle):
    """Config 1 run: Euler steps with the projected LOG operator approach z*exp(-E/T) (H-theorem)."""
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    g, l, C = oracle.collide(T, c["f"], 0)
    nu_max = (l[0] / c["f"][0]).max()

    def dist_to_mb(f):
        # least-squares fit of ln f = ln z - E/T on the populated bins
        msk = f > 1e-8 * f.max()
        A = np.stack([np.ones(msk.sum()), -T.E[msk]], axis=1)
        coef, res, *_ = np.linalg.lstsq(A, np.log(f[msk]), rcond=None)
        return float(np.sqrt(((A @ coef - np.log(f[msk])) ** 2).mean()))

    d0 = dist_to_mb(c["f"][0])
    f = c["f"]
    for S in (200, 2000):
        tau = np.arange(S + 1) * (0.2 / nu_max)
        f = oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=oracle.EULER, tau=tau)
        d = dist_to_mb(f[0])
        assert d < d0
        d0 = d
    assert (f > 0).all()


# ------------------------------------------------------------------ P7: normalisation against eq. 2.4 (closed form)
def test_P7_loss_frequency_closed_form(oracle):
    """m=0, contact, f = z exp(-p/T): eq. 2.4 with the massless two-body phase space 1/(8 pi) gives
    nu(p) = loss/f = |M|^2 z T^2 / (64 pi^3 p), and gain = nu f.  The discrete operator converges to it."""
    z, Tt, M2 = 0.8, 1.0, 2.5
    errs = []
    for N in (100, 200):
        D = 30.0 / N
        p = D * np.arange(1, N + 1)
        T = oracle.Tables(p, np.full(N, D), 0.0, 1.0, M2, 0.0)
        f = (z * np.exp(-p / Tt))[None, :]
        g, l, C = oracle.collide(T, f, 0)
        nu = l[0] / f[0]
        exact = M2 * z * Tt ** 2 / (64 * math.pi ** 3 * p)
        win = (p > 0.5) & (p < 8.0)
        errs.append(np.abs(nu[win] / exact[win] - 1).max())
        assert np.abs(g[0][win] / (exact * f[0])[win] - 1).max() < 0.09
    assert errs[0] < 0.08 and errs[1] < 0.025 and errs[1] < 0.4 * errs[0]


# ------------------------------------------------------------------ P8: residuals shrink with N
def test_P8_raw_residuals_decrease_with_N(oracle):
    res = []
    for N in (32, 64, 128):
        p = kin.log_grid(N, 1e-3, 1e2)
        dp = kin.trapezoid_widths(p)
        T = oracle.Tables(p, dp, 1.0)
        f = kin.two_bump_eq51(p)[None, :]
        g, l, C = oracle.collide(T, f, 0)
        Cp, diag = oracle.project(T, f, C)
        res.append(np.abs(diag[0]))
    assert res[2][0] < res[0][0] and res[2][1] < res[0][1]        # eps_N, eps_E
    assert res[2][2] < res[0][2] and res[2][3] < res[0][3]        # R_N, R_E (Fig. 9)


# ------------------------------------------------------------------ P9: brute-force angular quadrature (B.5-B.12) = B.17
@pytest.mark.parametrize("m_med", [0.0, 0.5])
def test_P9_closed_form_equals_mu_quadrature(oracle, m_med):
    mu, w = np.polynomial.legendre.leggauss(6000)
    rng = np.random.default_rng(11)
    done = 0
    while done < 12:
        pi, pn, pm = rng.uniform(0.1, 3.0, size=3)
        Fc = oracle.F_closed(pi, pn, pm, 1.0, 1.7, m_med)
        if Fc <= 0:
            continue
        Fq = oracle.F_quadrature(pi, pn, pm, 1.0, 1.7, m_med, mu, w)
        assert Fq == pytest.approx(Fc, rel=2e-3)
        done += 1


def test_P9_mediator_J_against_numerical_integration(oracle):
    """D5: F_closed(m_med)/F_closed(contact) = m_med^4 * int dQ/(Q^2+c^2)^2 / (Q+ - Q-), checked by adaptive quadrature (scipy QUADPACK)."""
    rng = np.random.default_rng(12)
    m = 1.0
    done = 0
    while done < 20:
        pi, pn, pm = rng.uniform(0.05, 6.0, size=3)
        m_med = float(rng.choice([0.05, 0.5, 3.0]))
        Fc0 = oracle.F_closed(pi, pn, pm, m, 1.0, 0.0)
        if Fc0 <= 0:
            continue
        Ei, En, Em = (math.sqrt(x * x + m * m) for x in (pi, pn, pm))
        pj = math.sqrt((En + Em - Ei) ** 2 - m * m)
        Qm, Qp = max(abs(pi - pn), abs(pm - pj)), min(pi + pn, pm + pj)
        dE2 = (Ei - En) ** 2
        integrand = lambda Q: 1.0 / (1.0 + (Q * Q - dE2) / m_med ** 2) ** 2
        simpson, _ = quad(integrand, Qm, Qp, epsabs=0, epsrel=1e-13, limit=400)
        ratio = oracle.F_closed(pi, pn, pm, m, 1.0, m_med) / Fc0
        assert ratio == pytest.approx(simpson / (Qp - Qm), rel=1e-8)
        done += 1


# ------------------------------------------------------------------ P10: the paper's printed projection sizes (soft)
def test_P10_paper_projection_correction_trend(oracle):
    rows = [ln.split() for ln in open(os.path.join(HERE, "golden", "paper_projection_correction.txt"))
            if ln.strip() and not ln.startswith("#")]
    paper = {int(r[0]): float(r[1]) for r in rows}
    got = {}
    for N in paper:
        p = kin.log_grid(N, 1e-3, 1e2)
        T = oracle.Tables(p, kin.trapezoid_widths(p), 1.0)
        f = kin.two_bump_eq51(p)[None, :]
        g, l, C = oracle.collide(T, f, 0)
        Cp, _ = oracle.project(T, f, C)
        got[N] = 100 * np.abs(Cp - C).max() / np.abs(C).max()
    # soft: same order of magnitude as PAPER.md:468 (Bose factors and eps_supp differ) and ~N^-2 trend
    for N, v in paper.items():
        assert v / 10 < got[N] < v * 10, (N, got[N], v)
    assert got[256] < got[96] / 3


# ------------------------------------------------------------------ moments: closed form (B.2)
def test_moments_closed_form(oracle):
    """n = g/(2 pi^2) sum h f: for f=exp(-p) on a fine uniform grid -> g/(2 pi^2) * 2 (int p^2 e^-p = 2);
    <p> = 3, <p^2> = 12 ; rho(m=0) = g/(2 pi^2) * 6."""
    N = 4000
    p = np.linspace(0.005, 40.0, N)
    dp = kin.trapezoid_widths(p)
    T = oracle.Tables.__new__(oracle.Tables)
    T.N, T.p, T.g_chi = N, p, 2.0
    T.E, T.K, T.h = oracle.kinematics(p, dp, 0.0)
    mo = oracle.moments(T, np.exp(-p)[None, :])[0]
    fac = 2.0 / (2 * math.pi ** 2)
    assert mo[0] == pytest.approx(fac * 2.0, rel=1e-4)
    assert mo[1] == pytest.approx(fac * 6.0, rel=1e-4)
    assert mo[2] == pytest.approx(3.0, rel=1e-4)
    assert mo[3] == pytest.approx(12.0, rel=1e-4)


# ------------------------------------------------------------------ integrator (O12): closed forms and convergence order
def test_evolve_sources_only_closed_form(oracle):
    """kappa = 0 switches the collision term off: f(S) = f(0) + sum_k amp[:,k] dtau_k G exactly, any method."""
    c = kin.config(5, N=24, B=3)
    sch = kin.config5_schedule(c["p"], c["p"] ** 2 * c["dp"], B=3, S=40)
    expect = (sch["amp"] * np.diff(sch["tau"])[None, :]).sum(axis=1) @ sch["G"]
    for method in (oracle.EULER, oracle.HEUN, oracle.RK4):
        f = oracle.evolve(c["p"], c["dp"], c["f"], method=method, tau=sch["tau"], rate=sch["rate"],
                          mass=None, kappa=np.zeros(3), G=sch["G"], amp=sch["amp"])
        assert np.allclose(f, expect[None, :], rtol=1e-13, atol=0)


def test_evolve_convergence_order_and_rate_scaling(oracle):
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    g, l, C = oracle.collide(T, c["f"], 0)
    t_end = 8.0 / (l[0] / c["f"][0]).max()

    def run(method, S, **kw):
        return oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=method, tau=np.linspace(0, t_end, S + 1), **kw)

    ref = run(oracle.RK4, 256)
    errs = {}
    for method, order in ((oracle.EULER, 1), (oracle.HEUN, 2), (oracle.RK4, 4)):
        e1 = np.abs(run(method, 8) - ref).max()
        e2 = np.abs(run(method, 16) - ref).max()
        errs[method] = (e1, e2)
        assert e1 / e2 > 0.6 * 2 ** order, (method, e1, e2)
    # a constant rate R and coupling kappa multiply the operator: (R=2, kappa=3, t) == (R=1, kappa=1, 6t)
    S = 16
    a = oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=oracle.RK4, tau=np.linspace(0, t_end / 6, S + 1),
                      rate=np.full(2 * S + 1, 2.0), kappa=np.array([3.0]))
    b = run(oracle.RK4, S)
    assert np.allclose(a, b, rtol=1e-12, atol=1e-300)
    # a mass schedule that is constant equals the static run (per-stage rebuild path)
    d = oracle.evolve(c["p"], c["dp"], c["f"], m=0.3, method=oracle.HEUN, tau=np.linspace(0, t_end, 5),
                      mass=np.full(9, c["m"]))
    e = run(oracle.HEUN, 4)
    assert np.array_equal(d, e)


# ------------------------------------------------------------------ row-sampled evaluator = full evaluator
@pytest.mark.parametrize("cfg,interp", [(1, 0), (3, 0), (3, 1)])
def test_collide_rows_equals_full_tables(oracle, cfg, interp):
    """okx_collide_rows (used to sample N=512) walks the same triples as the dense-table path: identical results."""
    c = kin.config(cfg, N=40 if cfg == 3 else None, B=3 if cfg == 3 else None)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g, l, C = oracle.collide(T, c["f"], interp)
    rows = np.array([0, 1, 7, T.N // 2, T.N - 2, T.N - 1])
    gr, lr, Cr = oracle.collide_rows(c["p"], c["dp"], c["f"], rows, m=c["m"], g_chi=c["g_chi"], M2_0=c["M2_0"],
                                     m_med=c["m_med"], interp=interp)
    assert np.array_equal(gr, g[:, rows]) and np.array_equal(lr, l[:, rows]) and np.array_equal(Cr, C[:, rows])


# ------------------------------------------------------------------ quantum-statistics operator
@pytest.mark.parametrize("eta,mu,Tchi", [(1, 0.0, 1.0), (1, -0.4, 0.7), (-1, 0.5, 1.0), (-1, 2.0, 0.3)])
def test_Q1_quantum_thermal_fixed_point(oracle, eta, mu, Tchi):
    """Fig. 11: N=96, T/m=1, mu=0 Bose-Einstein; the raw operator vanishes at round-off because
    y = ln(f/(1+eta f)) = (mu-E)/T is linear in E (eq. B.20).  Same for Fermi-Dirac and other (T, mu)."""
    p = kin.log_grid(96, 1e-3, 1e2)
    dp = kin.trapezoid_widths(p)
    T = oracle.Tables(p, dp, 1.0)
    f = 1.0 / (np.exp((T.E - mu) / Tchi) - eta)
    g, l, C = oracle.collide_q(T, f, eta)
    assert np.abs(C).max() <= 1e-13 * np.abs(g).max()
    # a distribution that is NOT of that form does not vanish (the test has teeth)
    g2, l2, C2 = oracle.collide_q(T, f * (1.0 - 0.3 * np.sin(p) ** 2), eta)
    assert np.abs(C2).max() >= 1e-4 * np.abs(g2).max()


@pytest.mark.parametrize("eta", [1, -1])
def test_Q2_dilute_limit_is_the_classical_operator(oracle, eta):
    """eq. 2.6: for f << 1 the quantum factors drop out; the difference is O(f) relative."""
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    for eps in (1e-4, 1e-7):
        f = eps * c["f"]
        g0, l0, C0 = oracle.collide(T, f, oracle.LOG)
        g, l, C = oracle.collide_q(T, f, eta)
        rel = np.abs(C - C0).max() / np.abs(g0).max()
        assert rel <= 20.0 * eps * np.abs(c["f"]).max(), (eps, rel)
        assert rel >= 1e-3 * eps            # and it is there: the quantum terms are not silently dropped


@pytest.mark.parametrize("eta", [1, -1])
def test_Q3_quantum_conservation_and_H_theorem_on_exact_grid(oracle, eta):
    """On the massless uniform grid of pin P4 every j~ is on-grid, Lambda is antisymmetric under (i,j~)<->(n,m) and
    h_i W_inm is symmetric, so the RAW quantum operator conserves number and energy at round-off and the discrete
    entropy production  -sum_i h_i C_i ln(f_i/(1+eta f_i))  is >= 0 (a wrong sign or a dropped factor breaks one)."""
    N = 40
    p = 0.25 * np.arange(1, N + 1)
    dp = np.full(N, 0.25)
    T = oracle.Tables(p, dp, 0.0)
    rng = np.random.default_rng(77)
    f = (0.4 + 0.3 * rng.uniform(size=N)) * np.exp(-0.5 * (p - 3.0) ** 2) + 0.05 * np.exp(-p / 4)
    if eta == -1:
        assert f.max() < 1.0
    g, l, C = oracle.collide_q(T, f, eta)
    h = T.h
    assert abs((h * C[0]).sum()) <= 1e-13 * (h * np.abs(C[0])).sum()
    assert abs((h * T.E * C[0]).sum()) <= 1e-13 * (h * T.E * np.abs(C[0])).sum()
    sigma = -(h * C[0] * np.log(f / (1.0 + eta * f))).sum()
    assert sigma > 0.0
    # eta enters: Bose enhancement and Pauli blocking move the operator in opposite directions from the classical one
    g0, l0, C0 = oracle.collide(T, f, oracle.LOG)
    assert np.abs(C[0] - C0[0]).max() > 1e-3 * np.abs(g0).max()


# ------------------------------------------------------------------ adaptive Heun
def test_A1_adaptive_heun_converges_to_rk4(oracle):
    """The adaptive Heun solution approaches a fine fixed-step RK4 solution as rtol -> 0, the error scales with the
    tolerance (second-order local estimate) and tighter tolerances take more steps; a first step far too large is rejected."""
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    g, l, C = oracle.collide(T, c["f"], oracle.LOG)
    nu = float((l[0] / c["f"][0]).max())
    u1 = 20.0 / nu
    ref = oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=oracle.RK4, tau=np.linspace(0.0, u1, 2001))
    errs, steps = [], []
    for rtol in (1e-3, 1e-4, 1e-5):
        f, info = oracle.evolve_adaptive(c["p"], c["dp"], c["f"], u0=0.0, u1=u1, du0=0.01 / nu, rtol=rtol, atol=1e-3 * rtol * 1e-6)
        assert info["done"] and abs(info["u"] - u1) <= 1e-12 * u1
        errs.append(np.abs(f - ref).max() / np.abs(ref).max())
        steps.append(info["accepted"])
    assert errs[0] < 1e-3 and errs[2] < 1e-5
    assert 3.0 < errs[0] / errs[1] < 30.0 and 3.0 < errs[1] / errs[2] < 30.0
    assert steps[0] < steps[1] < steps[2]
    f, info = oracle.evolve_adaptive(c["p"], c["dp"], c["f"], u0=0.0, u1=u1, du0=5.0 / nu, rtol=1e-3, atol=1e-12)
    assert info["rejected"] >= 2 and info["done"]
    # number and energy are conserved along the way (projected operator)
    m0, m1 = oracle.moments(T, c["f"]), oracle.moments(T, f)
    assert np.allclose(m0[:, :2], m1[:, :2], rtol=1e-11, atol=0)


def test_A2_adaptive_heun_sources_only_closed_form(oracle):
    """kappa = 0: df/du = sum_s amp_s G_s is constant, Heun is exact, the error estimate is 0, every step is accepted and
    grows by the maximal factor 5: n steps with du0 (5^n - 1)/4 >= u1 - u0, and f = f0 + (u1-u0) sum amp G exactly."""
    c = kin.config(1)
    N = c["p"].size
    G = np.stack([np.exp(-0.5 * (c["p"] - 3.0) ** 2), np.exp(-0.5 * ((c["p"] - 6.0) / 2.0) ** 2)])
    amp = np.array([0.3, 0.05])
    u0, u1, du0 = 1.0, 4.0, 1e-4
    f, info = oracle.evolve_adaptive(c["p"], c["dp"], c["f"], u0=u0, u1=u1, du0=du0, kappa=np.zeros(1), G=G, amp=amp)
    n = int(np.ceil(np.log(4.0 * (u1 - u0) / du0 + 1.0) / np.log(5.0)))
    assert info["accepted"] == n and info["rejected"] == 0 and info["done"]
    want = c["f"] + (u1 - u0) * (amp[:, None] * G).sum(axis=0)[None, :]
    assert np.abs(f - want).max() <= 1e-13 * np.abs(want).max()


# ------------------------------------------------------------------ monoenergetic source deposition (8(f) item 4)
@pytest.mark.parametrize("m", [0.0, 1.0, 300.0])
def test_S1_delta_source_moments_exact(oracle, m):
    """the deposited source reproduces the injected number and energy exactly; it sits on the two
    neighbours of p0, with the whole weight on a grid point when p0 hits one; the fractions are linear in ENERGY."""
    p = kin.log_grid(64, 1e-3, 1e2)
    dp = kin.trapezoid_widths(p)
    E, K, h = oracle.kinematics(p, dp, m)
    for p0 in (p[0], 0.5 * (p[10] + p[11]), p[30] * 1.0000001, 7.3, p[-1]):
        G = oracle.delta_source(p, dp, m, p0)
        E0 = np.sqrt(p0 * p0 + m * m)
        assert abs((h * G).sum() - 1.0) <= 1e-14
        assert abs((h * E * G).sum() - E0) <= 1e-13 * E0
        nz = np.nonzero(G)[0]
        assert 1 <= nz.size <= 2 and (nz.size == 1 or nz[1] == nz[0] + 1)
        assert p[nz[0]] <= p0 <= p[min(nz[0] + 1, p.size - 1)]
        assert (G >= 0).all()
    G = oracle.delta_source(p, dp, m, p[17])
    assert np.count_nonzero(G) == 1 and G[17] == 1.0 / h[17]
    # not linear in momentum: at the momentum midpoint the right fraction differs from 1/2 for a massive species
    if m == 1.0:
        j = 40
        G = oracle.delta_source(p, dp, m, 0.5 * (p[j] + p[j + 1]))
        assert abs(h[j + 1] * G[j + 1] - 0.5) > 1e-3


# ------------------------------------------------------------------ numerical angular kernel (8(f) item 3)
@pytest.mark.parametrize("cfg,N", [(1, None), (3, 40)])
def test_K1_numerical_kernel_converges_to_analytic(oracle, cfg, N):
    """for |M|^2 = const (and for the t-channel form of D5) the mu-quadrature of eq. B.5-B.12 reproduces
    the analytic kernel; the tables built with n_mu nodes approach the analytic ones like 1/n_mu (kinks of the integrand),
    and so does the operator.  The index map is the same."""
    c = kin.config(cfg, N=N, B=1)
    T0 = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T0, c["f"], oracle.LOG)
    devW, devC = [], []
    for n_mu in (64, 512, 4096):
        T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"], n_mu=n_mu)
        assert np.array_equal(T.jL, T0.jL) and np.array_equal(T.wR, T0.wR)
        devW.append(np.abs(T.W - T0.W).max() / np.abs(T0.W).max())
        g, l, C = oracle.collide(T, c["f"], oracle.LOG)
        devC.append(np.abs(C - C0).max() / np.abs(g0).max())
    assert devW[0] < 0.15 and devW[2] < 2e-3 and devW[0] > 3 * devW[1] > 9 * devW[2]
    assert devC[2] < 2e-4 and devC[0] > 3 * devC[2]


# ------------------------------------------------------------------ non-autonomous integrators: stage times of rate[] and mass[]
def test_E1_rate_stage_indexing_by_reparametrisation(oracle):
    """eq. 4.9: df/dtau = R(tau) C[f].  With R = e^{a tau} the substitution s = (e^{a tau} - 1)/a makes the
    problem autonomous, df/ds = C[f]: the run with rate[] sampled at nodes and midpoints must converge to the static-rate
    solution at s(T) with the order of the method (1/2/4).  Handing stages 2-3 of RK4 the node value, or Heun's second
    stage the start value, makes the scheme first order and fails the order and the magnitude checks."""
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    g, l, C = oracle.collide(T, c["f"], 0)
    s_end = 8.0 / (l[0] / c["f"][0]).max()
    a = 4.0 / s_end                               # R grows from 1 to 5 over the run
    t_end = math.log(5.0) / a
    ref = oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=oracle.RK4, tau=np.linspace(0.0, s_end, 513))
    scale = np.abs(ref).max()

    def run(method, S):
        tau = np.linspace(0.0, t_end, S + 1)
        th = np.empty(2 * S + 1)
        th[0::2] = tau
        th[1::2] = 0.5 * (tau[:-1] + tau[1:])
        return oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=method, tau=tau, rate=np.exp(a * th))

    for method, order, tol16 in ((oracle.EULER, 1, 1e-1), (oracle.HEUN, 2, 2e-2), (oracle.RK4, 4, 1e-4)):
        e1 = np.abs(run(method, 16) - ref).max() / scale
        e2 = np.abs(run(method, 32) - ref).max() / scale
        assert e1 / e2 > 0.7 * 2 ** order, (method, e1, e2)
        assert e1 < tol16, (method, e1)


def test_E2_stage_times_against_textbook_tableaux(oracle):
    """The arrays rate[2S+1], mass[2S+1] hold nodes and midpoints (eq. 4.9).  Independent check of which
    entry each stage reads: generic one-step methods for y' = F(t, y) written from their Butcher tableaux (Euler c=(0);
    Heun c=(0,1), b=(1/2,1/2); classical RK4 c=(0,1/2,1/2,1), b=(1/6,1/3,1/3,1/6)) with F(t, y) = kappa R(t) C_proj[y; m(t)]
    + amp G evaluated through FUNCTIONS of t, against okx_evolve fed the sampled arrays.  R and m take different values
    at every node and midpoint, so any mix-up of the positions changes the result at O(1)."""
    N, B, S = 24, 2, 3
    p = kin.log_grid(N, 2e-2, 20.0)
    dp = kin.trapezoid_widths(p)
    f0 = np.stack([kin._random_bimodal(p, 77 + b) for b in range(B)])
    kappa = np.array([1.0, 0.3])
    G = np.exp(-0.5 * (p - 2.0) ** 2)[None, :]
    tau = np.array([0.0, 0.7, 1.1, 2.0])
    Rfun = lambda t: 40.0 * math.exp(0.9 * t)
    mfun = lambda t: 0.5 * math.exp(0.6 * t)
    amp = np.array([[0.02, 0.0, 0.05]])
    th = np.empty(2 * S + 1)
    th[0::2] = tau
    th[1::2] = 0.5 * (tau[:-1] + tau[1:])
    rate = np.array([Rfun(t) for t in th])
    mass = np.array([mfun(t) for t in th])

    def F(t, y, k):
        T = oracle.Tables(p, dp, mfun(t))
        g, l, C = oracle.collide(T, y, oracle.LOG)
        Cp, _ = oracle.project(T, y, C)
        return kappa[:, None] * Rfun(t) * Cp + amp[0, k] * G

    tableaux = {oracle.EULER: ([0.0], [[]], [1.0]),
                oracle.HEUN: ([0.0, 1.0], [[], [1.0]], [0.5, 0.5]),
                oracle.RK4: ([0.0, 0.5, 0.5, 1.0], [[], [0.5], [0.0, 0.5], [0.0, 0.0, 1.0]], [1 / 6, 1 / 3, 1 / 3, 1 / 6])}
    for method, (cs, As, bs) in tableaux.items():
        y = f0.copy()
        for k in range(S):
            hstep = tau[k + 1] - tau[k]
            ks = []
            for cst, arow in zip(cs, As):
                yst = y + hstep * sum((aij * kj for aij, kj in zip(arow, ks)), np.zeros_like(y))
                ks.append(F(tau[k] + cst * hstep, yst, k))
            y = y + hstep * sum(bj * kj for bj, kj in zip(bs, ks))
        got = oracle.evolve(p, dp, f0, m=mfun(0.0), method=method, tau=tau, rate=rate, mass=mass, kappa=kappa,
                            G=G, amp=amp)
        assert np.abs(got - y).max() <= 1e-12 * np.abs(y).max(), method
        # teeth: the same arrays shifted by one position (midpoint <-> node) give a different answer
        bad = oracle.evolve(p, dp, f0, m=mfun(0.0), method=method, tau=tau, rate=np.roll(rate, 1), mass=mass, kappa=kappa,
                            G=G, amp=amp)
        assert np.abs(bad - y).max() > 1e-4 * np.abs(y).max()


def test_A3_adaptive_rate_slope_by_reparametrisation(oracle):
    """okx_evolve_adaptive's R(u) = rate0 e^{slope (u - u0)} (eq. 4.9 with 1/H a power of a): s = rate0 (e^{slope (u-u0)} - 1)
    / slope makes the problem autonomous, so the adaptive solution must approach the static-rate fine RK4 solution at s(u1)
    with an error proportional to rtol (Heun with R taken at u and u + du is second order; R taken at u for both stages is
    first order: error ~ sqrt(rtol) and far above the bound)."""
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    g, l, C = oracle.collide(T, c["f"], oracle.LOG)
    nu = float((l[0] / c["f"][0]).max())
    s_end = 12.0 / nu
    u0, u1, rate0 = -1.0, 1.0, 0.5
    slope = math.log(9.0) / (u1 - u0)                       # R grows ninefold
    rate0 = s_end * slope / (math.exp(slope * (u1 - u0)) - 1.0)
    ref = oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], method=oracle.RK4, tau=np.linspace(0.0, s_end, 1501))
    errs = []
    for rtol in (1e-4, 1e-5):
        f, info = oracle.evolve_adaptive(c["p"], c["dp"], c["f"], u0=u0, u1=u1, du0=1e-4, rtol=rtol, atol=rtol * 1e-9,
                                         rate0=rate0, rate_slope=slope)
        assert info["done"]
        errs.append(np.abs(f - ref).max() / np.abs(ref).max())
    assert errs[0] < 2e-4 and errs[1] < 2e-5, errs
    assert errs[0] / errs[1] > 5.0, errs


def test_A4_adaptive_mass_slope_against_fixed_step_reference(oracle):
    """okx_evolve_adaptive's kinematic mass m(u) = m e^{mass_slope (u - u0)} (comoving momenta: the kinematics see m a,
    PAPER.md:166).  Independent reference: the fixed-step RK4 integrator fed the sampled arrays mass[2S+1] (whose stage
    positions are pinned by E2) on a fine grid.  The adaptive solution approaches it with an error proportional to rtol;
    taking the mass at u for both Heun stages would be first order (error ~ sqrt(rtol)), and ignoring the slope is off at
    O(1)."""
    N = 24
    p = kin.log_grid(N, 2e-2, 20.0)
    dp = kin.trapezoid_widths(p)
    f0 = kin._random_bimodal(p, 91)[None, :]
    m0, slope = 0.4, 1.0
    T = oracle.Tables(p, dp, m0)
    g, l, C = oracle.collide(T, f0, oracle.LOG)
    nu = float((l[0] / f0[0]).max())
    u0, u1 = 0.0, 1.2                                     # the mass grows by e^1.2 = 3.3
    rate0 = 6.0 / nu / (u1 - u0)
    S = 600
    tau = np.linspace(u0, u1, S + 1)
    th = np.empty(2 * S + 1)
    th[0::2] = tau
    th[1::2] = 0.5 * (tau[:-1] + tau[1:])
    ref = oracle.evolve(p, dp, f0, m=m0, method=oracle.RK4, tau=tau, rate=np.full(2 * S + 1, rate0),
                        mass=m0 * np.exp(slope * (th - u0)))
    scale = np.abs(ref).max()
    errs = []
    for rtol in (1e-4, 1e-5):
        f, info = oracle.evolve_adaptive(p, dp, f0, m=m0, u0=u0, u1=u1, du0=1e-4, rtol=rtol, atol=rtol * 1e-9, rate0=rate0,
                                         mass_slope=slope)
        assert info["done"]
        errs.append(np.abs(f - ref).max() / scale)
    assert errs[0] < 3e-4 and errs[1] < 3e-5, errs
    assert errs[0] / errs[1] > 5.0, errs
    f_static, _ = oracle.evolve_adaptive(p, dp, f0, m=m0, u0=u0, u1=u1, du0=1e-4, rtol=1e-5, atol=1e-14, rate0=rate0)
    assert np.abs(f_static - ref).max() / scale > 1e-3


def test_R1_regime_switch_closed_form(oracle):
    """The Gamma_2->2/H switch of Sec. 4.2 (reading D16) where it has a closed form: before the switch f(u) = (u - u0) S
    with S = sum_s amp_s G_s (f0 = 0, sources only), the LOG-interpolated loss is homogeneous of degree two in f, so
        Gamma/H (u) = kappa R(u) (u - u0) nu_bar[S],   nu_bar[S] = sum h loss[S] / sum h S
    with one oracle.collide of S.  The whole batch switches at the first fixed step boundary where the LARGEST member ratio
    exceeds eps_switch; the monitor sees R(u) at the boundary."""
    c = kin.config(1)
    p, dp = c["p"], c["dp"]
    G = np.stack([np.exp(-0.5 * (p - 3.0) ** 2), np.exp(-0.5 * ((p - 6.0) / 2.0) ** 2)])
    amp = np.array([0.3, 0.05])
    Ssrc = (amp[:, None] * G).sum(axis=0)[None, :]
    T = oracle.Tables(p, dp, c["m"])
    g, l, C = oracle.collide(T, Ssrc, oracle.LOG)
    nubar = float((T.h * l[0]).sum() / (T.h * Ssrc[0]).sum())
    u0, u1, duf, eps = 0.5, 3.0, 0.05, 1e-2
    kappa = np.array([0.2, 1.0, 0.05])
    slope = 0.8
    rate0 = eps / (kappa.max() * nubar * 1.02)            # the largest member crosses eps near u - u0 = 0.6
    ks = np.arange(1, 60)
    ratio = kappa.max() * rate0 * np.exp(slope * ks * duf) * (ks * duf) * nubar
    k_star = int(ks[np.argmax(ratio > eps)])
    assert 5 < k_star < 40
    f0 = np.zeros((3, p.size))
    f, info = oracle.evolve_regimes(p, dp, f0, m=c["m"], u0=u0, u1=u1, du_fixed=duf, eps_switch=eps, du0=1e-3, rtol=1e-3,
                                    atol=1e-12, rate0=rate0, rate_slope=slope, kappa=kappa, G=G, amp=amp, max_steps=1)
    assert info["fixed_steps"] == k_star
    assert abs(info["u_switch"] - (u0 + k_star * duf)) <= 1e-12
    assert info["ratio"] == pytest.approx(float(ratio[k_star - 1]), rel=1e-10)
    # teeth: a rule based on the smallest member, or a monitor without R(u), switches at another step
    k_min = int(ks[np.argmax(kappa.min() * rate0 * np.exp(slope * ks * duf) * (ks * duf) * nubar > eps)]) if \
        (kappa.min() * rate0 * np.exp(slope * ks * duf) * (ks * duf) * nubar > eps).any() else 10 ** 9
    k_noR = int(ks[np.argmax(kappa.max() * rate0 * (ks * duf) * nubar > eps)])
    assert k_min != k_star and k_noR != k_star
    # never switching: sources only to the end, f = (u1 - u0) S exactly, no Heun step taken
    f2, info2 = oracle.evolve_regimes(p, dp, f0, m=c["m"], u0=u0, u1=u1, du_fixed=duf, eps_switch=1e30, rate0=rate0,
                                      rate_slope=slope, kappa=kappa, G=G, amp=amp)
    assert info2["done"] and info2["accepted"] == 0 and info2["u_switch"] == u1
    assert np.abs(f2 - (u1 - u0) * Ssrc).max() <= 1e-13 * np.abs(Ssrc).max() * (u1 - u0)


def test_R2_regimes_compose(oracle):
    """After the switch the run IS the adaptive Heun integration started from the switch state: regimes(u0 -> u1) equals
    sources-only to u_switch followed by okx_evolve_adaptive(u_switch -> u1) with the rate and the mass continued
    (rate0' = R(u_switch), m' = m(u_switch)); eps_switch <= 0 is plain adaptive Heun from u0.  With a mass slope the monitor
    uses the kinematics of m(u) (the monitored ratio moves when the slope is ignored)."""
    N = 24
    p = kin.log_grid(N, 2e-2, 20.0)
    dp = kin.trapezoid_widths(p)
    G = np.exp(-0.5 * ((p - 2.0) / 0.7) ** 2)[None, :]
    amp = np.array([0.4])
    m0, mslope, rslope = 0.3, 1.0, 0.5
    u0, u1, duf = 0.0, 1.5, 0.1
    f0 = np.zeros((2, N))
    kappa = np.array([1.0, 0.3])
    T = oracle.Tables(p, dp, m0)
    g, l, C = oracle.collide(T, amp[0] * G, oracle.LOG)
    nubar = float((T.h * l[0]).sum() / (T.h * amp[0] * G[0]).sum())
    rate0 = 1e-2 / (nubar * 0.45)
    kw = dict(du0=1e-3, rtol=1e-4, atol=1e-13, kappa=kappa, G=G, amp=amp)
    f, info = oracle.evolve_regimes(p, dp, f0, m=m0, u0=u0, u1=u1, du_fixed=duf, eps_switch=1e-2, rate0=rate0,
                                    rate_slope=rslope, mass_slope=mslope, **kw)
    assert info["done"] and 1 <= info["fixed_steps"] < 14 and info["accepted"] > 3
    us = info["u_switch"]
    start = f0 + (us - u0) * amp[0] * G
    f2, info2 = oracle.evolve_adaptive(p, dp, start, m=m0 * math.exp(mslope * (us - u0)), u0=us, u1=u1,
                                       rate0=rate0 * math.exp(rslope * (us - u0)), rate_slope=rslope, mass_slope=mslope, **kw)
    assert info2["accepted"] == info["accepted"] and info2["rejected"] == info["rejected"]
    assert np.abs(f - f2).max() <= 1e-12 * np.abs(f2).max()
    f3, info3 = oracle.evolve_regimes(p, dp, start, m=m0, u0=u0, u1=u1, du_fixed=duf, eps_switch=0.0, rate0=rate0,
                                      rate_slope=rslope, mass_slope=mslope, **kw)
    f4, info4 = oracle.evolve_adaptive(p, dp, start, m=m0, u0=u0, u1=u1, rate0=rate0, rate_slope=rslope, mass_slope=mslope, **kw)
    assert info3["fixed_steps"] == 0 and info3["accepted"] == info4["accepted"] and np.array_equal(f3, f4)
    _, info5 = oracle.evolve_regimes(p, dp, f0, m=m0, u0=u0, u1=u1, du_fixed=duf, eps_switch=1e-2, rate0=rate0,
                                     rate_slope=rslope, mass_slope=0.0, **kw)
    assert info5["fixed_steps"] != info["fixed_steps"] or abs(info5["ratio"] / info["ratio"] - 1.0) > 1e-2
