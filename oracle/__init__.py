"""CPU oracle of the KineticXGPU collision operator -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this package.  It shares no code with `paper_2607_00755_b200/` and never
imports it.  The arithmetic lives in `kx_oracle.c` (plain C, literal loops in the paper's
notation); this file only compiles it with gcc and marshals numpy arrays through ctypes.

Steps and citations: see the header of `kx_oracle.c` (eq. 4.4,
4.6, 4.7, B.15-B.20, C.1-C.9).  Pins: tests/test_oracle_pins.py.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "kx_oracle.c")
_LIB = os.path.join(_HERE, "libokx.so")
_lib = None

_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)


def build(force: bool = False) -> str:
    """Compile kx_oracle.c -> libokx.so (gcc -O2 -ffp-contract=off -fopenmp)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        build()
        _lib = C.CDLL(_LIB)
        _lib.okx_kinematics.argtypes = [C.c_int, _dp, _dp, C.c_double, _dp, _dp, _dp]
        _lib.okx_kinematics.restype = None
        _lib.okx_build.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_double, C.c_double, C.c_double,
                                   _dp, _ip, _dp]
        _lib.okx_build.restype = C.c_long
        _lib.okx_collide.argtypes = [C.c_int, C.c_int, _dp, _dp, _ip, _dp, C.c_int, C.c_double,
                                     _dp, _dp, _dp]
        _lib.okx_collide.restype = None
        _lib.okx_collide_q.argtypes = [C.c_int, C.c_int, _dp, _dp, _ip, _dp, C.c_int, C.c_double, _dp, _dp, _dp]
        _lib.okx_collide_q.restype = None
        _lib.okx_evolve_q.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp, C.c_double, C.c_double, C.c_double,
                                      C.c_double, C.c_double, C.c_double, _dp, C.c_int, C.c_int, _dp, _dp, _dp, _dp,
                                      C.c_int, C.c_int, _dp, _dp, _dp]
        _lib.okx_evolve_q.restype = C.c_int
        _lib.okx_evolve_adaptive.argtypes = [C.c_int, C.c_int, C.c_int, _dp, _dp] + [C.c_double] * 6 + [_dp] + \
            [C.c_double] * 9 + [_dp, C.c_int, C.c_int, _dp, _dp, C.c_int, _dp]
        _lib.okx_evolve_adaptive.restype = C.c_int
        _lib.okx_evolve_regimes.argtypes = [C.c_int, C.c_int, _dp, _dp] + [C.c_double] * 6 + [_dp] + \
            [C.c_double] * 11 + [_dp, C.c_int, C.c_int, _dp, _dp, C.c_int, _dp]
        _lib.okx_evolve_regimes.restype = C.c_int
        _lib.okx_delta_source.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_double, _dp]
        _lib.okx_delta_source.restype = C.c_int
        _lib.okx_requadrature.argtypes = [C.c_int, _dp, _dp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int,
                                          _dp, _dp, _dp, _ip]
        _lib.okx_requadrature.restype = None
        _lib.okx_collide_rows.argtypes = [C.c_int, C.c_int, _dp, _dp, C.c_double, C.c_double, C.c_double,
                                          C.c_double, _dp, C.c_int, _ip, C.c_int, C.c_double, _dp, _dp, _dp]
        _lib.okx_collide_rows.restype = None
        _lib.okx_project.argtypes = [C.c_int, _dp, _dp, _dp, _dp, _dp, C.c_double, _dp, _dp]
        _lib.okx_project.restype = None
        _lib.okx_moments.argtypes = [C.c_int, _dp, _dp, _dp, _dp, C.c_double, _dp]
        _lib.okx_moments.restype = None
        _lib.okx_evolve.argtypes = [C.c_int, C.c_int, _dp, _dp, C.c_double, C.c_double, C.c_double,
                                    C.c_double, C.c_int, C.c_double, C.c_double, _dp, C.c_int, C.c_int,
                                    _dp, _dp, _dp, _dp, C.c_int, C.c_int, _dp, _dp, _dp]
        _lib.okx_evolve.restype = C.c_int
        _lib.okx_F_quadrature.argtypes = [C.c_double] * 6 + [C.c_int, _dp, _dp]
        _lib.okx_F_quadrature.restype = C.c_double
        _lib.okx_F_closed.argtypes = [C.c_double] * 6
        _lib.okx_F_closed.restype = C.c_double
    return _lib


def _d(a):
    return None if a is None else a.ctypes.data_as(_dp)


def _c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


LOG, LINEAR = 0, 1
EULER, HEUN, RK4 = 0, 1, 2


def kinematics(p, dp, m):
    """O1: returns E, K, h."""
    p, dp = _c(p), _c(dp)
    n = p.size
    E, K, h = np.empty(n), np.empty(n), np.empty(n)
    _load().okx_kinematics(n, _d(p), _d(dp), float(m), _d(E), _d(K), _d(h))
    return E, K, h


class Tables:
    """Dense W[i,n,m], jL[i,n,m] (-1 = dropped), wR[i,n,m] from the quadruple loop (O2-O7)."""

    def __init__(self, p, dp, m=1.0, g_chi=1.0, M2_0=1.0, m_med=0.0, n_mu=0):
        """n_mu > 0: W from the numerical angular kernel (eq. B.5-B.12) with n_mu Gauss-Legendre nodes
        (numpy.polynomial.legendre.leggauss) instead of the analytic kernel of eq. B.17."""
        self.p, self.dp = _c(p), _c(dp)
        self.m, self.g_chi, self.M2_0, self.m_med = float(m), float(g_chi), float(M2_0), float(m_med)
        n = self.N = self.p.size
        self.W = np.empty((n, n, n))
        self.jL = np.empty((n, n, n), dtype=np.int32)
        self.wR = np.empty((n, n, n))
        self.kept = _load().okx_build(n, _d(self.p), _d(self.dp), self.m, self.g_chi, self.M2_0,
                                      self.m_med, _d(self.W), self.jL.ctypes.data_as(_ip), _d(self.wR))
        self.E, self.K, self.h = kinematics(self.p, self.dp, self.m)
        if n_mu:
            mu, wmu = np.polynomial.legendre.leggauss(int(n_mu))
            mu, wmu = _c(mu), _c(wmu)
            _load().okx_requadrature(n, _d(self.p), _d(self.dp), self.m, self.g_chi, self.M2_0, self.m_med, int(n_mu),
                                     _d(mu), _d(wmu), _d(self.W), self.jL.ctypes.data_as(_ip))


def collide(T: Tables, f, interp=LOG, f_floor=1e-300):
    """O8-O9: returns gain, loss, C_raw, each [B,N]."""
    f = _c(np.atleast_2d(f))
    B, n = f.shape
    assert n == T.N
    g, l, c = np.empty((B, n)), np.empty((B, n)), np.empty((B, n))
    _load().okx_collide(n, B, _d(f), _d(T.W), T.jL.ctypes.data_as(_ip), _d(T.wR), int(interp),
                        float(f_floor), _d(g), _d(l), _d(c))
    return g, l, c


def collide_q(T: Tables, f, eta, f_floor=1e-300):
    """Quantum-statistics operator (eq. 4.3 with B.20), eta = +1 Bose / -1 Fermi: returns gain, loss, C_raw [B,N]."""
    assert eta in (1, -1)
    f = _c(np.atleast_2d(f))
    B, n = f.shape
    assert n == T.N
    g, l, c = np.empty((B, n)), np.empty((B, n)), np.empty((B, n))
    _load().okx_collide_q(n, B, _d(f), _d(T.W), T.jL.ctypes.data_as(_ip), _d(T.wR), int(eta), float(f_floor),
                          _d(g), _d(l), _d(c))
    return g, l, c


def collide_rows(p, dp, f, rows, *, m=1.0, g_chi=1.0, M2_0=1.0, m_med=0.0, interp=LOG, f_floor=1e-300):
    """O2-O9 for the selected rows i only (no stored tables): returns gain, loss, C_raw, each [B, len(rows)]."""
    p, dp = _c(p), _c(dp)
    f = _c(np.atleast_2d(f))
    B, n = f.shape
    rows = np.ascontiguousarray(rows, dtype=np.int32)
    g, l, c = np.empty((B, rows.size)), np.empty((B, rows.size)), np.empty((B, rows.size))
    _load().okx_collide_rows(n, B, _d(p), _d(dp), float(m), float(g_chi), float(M2_0), float(m_med), _d(f),
                             rows.size, rows.ctypes.data_as(_ip), int(interp), float(f_floor), _d(g), _d(l), _d(c))
    return g, l, c


def project(T: Tables, f, Craw, eps_supp=1e-12):
    """O10: returns C_proj [B,N] and diag [B,4] = eps_N, eps_E, R_N, R_E."""
    f, Craw = _c(np.atleast_2d(f)), _c(np.atleast_2d(Craw))
    B, n = f.shape
    out, diag = np.empty((B, n)), np.empty((B, 4))
    for b in range(B):
        fb, cb, ob, db = f[b], Craw[b], out[b], diag[b]
        _load().okx_project(n, _d(fb), _d(cb), _d(T.h), _d(T.E), _d(T.K), float(eps_supp), _d(ob), _d(db))
    return out, diag


def moments(T: Tables, f):
    """O11: returns [B,4] = n, rho, <p>, <p^2>."""
    f = _c(np.atleast_2d(f))
    out = np.empty((f.shape[0], 4))
    for b in range(f.shape[0]):
        _load().okx_moments(T.N, _d(f[b]), _d(T.p), _d(T.h), _d(T.E), T.g_chi, _d(out[b]))
    return out


def evolve(p, dp, f, *, m=1.0, g_chi=1.0, M2_0=1.0, m_med=0.0, interp=LOG, f_floor=1e-300,
           eps_supp=1e-12, method=RK4, tau=None, rate=None, mass=None, kappa=None, project=True,
           G=None, amp=None, want_diag=False, eta=0):
    """O12: fixed-step integration; returns f_final [B,N] (and diag [S,B,6] if want_diag).
    eta = +1 / -1 integrates the quantum-statistics operator (collide_q) instead."""
    p, dp = _c(p), _c(dp)
    f = _c(np.atleast_2d(f)).copy()
    B, n = f.shape
    tau = _c(tau)
    S = tau.size - 1
    rate = None if rate is None else _c(rate)
    mass = None if mass is None else _c(mass)
    kappa = None if kappa is None else _c(kappa)
    nsrc = 0 if G is None else int(np.atleast_2d(G).shape[0])
    G = None if G is None else _c(np.atleast_2d(G))
    amp = None if amp is None else _c(np.atleast_2d(amp))
    diag = np.zeros((S, B, 6)) if want_diag else None
    if eta:
        rc = _load().okx_evolve_q(int(eta), n, B, _d(p), _d(dp), float(m), float(g_chi), float(M2_0), float(m_med),
                                  float(f_floor), float(eps_supp), _d(f), int(method), S,
                                  _d(tau), _d(rate), _d(mass), _d(kappa), int(bool(project)), nsrc,
                                  _d(G), _d(amp), _d(diag))
    else:
        rc = _load().okx_evolve(n, B, _d(p), _d(dp), float(m), float(g_chi), float(M2_0), float(m_med),
                                int(interp), float(f_floor), float(eps_supp), _d(f), int(method), S,
                                _d(tau), _d(rate), _d(mass), _d(kappa), int(bool(project)), nsrc,
                                _d(G), _d(amp), _d(diag))
    assert rc == 0
    return (f, diag) if want_diag else f


def evolve_adaptive(p, dp, f, *, u0, u1, du0=1e-4, rtol=1e-2, atol=2e-8, safety=0.9, rate0=1.0, rate_slope=0.0,
                    mass_slope=0.0, m=1.0, g_chi=1.0, M2_0=1.0, m_med=0.0, f_floor=1e-300, eps_supp=1e-12, kappa=None,
                    project=True, G=None, amp=None, max_steps=100000, eta=0):
    """Adaptive Heun of Sec. 4.2 (reading D15): returns f_final [B,N] and dict(u, du, accepted, rejected, done).
    Kinematic mass m(u) = m exp(mass_slope (u - u0))."""
    p, dp = _c(p), _c(dp)
    f = _c(np.atleast_2d(f)).copy()
    B, n = f.shape
    kappa = None if kappa is None else _c(kappa)
    nsrc = 0 if (G is None or amp is None) else int(np.atleast_2d(G).shape[0])
    G = None if nsrc == 0 else _c(np.atleast_2d(G))
    amp = None if nsrc == 0 else _c(np.atleast_1d(amp))
    out = np.zeros(5)
    rc = _load().okx_evolve_adaptive(int(eta), n, B, _d(p), _d(dp), float(m), float(g_chi), float(M2_0), float(m_med),
                                     float(f_floor), float(eps_supp), _d(f), float(u0), float(u1), float(du0),
                                     float(rtol), float(atol), float(safety), float(rate0), float(rate_slope),
                                     float(mass_slope), _d(kappa), int(bool(project)), nsrc, _d(G), _d(amp), int(max_steps),
                                     _d(out))
    assert rc == 0
    return f, dict(u=out[0], du=out[1], accepted=int(out[2]), rejected=int(out[3]), done=bool(out[4]))


def evolve_regimes(p, dp, f, *, u0, u1, du_fixed, eps_switch=1e-2, du0=1e-4, rtol=1e-2, atol=2e-8, safety=0.9, rate0=1.0,
                   rate_slope=0.0, mass_slope=0.0, m=1.0, g_chi=1.0, M2_0=1.0, m_med=0.0, f_floor=1e-300, eps_supp=1e-12,
                   kappa=None, project=True, G=None, amp=None, max_steps=100000):
    """The two regimes of Sec. 4.2 (reading D16): sources only on fixed intervals until Gamma_2->2/H > eps_switch, then
    adaptive Heun.  Returns f_final [B,N] and dict(u, du, accepted, rejected, done, u_switch, fixed_steps, ratio)."""
    p, dp = _c(p), _c(dp)
    f = _c(np.atleast_2d(f)).copy()
    B, n = f.shape
    kappa = None if kappa is None else _c(kappa)
    nsrc = 0 if (G is None or amp is None) else int(np.atleast_2d(G).shape[0])
    G = None if nsrc == 0 else _c(np.atleast_2d(G))
    amp = None if nsrc == 0 else _c(np.atleast_1d(amp))
    out = np.zeros(8)
    rc = _load().okx_evolve_regimes(n, B, _d(p), _d(dp), float(m), float(g_chi), float(M2_0), float(m_med),
                                    float(f_floor), float(eps_supp), _d(f), float(u0), float(u1), float(du_fixed),
                                    float(eps_switch), float(du0), float(rtol), float(atol), float(safety), float(rate0),
                                    float(rate_slope), float(mass_slope), _d(kappa), int(bool(project)), nsrc, _d(G),
                                    _d(amp), int(max_steps), _d(out))
    assert rc == 0
    return f, dict(u=out[0], du=out[1], accepted=int(out[2]), rejected=int(out[3]), done=bool(out[4]),
                   u_switch=out[5], fixed_steps=int(out[6]), ratio=out[7])


def delta_source(p, dp, m, p0):
    """Grid deposition of a monoenergetic source at p0: G [N] with sum h G = 1, sum h E G = E_0."""
    p, dp = _c(p), _c(dp)
    G = np.empty(p.size)
    rc = _load().okx_delta_source(p.size, _d(p), _d(dp), float(m), float(p0), _d(G))
    assert rc == 0, "p0 outside the grid"
    return G


def F_quadrature(pi, pn, pm, m, M2_0, m_med, mu, wmu):
    mu, wmu = _c(mu), _c(wmu)
    return _load().okx_F_quadrature(pi, pn, pm, m, M2_0, m_med, mu.size, _d(mu), _d(wmu))


def F_closed(pi, pn, pm, m, M2_0, m_med):
    return _load().okx_F_closed(pi, pn, pm, m, M2_0, m_med)
