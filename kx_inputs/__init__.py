"""Seeded synthetic input generators shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no kinematics, no kernel tensor, no
interpolation, no moments): only momentum grids, bin widths, seeded input distributions
and the schedule arrays of the five BASELINE.json configs.  Both `oracle/` (through the
tests) and `paper_2607_00755_b200/` (through the tests and `bench.py`) receive the arrays
produced here as plain inputs.

The inputs stand in for the paper's workloads: two-bump distributions on grids spanning
3-5 decades (eq. 5.1-5.2; N=64...512).  No public dataset
is involved.  Recipes: DESIGN.md "Input recipe", SURVEY.md section 8(d).
"""
from __future__ import annotations

import math
import numpy as np

__all__ = [
    "uniform_grid", "log_grid", "trapezoid_widths", "bimodal", "two_bump_eq51",
    "config", "config5_schedule", "CONFIG_NAMES",
]


# ----------------------------------------------------------------------------- grids
def uniform_grid(n: int, lo: float, hi: float) -> np.ndarray:
    """n points uniformly spaced on [lo, hi] (both ends included)."""
    return np.linspace(float(lo), float(hi), int(n), dtype=np.float64)


def log_grid(n: int, lo: float, hi: float) -> np.ndarray:
    """n points log-spaced on [lo, hi] (PAPER.md:190 'logarithmic grid', eq. 4.5)."""
    return np.exp(np.linspace(math.log(lo), math.log(hi), int(n), dtype=np.float64))


def trapezoid_widths(p: np.ndarray) -> np.ndarray:
    """Reading D1 (paper never defines Delta p_i): trapezoid node widths.

    dp_0=(p_1-p_0)/2, dp_{N-1}=(p_{N-1}-p_{N-2})/2, interior (p_{i+1}-p_{i-1})/2.
    """
    p = np.asarray(p, dtype=np.float64)
    dp = np.empty_like(p)
    dp[0] = 0.5 * (p[1] - p[0])
    dp[-1] = 0.5 * (p[-1] - p[-2])
    dp[1:-1] = 0.5 * (p[2:] - p[:-2])
    return dp


# ----------------------------------------------------------------------------- distributions
def bimodal(p: np.ndarray, c, s, w=(0.6, 0.4)) -> np.ndarray:
    """0.6*exp(-(p-c1)^2/2s1^2) + 0.4*exp(-(p-c2)^2/2s2^2), Gaussian in p (BASELINE.json configs)."""
    p = np.asarray(p, dtype=np.float64)
    return (w[0] * np.exp(-((p - c[0]) ** 2) / (2.0 * s[0] ** 2))
            + w[1] * np.exp(-((p - c[1]) ** 2) / (2.0 * s[1] ** 2)))


def two_bump_eq51(q: np.ndarray) -> np.ndarray:
    """The paper's validation input, eq. 5.1."""
    q = np.asarray(q, dtype=np.float64)
    return (np.exp(-(np.log(q / 0.3)) ** 2 / (2 * 0.18 ** 2))
            + 0.5 * np.exp(-(np.log(q / 8.0)) ** 2 / (2 * 0.22 ** 2)))


def _random_bimodal(p: np.ndarray, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    c = rng.uniform(0.5, 8.0, size=2)
    s = rng.uniform(0.2, 1.5, size=2)
    return bimodal(p, c, s)


# ----------------------------------------------------------------------------- configs
CONFIG_NAMES = {
    1: "cfg1_N32_B1_contact",
    2: "cfg2_N128_B1_contact",
    3: "cfg3_N256_B64_mediator",
    4: "cfg4_N512_contact",
    5: "cfg5_N256_B8_freezein",
}


def config(k: int, *, B: int | None = None, N: int | None = None) -> dict:
    """Inputs of BASELINE.json config k (1..5).  `B`/`N` override the batch / grid size
    (used for reduced parity copies).  Returns a dict of plain numpy arrays and floats:
    p, dp, m, g_chi, M2_0, m_med (<=0: contact), f[B,N], name.
    """
    if k == 1:
        n = N or 32
        p = uniform_grid(n, 0.05, 10.0)
        rng = np.random.default_rng(1001)
        f = bimodal(p, (1.0, 5.0), (0.3, 1.0)) * (1.0 + 0.01 * rng.uniform(-1.0, 1.0, size=n))
        f = f[None, :]
        m_med = 0.0
    elif k == 2:
        n = N or 128
        p = uniform_grid(n, 0.02, 20.0)
        f = _random_bimodal(p, 2001)[None, :]
        m_med = 0.0
    elif k == 3:
        n = N or 256
        nb = B or 64
        p = log_grid(n, 1e-3, 50.0)
        f = np.stack([_random_bimodal(p, 3000 + b) for b in range(nb)])
        m_med = 0.5
    elif k == 4:
        n = N or 512
        nb = B or 8
        p = log_grid(n, 1e-3, 100.0)
        f = np.stack([_random_bimodal(p, 4000 + b) for b in range(nb)])
        m_med = 0.0
    elif k == 5:
        n = N or 256
        nb = B or 8
        p = log_grid(n, 1e-3, 100.0)          # q = p/T, range proposed in SURVEY 8(d) / D11
        f = np.zeros((nb, n), dtype=np.float64)
        m_med = 0.0
    else:
        raise ValueError("config must be 1..5")
    if B is not None and k in (1, 2):
        f = np.repeat(f, B, axis=0)
    return dict(name=CONFIG_NAMES[k], p=p, dp=trapezoid_widths(p), m=1.0, g_chi=1.0,
                M2_0=1.0, m_med=m_med, f=np.ascontiguousarray(f, dtype=np.float64))


def config5_schedule(p: np.ndarray, w: np.ndarray, *, B: int = 8, S: int = 10_000) -> dict:
    """Schedule arrays of config 5 (reading D11; every constant is a stated proposal).

    u = ln x from x=1e-2 to 1e3 in S steps; kinematic mass m(u)=x; rate = R1*x with
    R1 = 128 pi^3 (radiation domination, H ~ x^-2, in the kernel's units); two Gaussian
    sources in q, centres (3, 30), widths (1, 3), each scaled so that sum_i w_i G_i = 1 for the
    weights w the caller hands in (the callers pass w_i = q_i^2 dq_i: unit injected number per unit
    amplitude; the generator itself holds none of the method's arithmetic);
    source 1 active while x<1, source 2 while 10<x<100, each adding 1e-3*G per step;
    kappa_b log-spaced 1e-4..1e2.
    """
    x0, x1 = 1e-2, 1e3
    u = np.linspace(math.log(x0), math.log(x1), S + 1)
    du = (u[-1] - u[0]) / S
    uh = np.empty(2 * S + 1)
    uh[0::2] = u
    uh[1::2] = 0.5 * (u[:-1] + u[1:])
    x = np.exp(uh)
    R1 = 128.0 * math.pi ** 3
    G = np.stack([np.exp(-((p - 3.0) ** 2) / (2 * 1.0 ** 2)),
                  np.exp(-((p - 30.0) ** 2) / (2 * 3.0 ** 2))])
    G /= (G * np.asarray(w, dtype=np.float64)).sum(axis=1, keepdims=True)
    xs = np.exp(u[:-1])                       # x at the start of each step
    amp = np.zeros((2, S))
    amp[0, xs < 1.0 - 1e-12] = 1e-3 / du
    amp[1, (xs >= 10.0 - 1e-9) & (xs < 100.0 - 1e-9)] = 1e-3 / du
    kappa = 10.0 ** (-4.0 + 6.0 * np.arange(B) / max(B - 1, 1))
    return dict(tau=u, rate=R1 * x, mass=x, kappa=kappa, G=np.ascontiguousarray(G),
                amp=np.ascontiguousarray(amp), S=S, du=du)
