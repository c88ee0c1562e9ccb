"""Quantum-statistics operator (eq. 4.3 with B.20) on the GPU against the oracle's literal
Lambda_inm loop: collide, gain/loss parts, projection, a short RK4 evolution, thermal fixed points."""
import numpy as np
import pytest

import kx_inputs as kin

pytestmark = pytest.mark.gpu
TOL = 1e-11


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return torch


def _dev(torch, a):
    return torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")


def _occupied(c, eta):
    """Occupations of order one (where the quantum factors matter); Fermi needs f < 1."""
    f = c["f"] / np.abs(c["f"]).max(axis=1, keepdims=True)
    return f * (0.8 if eta == -1 else 2.5)


@pytest.mark.parametrize("eta", [1, -1])
@pytest.mark.parametrize("cfg,N,B", [(1, None, 1), (3, 88, 11), (4, 72, 3)])
def test_quantum_collide_parity(torch_cuda, oracle, eta, cfg, N, B):
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(cfg, N=N, B=B)
    f = _occupied(c, eta)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide_q(T, f, eta)
    scale = np.abs(g0).max(axis=1, keepdims=True)
    h = kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"], statistics=eta)
    fd = _dev(torch, f)
    g, l = h.collide_parts(fd)
    assert (np.abs(g.cpu().numpy() - g0) / scale).max() <= TOL
    assert (np.abs(l.cpu().numpy() - l0) / scale).max() <= TOL
    assert (np.abs(h.collide(fd).cpu().numpy() - C0) / scale).max() <= TOL
    Cp0, _ = oracle.project(T, f, C0)
    assert (np.abs(h.collide(fd, flags=kx.PROJECT).cpu().numpy() - Cp0) / scale).max() <= TOL
    # the quantum factors are really there
    gc, lc, Cc = oracle.collide(T, f, oracle.LOG)
    assert np.abs(C0 - Cc).max() > 1e-3 * scale.max()
    h.close()


@pytest.mark.parametrize("eta,mu,Tchi", [(1, 0.0, 1.0), (-1, 0.5, 1.0)])
def test_quantum_fixed_point_on_gpu(torch_cuda, eta, mu, Tchi):
    """Fig. 11: N=96, T/m=1, mu=0: the raw operator of an exact Bose-Einstein (Fermi-Dirac)
    distribution is at round-off."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    p = kin.log_grid(96, 1e-3, 1e2)
    dp = kin.trapezoid_widths(p)
    h = kx.Handle(p, dp, 1.0, statistics=eta)
    E = np.sqrt(p * p + 1.0)
    f = 1.0 / (np.exp((E - mu) / Tchi) - eta)
    g, l = h.collide_parts(_dev(torch, f[None, :]))
    C = h.collide(_dev(torch, f[None, :])).cpu().numpy()
    assert np.abs(C).max() <= 1e-12 * np.abs(g.cpu().numpy()).max()
    h.close()


@pytest.mark.parametrize("eta", [1, -1])
def test_quantum_evolve_parity(torch_cuda, oracle, eta):
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(1)
    f0 = _occupied(c, eta)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    g0, l0, C0 = oracle.collide_q(T, f0, eta)
    nu = float((l0[0] / f0[0]).max())
    tau = np.arange(13) * (0.3 / nu)
    f_ref = oracle.evolve(c["p"], c["dp"], f0, m=c["m"], method=oracle.RK4, tau=tau, eta=eta)
    h = kx.Handle(c["p"], c["dp"], c["m"], statistics=eta)
    f = _dev(torch, f0)
    h.evolve(f, tau, method=kx.RK4)
    got = f.cpu().numpy()
    assert np.abs(got - f_ref).max() <= 1e-10 * np.abs(f_ref).max()
    # number and energy are conserved by the projected quantum operator
    m0, m1 = oracle.moments(T, f0), oracle.moments(T, got)
    assert np.allclose(m0[:, :2], m1[:, :2], rtol=1e-11, atol=0)
    h.close()


def test_quantum_rejects_linear_interpolation(torch_cuda):
    import paper_2607_00755_b200 as kx
    c = kin.config(1)
    with pytest.raises(kx.KxError):
        kx.Handle(c["p"], c["dp"], c["m"], statistics=1, interp=kx.INTERP_LINEAR)
    with pytest.raises(kx.KxError):
        kx.Handle(c["p"], c["dp"], c["m"], statistics=2)


@pytest.mark.parametrize("cfg,N,n_mu", [(1, None, 48), (3, 40, 32)])
def test_numerical_angular_kernel_parity(torch_cuda, oracle, cfg, N, n_mu):
    """n_mu > 0: the device builder evaluates F_inm by the Gauss-Legendre quadrature of eq.
    B.5-B.12; entries and operator against the oracle's quadrature tables (its nodes come from numpy, the library's from
    its own Newton iteration), on the streaming and the tensor-core storage."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(cfg, N=N, B=3)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"], n_mu=n_mu)
    n = T.N
    Wsym = T.W + np.transpose(T.W, (0, 2, 1))
    Wsym[:, np.arange(n), np.arange(n)] = T.W[:, np.arange(n), np.arange(n)]
    g0, l0, C0 = oracle.collide(T, c["f"], oracle.LOG)
    scale = np.abs(g0).max(axis=1, keepdims=True)
    for storage in (kx.STORE_SYM_ROWS, kx.STORE_TILED):
        h = kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"], n_mu=n_mu, storage=storage)
        ex = h.tensor_export()
        rowptr, W, nn, mm = ex["rowptr"], ex["W"], ex["n"], ex["m"]
        i_of = np.repeat(np.arange(n), np.diff(rowptr))
        # tolerance: B.11 takes asin at arguments clipped to +-1, where an ulp of the argument moves the result by
        # sqrt(ulp) ~ 1e-8 of a node's weight; measured 4e-10
        assert np.abs(W - Wsym[i_of, nn, mm]).max() <= 1e-8 * np.abs(Wsym).max()
        C = h.collide(_dev(torch, c["f"])).cpu().numpy()
        assert (np.abs(C - C0) / scale).max() <= 1e-8
        h.close()
    # and it is the quadrature, not the analytic kernel
    T0 = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    assert np.abs(T.W - T0.W).max() > 1e-5 * np.abs(T0.W).max()
