"""kx_evolve_adaptive (adaptive Heun of Sec. 4.2) against the oracle's integrator: the same
accepted / rejected counts, the same final u and f, on the tensor-core path, the streaming path and with Bose statistics."""
import numpy as np
import pytest

import kx_inputs as kin

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return torch


def _dev(torch, a):
    return torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")


def _nu(oracle, T, f):
    g, l, C = oracle.collide(T, f, oracle.LOG)
    return float((l / np.where(f > 0, f, 1.0)).max())


@pytest.mark.parametrize("storage", ["tiled", "rows"])
def test_adaptive_parity_cfg1(torch_cuda, oracle, storage):
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(1)
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    nu = _nu(oracle, T, c["f"])
    kw = dict(u0=0.0, u1=6.0 / nu, du0=2.0 / nu, rtol=1e-3, atol=1e-12)
    f_ref, info_ref = oracle.evolve_adaptive(c["p"], c["dp"], c["f"], **kw)
    assert info_ref["rejected"] >= 1          # the first step is too long: the reject path is exercised
    h = kx.Handle(c["p"], c["dp"], c["m"], storage=kx.STORE_TILED if storage == "tiled" else kx.STORE_SYM_ROWS)
    f = _dev(torch, c["f"])
    info = h.evolve_adaptive(f, **kw)
    assert (info["accepted"], info["rejected"], info["done"]) == (info_ref["accepted"], info_ref["rejected"], True)
    assert abs(info["u"] - info_ref["u"]) <= 1e-12 * abs(info_ref["u"])
    assert abs(info["du"] - info_ref["du"]) <= 1e-8 * abs(info_ref["du"])
    assert np.abs(f.cpu().numpy() - f_ref).max() <= 1e-10 * np.abs(f_ref).max()
    h.close()


def test_adaptive_batch_sources_rate_kappa(torch_cuda, oracle):
    """A batch with per-member couplings, two sources and an exponential rate; one common step for all members."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    B = 5
    c = kin.config(3, N=64, B=B)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    nu = _nu(oracle, T, c["f"])
    G = np.stack([np.exp(-0.5 * (c["p"] - 3.0) ** 2), np.exp(-0.5 * ((c["p"] - 8.0) / 2.0) ** 2)])
    amp = np.array([0.02, 0.01]) * nu
    kappa = np.array([0.0, 0.3, 1.0, 2.0, 0.1])
    kw = dict(u0=0.5, u1=0.5 + 3.0 / nu, du0=0.05 / nu, rtol=1e-2, atol=2e-8, rate0=1.0, rate_slope=0.2 * nu)
    f_ref, info_ref = oracle.evolve_adaptive(c["p"], c["dp"], c["f"], m=c["m"], M2_0=c["M2_0"], m_med=c["m_med"],
                                             kappa=kappa, G=G, amp=amp, **kw)
    h = kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    f = _dev(torch, c["f"])
    info = h.evolve_adaptive(f, kappa=kappa, G=_dev(torch, G), amp=amp, **kw)
    assert (info["accepted"], info["rejected"], info["done"]) == (info_ref["accepted"], info_ref["rejected"], True)
    assert np.abs(f.cpu().numpy() - f_ref).max() <= 1e-10 * np.abs(f_ref).max()
    h.close()


def test_adaptive_bose_and_step_budget(torch_cuda, oracle):
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(1)
    f0 = c["f"] / np.abs(c["f"]).max() * 2.0
    T = oracle.Tables(c["p"], c["dp"], c["m"])
    g, l, C = oracle.collide_q(T, f0, 1)
    nu = float((l[0] / f0[0]).max())
    kw = dict(u0=0.0, u1=4.0 / nu, du0=0.05 / nu, rtol=1e-3, atol=1e-12)
    f_ref, info_ref = oracle.evolve_adaptive(c["p"], c["dp"], f0, eta=1, **kw)
    h = kx.Handle(c["p"], c["dp"], c["m"], statistics=kx.STAT_BOSE)
    f = _dev(torch, f0)
    info = h.evolve_adaptive(f, **kw)
    assert (info["accepted"], info["rejected"]) == (info_ref["accepted"], info_ref["rejected"])
    assert np.abs(f.cpu().numpy() - f_ref).max() <= 1e-10 * np.abs(f_ref).max()
    # a step budget that is too small stops early, says so, and leaves a state the oracle reproduces
    f = _dev(torch, f0)
    info = h.evolve_adaptive(f, max_steps=5, **kw)
    f_ref5, info_ref5 = oracle.evolve_adaptive(c["p"], c["dp"], f0, eta=1, max_steps=5, **kw)
    assert not info["done"] and info["accepted"] + info["rejected"] == 5
    assert abs(info["u"] - info_ref5["u"]) <= 1e-12 * abs(info_ref5["u"])
    assert np.abs(f.cpu().numpy() - f_ref5).max() <= 1e-11 * np.abs(f_ref5).max()
    h.close()


@pytest.mark.parametrize("m", [0.0, 1.0, 300.0])
def test_delta_source_parity_and_injection(torch_cuda, oracle, m):
    """kx_delta_source against the oracle, element by element, also after kx_set_mass; used as a source of
    kx_evolve it injects exactly the prescribed number and energy per step."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    p = kin.log_grid(48, 1e-2, 50.0)
    dp = kin.trapezoid_widths(p)
    h = kx.Handle(p, dp, 2.0)
    h.set_mass(m)
    E, K, hw = oracle.kinematics(p, dp, m)
    for p0 in (p[0], 0.37, p[20], 11.0, p[-1]):
        G = h.delta_source(p0).cpu().numpy()
        G0 = oracle.delta_source(p, dp, m, p0)
        assert np.abs(G - G0).max() <= 1e-13 * np.abs(G0).max()
    with pytest.raises(kx.KxError):
        h.delta_source(2.0 * p[-1])
    # sources only (kappa = 0): 10 Euler steps inject 10 * amp * dtau particles of energy E_0 each
    p0 = 3.3
    G = h.delta_source(p0)
    f = torch.zeros((1, p.size), dtype=torch.float64, device="cuda")
    tau = np.linspace(0.0, 1.0, 11)
    h.evolve(f, tau, method=kx.EULER, kappa=np.zeros(1), G=G[None, :].contiguous(), amp=np.full((1, 10), 0.7), project=False)
    got = f.cpu().numpy()[0]
    assert abs((hw * got).sum() - 0.7) <= 1e-14
    assert abs((hw * E * got).sum() - 0.7 * np.sqrt(p0 * p0 + m * m)) <= 1e-13 * (1.0 + m)
    h.close()


def test_adaptive_mass_slope_parity(torch_cuda, oracle):
    """Adaptive Heun with the kinematic mass m(u) = m e^{u - u0} computed on the device from the controller's u (a1-a3
    rebuilt at every stage): the same accepted / rejected counts and final state as the oracle, and the handle is left with
    the tensor of m(u_final)."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    N, B = 48, 3
    p = kin.log_grid(N, 2e-2, 20.0)
    dp = kin.trapezoid_widths(p)
    f0 = np.stack([kin._random_bimodal(p, 91 + b) for b in range(B)])
    m0 = 0.4
    T = oracle.Tables(p, dp, m0)
    nu = _nu(oracle, T, f0)
    kappa = np.array([1.0, 0.4, 0.0])
    G = np.exp(-0.5 * ((p - 2.0) / 0.7) ** 2)[None, :]
    kw = dict(u0=-0.3, u1=0.6, du0=0.5, rtol=1e-3, atol=1e-12, rate0=5.0 / nu, rate_slope=0.7, mass_slope=1.0, kappa=kappa,
              amp=np.array([0.05]))
    f_ref, info_ref = oracle.evolve_adaptive(p, dp, f0, m=m0, G=G, **kw)
    assert info_ref["rejected"] >= 1 and info_ref["accepted"] >= 5
    for storage in (kx.STORE_TILED, kx.STORE_SYM_ROWS):
        h = kx.Handle(p, dp, m0, storage=storage)
        f = _dev(torch, f0)
        info = h.evolve_adaptive(f, G=_dev(torch, G), **kw)
        assert (info["accepted"], info["rejected"], info["done"]) == (info_ref["accepted"], info_ref["rejected"], True)
        assert abs(info["u"] - info_ref["u"]) <= 1e-12
        assert np.abs(f.cpu().numpy() - f_ref).max() <= 1e-10 * np.abs(f_ref).max()
        # the handle now holds m(u1) = m0 e^{0.9}: a plain collide equals the oracle's for that mass
        T1 = oracle.Tables(p, dp, m0 * np.exp(0.9))
        g1, l1, C1 = oracle.collide(T1, f_ref, oracle.LOG)
        C = h.collide(_dev(torch, f_ref)).cpu().numpy()
        assert (np.abs(C - C1) / np.abs(g1).max(axis=1, keepdims=True)).max() <= 1e-11
        h.close()


@pytest.mark.parametrize("mass_slope", [0.0, 1.0])
def test_two_regimes_parity(torch_cuda, oracle, mass_slope):
    """Sec. 4.2 end to end on the device: sources only on fixed intervals with Gamma_2->2/H monitored by device kernels, the
    switch at the same interval boundary as the oracle, then adaptive Heun with identical accept / reject counts."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    N, B = 40, 3
    p = kin.log_grid(N, 2e-2, 20.0)
    dp = kin.trapezoid_widths(p)
    G = np.stack([np.exp(-0.5 * ((p - 2.0) / 0.7) ** 2), np.exp(-0.5 * ((p - 6.0) / 1.5) ** 2)])
    amp = np.array([0.4, 0.02])
    m0 = 0.3
    T = oracle.Tables(p, dp, m0)
    S = (amp[:, None] * G).sum(axis=0)[None, :]
    g, l, C = oracle.collide(T, S, oracle.LOG)
    nubar = float((T.h * l[0]).sum() / (T.h * S[0]).sum())
    kappa = np.array([1.0, 0.3, 0.05])
    kw = dict(u0=0.0, u1=1.5, du_fixed=0.1, eps_switch=1e-2, du0=1e-3, rtol=1e-3, atol=1e-13, rate0=1e-2 / (nubar * 0.45),
              rate_slope=0.5, mass_slope=mass_slope, kappa=kappa, amp=amp)
    f0 = np.zeros((B, N))
    f_ref, info_ref = oracle.evolve_regimes(p, dp, f0, m=m0, G=G, **kw)
    assert 1 <= info_ref["fixed_steps"] < 14 and info_ref["accepted"] > 3 and info_ref["done"]
    h = kx.Handle(p, dp, m0)
    f = _dev(torch, f0)
    info = h.evolve_adaptive(f, G=_dev(torch, G), **kw)
    assert info["switched"] and info["fixed_steps"] == info_ref["fixed_steps"]
    assert abs(info["u_switch"] - info_ref["u_switch"]) <= 1e-12
    assert abs(info["ratio"] / info_ref["ratio"] - 1.0) <= 1e-10
    assert (info["accepted"], info["rejected"], info["done"]) == (info_ref["accepted"], info_ref["rejected"], True)
    assert np.abs(f.cpu().numpy() - f_ref).max() <= 1e-10 * np.abs(f_ref).max()
    # never switching: sources only to u1, exact
    f2 = _dev(torch, f0)
    info2 = h.evolve_adaptive(f2, G=_dev(torch, G), **{**kw, "eps_switch": 1e30})
    assert info2["done"] and not info2["switched"] and info2["accepted"] == 0 and info2["fixed_steps"] == 15
    assert np.abs(f2.cpu().numpy() - 1.5 * S).max() <= 1e-13 * np.abs(S).max() * 1.5
    h.close()
