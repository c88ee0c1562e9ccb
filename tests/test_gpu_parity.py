"""GPU-vs-oracle parity through the C ABI (libkx) on the seeded inputs of kx_inputs.

Bar (BASELINE.json north_star): max-abs error <= 1e-11 relative to max_i |gain_i| per distribution in fp64;
integer work (which triples are kept, the bracket index j_L) bit-exact.  The oracle (oracle/) is the CPU
reference; nothing here feeds a GPU value back into it.
"""
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


def _handle(c, **kw):
    import paper_2607_00755_b200 as kx
    return kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"], **kw)


def _dev(torch, a):
    return torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")


def _relerr(got, ref, gain):
    """max_i |got-ref| / max_i |gain_i|, per member, worst member."""
    scale = np.abs(gain).max(axis=1, keepdims=True)
    return float((np.abs(got - ref) / scale).max())


# --------------------------------------------------------------------------------------- a1-a3: builder
@pytest.mark.parametrize("cfg,N", [(1, None), (2, 96), (3, 72), (4, 80), (5, 64)])
def test_builder_entry_by_entry(torch_cuda, oracle, cfg, N):
    c = kin.config(cfg, N=N)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    h = _handle(c)
    t = h.tensor_export()
    n_, m_, j_, rp = t["n"], t["m"], t["jL"], t["rowptr"]
    nn = T.N
    i_ = np.repeat(np.arange(nn), np.diff(rp))
    # kinematics
    E, K, hw = h.kinematics_export()
    assert np.array_equal(K, T.K) and np.array_equal(E, T.E) and np.array_equal(hw, T.h)
    # which (i, n<=m) triples are kept: exact
    kept = T.jL >= 0
    iu, nu, mu = np.nonzero(kept & (np.arange(nn)[None, :, None] <= np.arange(nn)[None, None, :]))
    assert len(iu) == len(i_) == h.info()["nnz"]
    assert np.array_equal(i_, iu) and np.array_equal(n_, nu) and np.array_equal(m_, mu)   # same deterministic order
    assert (n_ <= m_).all()
    # bracket index: exact; omega_R and W: rounding level
    assert np.array_equal(j_, T.jL[i_, n_, m_])
    assert np.abs(t["omega"] - T.wR[i_, n_, m_]).max() <= 4e-16
    Wsym = np.where(n_ == m_, T.W[i_, n_, m_], T.W[i_, n_, m_] + T.W[i_, m_, n_])
    rowmax = np.array([Wsym[rp[i]:rp[i + 1]].max() if rp[i + 1] > rp[i] else 1.0 for i in range(nn)])[i_]
    tol = 1e-13 if c["m_med"] <= 0 else 2e-12        # mediator: closed form in double vs long double
    assert (np.abs(t["W"] - Wsym) <= tol * rowmax + 1e-14 * np.abs(Wsym)).all()
    assert np.median(np.abs(t["W"] - Wsym)[Wsym > 0] / Wsym[Wsym > 0]) < 1e-15
    h.close()


# --------------------------------------------------------------------------------------- a4-a6: operator
@pytest.mark.parametrize("cfg,N,B,interp", [
    (1, None, None, 0), (1, None, None, 1),
    (2, None, None, 0), (2, None, None, 1),
    (3, 96, 5, 0), (3, 96, 9, 1), (3, 33, 3, 0),
    (4, 100, 8, 0), (4, 100, 2, 0),
])
def test_collide_parity(torch_cuda, oracle, cfg, N, B, interp):
    torch = torch_cuda
    c = kin.config(cfg, N=N, B=B)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T, c["f"], interp)
    h = _handle(c, interp=interp)
    f = _dev(torch, c["f"])
    g, l = h.collide_parts(f)
    C = h.collide(f)
    assert _relerr(g.cpu().numpy(), g0, g0) <= TOL
    assert _relerr(l.cpu().numpy(), l0, g0) <= TOL
    assert _relerr(C.cpu().numpy(), C0, g0) <= TOL
    # typical error is far below the bar
    assert _relerr(C.cpu().numpy(), C0, g0) <= 2e-13
    h.close()


def test_collide_full_cfg3_all_members(torch_cuda, oracle):
    """BASELINE config 3 at full size (N=256, B=64, mediator |M|^2), every member, in the bench's launch configuration."""
    torch = torch_cuda
    c = kin.config(3)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T, c["f"], 0)
    h = _handle(c)
    f = _dev(torch, c["f"])
    o = h.collide_ex(f, flags=0, want=("C", "gain", "loss"))
    assert _relerr(o["gain"].cpu().numpy(), g0, g0) <= TOL
    assert _relerr(o["loss"].cpu().numpy(), l0, g0) <= TOL
    assert _relerr(o["C"].cpu().numpy(), C0, g0) <= TOL
    # projected
    Cp0, d0 = oracle.project(T, c["f"], C0)
    o = h.collide_ex(f, flags=1, want=("C", "diag"))
    assert _relerr(o["C"].cpu().numpy(), Cp0, g0) <= TOL
    assert np.allclose(o["diag"].cpu().numpy(), d0, rtol=1e-9, atol=1e-13)
    # library exp2 gives the same operator
    h2 = _handle(c, exp_impl=1)
    assert _relerr(h2.collide(f).cpu().numpy(), C0, g0) <= TOL
    h.close(); h2.close()


@pytest.mark.parametrize("B", [1, 8])
def test_collide_cfg4_full_size_sampled_rows(torch_cuda, oracle, B):
    """BASELINE config 4 (N=512): the dense oracle tables are too slow to build, so rows are sampled one by one."""
    torch = torch_cuda
    c = kin.config(4, B=B)
    rows = np.array([0, 1, 2, 31, 32, 100, 255, 256, 300, 400, 480, 509, 510, 511])
    g0, l0, C0 = oracle.collide_rows(c["p"], c["dp"], c["f"], rows, m=c["m"], M2_0=c["M2_0"], m_med=c["m_med"])
    h = _handle(c)
    f = _dev(torch, c["f"])
    o = h.collide_ex(f, flags=0, want=("C", "gain", "loss"))
    gmax = np.abs(o["gain"].cpu().numpy()).max(axis=1, keepdims=True)
    for key, ref in (("gain", g0), ("loss", l0), ("C", C0)):
        got = o[key].cpu().numpy()[:, rows]
        assert (np.abs(got - ref) / gmax).max() <= TOL, key
    # properties that hold at any size: projected operator has vanishing number and energy moments
    E, K, hw = h.kinematics_export()
    Cp = h.collide(f, flags=1).cpu().numpy()
    Craw = o["C"].cpu().numpy()
    assert (np.abs((hw * Cp).sum(axis=1)) <= 1e-13 * (hw * np.abs(Craw)).sum(axis=1)).all()
    assert (np.abs((hw * E * Cp).sum(axis=1)) <= 1e-13 * (hw * E * np.abs(Craw)).sum(axis=1)).all()
    info = h.info()
    assert 0.6 < info["nnz"] / (512 * 512 * 513 / 2) < 0.7
    h.close()


def test_thermal_fixed_point_on_gpu(torch_cuda):
    """P5 on the device: C_raw[z exp(-E/T)] vanishes term by term under LOG interpolation."""
    torch = torch_cuda
    c = kin.config(3)
    h = _handle(c)
    E, K, hw = h.kinematics_export()
    f = _dev(torch, np.stack([0.37 * np.exp(-E / 0.7), 2.0 * np.exp(-E / 3.0)]))
    o = h.collide_ex(f, want=("C", "gain"))
    assert (o["C"].abs().amax(dim=1) <= 3e-13 * o["gain"].abs().amax(dim=1)).all()
    h.close()


# --------------------------------------------------------------------------------------- edge cases
def test_edge_cases(torch_cuda, oracle):
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    # smallest grid, zeros / floor in f, negative values, ragged batch
    p = kin.uniform_grid(4, 0.5, 2.0)
    dp = kin.trapezoid_widths(p)
    f = np.array([[1.0, 0.5, 0.0, 1e-310], [0.0, 0.0, 0.0, 0.0], [1.0, -0.5, 0.3, 0.2]])
    T = oracle.Tables(p, dp, 0.3)
    h = kx.Handle(p, dp, 0.3)
    for interp in (0, 1):
        hh = kx.Handle(p, dp, 0.3, interp=interp)
        g0, l0, C0 = oracle.collide(T, f, interp)
        C = hh.collide(_dev(torch, f)).cpu().numpy()
        scale = max(np.abs(g0).max(), 1e-300)
        assert np.abs(C - C0).max() <= TOL * scale
        Cp0, d0 = oracle.project(T, f, C0)
        o = hh.collide_ex(_dev(torch, f), flags=1, want=("C", "diag"))
        assert np.abs(o["C"].cpu().numpy() - Cp0).max() <= TOL * scale       # includes the f == 0 member (D9)
        hh.close()
    # error behaviour
    fz = _dev(torch, f)
    with pytest.raises(kx.KxError):
        h.collide(fz, out=fz)                                 # in place
    with pytest.raises(ValueError):
        h.collide(_dev(torch, np.zeros((2, 5))))              # wrong N
    big = torch.zeros(3 * 4 + 1, dtype=torch.float64, device="cuda")
    mis = big[1:].view(3, 4)
    with pytest.raises(kx.KxError):
        h.collide(mis)                                        # misaligned pointer
    for bad in (dict(p=p[::-1].copy(), dp=dp), dict(p=p, dp=-dp), dict(p=p[:3], dp=dp[:3])):
        with pytest.raises(kx.KxError):
            kx.Handle(bad["p"], bad["dp"], 0.3)
    with pytest.raises(kx.KxError):
        kx.Handle(p, dp, 0.3, f_floor=0.0)
    h.close()


def test_host_buffer_call(torch_cuda, oracle):
    torch = torch_cuda
    c = kin.config(3, N=64, B=4)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T, c["f"], 0)
    h = _handle(c)
    fh = torch.tensor(c["f"]).pin_memory()
    Ch = torch.empty_like(fh).pin_memory()
    h.collide_host(fh, Ch)
    assert _relerr(Ch.numpy(), C0, g0) <= TOL
    Cn = np.empty_like(c["f"])
    h.collide_host(c["f"], Cn)                                # pageable numpy buffers work too
    assert np.array_equal(Cn, Ch.numpy())
    h.close()


def test_bitwise_reproducible(torch_cuda):
    torch = torch_cuda
    c = kin.config(3, N=128, B=16)
    h = _handle(c)
    f = _dev(torch, c["f"])
    a = h.collide(f, flags=1).clone()
    for _ in range(3):
        assert torch.equal(h.collide(f, flags=1), a)
    h2 = _handle(c)
    assert torch.equal(h2.collide(f, flags=1), a)
    # a member's result does not depend on its batch neighbours
    assert torch.equal(h.collide(f[3:4].contiguous(), flags=1)[0], a[3])
    h.close(); h2.close()


# --------------------------------------------------------------------------------------- a7, a9
@pytest.mark.parametrize("m", [1.0, 1000.0])
def test_projection_and_moments_parity(torch_cuda, oracle, m):
    torch = torch_cuda
    c = kin.config(5, N=96, B=3)
    p, dp = c["p"], c["dp"]
    f = np.stack([kin.bimodal(p, (3.0, 30.0), (1.0, 3.0)), kin.bimodal(p, (1.0, 8.0), (0.5, 2.0)),
                  kin.two_bump_eq51(p)])
    T = oracle.Tables(p, dp, m)
    g0, l0, C0 = oracle.collide(T, f, 0)
    Cp0, d0 = oracle.project(T, f, C0)
    import paper_2607_00755_b200 as kx
    h = kx.Handle(p, dp, m)
    o = h.collide_ex(_dev(torch, f), flags=1)
    assert _relerr(o["C"].cpu().numpy(), Cp0, g0) <= TOL
    assert np.allclose(o["diag"].cpu().numpy(), d0, rtol=1e-8, atol=1e-13)
    mo = h.moments(_dev(torch, f)).cpu().numpy().T
    assert np.allclose(mo, oracle.moments(T, f), rtol=1e-13, atol=0)
    # kx_set_mass: rebuilding for another mass equals a fresh build
    h.set_mass(2.5)
    T2 = oracle.Tables(p, dp, 2.5)
    g2, l2, C2 = oracle.collide(T2, f, 0)
    assert _relerr(h.collide(_dev(torch, f)).cpu().numpy(), C2, g2) <= TOL
    assert h.info()["nnz"] == int(((T2.jL >= 0) & (np.arange(96)[None, :, None] <= np.arange(96)[None, None, :])).sum())
    h.close()


# --------------------------------------------------------------------------------------- storage modes
@pytest.mark.parametrize("interp", [0, 1])
def test_streaming_storage_parity(torch_cuda, oracle, interp):
    """KX_STORE_SYM_ROWS: the exact streaming kernel alone (one exp per entry and member)."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(3, N=96, B=11)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T, c["f"], interp)
    h = _handle(c, interp=interp, storage=kx.STORE_SYM_ROWS)
    f = _dev(torch, c["f"])
    g, l = h.collide_parts(f)
    assert _relerr(g.cpu().numpy(), g0, g0) <= TOL
    assert _relerr(l.cpu().numpy(), l0, g0) <= TOL
    assert _relerr(h.collide(f).cpu().numpy(), C0, g0) <= 2e-13
    h.close()


@pytest.mark.parametrize("nodes", [8, 16, 24, 32])
def test_tiled_loss_nodes(torch_cuda, oracle, nodes):
    """Every Chebyshev order gives the oracle's operator: brackets the order cannot resolve to 1e-15 max f send
    their member to the streaming kernel (few nodes => many members fall back, the result stays within the bar)."""
    torch = torch_cuda
    c = kin.config(3, N=64, B=20)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T, c["f"], 0)
    h = _handle(c, loss_nodes=nodes)
    f = _dev(torch, c["f"])
    g, l = h.collide_parts(f)
    assert _relerr(g.cpu().numpy(), g0, g0) <= TOL
    assert _relerr(l.cpu().numpy(), l0, g0) <= TOL
    assert _relerr(l.cpu().numpy(), l0, g0) <= 1e-13
    h.close()


def test_tiled_fallback_sharp_features(torch_cuda, oracle):
    """Distributions the Chebyshev-moment loss cannot represent (cut-offs to exact zero, steps of 1e200, a single
    occupied bin) are routed per member to the exact streaming kernel; smooth neighbours stay on the DMMA path."""
    torch = torch_cuda
    c = kin.config(3, N=80, B=6)
    p = c["p"]
    f = c["f"].copy()
    f[1, p > 3.0] = 0.0                                  # sharp cut-off: ln(f_j+1/f_j) ~ -690 in one bracket
    f[2] = np.where((p > 0.5) & (p < 2.0), 1.0, 1e-200)  # step function
    f[3] = 0.0
    f[3, 40] = 2.5                                       # one occupied bin
    f[4] = 1e-250 * c["f"][4]                            # tiny but smooth: no fallback needed, still exact
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T, f, 0)
    h = _handle(c)
    fd = _dev(torch, f)
    g, l = h.collide_parts(fd)
    scale = np.maximum(np.abs(g0).max(axis=1, keepdims=True), 1e-300)
    assert (np.abs(g.cpu().numpy() - g0) / scale).max() <= TOL
    assert (np.abs(l.cpu().numpy() - l0) / scale).max() <= TOL
    Cp0, _ = oracle.project(T, f, C0)
    Cp = h.collide(fd, flags=1).cpu().numpy()
    assert (np.abs(Cp - Cp0) / scale).max() <= TOL
    # the same members in another order and batch size give the same bits (fallback is per member)
    perm = [3, 0, 5, 1]
    assert h.fallback_members() == 6                     # members 1, 2, 3 in each of the two calls above, nobody else
    Cq = h.collide(_dev(torch, f[perm]), flags=1).cpu().numpy()
    assert np.array_equal(Cq, Cp[perm])
    assert h.fallback_members() == 2                     # members 3 and 1 of the permuted batch
    # smooth members only: nobody takes the exact path
    h.collide(_dev(torch, c["f"]), flags=1)
    assert h.fallback_members() == 0
    h.close()


@pytest.mark.parametrize("N,log", [(6, False), (8, False), (12, False), (22, False), (32, True), (33, True), (44, True), (52, True)])
def test_tiled_small_grids_poisoned_workspace(torch_cuda, oracle, monkeypatch, N, log):
    """Grids with fewer gain groups than gain workers, on workspaces filled with NaN patterns (KX_POISON_WS) and after a
    larger handle was created and destroyed in the same process: every partial slot the finishing phase adds must have been
    written by the same launch.  Also across batch sizes on one handle, and bit-equal gain with the streaming storage."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    monkeypatch.setenv("KX_POISON_WS", "1")
    big = kin.config(3, N=96, B=16)
    hb = _handle(big)
    hb.collide(_dev(torch, big["f"]))
    hb.close()
    p = kin.log_grid(N, 1e-2, 20.0) if log else kin.uniform_grid(N, 0.05, 8.0)
    dp = kin.trapezoid_widths(p)
    T = oracle.Tables(p, dp, 1.0)
    h = kx.Handle(p, dp, 1.0, interp=kx.INTERP_LINEAR)
    hs = kx.Handle(p, dp, 1.0, interp=kx.INTERP_LINEAR, storage=kx.STORE_SYM_ROWS)
    for B in (3, 9, 1, 20):
        f = np.stack([kin._random_bimodal(p, 7000 + b) for b in range(B)])
        g0, l0, C0 = oracle.collide(T, f, 1)
        g, l = h.collide_parts(_dev(torch, f))
        assert torch.isfinite(g).all() and torch.isfinite(l).all()
        assert _relerr(g.cpu().numpy(), g0, g0) <= TOL
        assert _relerr(l.cpu().numpy(), l0, g0) <= TOL
        gs, ls = hs.collide_parts(_dev(torch, f))
        assert _relerr(gs.cpu().numpy(), g0, g0) <= TOL
    hl = kx.Handle(p, dp, 1.0)                           # LOG interpolation: the Chebyshev-moment loss on the same grids
    f = np.stack([kin._random_bimodal(p, 7100 + b) for b in range(5)])
    g0, l0, C0 = oracle.collide(T, f, 0)
    assert _relerr(hl.collide(_dev(torch, f)).cpu().numpy(), C0, g0) <= TOL
    h.close(); hs.close(); hl.close()


@pytest.mark.parametrize("B", [1, 7, 8, 9, 17, 33, 64, 65, 130])
def test_tiled_batch_sizes(torch_cuda, oracle, B):
    """Every MMA column-tile configuration (1, 2, 4, 8 tiles; several CTA column groups; ragged tails)."""
    torch = torch_cuda
    c = kin.config(3, N=40, B=B)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T, c["f"], 0)
    h = _handle(c)
    C = h.collide(_dev(torch, c["f"])).cpu().numpy()
    assert _relerr(C, C0, g0) <= 2e-13
    h.close()


def test_back_to_back_calls_are_ordered(torch_cuda):
    """The kernels of one call overlap through programmatic dependent launch and every call reuses the handle's
    workspaces (operand rows, partials, member statistics): calls enqueued back to back without a host sync must
    give the bits of calls run one at a time, also when smooth and flagged (fallback) members alternate."""
    torch = torch_cuda
    c = kin.config(3, N=96, B=24)
    h = _handle(c)
    fa = c["f"].copy()
    fb = c["f"][::-1].copy()
    fb[3, c["p"] > 2.0] = 0.0            # one member that takes the exact streaming path
    fb[10] *= 1e-120
    da, db = _dev(torch, fa), _dev(torch, fb)
    ref_a = h.collide(da, flags=1).clone()
    torch.cuda.synchronize()
    ref_b = h.collide(db, flags=1).clone()
    torch.cuda.synchronize()
    outs = [torch.empty_like(da) for _ in range(6)]
    for rep in range(10):
        for k, o in enumerate(outs):
            h.collide(da if k % 2 == 0 else db, flags=1, out=o)
        torch.cuda.synchronize()
        for k, o in enumerate(outs):
            assert torch.equal(o, ref_a if k % 2 == 0 else ref_b), (rep, k)
    h.close()


def test_collide_max_grid_sampled_rows(torch_cuda, oracle):
    """The ABI's largest grid, N = 1024 (n, m, j_L packed 10 bits each; 2.8 GB tiled operand), B = 3, mediator |M|^2:
    sampled rows against the oracle, conservation of the projected operator, and the packed index limits."""
    torch = torch_cuda
    N, B = 1024, 3
    p = kin.log_grid(N, 1e-3, 100.0)
    dp = kin.trapezoid_widths(p)
    f = np.stack([kin._random_bimodal(p, 9000 + b) for b in range(B)])
    rows = np.array([0, 1, 15, 16, 255, 256, 511, 777, 1008, 1022, 1023])
    g0, l0, C0 = oracle.collide_rows(p, dp, f, rows, m=1.0, M2_0=1.0, m_med=0.5)
    c = dict(p=p, dp=dp, m=1.0, g_chi=1.0, M2_0=1.0, m_med=0.5)
    h = _handle(c)
    fd = _dev(torch, f)
    o = h.collide_ex(fd, flags=0, want=("C", "gain", "loss"))
    gmax = np.abs(o["gain"].cpu().numpy()).max(axis=1, keepdims=True)
    for key, ref in (("gain", g0), ("loss", l0), ("C", C0)):
        assert (np.abs(o[key].cpu().numpy()[:, rows] - ref) / gmax).max() <= TOL, key
    E, K, hw = h.kinematics_export()
    Cp = h.collide(fd, flags=1).cpu().numpy()
    Craw = o["C"].cpu().numpy()
    assert (np.abs((hw * Cp).sum(axis=1)) <= 1e-13 * (hw * np.abs(Craw)).sum(axis=1)).all()
    assert (np.abs((hw * E * Cp).sum(axis=1)) <= 1e-13 * (hw * E * np.abs(Craw)).sum(axis=1)).all()
    h.close()


# --------------------------------------------------------------------------------------- eq. 5.1 validation workload
def test_two_bump_eq51_workload(torch_cuda, oracle):
    """SURVEY.md 8(f) item 4, second half: the paper's validation input (eq. 5.1-5.2; m = lambda = a = 1,
    log grid q in [1e-3, 1e2], analytical kernel) at N = 96, 128, 256.  C_raw, C_proj and the diagnostics eps_N, eps_E
    (C.1), R_N, R_E (C.9) from kx_collide_ex against the oracle; the Fig. 9-10 trends on the GPU values: the conservation
    residuals and the largest pointwise projection correction fall like N^-2, the latter in the range the paper prints
    (1.19 % at N=96, 0.16 % at N=256; soft, as in pin P10: the paper's run had Bose factors on)."""
    torch = torch_cuda
    import os
    import paper_2607_00755_b200 as kx
    here = os.path.dirname(os.path.abspath(__file__))
    rows = [ln.split() for ln in open(os.path.join(here, "golden", "paper_projection_correction.txt"))
            if ln.strip() and not ln.startswith("#")]
    paper = {int(r[0]): float(r[1]) for r in rows}
    corr, epsN, epsE = {}, {}, {}
    for N in (96, 128, 256):
        p = kin.log_grid(N, 1e-3, 1e2)
        dp = kin.trapezoid_widths(p)
        f = kin.two_bump_eq51(p)[None, :]
        T = oracle.Tables(p, dp, 1.0)
        g0, l0, C0 = oracle.collide(T, f, 0)
        Cp0, d0 = oracle.project(T, f, C0)
        h = kx.Handle(p, dp, 1.0)
        fd = _dev(torch, f)
        raw = h.collide_ex(fd, flags=0, want=("C", "gain", "loss"))
        pro = h.collide_ex(fd, flags=kx.PROJECT, want=("C", "diag"))
        assert _relerr(raw["gain"].cpu().numpy(), g0, g0) <= TOL
        assert _relerr(raw["loss"].cpu().numpy(), l0, g0) <= TOL
        assert _relerr(raw["C"].cpu().numpy(), C0, g0) <= TOL
        assert _relerr(pro["C"].cpu().numpy(), Cp0, g0) <= TOL
        dg = pro["diag"].cpu().numpy()
        assert np.allclose(dg, d0, rtol=1e-8, atol=1e-13)
        assert h.fallback_members() == 0                 # the two-bump input stays on the tensor-core path
        Cr, Cp = raw["C"].cpu().numpy()[0], pro["C"].cpu().numpy()[0]
        corr[N] = 100 * np.abs(Cp - Cr).max() / np.abs(Cr).max()
        epsN[N], epsE[N] = abs(dg[0, 0]), abs(dg[0, 1])
        # the projected operator conserves number and energy at round-off (C.2-C.8)
        hw, E = T.h, T.E
        assert abs((hw * Cp).sum()) <= 1e-13 * (hw * np.abs(Cr)).sum()
        assert abs((hw * E * Cp).sum()) <= 1e-13 * (hw * E * np.abs(Cr)).sum()
        h.close()
    for N, v in paper.items():
        assert v / 10 < corr[N] < v * 10, (N, corr[N], v)
    assert corr[256] < corr[128] < corr[96] and corr[256] < corr[96] / 3
    assert epsN[256] < epsN[96] / 3 and epsE[256] < epsE[96] / 3


# --------------------------------------------------------------------------------------- optional fp32 mode
@pytest.mark.parametrize("cfg,N,B,interp", [(1, None, None, 0), (3, 96, 9, 0), (3, 96, 9, 1), (4, 100, 3, 0)])
def test_fp32_mode_within_1e4(torch_cuda, oracle, cfg, N, B, interp):
    """KX_FP32 (BASELINE.json north_star: optional fp32 mode, max-abs error <= 1e-4 relative to max_i |gain_i|): the
    contraction in single precision against the fp64 oracle; the projected operator still conserves at fp64 round-off
    because the finishing phase stays in double."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(cfg, N=N, B=B)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    g0, l0, C0 = oracle.collide(T, c["f"], interp)
    h = _handle(c, interp=interp, precision=kx.FP32)
    f = _dev(torch, c["f"])
    o = h.collide_ex(f, flags=0, want=("C", "gain", "loss"))
    for key, ref in (("gain", g0), ("loss", l0), ("C", C0)):
        err = _relerr(o[key].cpu().numpy(), ref, g0)
        assert err <= 1e-4, (key, err)
        assert err >= 1e-12 or key == "C"                # it really is single precision
    Cp = h.collide(f, flags=1).cpu().numpy()
    Craw = o["C"].cpu().numpy()
    assert (np.abs((T.h * Cp).sum(axis=1)) <= 1e-12 * (T.h * np.abs(Craw)).sum(axis=1)).all()
    with pytest.raises(kx.KxError):
        _handle(c, precision=kx.FP32, statistics=kx.STAT_BOSE)
    # a few RK4 steps in fp32 stay within 1e-4 of the fp64 oracle's
    pos = c["f"] > 0
    nu = float((l0[pos] / c["f"][pos]).max())
    tau = np.arange(4) * (0.5 / nu)
    f_ref = oracle.evolve(c["p"], c["dp"], c["f"], m=c["m"], M2_0=c["M2_0"], m_med=c["m_med"], interp=interp, method=oracle.RK4, tau=tau)
    h.evolve(f, tau, method=kx.RK4)
    assert np.abs(f.cpu().numpy() - f_ref).max() <= 1e-4 * np.abs(f_ref).max()
    h.close()


def test_nonfinite_member_takes_the_exact_path(torch_cuda):
    """structural zeros of the tiled operand are stored as A = 0, and 0 x Inf = NaN would leak into rows whose
    (i, n, m) triple is dropped.  A member holding an Inf or a NaN is routed to the exact fallback (its max |f| statistic is
    not finite), so the tiled and the row storage agree bit for bit on it, and its batch neighbours are untouched."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(3, N=64, B=4)
    f = c["f"].copy()
    f[1, 50] = np.inf
    f[2, 3] = np.nan
    ht, hr = _handle(c), _handle(c, storage=kx.STORE_SYM_ROWS)
    fd = _dev(torch, f)
    Ct = ht.collide(fd).cpu().numpy()
    assert ht.fallback_members() == 2
    Cr = hr.collide(fd).cpu().numpy()
    for b in (1, 2):
        assert np.array_equal(np.isnan(Ct[b]), np.isnan(Cr[b])) and np.array_equal(np.isinf(Ct[b]), np.isinf(Cr[b]))
        ok = np.isfinite(Cr[b])
        assert np.array_equal(Ct[b][ok], Cr[b][ok])
    clean = ht.collide(_dev(torch, c["f"])).cpu().numpy()
    assert np.array_equal(Ct[0], clean[0]) and np.array_equal(Ct[3], clean[3])
    ht.close(); hr.close()
