"""kx_collide_static: the evaluation entry point that allocates nothing (its scratch is a static __device__ array shared by
all calls, kx_static.cu).  Collected last on purpose (the file name sorts after every other test file): the suite runs with
pytest -x, and a failure here must not hide the other tests.  Passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

import kx_inputs as kin

pytestmark = pytest.mark.gpu

TOL = 1e-11          # the bar of tests/test_gpu_parity.py: max-abs error relative to max_i |gain_i| per member


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    return torch


def _dev(torch, a):
    return torch.tensor(np.ascontiguousarray(a), dtype=torch.float64, device="cuda")


def _relerr(got, ref, gain):
    scale = np.abs(gain).max(axis=1, keepdims=True)
    return float((np.abs(got - ref) / scale).max())


@pytest.mark.parametrize("storage", ["tiled", "rows"])
def test_static_entry_matches_existing_path_two_calls_in_a_row(torch_cuda, storage):
    """Two calls in a row on the shared static scratch (different inputs and batch sizes, so the second call meets the first
    one's leftovers) against the existing path kx_collide / kx_collide_parts on the same handle, raw and projected."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(3, N=96, B=11)
    h = kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"],
                  storage=kx.STORE_TILED if storage == "tiled" else kx.STORE_SYM_ROWS)
    f1 = _dev(torch, c["f"])
    f2 = _dev(torch, c["f"][::-1][:5] * 3.0)
    refs = []
    for f in (f1, f2):
        gain = h.collide_parts(f)[0].cpu().numpy()
        refs.append((gain, h.collide(f).cpu().numpy(), h.collide(f, flags=kx.PROJECT).cpu().numpy()))
    torch.cuda.synchronize()
    out1, out2 = torch.empty_like(f1), torch.empty_like(f2)
    out1p, out2p = torch.empty_like(f1), torch.empty_like(f2)
    # back to back on one stream, no synchronisation in between: stream order is all the entry point needs
    h.collide_static(f1, out=out1)
    h.collide_static(f2, out=out2)
    h.collide_static(f1, flags=kx.PROJECT, out=out1p)
    h.collide_static(f2, flags=kx.PROJECT, out=out2p)
    torch.cuda.synchronize()
    for (gain, Craw, Cproj), o, op in ((refs[0], out1, out1p), (refs[1], out2, out2p)):
        assert torch.isfinite(o).all() and torch.isfinite(op).all()
        assert _relerr(o.cpu().numpy(), Craw, gain) <= TOL
        assert _relerr(op.cpu().numpy(), Cproj, gain) <= TOL
    # the same call twice gives the same bits (fixed summation order, nothing left over from the call before)
    again = torch.empty_like(f1)
    h.collide_static(f1, out=again)
    assert torch.equal(again, out1)
    h.close()


def test_static_entry_other_modes_and_limits(torch_cuda, oracle):
    """LINEAR interpolation and a grid with N > 256 against the oracle; sizes beyond the static scratch and unsupported
    options are rejected with a clear error and nothing is launched."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(4, N=300, B=3)
    T = oracle.Tables(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    for interp in (kx.INTERP_LOG, kx.INTERP_LINEAR):
        g0, l0, C0 = oracle.collide(T, c["f"], interp)
        h = kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"], interp=interp)
        C = h.collide_static(_dev(torch, c["f"])).cpu().numpy()
        assert _relerr(C, C0, g0) <= TOL
        h.close()
    big = kin.config(3, B=2)                                # N = 256: 131072 pairs hold at most 385 members (chunk 65536)
    h = kx.Handle(big["p"], big["dp"], big["m"], big["g_chi"], big["M2_0"], big["m_med"])
    f = _dev(torch, np.repeat(big["f"], 300, axis=0))       # B = 600
    with pytest.raises(kx.KxError) as ei:
        h.collide_static(f)
    assert ei.value.status == 4 and "static scratch" in str(ei.value)
    ok = h.collide_static(f[:64].contiguous())              # the headline batch fits
    assert _relerr(ok.cpu().numpy(), h.collide(f[:64].contiguous()).cpu().numpy(),
                   h.collide_parts(f[:64].contiguous())[0].cpu().numpy()) <= TOL
    h.close()
    hb = kx.Handle(big["p"][:32] * 1.0, kin.trapezoid_widths(big["p"][:32]), 1.0, statistics=kx.STAT_BOSE)
    with pytest.raises(kx.KxError):
        hb.collide_static(_dev(torch, np.full((1, 32), 0.1)))
    hb.close()


def test_static_entry_leaves_device_memory_alone(torch_cuda):
    """What "allocates nothing" means, observed from outside: after a first call (CUDA loads a kernel's code lazily on its
    first launch), the free device memory reported by the driver does not move over further calls with new batch sizes --
    whereas the ordinary entry point grows the handle's workspace when it first sees a larger batch."""
    torch = torch_cuda
    import paper_2607_00755_b200 as kx
    c = kin.config(3, N=128, B=48)
    h = kx.Handle(c["p"], c["dp"], c["m"], c["g_chi"], c["M2_0"], c["m_med"])
    f = _dev(torch, c["f"])
    outs = {B: torch.empty((B, 128), dtype=torch.float64, device="cuda") for B in (2, 7, 48)}
    h.collide_static(f[:2].contiguous(), out=outs[2])
    h.collide_static(f[:2].contiguous(), flags=kx.PROJECT, out=outs[2])
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for B in (7, 48, 2, 48):
        fb = f[:B]                                           # a view of the leading rows: contiguous, no torch allocation
        h.collide_static(fb, out=outs[B])
        h.collide_static(fb, flags=kx.PROJECT, out=outs[B])
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    h.collide(f)                                             # the ordinary path allocates its workspace for B = 48 now
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] < free0
    h.close()
