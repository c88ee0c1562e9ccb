"""Host logic of the tensor-core kernel's launch plan (kx_plan_probe: no device needed).  The kernel relies on these
invariants: every gain warp owns at least one group (so every partial slot the finishing phase adds was written by the same
launch: ADVICE r1, the unwritten gpart slot), the CTAs of a tile form a contiguous range, every loss CTA has at least one
chunk, the supertile -> loss CTA ranges tile [0, GL), and the grid fits the device."""
import numpy as np
import pytest

import kx_inputs as kin


def _groups_per_tile(p, m):
    """Gain groups of every 16-row tile for a grid: runs (tile, n) -> union over the tile's rows of the kept m >= n interval,
    padded to quads of 4 m, quads per tile padded to groups of 4 (the layout of kx_tiled_build.cu, counted here in numpy)."""
    N = p.size
    E = np.sqrt(p * p + m * m)
    K = p * p / (E + m)
    NT = (N + 15) // 16
    out = np.zeros(NT, dtype=np.uint32)
    for t in range(NT):
        quads = 0
        rows = range(16 * t, min(N, 16 * t + 16))
        for n in range(N):
            lo, hi = N, -1
            for i in rows:
                Kt = K[n] + K[n:] - K[i]
                tau = 32 * 2.0 ** -52 * (K[n] + K[n:] + K[i])
                ok = np.nonzero((Kt >= K[0] - tau) & (Kt <= K[-1] + tau))[0]
                if ok.size:
                    lo, hi = min(lo, n + ok[0]), max(hi, n + ok[-1] + 1)
            if hi > lo:
                quads += (hi - lo + 3) // 4
        out[t] = (quads + 3) // 4
    return out


def _check(plan, g, B):
    GG, GL, NT, RS, LC = plan["GG"], plan["GL"], plan["NT"], plan["RS"], plan["LC"]
    w = plan["wstart"]
    assert GG >= 1 and GL >= 1 and GG + GL <= 148
    assert plan["smem"] <= 226 * 1024
    assert plan["nbt"] in (1, 2, 4, 8) and plan["nbt"] * 8 >= min(B, 64) or plan["nbt"] < 8
    assert (np.diff(w) >= 0).all() and w[0] == 0 and w[NT] <= GG * 8
    for t in range(NT):
        wt = w[t + 1] - w[t]
        if g[t] == 0:
            assert wt == 0
            continue
        assert 1 <= wt <= g[t], (t, wt, g[t])            # at least one group for every warp of the tile
        # the device-side split: warp r of the tile takes groups [r g / wt, (r + 1) g / wt): never empty
        cuts = (np.arange(wt + 1) * int(g[t])) // int(wt)
        assert (np.diff(cuts) >= 1).all()
        # every CTA of the tile's range c0..c1 holds at least one of its warps: its slot c + t is written
        c0, c1 = w[t] // 8, (w[t + 1] - 1) // 8
        for c in range(c0, c1 + 1):
            assert max(w[t], 8 * c) < min(w[t + 1], 8 * c + 8)
    # loss: chunk units [sp LC, (sp + 1) LC) of the RS LC units; CTA c takes [c U / GL, (c + 1) U / GL)
    U = RS * LC
    assert GL <= U
    cuts = (np.arange(GL + 1) * U) // GL
    assert (np.diff(cuts) >= 1).all()
    for sp in range(RS):
        first = int(np.searchsorted(cuts, sp * LC, side="right") - 1)
        last = int(np.searchsorted(cuts, (sp + 1) * LC - 1, side="right") - 1)
        assert plan["ld0"][sp] == first and plan["ld1"][sp] == last, (sp, plan["ld0"], plan["ld1"], first, last)
    assert plan["ld0"][0] == 0 and plan["ld1"][RS - 1] == GL - 1


@pytest.mark.parametrize("N,log", [(6, False), (8, False), (12, False), (22, False), (32, True), (33, True), (44, True), (52, True),
                                   (96, True), (256, True), (300, False), (512, True)])
def test_plan_invariants_on_real_grids(N, log):
    import paper_2607_00755_b200 as kx
    p = kin.log_grid(N, 1e-3, 50.0) if log else kin.uniform_grid(N, 0.05, 10.0)
    g = _groups_per_tile(p, 1.0) if N <= 300 else None
    if g is None:                                         # N = 512: a synthetic profile of the same shape, cheaper than counting
        t = np.arange((N + 15) // 16)
        g = np.maximum(1, (16000 * (1.0 - (t / t.size) ** 2)).astype(np.uint32))
    for B in (1, 3, 8, 9, 16, 33, 64, 65, 200):
        for Q in (2, 24):
            _check(kx.plan_probe(N, B, g, Q=Q), g, B)


def test_plan_invariants_on_adversarial_profiles():
    import paper_2607_00755_b200 as kx
    rng = np.random.default_rng(5)
    for N in (16, 17, 48, 130, 256, 1024):
        NT = (N + 15) // 16
        for trial in range(20):
            kind = trial % 4
            if kind == 0:
                g = rng.integers(1, 5, size=NT)                       # fewer groups than warps
            elif kind == 1:
                g = rng.integers(0, 3, size=NT); g[rng.integers(NT)] = 1   # empty tiles
            elif kind == 2:
                g = rng.integers(1, 40000, size=NT)                   # wildly uneven
            else:
                g = np.full(NT, 1 + trial)
            g = g.astype(np.uint32)
            for B in (1, 8, 64):
                _check(kx.plan_probe(N, B, g, Q=24), g, B)
