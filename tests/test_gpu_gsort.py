"""f2 on the GPU -- the paper's gapped in-place fine sort fused with the pusher (include/pic1d_gsort.h) against
the oracle's statement of it: N_i of every sort cell and the per-cell MULTISETS of particles bit for bit (the
order inside a cell is undefined in the paper: atomic counters), wall losses and mover counts exactly."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _case(Nc, n, vth, seed):
    rng = np.random.default_rng(seed)
    x = (rng.random(n, dtype=np.float32) * Nc).astype(np.float32)
    v = (rng.normal(size=(3, n)) * vth).astype(np.float32)
    E = rng.normal(size=Nc + 1).astype(np.float32)
    return x, v, E


def _same(go, gg):
    from oracle import oracle as O
    No, ao, so = go.get()
    Ng, ag, sg = gg.get()
    assert np.array_equal(No, Ng)
    assert so == {k: sg[k] for k in so} or (so["error"], sg["error"]) == (-2, -2)
    mo, mg = O.cell_multisets(No, ao), O.cell_multisets(Ng, ag)
    for k in range(len(mo)):
        assert np.array_equal(mo[k], mg[k]), k


@pytest.mark.parametrize("Nc,n,inv_ratio,vth,steps", [
    (64, 6000, 1.0, 0.3, 6), (64, 6000, 1.0, 3.0, 4), (128, 40000, 0.5, 0.4, 4), (100, 9000, 2.0, 0.2, 4),
    (256, 300000, 1.0, 0.03, 3),        # ~1170 particles per cell, Eq. 5 well satisfied (ions, Courant twins)
    (16, 60000, 1.0, 0.5, 3),           # 3750 particles per cell: several passes per thread
    (128, 2000, 0.0625, 2.0, 3), (8, 5, 1.0, 0.1, 2)])
def test_gapped_sort_matches_the_oracle_cell_by_cell(Nc, n, inv_ratio, vth, steps):
    from oracle import oracle as O
    from paper_1104_3998_b200 import gsort as GS
    kappa = -0.05
    x, v, E = _case(Nc, n, vth, 3)
    n_max = min(8192, int(2.5 * n / (Nc * inv_ratio)) + 64)
    go, gg = O.Gapped(Nc, inv_ratio, n_max, kappa), GS.GappedSort(Nc, inv_ratio, n_max, kappa)
    assert go.load(x, v[0], v[1], v[2]) == 0
    gg.load(x, v[0], v[1], v[2])
    _same(go, gg)
    for s in range(steps):
        go.set_E32(E); gg.set_E32(E)
        assert go.step() == 0
        gg.step(1)
        _same(go, gg)
    assert gg.get(arrays=False)[2]["error"] == 0
    go.close(); gg.close()


def test_gapped_sort_cell_overflow_is_flagged():
    from paper_1104_3998_b200 import gsort as GS
    from paper_1104_3998_b200 import pic1d as G
    Nc = 8
    x = np.array([2.5, 2.6, 2.7, 2.8, 3.1, 3.2, 3.3], np.float32)
    v = np.array([1.0, 1.0, 1.0, 1.0, 0.0, 0.0, 0.0], np.float32)
    gg = GS.GappedSort(Nc, 1.0, 4, 0.0)
    gg.load(x, v, 0 * x, 0 * x)
    gg.set_E32(np.zeros(Nc + 1, np.float32))
    gg.step(1)
    N, _, st = gg.get()
    assert st["error"] == G.ERR_CAPACITY and N.max() <= 4
    gg.close()
