"""f2 -- the paper's gapped in-place fine sort (steps 1a / 1b / 2 / 3) as the oracle
states it, pinned by the plain definition of its result: afterwards sort cell k holds exactly the surviving
particles whose key is k ("all particles are arranged in correct sorting cells", L192) -- taken from the compact
stable counting sort of the same particles, which is itself pinned by brute force (test_oracle_particles.py)."""
import numpy as np
import pytest

from oracle import oracle as O
from helpers import params, load


def _compact(Nc, inv_ratio, kappa, n):
    p = params(0, n_cells=Nc, ppc=1, mcc=False, n_species=1, bc=0, capacity_factor=2.0 * n / Nc + 2)
    p["species"][0].update(kappa=kappa)
    p["sort_inv_ratio"] = inv_ratio
    return O.Oracle(p)


def _case(Nc, n, vth, seed):
    rng = np.random.default_rng(seed)
    x = (rng.random(n, dtype=np.float32) * Nc).astype(np.float32)
    v = (rng.normal(size=(3, n)) * vth).astype(np.float32)
    E = rng.normal(size=Nc + 1).astype(np.float32)
    return x, v, E


@pytest.mark.parametrize("inv_ratio,vth", [(1.0, 0.3), (1.0, 3.0), (0.5, 0.4), (2.0, 0.2), (0.0625, 2.0)])
def test_gapped_sort_reaches_the_defined_cell_membership(inv_ratio, vth):
    Nc, n, kappa = 64, 6000, -0.05
    x, v, E = _case(Nc, n, vth, 11)
    o = _compact(Nc, inv_ratio, kappa, n)
    load(o, [(x, v[0], v[1], v[2])])
    g = O.Gapped(Nc, inv_ratio, int(2.5 * n / (Nc * inv_ratio)) + 64, kappa)
    assert g.load(x, v[0], v[1], v[2]) == 0
    for step in range(5):
        o.set_E32(E); g.set_E32(E)
        keys_before = [np.repeat(np.arange(g.n_sc), g.get()[0])]
        assert o.step(1) == 0 and g.step() == 0
        N, arr, st = g.get()
        off = o.debug_get(O.OFFSETS)
        assert np.array_equal(N, np.diff(off))                                  # N_i of every sort cell
        ref = [o.debug_get(w) for w in (O.X, O.VX, O.VY, O.VZ)]
        mine = O.cell_multisets(N, arr)
        for k in range(g.n_sc):                                                 # the cell's particles, as a multiset
            t = np.stack([a[off[k]:off[k + 1]] for a in ref], 1)
            assert np.array_equal(mine[k], t[np.lexsort(t.T[::-1])]), (step, k)
            kk = np.floor(mine[k][:, 0].astype(np.float64) * inv_ratio)
            assert np.all(kk == k)                                              # ... all in the right cell
        m = o.moments(0)
        assert (st["absorbed_left"], st["absorbed_right"]) == (m["absorbed_left"], m["absorbed_right"])
        assert N.sum() == m["count"]
    if vth * inv_ratio < 0.5:
        assert st["moved_far"] * 20 < st["moved_near"]     # Eq. 5 holds: step 3 is the rare case (L186)
    else:
        assert st["moved_far"] > 0                          # ... and it is exercised when it does not
    o.close(); g.close()


def test_gapped_load_keeps_input_order_inside_a_cell_and_overflow_is_flagged():
    Nc = 8
    x = np.array([3.5, 0.25, 3.25, 7.9, 3.75], np.float32)
    tag = np.arange(5, dtype=np.float32)
    g = O.Gapped(Nc, 1.0, 3, 0.0)
    assert g.load(x, 0 * x, tag, tag) == 0
    N, arr, _ = g.get()
    assert N.tolist() == [1, 0, 0, 3, 0, 0, 0, 1] and arr[2][3, :3].tolist() == [0.0, 2.0, 4.0]
    g.close()
    g = O.Gapped(Nc, 1.0, 2, 0.0)
    assert g.load(x, 0 * x, tag, tag) == -2            # cell 3 would need 3 slots
    g.close()
    # a cell that receives more than its free slots during a step: flagged, nothing written out of bounds
    g = O.Gapped(Nc, 1.0, 4, 0.0)
    x = np.array([2.5, 2.6, 2.7, 2.8, 3.1, 3.2, 3.3], np.float32)
    v = np.array([1.0, 1.0, 1.0, 1.0, 0.0, 0.0, 0.0], np.float32)   # four particles enter cell 3, which has one free slot
    assert g.load(x, v, 0 * x, 0 * x) == 0
    g.set_E32(np.zeros(Nc + 1, np.float32))
    assert g.step() == -2                               # cell 2 is full: no free slot to buffer its rejected particles
    N, _, _ = g.get()
    assert N.max() <= 4 and N[2] == 0 and N.sum() < 7
    g.close()


def test_step_1b_fills_gaps_from_the_end():
    """six particles in cell 2; #1 and #4 leave to the right, #0 leaves the box: the valid ones end up compact"""
    Nc = 4
    x = np.array([2.1, 2.2, 2.3, 2.4, 2.5, 2.6], np.float32)
    v = np.array([-3.0, 1.0, 0.0, 0.0, 1.0, 0.0], np.float32)
    tag = np.arange(6, dtype=np.float32)
    g = O.Gapped(Nc, 1.0, 8, 0.0)
    g.load(x, v, tag, tag)
    g.set_E32(np.zeros(Nc + 1, np.float32))
    assert g.step() == 0
    N, arr, st = g.get()
    assert N.tolist() == [0, 0, 3, 2] and st["absorbed_left"] == 1 and st["moved_near"] == 2 and st["moved_far"] == 0
    assert sorted(arr[2][2, :3].tolist()) == [2.0, 3.0, 5.0] and sorted(arr[2][3, :2].tolist()) == [1.0, 4.0]
    g.close()
