"""f3 -- binary Coulomb collisions inside sort cells (Takizuka-Abe model,
DESIGN.md R23): pairing, per-pair conservation, scattering-angle statistics and the isotropisation rate of
an anisotropic Maxwellian against the analytic (NRL formulary) rate."""
import numpy as np
import pytest

from oracle import oracle as O
from helpers import params, load


def _box(n, coul_A, n_cells=8, sort_ratio=8.0, seed=3):
    """periodic box, electrons only, no field push (kappa = 0), no MCC: only the binary collisions act"""
    p = params(1, n_cells=n_cells, ppc=1, sort_ratio=sort_ratio, seed=seed, capacity_factor=2.0 * n / n_cells + 2)
    p["species"][0]["kappa"] = 0.0
    p["coul_A"] = [coul_A, 0.0]
    return p


def _state(o):
    return np.stack([o.debug_get(w) for w in (O.VX, O.VY, O.VZ)], 1).astype(np.float64)


@pytest.mark.parametrize("n_cells,ratio,n", [(8, 8.0, 1001), (8, 1.0, 4000), (16, 2.0, 777)])
def test_pairing_is_a_perfect_matching_inside_each_cell(n_cells, ratio, n):
    rng = np.random.default_rng(1)
    p = _box(n, 1e-3, n_cells, ratio)
    o = O.Oracle(p)
    x = (rng.random(n, dtype=np.float32) * n_cells).astype(np.float32)
    v = (rng.normal(size=(3, n)) * 0.01).astype(np.float32)
    load(o, [(x, v[0], v[1], v[2])])
    seen, want_pairs = [], 0
    for step in range(3):
        o.step(1)
        part = o.debug_get(O.PARTNER)
        off = o.debug_get(O.OFFSETS)
        idx = np.arange(part.shape[0])
        paired = part >= 0
        assert np.array_equal(part[part[paired]], idx[paired])          # an involution without fixed points
        assert np.all(part[paired] != idx[paired])
        cell = np.searchsorted(off, idx, side="right") - 1
        assert np.array_equal(cell[paired], cell[part[paired]])          # partners share the sort cell
        counts = np.diff(off)
        unpaired = np.bincount(cell[~paired], minlength=counts.shape[0])
        assert np.array_equal(unpaired, counts % 2)                      # everybody once; odd cells leave one out
        want_pairs += int((counts // 2).sum())
        assert o.moments(0)["n_pairs"] == want_pairs
        seen.append(part.copy())
    assert np.mean(seen[0] == seen[1]) < 0.2 and np.mean(seen[1] == seen[2]) < 0.2   # new partners every step


def _partners_of_one_cell(n, steps, seed=5):
    """partner arrays (slot numbers inside the cell) of a single sort cell of n particles over `steps` steps"""
    rng = np.random.default_rng(seed)
    p = _box(n, 1e-9, n_cells=8, sort_ratio=8.0, seed=seed)
    o = O.Oracle(p)
    x = (rng.random(n, dtype=np.float32) * 8).astype(np.float32)
    v = (rng.normal(size=(3, n)) * 1e-4).astype(np.float32)
    load(o, [(x, v[0], v[1], v[2])])
    out = []
    for _ in range(steps):
        o.step(1)
        out.append(o.debug_get(O.PARTNER).copy())
    return out


def test_every_pairing_of_four_particles_comes_out_equally_often():
    """n = 4 has three perfect matchings, 01|23, 02|13, 03|12; random pairing (Takizuka-Abe) draws each with
    probability 1/3.  (An affine map (a m + b) mod 4 can never pair slots 0 and 2: this pin rejects it.)"""
    steps = 600
    count = {1: 0, 2: 0, 3: 0}
    for part in _partners_of_one_cell(4, steps):
        assert sorted(part[part]) == [0, 1, 2, 3]
        count[int(part[0])] += 1
    for k in (1, 2, 3):
        assert abs(count[k] - steps / 3) <= 4.5 * np.sqrt(steps * (1 / 3) * (2 / 3)), count


def test_pair_distances_in_a_cell_are_not_a_single_stride():
    """the slot distance |i - partner(i)| of random pairs of n slots has the triangular law P(d) = 2 (n - d) /
    (n (n - 1)); pairs built from one stride would all share one or two distances"""
    n, steps = 101, 40
    d = np.concatenate([np.abs(np.arange(n) - part)[part >= 0] for part in _partners_of_one_cell(n, steps)])
    assert d.shape[0] == steps * (n - 1)
    for part in _partners_of_one_cell(n, 3):
        assert np.unique(np.abs(np.arange(n) - part)[part >= 0]).shape[0] > 25
    hist = np.bincount(d, minlength=n)[1:] / 2                      # pairs per distance (each pair counted twice)
    want = steps * (n // 2) * 2 * (n - np.arange(1, n)) / (n * (n - 1))
    # chi-square over 10 bands of distances (each band has dozens of expected pairs)
    bands = np.array_split(np.arange(n - 1), 10)
    chi2 = sum((hist[b].sum() - want[b].sum()) ** 2 / want[b].sum() for b in bands)
    assert chi2 < 35.0, chi2                                        # 9 degrees of freedom: P(chi2 > 35) < 1e-4
    # who sits out of an odd cell is uniform too: not always the same slot
    out = [int(np.nonzero(part < 0)[0][0]) for part in _partners_of_one_cell(n, steps)]
    assert len(set(out)) > steps // 2


def test_every_pair_conserves_momentum_and_energy():
    n = 20000
    rng = np.random.default_rng(2)
    p = _box(n, 2e-6)
    o = O.Oracle(p)
    x = (rng.random(n, dtype=np.float32) * 8).astype(np.float32)
    v = (rng.normal(size=(3, n)) * 0.02).astype(np.float32)
    load(o, [(x, v[0], v[1], v[2])])
    o.set_E32(np.zeros(8, np.float32))
    # the step sorts (a permutation that depends on x only), then collides: recover the pre-collision velocities
    # of the sorted slots from a twin run without collisions
    p0 = dict(p, coul_A=[0.0, 0.0])
    o0 = O.Oracle(p0)
    load(o0, [(x, v[0], v[1], v[2])])
    o0.set_E32(np.zeros(8, np.float32))
    o.step(1); o0.step(1)
    before, after = _state(o0), _state(o)
    part = o.debug_get(O.PARTNER)
    a = np.nonzero(part > np.arange(n))[0]
    b = part[a]
    assert a.shape[0] == n // 2
    scale = np.abs(before).max()
    assert np.max(np.abs((after[a] + after[b]) - (before[a] + before[b]))) < 4e-7 * scale      # momentum
    u0, u1 = before[a] - before[b], after[a] - after[b]
    assert np.max(np.abs(np.linalg.norm(u1, axis=1) / np.linalg.norm(u0, axis=1) - 1)) < 2e-6    # |u| kept
    e0, e1 = (before[a] ** 2 + before[b] ** 2).sum(1), (after[a] ** 2 + after[b] ** 2).sum(1)
    assert np.max(np.abs(e1 / e0 - 1)) < 3e-6                                                     # energy
    assert np.mean(np.abs(u1 - u0).max(1) > 1e-4 * scale) > 0.9                                   # and they did collide


@pytest.mark.parametrize("axis", [0, 2])
def test_scattering_angle_variance_and_azimuth(axis):
    """counter-streaming beams +-v0 along one axis: every pair of opposite particles has u = 2 v0, so
    tan^2(theta/2) ~ <delta^2> = coul_A n / u^3 and the azimuth is uniform (axis 2: the u_perp = 0 branch)"""
    n, v0, var = 40000, 0.25, 0.02
    u = 2 * v0
    p = _box(n, var * u ** 3 / n)
    o = O.Oracle(p)
    rng = np.random.default_rng(5)
    x = (rng.random(n, dtype=np.float32) * 8).astype(np.float32)
    v = np.zeros((3, n), np.float32)
    v[axis] = np.where(rng.random(n) < 0.5, v0, -v0)
    load(o, [(x, v[0], v[1], v[2])])
    p0 = dict(p, coul_A=[0.0, 0.0])
    o0 = O.Oracle(p0)
    load(o0, [(x, v[0], v[1], v[2])])
    o.step(1); o0.step(1)
    before, after = _state(o0), _state(o)
    part = o.debug_get(O.PARTNER)
    a = np.nonzero(part > np.arange(n))[0]
    b = part[a]
    u0, u1 = before[a] - before[b], after[a] - after[b]
    hit = np.abs(u0[:, axis]) > v0                      # opposite beams (equal beams have u = 0: no collision)
    assert np.array_equal(after[a][~hit], before[a][~hit])
    u0, u1 = u0[hit], u1[hit]
    k = hit.sum()
    cos_t = (u0 * u1).sum(1) / (u ** 2)
    d2 = (1 - cos_t) / (1 + cos_t)
    assert abs(d2.mean() / var - 1) < 4 * np.sqrt(2.0 / k)          # delta ~ N(0, var): var(delta^2) = 2 var^2
    assert abs((d2 ** 2).mean() / (3 * var ** 2) - 1) < 0.1         # Gaussian: <delta^4> = 3 var^2
    perp = [q for q in range(3) if q != axis]
    kick = (u1 - u0)[:, perp] * np.sign(u0[:, axis])[:, None]
    assert np.all(np.abs(kick.mean(0)) < 4 * kick.std(0) / np.sqrt(k))          # azimuth: no preferred direction
    assert abs(kick[:, 0].var() / kick[:, 1].var() - 1) < 0.06


def test_anisotropic_maxwellian_relaxes_at_the_analytic_rate():
    """T_x = 2 T_perp relaxes as d(T_perp - T_par)/dt = -3 nu_T (T_perp - T_par) with the NRL-formulary rate
    nu_T dt = coul_A n F(A) / (4 sqrt(pi) v_par^3),  A = T_perp/T_par - 1,
    F = A^-2 [-3 + (A + 3) atanh(sqrt(-A)) / sqrt(-A)] for A < 0; the energy is conserved."""
    n, vpar, ratio = 200000, 0.02 * np.sqrt(2.0), 0.5
    vperp = vpar * np.sqrt(ratio)
    A = ratio - 1.0
    F = (-3 + (A + 3) * np.arctanh(np.sqrt(-A)) / np.sqrt(-A)) / A ** 2
    nu_dt = 2.0e-3                                      # per step
    coul_A = nu_dt * 4 * np.sqrt(np.pi) * vpar ** 3 / (n * F)
    p = _box(n, coul_A)
    o = O.Oracle(p)
    rng = np.random.default_rng(7)
    x = (rng.random(n, dtype=np.float32) * 8).astype(np.float32)
    v = np.stack([rng.normal(size=n) * vpar, rng.normal(size=n) * vperp, rng.normal(size=n) * vperp]).astype(np.float32)
    load(o, [(x, v[0], v[1], v[2])])
    steps = 12
    d, en = [], []
    for s in range(steps + 1):
        w = _state(o)
        T = (w ** 2).mean(0)
        d.append(0.5 * (T[1] + T[2]) - T[0])
        en.append((w ** 2).sum())
        if s < steps:
            o.step(1)
    d, en = np.array(d), np.array(en)
    assert np.max(np.abs(en / en[0] - 1)) < 2e-5                    # energy conserved
    assert np.all(np.diff(np.abs(d)) < 0)                           # monotonic towards isotropy
    rate = -np.polyfit(np.arange(4), np.log(d[:4] / d[0]), 1)[0]    # initial decay rate of the anisotropy
    assert abs(rate / (3 * nu_dt) - 1) < 0.15, rate / (3 * nu_dt)
