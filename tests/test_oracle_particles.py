"""P2 / P5 / P7 / P8 -- oracle push, deposit, boundary and sort against closed forms, invariants
and brute force.  PAPER.md L35, L41, L63-67, L128-138, L150-156, L160-192."""
import numpy as np
import pytest

from oracle import oracle as O
from helpers import params, load


def _one_species(Nc, kappa, bc=0, cap=4096, inv_ratio=1.0, **kw):
    p = params(0, n_cells=Nc, ppc=1, mcc=False, n_species=1, bc=bc, **kw)
    p["species"][0].update(kappa=kappa, capacity=cap)
    p["sort_inv_ratio"] = inv_ratio
    return p


# ---- P5 push ---------------------------------------------------------------------------------
def test_push_constant_field_closed_form():
    Nc, kappa, E0 = 64, -0.25, 0.125          # all dyadic: the closed form is exact in fp32
    o = O.Oracle(_one_species(Nc, kappa))
    x0 = np.array([10.5, 30.25, 50.0], np.float32)
    v0 = np.array([0.5, -0.25, 0.0], np.float32)
    z = np.zeros(3, np.float32)
    load(o, [(x0, v0, z + 1, z + 2)])
    for n in range(1, 9):
        o.set_E32(np.full(Nc + 1, E0, np.float32))
        o.step(1)
        assert np.array_equal(o.debug_get(O.VX), v0 + n * kappa * E0)
        xs = np.sort(x0 + n * v0 + kappa * E0 * n * (n + 1) / 2)
        assert np.array_equal(np.sort(o.debug_get(O.X)), xs.astype(np.float32))
        assert np.array_equal(np.sort(o.debug_get(O.VY)), z + 1)      # vy, vz untouched
        assert np.array_equal(np.sort(o.debug_get(O.VZ)), z + 2)


def test_push_linear_field_leapfrog_oscillator():
    # E = alpha (x - c): x_{n+1} - 2 x_n + x_{n-1} = kappa alpha (x_n - c); cos(w dt) = 1 + kappa alpha / 2
    Nc, kappa, alpha, c = 128, -1.0, 0.01, 64.0
    o = O.Oracle(_one_species(Nc, kappa))
    E = (alpha * (np.arange(Nc + 1) - c)).astype(np.float32)
    load(o, [(np.array([70.3], np.float32), np.zeros(1, np.float32), np.zeros(1, np.float32),
              np.zeros(1, np.float32))])
    xs = [70.3]
    for n in range(200):
        o.set_E32(E)
        o.step(1)
        xs.append(float(o.debug_get(O.X)[0]))
    xs = np.array(xs)
    res = xs[2:] - 2 * xs[1:-1] + xs[:-2] - kappa * alpha * (xs[1:-1] - c)
    assert np.max(np.abs(res)) < 3e-5                      # fp32 rounding at x ~ 64
    d = xs - c
    zc = np.nonzero((d[:-1] > 0) & (d[1:] <= 0))[0]
    tz = zc + d[zc] / (d[zc] - d[zc + 1])
    w = 2 * np.pi / np.mean(np.diff(tz))
    assert abs(w - np.arccos(1 + kappa * alpha / 2)) < 2e-4


def test_gather_is_linear_interpolation():
    Nc = 16
    o = O.Oracle(_one_species(Nc, 1.0))
    E = np.arange(Nc + 1, dtype=np.float32) ** 2
    x0 = np.array([3.25, 7.5, 0.0, 15.75], np.float32)
    z = np.zeros(4, np.float32)
    load(o, [(x0, z, z, z)])
    o.set_E32(E * np.float32(2.0 ** -10))
    o.step(1)
    j = np.floor(x0)
    f = x0 - j
    want = ((1 - f) * j ** 2 + f * (j + 1) ** 2) * 2.0 ** -10
    assert np.allclose(np.sort(o.debug_get(O.VX)), np.sort(want), rtol=1e-6)


# ---- P2 deposit ------------------------------------------------------------------------------
def test_deposit_single_particle_and_sum():
    Nc = 32
    p = params(0, n_cells=Nc, ppc=1, mcc=False)
    o = O.Oracle(p)
    z1 = np.zeros(1, np.float32)
    load(o, [(np.array([5.25], np.float32), z1, z1, z1), (np.array([31.75], np.float32), z1, z1, z1)])
    rho, _, _ = o.get_rho_phi_E()
    want = np.zeros(Nc + 1)
    want[5], want[6] = -0.75, -0.25          # electron: sign -1
    want[31], want[32] = 0.25, 0.75          # ion at the last cell touches the wall node
    assert np.array_equal(rho, want)
    assert np.array_equal(o.moments(0)["density"], -np.minimum(want, 0))


def test_deposit_exact_total_and_bruteforce_hat():
    Nc, n = 24, 5000
    rng = np.random.default_rng(3)
    p = params(0, n_cells=Nc, ppc=1, mcc=False, capacity_factor=300)
    o = O.Oracle(p)
    xe = np.minimum(rng.random(n, dtype=np.float32) * Nc, np.nextafter(np.float32(Nc), np.float32(0)))
    xi = np.minimum(rng.random(n // 2, dtype=np.float32) * Nc, np.float32(Nc - 0.001))
    load(o, [(xe, 0 * xe, 0 * xe, 0 * xe), (xi, 0 * xi, 0 * xi, 0 * xi)])
    de, di = o.moments(0)["density"], o.moments(1)["density"]
    assert de.sum() == n and di.sum() == n // 2           # exact: weights are dyadic
    nodes = np.arange(Nc + 1)[:, None]
    hat = lambda x: np.maximum(0.0, 1.0 - np.abs(x.astype(np.float64)[None, :] - nodes)).sum(1)
    assert np.allclose(de, hat(xe), atol=1e-9) and np.allclose(di, hat(xi), atol=1e-9)
    rho, _, _ = o.get_rho_phi_E()
    assert np.allclose(rho, di - de, atol=1e-12)


def test_deposit_periodic_wrap_and_background():
    Nc = 8
    p = params(1, n_cells=Nc, ppc=1)
    o = O.Oracle(p)
    x = np.array([7.5, 0.25], np.float32)
    load(o, [(x, 0 * x, 0 * x, 0 * x)])
    rho, _, _ = o.get_rho_phi_E()
    want = np.full(Nc, p["background_rho"])
    want[7] -= 0.5
    want[0] -= 0.5 + 0.75
    want[1] -= 0.25
    assert np.allclose(rho, want, atol=1e-15)


# ---- P7 boundary ----------------------------------------------------------------------------
def test_absorption_bookkeeping_order_and_ties():
    Nc = 16
    o = O.Oracle(_one_species(Nc, 0.0))
    x0 = np.array([0.5, 15.5, 8.0, 0.25, 15.0, 3.0, 1.0], np.float32)
    v0 = np.array([-1.0, 1.0, 0.5, -0.25, 1.0, -3.0, 0.0], np.float32)   # x' = -.5, 16.5, 8.5, 0, 16, 0, 1
    tag = np.arange(7, dtype=np.float32)
    load(o, [(x0, v0, tag, tag)])
    # the load sorted the particles; remember which tag sits where, then step
    o.set_E32(np.zeros(Nc + 1, np.float32))
    o.step(1)
    m = o.moments(0)
    assert (m["absorbed_left"], m["absorbed_right"], m["count"]) == (1, 2, 4)   # x'=16 exactly is absorbed
    xs, tg = o.debug_get(O.X), o.debug_get(O.VY)
    assert np.all((xs >= 0) & (xs < Nc))
    got = dict(zip(tg.tolist(), xs.tolist()))
    assert got == {2.0: 8.5, 3.0: 0.0, 5.0: 0.0, 6.0: 1.0}                 # x' = 0 survives (cell 0)
    keys = o.debug_get(O.KEYS)
    assert sorted(keys.tolist()) == [-1, -1, -1, 0, 0, 1, 8]


def test_periodic_wrap():
    Nc = 16
    o = O.Oracle(_one_species(Nc, 0.0, bc=1))
    x0 = np.array([0.5, 15.5, 8.0], np.float32)
    v0 = np.array([-1.0, 1.0, 0.5], np.float32)
    load(o, [(x0, v0, 0 * x0, 0 * x0)])
    o.set_E32(np.zeros(Nc, np.float32))
    o.step(1)
    assert sorted(o.debug_get(O.X).tolist()) == [0.5, 8.5, 15.5]
    assert o.moments(0)["count"] == 3


def test_secondary_emission_binomial_and_placement():
    Nc, n = 64, 40000
    p = params(2, n_cells=Nc, ppc=1, mcc=False, gamma=0.1, capacity_factor=2000)
    o = O.Oracle(p)
    rng = np.random.default_rng(1)
    xi = np.where(np.arange(n) % 2 == 0, 0.5, Nc - 0.5).astype(np.float32)
    vi = np.where(np.arange(n) % 2 == 0, -1.0, 1.0).astype(np.float32)     # every ion hits a wall
    z = np.zeros(0, np.float32)
    load(o, [(z, z, z, z), (xi, vi, 0 * xi, 0 * xi)])
    o.set_E32(np.zeros(Nc + 1, np.float32))
    o.step(1)
    me, mi = o.moments(0), o.moments(1)
    assert mi["absorbed_left"] == n // 2 and mi["absorbed_right"] == n // 2 and mi["count"] == 0
    k = me["injected"]
    assert k == me["count"] and abs(k - 0.1 * n) < 4 * np.sqrt(n * 0.1 * 0.9)
    x, vx = o.debug_get(O.X), o.debug_get(O.VX)
    left = x < 1
    assert np.all(left | (x >= Nc - 1)) and np.all(x < Nc) and np.all(x >= 0)
    assert np.all(vx[left] >= 0) and np.all(vx[~left] <= 0)                # pointing into the plasma
    assert abs(left.mean() - 0.5) < 0.06
    vy = o.debug_get(O.VY)
    # vx = vth sqrt(-2 ln(1-u)) is Rayleigh (flux-weighted half-Maxwellian): <vx^2> = 2 vth^2,
    # <|vx|> = vth sqrt(pi/2); (vy, vz) is a 2-D Maxwellian: <vy^2> = vth^2
    assert abs(np.mean(vx.astype(np.float64) ** 2) / (2 * p["see_vth"] ** 2) - 1) < 0.1
    assert abs(np.mean(np.abs(vx)) / (p["see_vth"] * np.sqrt(np.pi / 2)) - 1) < 0.05
    assert abs(np.mean(vy.astype(np.float64) ** 2) / p["see_vth"] ** 2 - 1) < 0.1
    assert abs(np.mean(vy)) < 4 * p["see_vth"] / np.sqrt(k)


def test_secondary_emission_capacity_drop_keeps_the_first_emitters():
    """The capacity-drop branch of the injection (L41; R10/R19): when the electron arrays fill up,
    the emitters that still fit -- in the order of the absorbed-ion list -- are injected, the rest are counted
    as dropped and the sticky capacity error is raised.  Pinned against the SAME step with room for everybody:
    injected = the free slots exactly, kept electrons = the first `free` of the unlimited run bit for bit,
    injected + dropped = the unlimited run's emitters."""
    Nc, n_i, n_e = 64, 30000, 7900
    xi = np.where(np.arange(n_i) % 3 == 0, 0.5, Nc - 0.5).astype(np.float32)
    vi = np.where(np.arange(n_i) % 3 == 0, -1.0, 1.0).astype(np.float32)   # every ion hits a wall
    xe = (np.arange(n_e, dtype=np.float32) % 60 + 2.25).astype(np.float32)  # electrons at rest, away from the walls
    ze = np.zeros(n_e, np.float32)
    res = {}
    for name, cap_e in (("room", 16384), ("full", 8192)):
        p = params(2, n_cells=Nc, ppc=1, mcc=False, gamma=0.1, capacity_factor=600)
        p["species"][0]["capacity"] = cap_e
        for s in range(2):
            p["species"][s]["kappa"] = 0.0
        o = O.Oracle(p)
        load(o, [(xe, ze, ze, ze), (xi, vi, 0 * xi, 0 * xi)])
        o.set_E32(np.zeros(Nc + 1, np.float32))
        rc = o.step(1)
        m = o.moments(0)
        # the secondaries go through the step's sort with the survivors; no resting electron sits in the two wall
        # cells, so the left-wall secondaries are cell 0 and the right-wall ones cell N_c - 1, each in emission
        # order (the sort is stable).  The ions of cell 0 precede those of cell N_c - 1 in the absorbed list.
        arr = [o.debug_get(w) for w in (O.X, O.VX, O.VY, O.VZ)]
        lft, rgt = arr[0] < 1.0, arr[0] >= Nc - 1.0
        res[name] = (rc, m, [a[lft] for a in arr], int(rgt.sum()))
        assert m["count"] == n_e + m["injected"] and lft.sum() + rgt.sum() == m["injected"]
    (rc_r, m_r, l_r, nr_r), (rc_f, m_f, l_f, nr_f) = res["room"], res["full"]
    free = 8192 - n_e
    assert rc_r == 0 and m_r["dropped"] == 0 and l_r[0].shape[0] > 2 * free and nr_r > 2 * free
    assert rc_f == -2 and m_f["injected"] == free and m_f["dropped"] == m_r["injected"] - free
    assert nr_f == 0                       # the free slots went to the FIRST emitters: all at the left wall
    for a, b in zip(l_r, l_f):
        assert np.array_equal(a[:free], b)


def test_periodic_clamp_faster_than_a_box_length_and_nan():
    """DESIGN.md R21 (L41 says only "removed"/"inserted" for bounded runs; periodic comes from
    BASELINE.json): ONE wrap is applied per step; a particle that is still outside [0, N_c)
    afterwards (|v| > N_c, or a non-finite position) is put at x = 0, so every later array index
    stays inside the grid."""
    Nc = 16
    o = O.Oracle(_one_species(Nc, 0.0, bc=1))
    x0 = np.array([8.0, 8.0, 8.0, 8.0, 8.0, 15.5], np.float32)
    v0 = np.array([20.0, 40.0, -40.0, -20.0, np.inf, 0.5], np.float32)
    tag = np.arange(6, dtype=np.float32)
    load(o, [(x0, v0, tag, tag)])
    o.set_E32(np.zeros(Nc, np.float32))
    o.step(1)
    got = dict(zip(o.debug_get(O.VY).tolist(), o.debug_get(O.X).tolist()))
    #   28 - 16 = 12 | 48 - 16 = 32 -> 0 | -32 + 16 = -16 -> 0 | -12 + 16 = 4 | inf -> 0 | 16 - 16 = 0
    assert got == {0.0: 12.0, 1.0: 0.0, 2.0: 0.0, 3.0: 4.0, 4.0: 0.0, 5.0: 0.0}
    assert o.moments(0)["count"] == 6 and o.moments(0)["absorbed_left"] == 0
    # NaN field -> NaN position -> x = 0 (periodic runs never lose a particle)
    o = O.Oracle(_one_species(Nc, 1.0, bc=1))
    load(o, [(np.array([3.5], np.float32),) + (np.zeros(1, np.float32),) * 3])
    e = np.zeros(Nc, np.float32)
    e[3] = np.nan
    o.set_E32(e)
    o.step(1)
    assert o.debug_get(O.X).tolist() == [0.0] and o.moments(0)["count"] == 1


# ---- f4: electron reflection at the walls (L41; R22) ---------------------------------------
def test_electron_reflection_mirror_positions_order_and_binomial():
    Nc, n = 32, 30000
    rng = np.random.default_rng(4)
    xe = np.where(np.arange(n) % 2 == 0, 0.25, Nc - 0.5).astype(np.float32)
    ve = np.where(np.arange(n) % 2 == 0, -1.0, 2.0).astype(np.float32)      # x' = -0.75 / N_c + 1.5: all cross a wall
    tag = np.arange(n, dtype=np.float32)
    xi = np.full(100, 0.25, np.float32)
    vi = np.full(100, -1.0, np.float32)                                        # ions cross too: never reflected
    for R in (1.0, 0.3, 0.0):
        p = params(2, n_cells=Nc, ppc=1, mcc=False, gamma=0.0, capacity_factor=1200, e_reflect=R)
        for s in range(2):
            p["species"][s]["kappa"] = 0.0
        o = O.Oracle(p)
        load(o, [(xe, ve, tag, tag), (xi, vi, 0 * xi, 0 * xi)])
        o.step(1)
        me, mi = o.moments(0), o.moments(1)
        assert mi["count"] == 0 and mi["reflected"] == 0 and mi["absorbed_left"] == 100
        assert me["reflected"] + me["absorbed_left"] + me["absorbed_right"] == n and me["count"] == me["reflected"]
        if R == 1.0:
            assert me["reflected"] == n
        elif R == 0.0:
            assert me["reflected"] == 0
        else:
            assert abs(me["reflected"] - R * n) < 4 * np.sqrt(n * R * (1 - R))
            assert abs(me["absorbed_left"] - (1 - R) * n / 2) < 4 * np.sqrt(n / 2 * R * (1 - R))
        x, vx, tg = o.debug_get(O.X), o.debug_get(O.VX), o.debug_get(O.VY)
        left = tg % 2 == 0
        assert np.all(x[left] == 0.75) and np.all(vx[left] == 1.0)             # mirror of -0.75, vx reversed
        assert np.all(x[~left] == Nc - 1.5) and np.all(vx[~left] == -2.0)      # mirror of N_c + 1.5 at the wall N_c
        assert np.all(np.diff(tg[left]) > 0) and np.all(np.diff(tg[~left]) > 0)  # survivors keep their order
    # a particle flung further than a box length beyond the wall is absorbed even with R = 1
    p = params(2, n_cells=Nc, ppc=1, mcc=False, gamma=0.0, e_reflect=1.0)
    p["species"][0]["kappa"] = 0.0
    o = O.Oracle(p)
    z = np.zeros(0, np.float32)
    load(o, [(np.array([1.0, 1.0], np.float32), np.array([-40.0, -3.0], np.float32), np.zeros(2, np.float32),
              np.zeros(2, np.float32)), (z, z, z, z)])
    o.step(1)
    assert o.moments(0)["count"] == 1 and o.debug_get(O.X).tolist() == [2.0] and o.moments(0)["absorbed_left"] == 1


def test_reflecting_walls_conserve_electrons_and_their_energy():
    p = params(2, n_cells=64, ppc=50, mcc=False, gamma=0.0, e_reflect=1.0)
    from paper_1104_3998_b200 import workloads as W
    parts = W.make_particles(p)
    for s in range(2):
        p["species"][s]["kappa"] = 0.0          # free streaming between two mirrors
    o = O.Oracle(p)
    load(o, parts)
    e0 = o.moments(0)["sum_v2"]
    o.step(30)
    m = o.moments(0)
    assert m["count"] == 64 * 50 and m["reflected"] > 200 and abs(m["sum_v2"] / e0 - 1) < 1e-12


# ---- moments / EEDF (diagnostics of pic1d_moments) ---------------------------------------------
def test_moments_and_eedf_against_numpy():
    """oracle_moments() against numpy on the arrays debug_get returns: sums of v, |v|^2, |v|^4 over ALL
    live slots (sorted part + birth tail) and the histogram of E = c_eV |v|^2 on [0, E_max)."""
    p = params(2, n_cells=32, ppc=400)
    o = O.Oracle(p)
    from paper_1104_3998_b200 import workloads as W
    p["vth"] = [3 * p["vth"][0], p["vth"][1]]     # 18 eV electrons: ionisation births within 3 steps
    load(o, W.make_particles(p))
    o.step(3)                                     # births in the tail, collided velocities
    for s in range(2):
        n_bins, E_max = 37, (60.0 if s == 0 else 0.2)
        m = o.moments(s, n_bins=n_bins, E_max=E_max)
        v = np.stack([o.debug_get(w, s) for w in (O.VX, O.VY, O.VZ)], 1).astype(np.float64)
        assert m["count"] == v.shape[0] and m["count"] >= m["n_sorted"] > 0
        if s == 0:
            assert m["count"] > m["n_sorted"]     # the case has a birth tail
        g2 = (v ** 2).sum(1)
        for k, want in (("sum_vx", v[:, 0].sum()), ("sum_vy", v[:, 1].sum()), ("sum_vz", v[:, 2].sum())):
            assert abs(m[k] - want) <= 1e-12 * np.abs(v).sum(), k
        assert abs(m["sum_v2"] / g2.sum() - 1) < 1e-12 and abs(m["sum_v4"] / (g2 ** 2).sum() - 1) < 1e-12
        En = p["species"][s]["c_eV"] * g2
        h, _ = np.histogram(En[En < E_max], bins=n_bins, range=(0.0, E_max))
        assert m["eedf"].sum() == (En < E_max).sum() > 0
        # bin edges are floating-point: allow a particle sitting on an edge to fall either side
        assert np.abs(np.cumsum(m["eedf"]) - np.cumsum(h)).max() <= 1
        dens = m["density"]
        assert dens.sum() == m["n_sorted"]        # density = rho_s of the last deposit (sorted part only)
    # a Maxwellian's moments: <v^2> = 3 vth^2, <v^4> = 15 vth^4 (fresh load, nothing collided yet)
    o = O.Oracle(p)
    load(o, W.make_particles(p))
    m = o.moments(1)
    assert m["count"] == m["n_sorted"] == p["n_per_species"]
    vt = p["vth"][1]
    assert abs(m["sum_v2"] / m["count"] / (3 * vt ** 2) - 1) < 0.03
    assert abs(m["sum_v4"] / m["count"] / (15 * vt ** 4) - 1) < 0.08


# ---- P8 sort ---------------------------------------------------------------------------------
@pytest.mark.parametrize("inv_ratio", [2.0, 1.0, 0.5, 0.0625])
def test_sort_is_stable_permutation_with_bruteforce_offsets(inv_ratio):
    Nc, n = 32, 3000
    rng = np.random.default_rng(11)
    o = O.Oracle(_one_species(Nc, 0.0, inv_ratio=inv_ratio))
    x0 = (rng.random(n, dtype=np.float32) * Nc).astype(np.float32)
    x0[:5] = [0.0, 31.999, 16.0, 15.999, 0.5]
    v0 = rng.normal(size=n).astype(np.float32) * 3
    tag = np.arange(n, dtype=np.float32)
    load(o, [(x0, v0, tag, -tag)])
    o.set_E32(np.zeros(Nc + 1, np.float32))
    # after load: stable sort of the input by key
    for it in range(2):
        xs, vs, tg, tz = (o.debug_get(w) for w in (O.X, O.VX, O.VY, O.VZ))
        off = o.debug_get(O.OFFSETS)
        n_sc = int(np.ceil(Nc * inv_ratio))
        assert off.shape[0] == n_sc + 1 and off[0] == 0 and off[-1] == xs.shape[0]
        keys = np.floor(xs.astype(np.float64) * inv_ratio).astype(np.int64)
        assert np.all(np.diff(keys) >= 0)
        assert np.array_equal(off, [(keys < k).sum() for k in range(n_sc + 1)])
        assert np.array_equal(tg, -tz)                         # 4-tuples stay together
        if it == 0:
            assert np.array_equal(np.sort(tg), tag)            # permutation
            for k in range(n_sc):
                seg = tg[off[k]:off[k + 1]]
                assert np.all(np.diff(seg) > 0)                # stable: source order kept
            order = np.argsort(np.floor(x0.astype(np.float64) * inv_ratio), kind="stable")
            assert np.array_equal(tg, tag[order]) and np.array_equal(xs, x0[order])
            prev = (xs.copy(), vs.copy(), tg.copy())
            o.step(1)
        else:
            # second pass: survivors of a real push, again stable w.r.t. the previous order
            px, pv, pt = prev
            nx = px + pv
            alive = (nx >= 0) & (nx < Nc)
            order = np.argsort(np.floor(nx[alive].astype(np.float64) * inv_ratio), kind="stable")
            assert np.array_equal(tg, pt[alive][order]) and np.array_equal(xs, nx[alive][order])
