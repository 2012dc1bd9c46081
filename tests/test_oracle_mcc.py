"""P9 / P10 -- oracle null-collision MCC (L196-209, Eq. 6) statistics and kinematic invariants.
Selection and kinematics: DESIGN.md R11-R14."""
import numpy as np

from oracle import oracle as O
from helpers import params, load


def _beam(energy_eV, n=60000, species=0, **over):
    """n particles of one species at rest in x (vx = 0), speed along +y, so nobody moves."""
    p = params(2, n_cells=8, ppc=1, gamma=0.0, capacity_factor=40000, **over)
    g = np.sqrt(energy_eV / p["species"][species]["c_eV"])
    x = (np.arange(n, dtype=np.float32) % 8 + 0.5).astype(np.float32)
    z = np.zeros(n, np.float32)
    part = (x, z, np.full(n, g, np.float32), z)
    empty = (np.zeros(0, np.float32),) * 4
    for s in range(2):
        p["species"][s]["kappa"] = 0.0            # no field push: the beam stays a beam
    o = O.Oracle(p)
    load(o, [part, empty] if species == 0 else [empty, part])
    return o, p, g


def test_null_collision_candidate_rate_eq6():
    o, p, g = _beam(3.0)
    n = o.moments(0)["count"]
    o.step(1)
    m = o.moments(0)
    P0 = np.float32(p["species"][0]["P0"])
    assert abs(m["n_candidates"] - n * P0) < 4 * np.sqrt(n * P0 * (1 - P0))      # Eq. 6: N0 = P0 N_p
    assert sum(m["n_events"]) == m["n_candidates"]
    mask = o.debug_get(O.MASK)
    assert [(mask == k).sum() for k in (1, 2, 3)] == m["n_events"][1:]


def test_beam_fractions_follow_sigma_v_over_numax():
    """mono-energetic beam: the fraction of particles that suffer process k in one step is
    P0 nu_k(E) / nu_max (Eq. 6: N0 = P0 N_p enter the selection, which accepts process k
    with probability nu_k / nu_max).  The expected value is built HERE from the physical inputs of
    BASELINE.json config 2 -- n_g = p / (k_B T), the synthetic sigma_k(E), v = sqrt(2 E / m), dt --
    and not from the normalised ratios the oracle is handed."""
    kB, qe, me = 1.380649e-23, 1.602176634e-19, 9.1093837015e-31
    n_g = 10.0 / (kB * 300.0)                      # 10 Pa, 300 K
    dt = 1.0 / (400 * 13.56e6)
    E_cap = 500.0                                  # DESIGN.md R11
    sig = lambda E: (1e-19, 1e-21 * max(0.0, 1 - 11.5 / E), 3e-21 * max(0.0, 1 - 15.8 / E))
    speed = lambda E: np.sqrt(2 * E * qe / me)
    nu_max = n_g * sum(sig(E_cap)) * speed(E_cap)
    P0 = 1 - np.exp(-nu_max * dt)
    n = 200000
    for E in (3.0, 14.0, 60.0, 200.0):
        o, p, g = _beam(E, n=n)
        o.step(1)
        m = o.moments(0)
        want = [P0 * n_g * s_k * speed(E) / nu_max for s_k in sig(E)]
        for k, w in enumerate(want, start=1):
            assert abs(m["n_events"][k] - n * w) <= 4.5 * np.sqrt(n * w * (1 - w)) + 1e-9, (E, k, m["n_events"][k], n * w)
        # the null-collision fraction itself (Eq. 6)
        assert abs(m["n_candidates"] - n * P0) <= 4.5 * np.sqrt(n * P0 * (1 - P0))
        # and the method agrees with the exact per-step probability 1 - exp(-nu dt) to first order in
        # nu_max dt (0.61 here): the ratio is P0 / (nu_max dt) (1 + O(nu dt)) -- checked, not assumed
        nu_el = n_g * sig(E)[0] * speed(E)
        exact = 1 - np.exp(-nu_el * dt)
        assert abs(want[0] / exact / (P0 / (nu_max * dt)) - 1) < 0.6 * nu_el * dt + 1e-3


def test_electron_kinematics_invariants():
    E0 = 40.0
    o, p, g = _beam(E0, n=120000)
    c_e = p["species"][0]["c_eV"]
    o.step(1)
    mask = o.debug_get(O.MASK)
    n_s = mask.shape[0]
    v = np.stack([o.debug_get(w)[:n_s] for w in (O.VX, O.VY, O.VZ)], 1).astype(np.float64)
    sp = np.linalg.norm(v, axis=1)
    En = c_e * sp ** 2
    assert np.allclose(En[mask == 0], E0, rtol=1e-5)                   # untouched
    el = mask == 1
    cchi = v[el, 1] / sp[el]                                           # incoming direction = +y
    assert np.allclose(sp[el] / g, np.sqrt(1 - 2 * p["mass_ratio"] * (1 - cchi)), rtol=2e-6)
    nhat = v[el] / sp[el, None]
    assert np.all(np.abs(nhat.mean(0)) < 4 / np.sqrt(3 * el.sum()))    # isotropic
    assert abs(np.mean(nhat[:, 0] ** 2) - 1 / 3) < 0.03
    assert np.allclose(En[mask == 2], E0 - 11.5, rtol=1e-5)            # excitation loss
    ion = mask == 3
    m_e, m_i = o.moments(0), o.moments(1)
    nb = int(ion.sum())
    assert nb > 50 and m_e["births"] == nb == m_i["births"] == m_i["count"]
    assert m_e["count"] == n_s + nb
    tail = np.stack([o.debug_get(w)[n_s:] for w in (O.VX, O.VY, O.VZ)], 1).astype(np.float64)
    E_tail = c_e * (tail ** 2).sum(1)
    assert np.allclose(En[ion] + E_tail, E0 - 15.8, rtol=1e-5)         # energy bookkeeping, in order
    # births sit at the parent's x, appended in ascending parent-slot order (L203)
    assert np.array_equal(o.debug_get(O.X)[n_s:], o.debug_get(O.X)[:n_s][ion])
    assert np.array_equal(o.debug_get(O.X, 1), o.debug_get(O.X)[:n_s][ion])
    # net charge unchanged by a co-located pair: deposit after the NEXT step's sort still neutral
    vi = np.stack([o.debug_get(w, 1) for w in (O.VX, O.VY, O.VZ)], 1).astype(np.float64)
    assert abs(vi.std() / p["gas_vth_ion"] - 1) < 5 / np.sqrt(2 * 3 * nb) + 0.02


def test_ion_charge_exchange_maxwellian():
    o, p, g = _beam(400.0, n=200000, species=1)
    o.step(1)
    m = o.moments(1)
    a = min(1.0, g * p["species"][1]["inv_g_cap"])
    P0 = p["species"][1]["P0"]
    n = 200000
    assert abs(m["n_candidates"] - n * P0) < 4 * np.sqrt(n * P0)
    assert abs(m["n_events"][1] - n * P0 * a) < 4 * np.sqrt(n * P0 * a)
    mask = o.debug_get(O.MASK, 1).astype(bool)
    v = np.stack([o.debug_get(w, 1) for w in (O.VX, O.VY, O.VZ)], 1).astype(np.float64)
    assert np.allclose(np.linalg.norm(v[~mask], axis=1), g, rtol=1e-6)
    k = mask.sum()
    vt = p["gas_vth_ion"]
    assert np.all(np.abs(v[mask].mean(0)) < 4.5 * vt / np.sqrt(k))
    assert np.all(np.abs(v[mask].var(0) / vt ** 2 - 1) < 5 * np.sqrt(2 / k))


def test_ionisation_pair_keeps_rho_neutral():
    o, p, g = _beam(80.0, n=50000)
    rho0, _, _ = o.get_rho_phi_E()
    o.step(1)
    o.step(1)                    # births of step 0 are sorted and deposited in step 1
    me, mi = o.moments(0), o.moments(1)
    assert mi["count"] > 0
    assert me["density"].sum() - mi["density"].sum() == 50000 - (me["absorbed_left"] + me["absorbed_right"])


def test_ionisation_capacity_drop_keeps_the_first_births():
    """The capacity-drop branch of the ionisation births (L203; R14): a pair is born only while BOTH
    arrays have a free slot; the births that fit are the ones of the lowest parent slots, the rest are counted as
    dropped (once per species) and the sticky capacity error is raised; the parent's own collision happens either
    way.  Pinned against the SAME step with room for everybody."""
    n = 12288 - 20                           # ~50 ionisations per step at this pressure: 20 slots do not hold them
    res = {}
    for name, cap_e in (("room", 16384), ("full", 12288)):
        o, p, g = _beam(60.0, n=n)           # well above the ionisation threshold
        o.close()
        p["species"][0]["capacity"] = cap_e
        p["species"][1]["capacity"] = 4096 * 4
        o = O.Oracle(p)
        x = (np.arange(n, dtype=np.float32) % 8 + 0.5).astype(np.float32)
        z = np.zeros(n, np.float32)
        empty = (np.zeros(0, np.float32),) * 4
        load(o, [(x, z, np.full(n, g, np.float32), z), empty])
        rc = o.step(1)
        me, mi = o.moments(0), o.moments(1)
        arr = [o.debug_get(w, 0) for w in (O.X, O.VX, O.VY, O.VZ)]
        ions = [o.debug_get(w, 1) for w in (O.X, O.VX, O.VY, O.VZ)]
        res[name] = (rc, me, mi, arr, ions, o.debug_get(O.MASK, 0))
    (rc_r, me_r, mi_r, a_r, i_r, k_r), (rc_f, me_f, mi_f, a_f, i_f, k_f) = res["room"], res["full"]
    free = 12288 - n
    assert rc_r == 0 and me_r["dropped"] == 0 and me_r["births"] == me_r["n_events"][3] > 2 * free
    assert rc_f == -2 and me_f["births"] == free and mi_f["births"] == free
    assert me_f["dropped"] == me_r["births"] - free and mi_f["dropped"] == me_f["dropped"]
    assert np.array_equal(k_r, k_f) and me_f["n_events"] == me_r["n_events"]     # every parent still collides
    assert me_f["count"] == n + free and mi_f["count"] == free
    for a, b in zip(a_r, a_f):          # parents (all n slots) and the first `free` new electrons: identical
        assert np.array_equal(a[:n + free], b)
    for a, b in zip(i_r, i_f):
        assert np.array_equal(a[:free], b)
