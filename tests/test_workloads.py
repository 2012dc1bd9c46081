"""Input generator vs the constants table of SURVEY.md 8(d)-D2 (tests/golden/constants_D2.txt)."""
import os

import numpy as np

from paper_1104_3998_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden", "constants_D2.txt")


def test_constants_match_survey_table():
    for line in open(GOLD):
        if line.startswith("#") or not line.strip():
            continue
        t = line.split()
        cfg = int(t[0])
        g = [float(v) for v in t[1:]]
        p = W.make_params(cfg)
        e, i = p["species"]
        got = [p["wpe_dt"], e["kappa"], i["kappa"], e["c_eV"], i["c_eV"], e["P0"], i["P0"],
               e["g_cap"], p["vth"][0], p["vth"][1], p["see_vth"], p["gas_vth_ion"], p["V0_norm"]]
        for a, b in zip(got, g):
            assert abs(a - b) <= 6e-3 * abs(b) + 1e-300, (cfg, a, b)


def test_particles_seeded_and_in_range():
    p = W.make_params(0)
    a = W.make_particles(p)
    b = W.make_particles(p)
    for (xa, *va), (xb, *vb) in zip(a, b):
        assert np.array_equal(xa, xb) and all(np.array_equal(u, v) for u, v in zip(va, vb))
        assert xa.dtype == np.float32 and xa.min() >= 0 and xa.max() < p["n_cells"]
    assert abs(np.std(a[0][1]) / p["vth"][0] - 1) < 0.05


def test_quiet_start_config1():
    p = W.make_params(1, ppc=50)
    (x, vx, vy, vz), = W.make_particles(p)
    assert x.shape[0] == 512 * 50 and not vx.any()
    s = (np.arange(x.shape[0]) + 0.5) / 50
    assert np.max(np.abs(x - s)) <= 0.01 + 1e-4
    assert p["species"][0]["kappa"] == -(0.1 ** 2) / 50 and p["background_rho"] == 50
