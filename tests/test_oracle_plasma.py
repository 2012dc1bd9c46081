"""P6 -- the whole collisionless loop of the oracle: cold-plasma oscillation at omega_p (config 1,
scaled in ppc) and momentum conservation of a periodic run."""
import numpy as np

from oracle import oracle as O
from paper_1104_3998_b200 import workloads as W
from helpers import load


def _mode1(E):
    k = 2 * np.pi * np.arange(E.shape[0]) / E.shape[0]
    return 2 * np.mean(E * np.cos(k)), 2 * np.mean(E * np.sin(k))


def test_cold_plasma_frequency_within_1pct_of_omega_p():
    p = W.make_params(1, ppc=100)
    o = O.Oracle(p)
    load(o, W.make_particles(p))
    steps = 1000
    amp = np.zeros(steps + 1)
    _, _, E = o.get_rho_phi_E()
    amp[0] = _mode1(E)[1]
    mom = []
    for n in range(1, steps + 1):
        o.step(1)
        _, _, E = o.get_rho_phi_E()
        amp[n] = _mode1(E)[1]
        if n % 100 == 0:
            mom.append(o.moments(0)["sum_vx"])
    assert np.abs(amp).max() > 0
    # zero crossings of the mode-1 amplitude, linearly interpolated
    zc = np.nonzero(amp[:-1] * amp[1:] < 0)[0]
    tz = zc + amp[zc] / (amp[zc] - amp[zc + 1])
    w = np.pi / np.mean(np.diff(tz))               # rad per step
    assert len(zc) >= 30
    assert abs(w / p["wpdt"] - 1) < 0.01                                  # north_star: within 1 %
    assert abs(w / (2 * np.arcsin(p["wpdt"] / 2)) - 1) < 2e-3              # leapfrog dispersion
    # amplitude stays put (no damping / growth in a cold collisionless plasma)
    pk = np.abs(amp[:200]).max(), np.abs(amp[-200:]).max()
    assert abs(pk[1] / pk[0] - 1) < 0.02
    # total momentum: same weighting for gather and deposit => conserved up to fp32 rounding
    vmax = 0.01 * p["wpdt"]
    assert np.max(np.abs(mom)) < 1e-4 * vmax * p["n_per_species"]
