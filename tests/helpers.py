"""Shared test helpers: parameter dicts for small cases, comparison utilities."""
import copy

import numpy as np

from paper_1104_3998_b200 import workloads as W


def params(cfg_id=0, **kw):
    over = {k: kw.pop(k) for k in list(kw) if k in (
        "bc", "background_rho", "V0_norm", "omega_dt", "see_gamma", "see_vth", "r_el", "r_exc",
        "r_ion", "E_exc", "E_ion", "gas_vth_ion", "mass_ratio", "n_species", "coul_A")}
    sp_over = kw.pop("species_over", None)
    p = copy.deepcopy(W.make_params(cfg_id, **kw))
    p.update(over)
    if sp_over:
        for s, d in sp_over.items():
            p["species"][s].update(d)
    if "n_species" in over:
        p["species"] = p["species"][:over["n_species"]]
    return p


def load(sim, parts):
    for s, a in enumerate(parts):
        sim.load_particles(s, *a)


def rel_linf(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    d = np.max(np.abs(a - b)) if a.size else 0.0
    return d / max(np.max(np.abs(b)) if b.size else 0.0, 1e-300)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)
