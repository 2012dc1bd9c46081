"""Seeded synthetic workloads shaped like the paper's argon discharges (BASELINE.json configs 0-4).

This module serves BOTH the oracle and the CUDA path and therefore holds none of the method's
arithmetic: it only turns physical inputs (gap, grid, pressure, voltages) into the normalised
parameter set of PAPER.md section 3.3 (L79-124) and draws seeded initial particle arrays with
numpy.  Recipe and constants: DESIGN.md "Inputs"; SURVEY.md section 8(d) D1/D2.
"""
import math

import numpy as np

# CODATA 2018
QE = 1.602176634e-19
EPS0 = 8.8541878128e-12
ME = 9.1093837015e-31
KB = 1.380649e-23
M_AR = 6.6334e-26          # Ar+ mass [kg]
N0 = 1.0e14                # initial plasma density [m^-3]   (R20)
A_E = 1.0                  # electrode area [m^2]
E_CAP = 500.0              # energy cap for nu_max [eV]       (R11)
GAP = 0.025                # electrode gap [m]
F_RF = 13.56e6
DX_COURANT = GAP / 128     # cell size of config 0; used by the Courant-respecting twins

SIG_EL, SIG_EXC0, E_EXC, SIG_ION0, E_ION, SIG_CX = 1e-19, 1e-21, 11.5, 3e-21, 15.8, 5e-19

CONFIGS = {
    0: dict(name="cfg0_tiny_bounded", n_cells=128, ppc=64, dt=1e-11, bc=0, V0=0.0, p_Pa=10.0,
            gamma=0.0, Te=2.0, Ti=0.026, steps=100, seed=1, ions=True, mcc=True),
    1: dict(name="cfg1_cold_plasma_periodic", n_cells=512, ppc=2000, dt=None, bc=1, V0=0.0,
            p_Pa=0.0, gamma=0.0, Te=0.0, Ti=0.0, steps=1000, seed=0, ions=False, mcc=False),
    2: dict(name="cfg2_rf_ccp", n_cells=1024, ppc=200, dt=1.0 / (400 * F_RF), bc=0, V0=200.0,
            p_Pa=10.0, gamma=0.1, Te=2.0, Ti=0.026, steps=2000, seed=7, ions=True, mcc=True),
    3: dict(name="cfg3_sort_sweep", n_cells=4096, ppc=1000, dt=1.0 / (400 * F_RF), bc=0, V0=200.0,
            p_Pa=10.0, gamma=0.1, Te=2.0, Ti=0.026, steps=500, seed=7, ions=True, mcc=True),
    4: dict(name="cfg4_large_stress", n_cells=16384, ppc=4000, dt=1.0 / (400 * F_RF), bc=0,
            V0=200.0, p_Pa=20.0, gamma=0.1, Te=2.0, Ti=0.026, steps=200, seed=7, ions=True,
            mcc=True),
}


def _round_up(n, m):
    return (n + m - 1) // m * m


LN_LAMBDA = 10.0           # Coulomb logarithm of the binary collisions (f3)


def make_params(cfg_id, n_cells=None, ppc=None, sort_ratio=1.0, courant=False, seed=None,
                capacity_factor=1.25, flags=0, mcc=None, gamma=None, coulomb=False, e_reflect=0.0):
    """Normalised parameter dict for config `cfg_id` (optionally scaled by n_cells / ppc).

    courant=True gives the Courant-respecting twin (same N_c, ppc, dt; dx = config 0's), see
    DESIGN.md "Inputs".
    """
    c = dict(CONFIGS[cfg_id])
    if n_cells is not None:
        c["n_cells"] = n_cells
    if ppc is not None:
        c["ppc"] = ppc
    if seed is not None:
        c["seed"] = seed
    if mcc is not None:
        c["mcc"] = mcc
    if gamma is not None:
        c["gamma"] = gamma
    Nc, ppc_ = c["n_cells"], c["ppc"]
    n_per_species = Nc * ppc_
    cap = _round_up(int(math.ceil(capacity_factor * n_per_species)) + 4096, 4096)
    p = dict(cfg_id=cfg_id, name=c["name"], n_cells=Nc, ppc=ppc_, bc=c["bc"], steps=c["steps"],
             n_per_species=n_per_species, sort_ratio=float(sort_ratio),
             sort_inv_ratio=1.0 / float(sort_ratio), seed=int(c["seed"]), flags=int(flags),
             courant=bool(courant), e_reflect=float(e_reflect), coul_A=[0.0, 0.0])
    # performance hint for the library (PIC1D_FLAG_EQ5_ELECTRONS = 4): electron thermal displacement below
    # one cell per step -- configs 0, 1 and the Courant-respecting twins
    if cfg_id in (0, 1) or courant:
        p["flags"] |= 4
    if cfg_id == 1:
        wpdt = 0.1
        p.update(n_species=1, background_rho=float(ppc_), V0_norm=0.0, omega_dt=0.0,
                 see_gamma=0.0, see_vth=0.0, r_el=0.0, r_exc=0.0, r_ion=0.0, E_exc=E_EXC,
                 E_ion=E_ION, gas_vth_ion=0.0, mass_ratio=ME / M_AR, wpdt=wpdt, vth=[0.0],
                 species=[dict(kappa=-(wpdt ** 2) / ppc_, c_eV=1.0, P0=0.0, inv_g_cap=0.0,
                               capacity=cap, charge_sign=-1, mcc_kind=0)])
        return p
    dt = c["dt"]
    dx = DX_COURANT if courant else GAP / Nc
    w = N0 * A_E * dx / ppc_                    # real particles per super-particle
    n_g = c["p_Pa"] / (KB * 300.0)
    species = []
    vth = []
    for (m, sign, T, kind) in ((ME, -1, c["Te"], 1), (M_AR, +1, c["Ti"], 2)):
        kappa = sign * QE * QE * w * dt * dt / (EPS0 * dx * m * A_E)        # Eq. 3 (L119)
        c_eV = 0.5 * m * (dx / dt) ** 2 / QE
        g_cap = math.sqrt(E_CAP / c_eV)                                    # cells/step
        v_cap = g_cap * dx / dt                                            # m/s
        if kind == 1:
            sig_cap = SIG_EL + SIG_EXC0 * (1 - E_EXC / E_CAP) + SIG_ION0 * (1 - E_ION / E_CAP)
        else:
            sig_cap = SIG_CX
        nu_max = n_g * sig_cap * v_cap
        P0 = 1.0 - math.exp(-nu_max * dt)                                  # Eq. 6 (L200)
        species.append(dict(kappa=kappa, c_eV=c_eV, P0=P0 if c["mcc"] else 0.0,
                            inv_g_cap=1.0 / g_cap, capacity=cap, charge_sign=sign,
                            mcc_kind=kind if c["mcc"] else 0, g_cap=g_cap, nu_max=nu_max))
        vth.append(math.sqrt(QE * T / m) * dt / dx)
        if coulomb:
            # Takizuka-Abe: <tan^2(theta/2)> = q^4 n_L lnL dt / (8 pi eps0^2 m_r^2 u^3), m_r = m / 2, with
            # n_L = n_cell w / (A_e r dx) and u in cells/step: coul_A multiplies n_cell / u^3
            m_r = 0.5 * m
            p["coul_A"][len(vth) - 1] = (QE ** 4 * LN_LAMBDA * dt * w / (8.0 * math.pi * EPS0 ** 2 * m_r ** 2 * A_E * sort_ratio * dx)
                                         * (dt / dx) ** 3)
    sig_cap_e = SIG_EL + SIG_EXC0 * (1 - E_EXC / E_CAP) + SIG_ION0 * (1 - E_ION / E_CAP)
    p.update(n_species=2, background_rho=0.0,
             V0_norm=c["V0"] * EPS0 * A_E / (QE * w * dx),
             omega_dt=2.0 * math.pi * F_RF * dt if c["V0"] != 0.0 else 0.0,
             see_gamma=c["gamma"], see_vth=math.sqrt(QE * 1.0 / ME) * dt / dx,
             r_el=SIG_EL / sig_cap_e, r_exc=SIG_EXC0 / sig_cap_e, r_ion=SIG_ION0 / sig_cap_e,
             E_exc=E_EXC, E_ion=E_ION, gas_vth_ion=math.sqrt(KB * 300.0 / M_AR) * dt / dx,
             mass_ratio=ME / M_AR, species=species, vth=vth, dx=dx, dt=dt,
             wpe_dt=math.sqrt(N0 * QE * QE / (EPS0 * ME)) * dt)
    return p


def make_particles(params):
    """[(x, vx, vy, vz)] fp32 arrays per species, from numpy.random.default_rng(seed)."""
    Nc, n = params["n_cells"], params["n_per_species"]
    out = []
    if params["cfg_id"] == 1:
        # quiet start: x_i = s_i + 0.01 sin(2 pi s_i / N_c), s_i = (i + 1/2) / ppc
        s = (np.arange(n, dtype=np.float64) + 0.5) / params["ppc"]
        x = s + 0.01 * np.sin(2.0 * np.pi * s / Nc)
        x = np.mod(x, Nc).astype(np.float32)
        x[x >= Nc] = 0.0
        z = np.zeros(n, dtype=np.float32)
        return [(x, z.copy(), z.copy(), z.copy())]
    rng = np.random.default_rng(params["seed"])
    top = np.nextafter(np.float32(Nc), np.float32(0))
    for s in range(params["n_species"]):
        x = (rng.random(n, dtype=np.float32) * np.float32(Nc)).astype(np.float32)
        np.minimum(x, top, out=x)
        v = [(rng.standard_normal(n, dtype=np.float32) * np.float32(params["vth"][s]))
             for _ in range(3)]
        out.append((x, v[0], v[1], v[2]))
    return out
