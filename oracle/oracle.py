"""ctypes wrapper around oracle/pic1d_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
may import this module.  It imports nothing from paper_1104_3998_b200 (the CUDA path) and
the CUDA path imports nothing from here.  The arithmetic lives in pic1d_oracle.c; this file
only marshals arguments.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "pic1d_oracle.c")
_LIB = os.path.join(_HERE, "libpic1d_oracle.so")

X, VX, VY, VZ, KEYS, OFFSETS, MASK, E32, RHO_S, PARTNER = range(10)
_DTYPES = {X: np.float32, VX: np.float32, VY: np.float32, VZ: np.float32, KEYS: np.int32,
           OFFSETS: np.int32, MASK: np.uint8, E32: np.float32, RHO_S: np.float64, PARTNER: np.int32}


_EXTRA = os.environ.get("ORACLE_CFLAGS", "").split()  # e.g. -fsanitize=address,undefined -g (profiles/r2_sanitizers.md)
if _EXTRA:
    _LIB = os.path.join(_HERE, "libpic1d_oracle_san.so")   # an instrumented build never replaces the plain one


def build(force=False):
    """gcc -O2 -ffp-contract=off: every fp32 op is the IEEE op that is written."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math"] + _EXTRA +
                              ["-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


class SpeciesCfg(C.Structure):
    _fields_ = [("kappa", C.c_double), ("c_eV", C.c_double), ("P0", C.c_double),
                ("inv_g_cap", C.c_double), ("capacity", C.c_int64),
                ("charge_sign", C.c_int32), ("mcc_kind", C.c_int32)]


class Config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_cells", C.c_int32), ("bc", C.c_int32),
                ("n_species", C.c_int32), ("sp", SpeciesCfg * 2),
                ("background_rho", C.c_double), ("sort_inv_ratio", C.c_double),
                ("V0_norm", C.c_double), ("omega_dt", C.c_double),
                ("see_gamma", C.c_double), ("see_vth", C.c_double),
                ("r_el", C.c_double), ("r_exc", C.c_double), ("r_ion", C.c_double),
                ("E_exc", C.c_double), ("E_ion", C.c_double),
                ("gas_vth_ion", C.c_double), ("mass_ratio", C.c_double),
                ("seed", C.c_uint64), ("flags", C.c_uint32), ("pad_", C.c_uint32),
                ("e_reflect", C.c_double), ("coul_A", C.c_double * 2)]


class Moments(C.Structure):
    _fields_ = [("count", C.c_int64), ("n_sorted", C.c_int64),
                ("sum_vx", C.c_double), ("sum_vy", C.c_double), ("sum_vz", C.c_double),
                ("sum_v2", C.c_double), ("sum_v4", C.c_double),
                ("absorbed_left", C.c_int64), ("absorbed_right", C.c_int64),
                ("injected", C.c_int64), ("n_candidates", C.c_int64),
                ("n_events", C.c_int64 * 4), ("births", C.c_int64),
                ("dropped", C.c_int64), ("over_cap", C.c_int64),
                ("reflected", C.c_int64), ("n_pairs", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.oracle_debug_count.restype = C.c_int64
        _lib.oracle_step_index.restype = C.c_uint32
    return _lib


def make_config(params):
    """params: the plain dict produced by the workload generators (numbers only)."""
    c = Config()
    c.struct_size = C.sizeof(Config)
    for k in ("n_cells", "bc", "n_species", "background_rho", "sort_inv_ratio", "V0_norm",
              "omega_dt", "see_gamma", "see_vth", "r_el", "r_exc", "r_ion", "E_exc", "E_ion",
              "gas_vth_ion", "mass_ratio", "seed", "flags"):
        setattr(c, k, params[k])
    c.e_reflect = params.get("e_reflect", 0.0)
    for s, a in enumerate(params.get("coul_A", [])):
        c.coul_A[s] = a
    for s, sp in enumerate(params["species"]):
        for k in ("kappa", "c_eV", "P0", "inv_g_cap", "capacity", "charge_sign", "mcc_kind"):
            setattr(c.sp[s], k, sp[k])
    return c


def _fp(a):
    return a.ctypes.data_as(C.c_void_p)


class Oracle:
    def __init__(self, params):
        self.cfg = make_config(params)
        self.h = C.c_void_p()
        rc = lib().oracle_create(C.byref(self.cfg), C.byref(self.h))
        if rc != 0:
            raise ValueError("oracle_create failed: %d" % rc)
        self.n_nodes = lib().oracle_n_nodes(self.h)
        self.n_sc = lib().oracle_n_sort_cells(self.h)

    def close(self):
        if self.h:
            lib().oracle_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def load_particles(self, s, x, vx, vy, vz):
        arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in (x, vx, vy, vz)]
        n = arrs[0].shape[0]
        rc = lib().oracle_load_particles(self.h, C.c_int(s), C.c_int64(n), *[_fp(a) for a in arrs])
        if rc != 0:
            raise ValueError("oracle_load_particles failed: %d" % rc)

    def step(self, n_steps=1):
        return lib().oracle_step(self.h, C.c_int(n_steps))

    def get_rho_phi_E(self):
        out = [np.zeros(self.n_nodes, dtype=np.float64) for _ in range(3)]
        lib().oracle_get_rho_phi_E(self.h, *[_fp(a) for a in out], C.c_int(self.n_nodes))
        return tuple(out)

    def moments(self, s, n_bins=0, E_max=0.0):
        m = Moments()
        dens = np.zeros(self.n_nodes, dtype=np.float64)
        eedf = np.zeros(max(n_bins, 1), dtype=np.int64)
        rc = lib().oracle_moments(self.h, C.c_int(s), C.byref(m), _fp(dens), C.c_int(self.n_nodes),
                                  _fp(eedf) if n_bins > 0 else None, C.c_int(n_bins),
                                  C.c_double(E_max))
        if rc == -1:
            raise ValueError("oracle_moments failed")
        d = {k: getattr(m, k) for k, _ in Moments._fields_ if k != "n_events"}
        d["n_events"] = list(m.n_events)
        d["density"] = dens
        d["eedf"] = eedf[:n_bins]
        return d

    def debug_get(self, what, s=0):
        n = lib().oracle_debug_count(self.h, C.c_int(what), C.c_int(s))
        out = np.zeros(int(n), dtype=_DTYPES[what])
        rc = lib().oracle_debug_get(self.h, C.c_int(what), C.c_int(s), _fp(out),
                                    C.c_size_t(out.nbytes))
        if rc != 0:
            raise ValueError("oracle_debug_get failed")
        return out

    def set_E32(self, e32):
        a = np.ascontiguousarray(e32, dtype=np.float32)
        rc = lib().oracle_debug_set_E32(self.h, _fp(a), C.c_int(a.shape[0]))
        if rc != 0:
            raise ValueError("oracle_debug_set_E32 failed")

    @property
    def step_index(self):
        return int(lib().oracle_step_index(self.h))


def philox(seed, c0, c1, c2, c3):
    out = (C.c_uint32 * 4)()
    lib().oracle_philox(C.c_uint64(seed), C.c_uint32(c0), C.c_uint32(c1), C.c_uint32(c2),
                        C.c_uint32(c3), out)
    return [int(v) for v in out]


def solve_field(n_cells, bc, rho, phi0=0.0, phiN=0.0):
    nodes = n_cells if bc == 1 else n_cells + 1
    rho = np.ascontiguousarray(rho, dtype=np.float64)
    assert rho.shape[0] == nodes
    phi = np.zeros(nodes + 1, dtype=np.float64)
    E = np.zeros(nodes + 1, dtype=np.float64)
    lib().oracle_solve_field(C.c_int(n_cells), C.c_int(bc), _fp(rho), C.c_double(phi0),
                             C.c_double(phiN), _fp(phi), _fp(E))
    return phi[:nodes], E[:nodes]


class Gapped:
    """the paper's gapped in-place fine sort (f2), stated step by step in pic1d_oracle.c"""

    def __init__(self, n_cells, sort_inv_ratio, n_max, kappa):
        self.h = C.c_void_p()
        rc = lib().oracle_gapped_create(C.c_int(n_cells), C.c_double(sort_inv_ratio), C.c_int(n_max),
                                        C.c_double(kappa), C.byref(self.h))
        if rc:
            raise ValueError("oracle_gapped_create failed")
        self.n_cells, self.n_max = n_cells, n_max
        self.n_sc = lib().oracle_gapped_n_sort_cells(self.h)

    def close(self):
        if self.h:
            lib().oracle_gapped_destroy(self.h)
            self.h = C.c_void_p()

    def load(self, x, vx, vy, vz):
        a = [np.ascontiguousarray(v, dtype=np.float32) for v in (x, vx, vy, vz)]
        return lib().oracle_gapped_load(self.h, C.c_int64(a[0].shape[0]), *[_fp(v) for v in a])

    def set_E32(self, e32):
        a = np.ascontiguousarray(e32, dtype=np.float32)
        assert lib().oracle_gapped_set_E32(self.h, _fp(a), C.c_int(a.shape[0])) == 0

    def step(self):
        return lib().oracle_gapped_step(self.h)

    def get(self):
        """(N_i, [x, vx, vy, vz] as (n_sc, n_max) arrays, stats dict)"""
        N = np.zeros(self.n_sc, np.int32)
        arr = [np.zeros((self.n_sc, self.n_max), np.float32) for _ in range(4)]
        st = np.zeros(4, np.int64)
        rc = lib().oracle_gapped_get(self.h, _fp(N), *[_fp(a) for a in arr], _fp(st))
        return N, arr, dict(absorbed_left=int(st[0]), absorbed_right=int(st[1]), moved_near=int(st[2]),
                            moved_far=int(st[3]), error=rc)


def cell_multisets(N, arr):
    """per sort cell: the valid 4-tuples, sorted lexicographically (the order inside a cell is undefined)"""
    out = []
    for k in range(N.shape[0]):
        t = np.stack([a[k, :N[k]] for a in arr], 1)
        out.append(t[np.lexsort(t.T[::-1])] if t.shape[0] else t)
    return out
