"""Thin Python binding of the C-ABI in include/pic1d.h (argument marshalling only).

Every step of the hot path runs in the CUDA kernels of libpic1d.so; PyTorch is used for device
memory (the workspace tensor) and the stream.  There is no CPU fallback: if the library is missing
or no CUDA device is present, construction fails loudly.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpic1d.so")

OK, ERR_ARG, ERR_CAPACITY, ERR_CUDA, ERR_NONFINITE, ERR_WORKSPACE, ERR_ORDER = 0, -1, -2, -3, -4, -5, -6
FLAG_CAPTURE = 1
FLAG_VERIFY_ORDER = 2
FLAG_EQ5_ELECTRONS = 4
FLAG_NO_FOLD = 8
FLAG_FOLD_ALL = 16
FLAG_MCC_GATHER = 32
FLAG_NO_OVERLAP = 64
FLAG_NO_GRAPH = 128
DBG_X, DBG_VX, DBG_VY, DBG_VZ, DBG_KEYS, DBG_OFFSETS, DBG_MASK, DBG_E32, DBG_RHO_S, DBG_TILE_W, DBG_PARTNER = range(11)
_DBG_DTYPE = {DBG_X: np.float32, DBG_VX: np.float32, DBG_VY: np.float32, DBG_VZ: np.float32,
              DBG_KEYS: np.int32, DBG_OFFSETS: np.int32, DBG_MASK: np.uint8, DBG_E32: np.float32,
              DBG_RHO_S: np.float64, DBG_TILE_W: np.int32, DBG_PARTNER: np.int32}

ABI_VERSION = 3   # PIC1D_ABI_VERSION of include/pic1d.h this binding was written against

EXPORTS = ["pic1d_abi_version", "pic1d_workspace_bytes", "pic1d_create", "pic1d_load_particles", "pic1d_step",
           "pic1d_get_rho_phi_E", "pic1d_moments", "pic1d_destroy", "pic1d_n_nodes",
           "pic1d_n_sort_cells", "pic1d_step_index", "pic1d_last_cuda_error", "pic1d_launch_count",
           "pic1d_graph_launch_count", "pic1d_step_timed", "pic1d_debug_count", "pic1d_debug_get", "pic1d_debug_set_E32",
           "pic1d_debug_set_state"]


class SpeciesConfig(C.Structure):
    _fields_ = [("kappa", C.c_double), ("c_eV", C.c_double), ("P0", C.c_double),
                ("inv_g_cap", C.c_double), ("capacity", C.c_int64),
                ("charge_sign", C.c_int32), ("mcc_kind", C.c_int32)]


class Config(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("n_cells", C.c_int32), ("bc", C.c_int32),
                ("n_species", C.c_int32), ("sp", SpeciesConfig * 2),
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


class KernelTime(C.Structure):
    _fields_ = [("name", C.c_char * 48), ("ms", C.c_float), ("species", C.c_int32)]


_lib = None


def load_library():
    """dlopen libpic1d.so (built by paper_1104_3998_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError("CUDA library %s is missing: run `python -m paper_1104_3998_b200.build` "
                               "(there is no CPU fallback)" % LIB_PATH)
        lib = C.CDLL(LIB_PATH)
        have = lib.pic1d_abi_version() if hasattr(lib, "pic1d_abi_version") else 2
        if have != ABI_VERSION:     # a stale in-tree build: struct layouts may differ, refuse instead of guessing
            raise RuntimeError("%s was built for ABI version %d, this binding needs %d: rebuild it with "
                               "`python -m paper_1104_3998_b200.build`" % (LIB_PATH, have, ABI_VERSION))
        lib.pic1d_last_cuda_error.restype = C.c_char_p
        lib.pic1d_launch_count.restype = C.c_int64
        lib.pic1d_graph_launch_count.restype = C.c_int64
        lib.pic1d_step_index.restype = C.c_uint32
        _lib = lib
    return _lib


def make_config(params):
    """params: the plain dict produced by paper_1104_3998_b200.workloads.make_params."""
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


class Pic1DError(RuntimeError):
    def __init__(self, where, code, detail=""):
        super().__init__("%s failed with code %d %s" % (where, code, detail))
        self.code = code


def _ptr(a):
    """pointer of a numpy array / torch tensor / None"""
    if a is None:
        return None
    if isinstance(a, np.ndarray):
        return C.c_void_p(a.ctypes.data)
    return C.c_void_p(a.data_ptr())


def _adopt(torch, stream, device, tensors):
    """Order `stream` after torch's current stream and tell the caching allocator that `stream` uses `tensors`.

    The handle runs on a stream of its own, but CUDA tensors handed to it (and its workspace) are produced or
    allocated on torch's current stream.  Without the wait a device-to-device copy could read a tensor before
    the kernel that fills it has run; without record_stream a temporary (.contiguous()) or the workspace could be
    handed out again by the allocator while our stream still reads or writes it."""
    cur = torch.cuda.current_stream(device)
    if cur != stream:
        stream.wait_stream(cur)
        for t in tensors:
            t.record_stream(stream)


class Pic1D:
    """One simulation handle on the current CUDA device; methods mirror the C calls."""

    def __init__(self, params, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("pic1d needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        self.cfg = make_config(params)
        nbytes = C.c_size_t()
        rc = self.lib.pic1d_workspace_bytes(C.byref(self.cfg), C.byref(nbytes))
        if rc:
            raise Pic1DError("pic1d_workspace_bytes", rc)
        self.workspace_bytes = nbytes.value
        self.workspace = torch.empty(nbytes.value, dtype=torch.uint8, device=self.device)
        # a stream of its own: the legacy default stream cannot be captured into a CUDA graph
        self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
        _adopt(torch, self.stream, self.device, [self.workspace])
        self.h = C.c_void_p()
        rc = self.lib.pic1d_create(C.byref(self.cfg), C.c_void_p(self.workspace.data_ptr()), nbytes,
                                   C.c_void_p(self.stream.cuda_stream), C.byref(self.h))
        if rc:
            raise Pic1DError("pic1d_create", rc)
        self.n_nodes = self.lib.pic1d_n_nodes(self.h)
        self.n_sc = self.lib.pic1d_n_sort_cells(self.h)

    def close(self):
        if getattr(self, "h", None):
            self.stream.synchronize()       # the workspace goes back to torch's allocator: nothing may still use it
            self.lib.pic1d_destroy(self.h)
            self.h = C.c_void_p()
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _err(self, where, rc):
        detail = self.lib.pic1d_last_cuda_error(self.h).decode() if rc == ERR_CUDA else ""
        raise Pic1DError(where, rc, detail)

    def load_particles(self, s, x, vx, vy, vz):
        """x, vx, vy, vz: fp32 numpy arrays (host, may be pinned torch tensors) or CUDA tensors."""
        arrs = [x, vx, vy, vz]
        on_device = 0
        if all(hasattr(a, "is_cuda") for a in arrs):
            on_device = 1 if arrs[0].is_cuda else 0
            arrs = [a.contiguous() for a in arrs]
            assert all(a.dtype == self._torch.float32 for a in arrs)
            if on_device:   # produced on torch's current stream, copied on ours
                _adopt(self._torch, self.stream, self.device, arrs)
        else:
            arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in arrs]
        n = int(arrs[0].shape[0])
        rc = self.lib.pic1d_load_particles(self.h, C.c_int(s), C.c_int64(n), *[_ptr(a) for a in arrs],
                                           C.c_int(on_device))
        if rc:
            self._err("pic1d_load_particles", rc)

    def step(self, n_steps=1):
        rc = self.lib.pic1d_step(self.h, C.c_int(n_steps))
        if rc:
            self._err("pic1d_step", rc)

    def step_timed(self):
        buf = (KernelTime * 64)()
        n = self.lib.pic1d_step_timed(self.h, buf, C.c_int(64))
        if n < 0:
            self._err("pic1d_step_timed", n)
        return [(buf[i].name.decode(), buf[i].species, float(buf[i].ms)) for i in range(n)]

    def get_rho_phi_E(self, out=None):
        """returns (rho, phi, E) as fp64 numpy arrays; `out` = optional tuple of pinned host tensors"""
        if out is None:
            out = [np.zeros(self.n_nodes, dtype=np.float64) for _ in range(3)]
        rc = self.lib.pic1d_get_rho_phi_E(self.h, *[_ptr(a) for a in out], C.c_int(self.n_nodes),
                                          C.c_int(0))
        if rc in (ERR_ARG, ERR_CUDA):
            self._err("pic1d_get_rho_phi_E", rc)
        self.sticky = rc
        return tuple(out)

    def moments(self, s, n_bins=0, E_max=0.0):
        m = Moments()
        dens = np.zeros(self.n_nodes, dtype=np.float64)
        eedf = np.zeros(max(n_bins, 1), dtype=np.int64)
        rc = self.lib.pic1d_moments(self.h, C.c_int(s), C.byref(m), _ptr(dens), C.c_int(self.n_nodes),
                                    _ptr(eedf) if n_bins > 0 else None, C.c_int(n_bins),
                                    C.c_double(E_max))
        if rc in (ERR_ARG, ERR_CUDA):
            self._err("pic1d_moments", rc)
        d = {k: getattr(m, k) for k, _ in Moments._fields_ if k != "n_events"}
        d["n_events"] = list(m.n_events)
        d["density"] = dens
        d["eedf"] = eedf[:n_bins]
        d["sticky"] = rc
        return d

    def debug_get(self, what, s=0):
        n = C.c_int64()
        rc = self.lib.pic1d_debug_count(self.h, C.c_int(what), C.c_int(s), C.byref(n))
        if rc:
            self._err("pic1d_debug_count", rc)
        out = np.zeros(int(n.value), dtype=_DBG_DTYPE[what])
        rc = self.lib.pic1d_debug_get(self.h, C.c_int(what), C.c_int(s), _ptr(out), C.c_size_t(out.nbytes))
        if rc:
            self._err("pic1d_debug_get", rc)
        return out

    def set_E32(self, e32):
        a = np.ascontiguousarray(e32, dtype=np.float32)
        rc = self.lib.pic1d_debug_set_E32(self.h, _ptr(a), C.c_int(a.shape[0]))
        if rc:
            self._err("pic1d_debug_set_E32", rc)

    def set_state(self, s, n_sorted, x, vx, vy, vz, step=-1):
        """debug: overwrite the live particles of species s in place (order kept); see pic1d_debug_set_state"""
        arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in (x, vx, vy, vz)]
        rc = self.lib.pic1d_debug_set_state(self.h, C.c_int(s), C.c_int64(arrs[0].shape[0]), C.c_int64(n_sorted),
                                            *[_ptr(a) for a in arrs], C.c_int64(step))
        if rc:
            self._err("pic1d_debug_set_state", rc)

    @property
    def step_index(self):
        return int(self.lib.pic1d_step_index(self.h))

    @property
    def launch_count(self):
        return int(self.lib.pic1d_launch_count(self.h))

    @property
    def graph_launch_count(self):
        """CUDA-graph replays (two steps each) so far; -1 = capture failed once, plain launches since"""
        return int(self.lib.pic1d_graph_launch_count(self.h))

    def synchronize(self):
        self.stream.synchronize()
