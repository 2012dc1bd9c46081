"""Thin Python binding of include/pic1d_gsort.h: the paper's gapped in-place fine sort fused with the pusher
(argument marshalling only; PyTorch for the workspace and the stream)."""
import ctypes as C

import numpy as np

from .pic1d import load_library, Pic1DError, _ptr, _adopt

EXPORTS = ["pic1d_gsort_workspace_bytes", "pic1d_gsort_create", "pic1d_gsort_load", "pic1d_gsort_set_E32",
           "pic1d_gsort_step", "pic1d_gsort_get", "pic1d_gsort_n_sort_cells", "pic1d_gsort_destroy"]


class GappedSort:
    def __init__(self, n_cells, sort_inv_ratio, n_max, kappa, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("pic1d_gsort needs a CUDA device (no CPU fallback)")
        self.lib = load_library()
        self.device = torch.device(device)
        torch.cuda.set_device(self.device)
        nbytes = C.c_size_t()
        rc = self.lib.pic1d_gsort_workspace_bytes(C.c_int(n_cells), C.c_double(sort_inv_ratio), C.c_int(n_max), C.byref(nbytes))
        if rc:
            raise Pic1DError("pic1d_gsort_workspace_bytes", rc)
        self.workspace = torch.empty(nbytes.value, dtype=torch.uint8, device=self.device)
        self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
        self._torch = torch
        _adopt(torch, self.stream, self.device, [self.workspace])
        self.h = C.c_void_p()
        rc = self.lib.pic1d_gsort_create(C.c_int(n_cells), C.c_double(sort_inv_ratio), C.c_int(n_max), C.c_double(kappa),
                                         C.c_void_p(self.workspace.data_ptr()), nbytes, C.c_void_p(self.stream.cuda_stream),
                                         C.byref(self.h))
        if rc:
            raise Pic1DError("pic1d_gsort_create", rc)
        self.n_cells, self.n_max = n_cells, n_max
        self.n_sc = self.lib.pic1d_gsort_n_sort_cells(self.h)

    def close(self):
        if getattr(self, "h", None):
            self.stream.synchronize()       # the workspace goes back to torch's allocator
            self.lib.pic1d_gsort_destroy(self.h)
            self.h = C.c_void_p()
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def load(self, x, vx, vy, vz):
        arrs = [x, vx, vy, vz]
        on_device = 1 if all(hasattr(a, "is_cuda") and a.is_cuda for a in arrs) else 0
        if not on_device:
            arrs = [np.ascontiguousarray(a, dtype=np.float32) for a in arrs]
        else:   # produced on torch's current stream, copied on ours
            arrs = [a.contiguous() for a in arrs]
            assert all(a.dtype == self._torch.float32 for a in arrs)
            _adopt(self._torch, self.stream, self.device, arrs)
        rc = self.lib.pic1d_gsort_load(self.h, C.c_int64(int(arrs[0].shape[0])), *[_ptr(a) for a in arrs], C.c_int(on_device))
        if rc:
            raise Pic1DError("pic1d_gsort_load", rc)

    def set_E32(self, e32):
        on_device = 1 if hasattr(e32, "is_cuda") and e32.is_cuda else 0
        a = e32.contiguous() if on_device else np.ascontiguousarray(e32, dtype=np.float32)
        if on_device:
            assert a.dtype == self._torch.float32
            _adopt(self._torch, self.stream, self.device, [a])
        rc = self.lib.pic1d_gsort_set_E32(self.h, _ptr(a), C.c_int(int(a.shape[0])), C.c_int(on_device))
        if rc:
            raise Pic1DError("pic1d_gsort_set_E32", rc)

    def step(self, n_steps=1):
        rc = self.lib.pic1d_gsort_step(self.h, C.c_int(n_steps))
        if rc:
            raise Pic1DError("pic1d_gsort_step", rc)

    def get(self, arrays=True):
        """(N_i, [x, vx, vy, vz] as (n_sc, n_max) arrays or None, stats dict)"""
        N = np.zeros(self.n_sc, np.int32)
        arr = [np.zeros((self.n_sc, self.n_max), np.float32) for _ in range(4)] if arrays else [None] * 4
        st = np.zeros(5, np.int64)
        rc = self.lib.pic1d_gsort_get(self.h, _ptr(N), *[_ptr(a) for a in arr], _ptr(st))
        if rc == -3 or rc == -1:
            raise Pic1DError("pic1d_gsort_get", rc)
        return N, (arr if arrays else None), dict(absorbed_left=int(st[0]), absorbed_right=int(st[1]),
                                                  moved_near=int(st[2]), moved_far=int(st[3]), error=int(st[4]))
