"""Thin Python binding of include/pic1d_static.h: the Poisson + E solve for callers that may not allocate
device memory (argument marshalling only; the solve runs in k_field_static of libpic1d.so).

The caller brings rho, phi and E (and optionally the fp32 copy E32) as CUDA tensors; the two temporary arrays
the solver needs sit in a fixed 1 MiB array inside the library, so the call itself allocates nothing.  Grids of
more than MAX_CELLS cells are refused.  All calls on one GPU share that array: keep them on one stream.
"""
import ctypes as C

from .pic1d import load_library, Pic1DError

EXPORTS = ["pic1d_field_solve_static", "pic1d_field_solve_static_error"]
MAX_CELLS = 65536   # PIC1D_FIELD_STATIC_MAX_CELLS


def _lib():
    lib = load_library()
    lib.pic1d_field_solve_static_error.restype = C.c_char_p
    return lib


def last_error():
    return _lib().pic1d_field_solve_static_error().decode()


def field_solve_static(rho, phi, E, n_cells, bc, phi0=0.0, E32=None, stream=None):
    """Enqueue pic1d_field_solve_static on `stream` (default: torch's current stream on rho's device).

    rho, phi, E: contiguous float64 CUDA tensors of n_cells + 1 (bc = 0) or n_cells (bc = 1) values on one
    device; E32: float32 or None.  Nothing is returned: phi, E (and E32) are written when the stream gets there.
    Raises Pic1DError with the library's own message on a refused call."""
    import torch
    nodes = n_cells + 1 if bc == 0 else n_cells
    for name, t, dt in (("rho", rho, torch.float64), ("phi", phi, torch.float64), ("E", E, torch.float64),
                        ("E32", E32, torch.float32)):
        if t is None and name == "E32":
            continue
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous() and t.numel() >= nodes and t.device == rho.device):
            raise ValueError("%s: need a contiguous %s CUDA tensor of at least %d values on %s" % (name, dt, nodes, rho.device))
    with torch.cuda.device(rho.device):     # the library resolves its scratch array for the CURRENT device
        st = stream if stream is not None else torch.cuda.current_stream()
        rc = _lib().pic1d_field_solve_static(C.c_void_p(rho.data_ptr()), C.c_void_p(phi.data_ptr()),
                                             C.c_void_p(E.data_ptr()),
                                             C.c_void_p(E32.data_ptr()) if E32 is not None else None,
                                             C.c_int(n_cells), C.c_int(bc), C.c_double(phi0),
                                             C.c_void_p(st.cuda_stream))
    if rc:
        raise Pic1DError("pic1d_field_solve_static", rc, last_error())
