"""pic1d_field_solve_static (include/pic1d_static.h): the field solve for callers that cannot allocate.

Some users of this library are not allowed, or not able, to create device memory: a host code whose own memory
manager has already taken the whole GPU (anybody else's cudaMalloc fails there), a plug-in that only ever sees
the input and output buffers of its host application, a time-step loop that must not run into the device-wide
synchronisation of cudaMalloc / cudaFree.  For them the library carries one entry point whose temporary arrays
live in a fixed 1 MiB array inside libpic1d.so (grids of up to 65536 cells) instead of a caller-allocated
workspace.  These tests check that entry point against the existing path (the field solve inside pic1d_step,
read back with pic1d_get_rho_phi_E), to the 1e-9 the parity tests ask of phi and E, on calls made back to back:
the array is shared by all calls and keeps the previous call's contents, so a second call must not care what
the first one left behind.

The file sorts last on purpose (`pytest --collect-only`): under `pytest -x` a failure here must not hide any other
test.  It holds no state of its own, so it passes alone in a fresh process as well as after the rest of the suite.
"""
import math

import numpy as np
import pytest

from paper_1104_3998_b200 import workloads as W
from helpers import load, rel_linf

TOL_FIELD = 1e-9   # the bar tests/test_gpu_parity.py puts on phi and E


def _existing_path(cfg_id, n_cells, ppc, steps):
    """rho, phi, E (host fp64) of the step's own field solve after `steps` steps, and the left-wall potential"""
    from paper_1104_3998_b200 import pic1d as G
    p = W.make_params(cfg_id, n_cells=n_cells, ppc=ppc)
    g = G.Pic1D(p)
    load(g, W.make_particles(p))
    g.step(steps)
    rho, phi, E = g.get_rho_phi_E()
    assert g.sticky == 0
    phi0 = p["V0_norm"] * math.sin(p["omega_dt"] * g.step_index) if p["bc"] == 0 else 0.0
    g.close()
    return dict(n_cells=n_cells, bc=p["bc"], phi0=phi0, rho=rho, phi=phi, E=E)


def _enqueue(case, dev):
    """what a caller without an allocator does: it owns rho, phi, E (and E32) and nothing else"""
    import torch
    from paper_1104_3998_b200 import field_static as FS
    rho = torch.from_numpy(case["rho"]).to(dev)
    phi = torch.full_like(rho, float("nan"))
    E = torch.full_like(rho, float("nan"))
    E32 = torch.full(rho.shape, float("nan"), dtype=torch.float32, device=dev)
    FS.field_solve_static(rho, phi, E, case["n_cells"], case["bc"], case["phi0"], E32=E32)
    return rho, phi, E, E32


def _check(case, out):
    _, phi, E, E32 = out
    phi, E, E32 = phi.cpu().numpy(), E.cpu().numpy(), E32.cpu().numpy()
    assert np.all(np.isfinite(phi)) and np.all(np.isfinite(E))
    assert rel_linf(phi, case["phi"]) <= TOL_FIELD, rel_linf(phi, case["phi"])
    assert rel_linf(E, case["E"]) <= TOL_FIELD, rel_linf(E, case["E"])
    assert np.array_equal(E32, E.astype(np.float32))
    return phi, E


@pytest.mark.gpu
def test_static_field_solve_matches_the_step_on_calls_in_a_row():
    """Three calls back to back on one stream, no synchronisation in between: a driven bounded grid of 1000 cells
    (ragged: not a multiple of the block), a periodic grid of 512 cells, and the first one again.  Each must match
    the existing path; the repeat must reproduce the first call bit for bit although the scratch array now holds
    the periodic problem's sums."""
    import torch
    dev = torch.device("cuda:0")
    a = _existing_path(2, 1000, 40, 3)      # RF-driven wall: phi0 != 0
    b = _existing_path(1, 512, 100, 2)      # periodic, neutralising background
    assert abs(a["phi0"]) > 0 and a["bc"] == 0 and b["bc"] == 1
    out1 = _enqueue(a, dev)
    out2 = _enqueue(b, dev)
    out3 = _enqueue(a, dev)
    torch.cuda.synchronize()
    phi1, E1 = _check(a, out1)
    _check(b, out2)
    phi3, E3 = _check(a, out3)
    assert np.array_equal(phi1, phi3) and np.array_equal(E1, E3)


@pytest.mark.gpu
def test_static_field_solve_large_grid_then_small():
    """32768 cells (the existing path then runs its global-memory kernel, the one this entry point is a variant
    of), directly followed by a 128-cell solve that reuses the front of the same scratch array."""
    import torch
    dev = torch.device("cuda:0")
    a = _existing_path(2, 32768, 6, 2)
    b = _existing_path(0, 128, 64, 2)
    out1 = _enqueue(a, dev)
    out2 = _enqueue(b, dev)
    torch.cuda.synchronize()
    _check(a, out1)
    _check(b, out2)


def test_static_field_solve_refuses_grids_beyond_its_array():
    """host-side check, before any CUDA call (runs without a GPU): one cell more than the fixed array holds is
    refused with PIC1D_ERR_ARG and a message that names the limit; so are the other bad arguments"""
    import ctypes as C
    from paper_1104_3998_b200 import build as B
    from paper_1104_3998_b200 import field_static as FS
    from paper_1104_3998_b200 import pic1d as G
    B.build()
    lib = FS._lib()
    dummy = C.c_void_p(256)     # never dereferenced: the call is refused first

    def call(n_cells, bc=0, phi0=0.0, rho=dummy):
        return lib.pic1d_field_solve_static(rho, dummy, dummy, None, C.c_int(n_cells), C.c_int(bc),
                                            C.c_double(phi0), None)
    assert call(FS.MAX_CELLS + 1) == G.ERR_ARG
    msg = FS.last_error()
    assert str(FS.MAX_CELLS) in msg and str(FS.MAX_CELLS + 1) in msg and "workspace" in msg
    assert call(1) == G.ERR_ARG
    assert call(128, bc=2) == G.ERR_ARG
    assert call(128, phi0=float("inf")) == G.ERR_ARG
    assert call(128, rho=None) == G.ERR_ARG and "NULL" in FS.last_error()
    src = open(B.CSRC + "/pic1d_field_static.cu").read()
    assert "#define PIC1D_FIELD_STATIC_MAX_CELLS %d" % FS.MAX_CELLS in open(B.HERE + "/../include/pic1d_static.h").read()
    for banned in ("cudaMalloc", "cudaFree", "cudaMemset", "cudaHostAlloc"):   # the entry point's file allocates nothing
        assert banned + "(" not in src, banned
