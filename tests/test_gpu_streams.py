"""The handles run on a stream of their own; CUDA tensors handed to them are produced on torch's current stream.
Loading tensors whose producer kernels are still queued must see the produced values, not what the memory held
before (the binding orders its stream after the current one and records the use with the caching allocator)."""
import numpy as np
import pytest

from paper_1104_3998_b200 import workloads as W
from helpers import load

pytestmark = pytest.mark.gpu


def _pending(torch, host_arrays, dev):
    """device tensors whose final values are written by kernels queued BEHIND ~100 ms of other work on the current
    stream, as non-contiguous views (so the binding also has to make contiguous temporaries)"""
    staged = [torch.from_numpy(np.ascontiguousarray(a)).to(dev) for a in host_arrays]
    out = [torch.full((a.shape[0], 2), -7.0, dtype=torch.float32, device=dev) for a in host_arrays]
    torch.cuda.synchronize()
    busy = torch.ones(8192, 8192, device=dev)
    for _ in range(12):
        busy = (busy @ busy) * 1e-4      # fp32 GEMMs: keeps the current stream busy
    for o, s in zip(out, staged):
        o[:, 0] = s                      # the values the load must see
    return [o[:, 0] for o in out], busy


def test_load_particles_from_cuda_tensors_still_being_produced():
    import torch
    from paper_1104_3998_b200 import pic1d as G
    dev = torch.device("cuda:0")
    p = W.make_params(2, n_cells=256, ppc=300)
    parts = W.make_particles(p)
    ref = G.Pic1D(p)
    load(ref, parts)                     # host arrays: the path every other test takes
    g = G.Pic1D(p)
    keep = []
    for s, a in enumerate(parts):
        views, busy = _pending(torch, a, dev)
        assert not views[0].is_contiguous()
        g.load_particles(s, *views)
        keep.append(busy)
        del views                        # the binding's temporaries and these views may be freed right away
        junk = [torch.full((a[0].shape[0], 2), 123.0, device=dev) for _ in range(4)]  # ... and their memory reused
        keep.append(junk)
    for s in range(p["n_species"]):
        for w in (G.DBG_X, G.DBG_VX, G.DBG_VY, G.DBG_VZ, G.DBG_OFFSETS):
            assert np.array_equal(ref.debug_get(w, s), g.debug_get(w, s)), (s, w)
    for a, b in zip(ref.get_rho_phi_E(), g.get_rho_phi_E()):
        assert np.array_equal(a, b)
    g.step(2); ref.step(2)
    for s in range(p["n_species"]):
        assert np.array_equal(ref.debug_get(G.DBG_X, s), g.debug_get(G.DBG_X, s))
    ref.close(); g.close()


def test_gapped_sort_load_from_cuda_tensors_still_being_produced():
    import torch
    from paper_1104_3998_b200 import gsort as GS
    dev = torch.device("cuda:0")
    rng = np.random.default_rng(11)
    Nc, n = 128, 60000
    x = (rng.random(n, dtype=np.float32) * Nc).astype(np.float32)
    v = (rng.normal(size=(3, n)) * 0.2).astype(np.float32)
    E = rng.normal(size=Nc + 1).astype(np.float32)
    ref, g = GS.GappedSort(Nc, 1.0, 1024, -0.05), GS.GappedSort(Nc, 1.0, 1024, -0.05)
    ref.load(x, v[0], v[1], v[2]); ref.set_E32(E)
    views, busy = _pending(torch, [x, v[0], v[1], v[2]], dev)
    g.load(*views)
    (Ev,), busy2 = _pending(torch, [E], dev)
    g.set_E32(Ev)
    del views, Ev
    ref.step(2); g.step(2)
    Nr, ar, sr = ref.get()
    Ng, ag, sg = g.get()
    assert np.array_equal(Nr, Ng) and sr == sg and sg["error"] == 0
    for c in range(Nc):                 # order inside a cell is undefined: compare the cells as multisets
        for q in range(4):
            assert np.array_equal(np.sort(ar[q][c, :Nr[c]]), np.sort(ag[q][c, :Ng[c]])), (c, q)
    ref.close(); g.close()
