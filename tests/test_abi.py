"""The C-ABI library builds, loads and exports every symbol include/pic1d.h declares (no compute
calls: there is no GPU on the CPU box); host-side argument validation."""
import ctypes as C
import os
import re

from paper_1104_3998_b200 import build as B
from paper_1104_3998_b200 import pic1d as G
from paper_1104_3998_b200 import gsort as GS
from paper_1104_3998_b200 import field_static as FS
from paper_1104_3998_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    names = set()
    for h in ("pic1d.h", "pic1d_gsort.h", "pic1d_static.h"):
        src = open(os.path.join(ROOT, "include", h)).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names |= set(re.findall(r"\b(pic1d_[a-z0-9_E]+)\s*\(", src))
    return sorted(names)


def test_library_exports_every_declared_symbol():
    B.build()
    lib = G.load_library()
    names = _declared()
    assert len(names) >= 22 and set(G.EXPORTS) | set(GS.EXPORTS) | set(FS.EXPORTS) == set(names)
    for n in names:
        assert getattr(lib, n) is not None


def test_struct_sizes_and_workspace_query():
    lib = G.load_library()
    assert C.sizeof(G.Config) == 16 + 2 * 48 + 13 * 8 + 8 + 8 + 3 * 8
    for cfg in (0, 1, 2):
        c = G.make_config(W.make_params(cfg))
        n = C.c_size_t()
        assert lib.pic1d_workspace_bytes(C.byref(c), C.byref(n)) == 0
        p = W.make_params(cfg)
        state = sum(sp["capacity"] for sp in p["species"]) * 16 * 2
        assert n.value >= state and n.value < state * 3 + (64 << 20)
    c = G.make_config(W.make_params(0))
    c.struct_size = 12
    assert lib.pic1d_workspace_bytes(C.byref(c), C.byref(n)) == G.ERR_ARG
    c = G.make_config(W.make_params(0))
    c.sort_inv_ratio = 0.3      # not a power of two
    assert lib.pic1d_workspace_bytes(C.byref(c), C.byref(n)) == G.ERR_ARG
    c = G.make_config(W.make_params(0))
    c.sp[0].capacity = 5000     # not a multiple of 4096
    assert lib.pic1d_workspace_bytes(C.byref(c), C.byref(n)) == G.ERR_ARG
    for field, bad in (("e_reflect", -0.1), ("e_reflect", 1.5), ("e_reflect", float("nan"))):
        c = G.make_config(W.make_params(0))
        setattr(c, field, bad)   # a probability
        assert lib.pic1d_workspace_bytes(C.byref(c), C.byref(n)) == G.ERR_ARG, (field, bad)
    for s in (0, 1):
        for bad in (-1.0, float("inf"), float("nan")):
            c = G.make_config(W.make_params(0))
            c.coul_A[s] = bad
            assert lib.pic1d_workspace_bytes(C.byref(c), C.byref(n)) == G.ERR_ARG, (s, bad)
    c = G.make_config(W.make_params(0))
    c.e_reflect, c.coul_A[0], c.coul_A[1] = 1.0, 0.0, 2.5
    assert lib.pic1d_workspace_bytes(C.byref(c), C.byref(n)) == 0
    h = C.c_void_p()            # pic1d_create validates the same way, before touching the device
    c.e_reflect = 2.0
    assert lib.pic1d_create(C.byref(c), C.c_void_p(256), C.c_size_t(1 << 30), None, C.byref(h)) == G.ERR_ARG


def test_product_path_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_1104_3998_b200")
    pat = re.compile(r"(^\s*(from|import)\s+oracle\b)|(oracle/)|(libpic1d_oracle)|(#include.*oracle)", re.M)
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dirpath, f)).read()), f
