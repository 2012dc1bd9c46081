"""P1 -- Philox4x32-10 of the oracle against an independent implementation (cuRAND's HOST
generator, runs on the CPU), bijectivity and uniformity.  DESIGN.md R12."""
import ctypes as C
import glob

import numpy as np
import pytest

from oracle import oracle as O


def _curand():
    for pat in ("/usr/local/cuda/targets/x86_64-linux/lib/libcurand.so.10",
                "/usr/local/cuda*/lib64/libcurand.so*",
                "/opt/prime-rl/.venv/lib/python3*/site-packages/nvidia/curand/lib/libcurand.so*"):
        for f in glob.glob(pat):
            try:
                return C.CDLL(f)
            except OSError:
                pass
    return None


@pytest.mark.parametrize("seed", [0, 1, 7, 0x123456789ABCDEF1])
def test_philox_matches_curand_host(seed):
    cr = _curand()
    if cr is None:
        pytest.skip("libcurand not found")
    gen = C.c_void_p()
    assert cr.curandCreateGeneratorHost(C.byref(gen), 161) == 0   # CURAND_RNG_PHILOX4_32_10
    assert cr.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    n = 3 * 4 * 65536
    out = np.zeros(n, dtype=np.uint32)
    assert cr.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(n)) == 0
    cr.curandDestroyGenerator(gen)
    # cuRAND host ordering (found empirically): word w of counter (k, 0, t, 0)
    # sits at out[4*65536*k + 4*t + w], key = (seed_lo, seed_hi).
    rng = np.random.default_rng(5)
    cases = [(0, 0), (1, 0), (0, 1), (2, 65535)] + [(int(rng.integers(3)), int(rng.integers(65536)))
                                                     for _ in range(200)]
    for k, t in cases:
        assert O.philox(seed, k, 0, t, 0) == [int(v) for v in out[4 * 65536 * k + 4 * t:][:4]]


def test_philox_counter_words_all_matter_and_bijective():
    base = O.philox(3, 10, 20, 30, 40)
    seen = {tuple(base)}
    for d in range(4):
        c = [10, 20, 30, 40]
        c[d] += 1
        w = tuple(O.philox(3, *c))
        assert w not in seen
        seen.add(w)
    assert tuple(O.philox(4, 10, 20, 30, 40)) not in seen
    assert tuple(O.philox(3 + (1 << 32), 10, 20, 30, 40)) not in seen
    # bijective per key: no collision on a 2^16 sub-cube of the counter space
    outs = {tuple(O.philox(9, a, b, 0, 0)) for a in range(256) for b in range(256)}
    assert len(outs) == 1 << 16
    outs = {tuple(O.philox(9, 5, 0, c, d)) for c in range(256) for d in range(256)}
    assert len(outs) == 1 << 16


def test_uniformity_chi2():
    w = np.array([O.philox(11, i, 5, 0, 0) for i in range(20000)], dtype=np.uint64).ravel()
    u = (w >> 8).astype(np.float64) * 2.0 ** -24
    assert u.min() >= 0 and u.max() < 1
    h, _ = np.histogram(u, bins=64, range=(0, 1))
    chi2 = np.sum((h - u.size / 64) ** 2 / (u.size / 64))
    assert chi2 < 63 + 5 * np.sqrt(2 * 63)
    assert abs(u.mean() - 0.5) < 4 / np.sqrt(12 * u.size)
