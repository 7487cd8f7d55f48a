"""Pin R-R1/R-R3: the oracle's Philox4x32-10 against cuRAND's HOST generator
(CURAND_RNG_PSEUDO_PHILOX4_32_10, an independent library implementation that runs on
the CPU).  cuRAND's host stream interleaves 65536 subsequences: output block g (4 words)
is Philox(counter = (g>>16 lo, g>>16 hi, g & 0xFFFF, 0), key = seed), which exercises
counter words c0, c1, c2 and both key words.
"""
import ctypes as C
import ctypes.util
import glob

import numpy as np
import pytest
from scipy import stats


def _curand():
    cands = ["/usr/local/cuda/lib64/libcurand.so"] + sorted(glob.glob("/usr/local/cuda*/lib64/libcurand.so*"))
    name = ctypes.util.find_library("curand")
    if name:
        cands.append(name)
    for c in cands:
        try:
            return C.CDLL(c)
        except OSError:
            continue
    return None


def _curand_words(cu, seed, offset_words, n):
    gen = C.c_void_p()
    assert cu.curandCreateGeneratorHost(C.byref(gen), 161) == 0
    assert cu.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    assert cu.curandSetGeneratorOffset(gen, C.c_ulonglong(offset_words)) == 0
    out = np.zeros(n, dtype=np.uint32)
    assert cu.curandGenerate(gen, out.ctypes.data_as(C.c_void_p), C.c_size_t(n)) == 0
    cu.curandDestroyGenerator(gen)
    return out


def _philox(L, seed, ctr):
    key = (C.c_uint32 * 2)(seed & 0xFFFFFFFF, (seed >> 32) & 0xFFFFFFFF)
    c = (C.c_uint32 * 4)(*ctr)
    o = (C.c_uint32 * 4)()
    L.orc_philox4x32_10(c, key, o)
    return np.array(list(o), dtype=np.uint32)


def test_philox_matches_curand_host(orc):
    cu = _curand()
    if cu is None:
        pytest.skip("libcurand not found")
    L = orc.lib()
    rng = np.random.default_rng(12345)
    # sequential blocks: subsequence index = c2
    for seed in (0, 1, 0xDEADBEEFCAFEF00D):
        words = _curand_words(cu, seed, 0, 4 * 300).reshape(-1, 4)
        for g in range(300):
            assert (words[g] == _philox(L, seed, (0, 0, g, 0))).all()
    # random far offsets: c0 and c1 non-zero, random 64-bit keys
    for t in range(200):
        g = int(rng.integers(0, 2**61)) if t % 2 else int(rng.integers(0, 2**36))
        seed = int(rng.integers(0, 2**63)) * 2 + int(rng.integers(0, 2))
        words = _curand_words(cu, seed, 4 * g, 4)
        q = g >> 16
        ctr = (q & 0xFFFFFFFF, (q >> 32) & 0xFFFFFFFF, g & 0xFFFF, 0)
        assert (words == _philox(L, seed, ctr)).all(), (g, seed)


def test_philox_counter_words_all_matter(orc):
    """Every counter/key word changes the output (a dropped word would collide)."""
    L = orc.lib()
    base = _philox(L, 7, (1, 2, 3, 4))
    for i in range(4):
        c = [1, 2, 3, 4]
        c[i] += 1
        assert (base != _philox(L, 7, tuple(c))).any()
    assert (base != _philox(L, 8, (1, 2, 3, 4))).any()
    assert (base != _philox(L, 7 + (1 << 32), (1, 2, 3, 4))).any()


def test_u01_open_interval_and_uniform(orc):
    L = orc.lib()
    assert L.orc_u01(0) == 0.5 / 2**32
    assert L.orc_u01(0xFFFFFFFF) == (2**32 - 0.5) / 2**32 < 1.0
    u = []
    for g in range(5000):
        u.extend(L.orc_u01(int(w)) for w in _philox(L, 99, (g, 0, 5, 0)))
    u = np.array(u)
    assert stats.kstest(u, "uniform").pvalue > 1e-3
    # lag-1 correlation inside blocks
    assert abs(np.corrcoef(u[:-1], u[1:])[0, 1]) < 0.03
