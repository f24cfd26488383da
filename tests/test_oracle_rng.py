"""Pins for the oracle's counter-based noise."""
import ctypes as C
import ctypes.util
import os

import numpy as np
import pytest
from scipy import stats


def _curand():
    for cand in ("/usr/local/cuda/lib64/libcurand.so", "/usr/local/cuda/lib64/libcurand.so.10", ctypes.util.find_library("curand")):
        if cand and os.path.exists(cand):
            return C.CDLL(cand)
    return None


@pytest.mark.parametrize("seed", [0, 0x0123456789ABCDEF, 2**64 - 1])
def test_philox_matches_curand_host_generator(orc, seed):
    """Library pin: cuRAND's *host* CURAND_RNG_PSEUDO_PHILOX4_32_10 (runs on the CPU, no GPU needed) emits
    4-word blocks; block i is Philox4x32-10(counter = (i // 65536, 0, i % 65536, 0), key = seed)
    (65536 interleaved subsequences; mapping found by search)."""
    cr = _curand()
    if cr is None:
        pytest.skip("libcurand not found")
    gen = C.c_void_p()
    assert cr.curandCreateGeneratorHost(C.byref(gen), 161) == 0       # CURAND_RNG_PSEUDO_PHILOX4_32_10 = 161
    assert cr.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
    n = 65536 + 8
    out = (C.c_uint32 * (4 * n))()
    assert cr.curandGenerate(gen, out, C.c_size_t(4 * n)) == 0
    got = np.frombuffer(out, dtype=np.uint32).reshape(n, 4)
    key = (seed & 0xFFFFFFFF, seed >> 32)
    for i in list(range(48)) + [4095, 4096, 65535, 65536, 65537, 65543]:
        assert got[i].tolist() == orc.philox4x32_10((i // 65536, 0, i % 65536, 0), key), i
    cr.curandDestroyGenerator(gen)


def test_philox_counter_words_all_matter(orc):
    base = orc.philox4x32_10((1, 2, 3, 4), (5, 6))
    for pos in range(4):
        c = [1, 2, 3, 4]
        c[pos] += 1
        assert orc.philox4x32_10(c, (5, 6)) != base
    assert orc.philox4x32_10((1, 2, 3, 4), (5, 7)) != base
    assert orc.philox4x32_10((1, 2, 3, 4), (6, 6)) != base


def test_normals_are_standard_normal(orc):
    """Invariant pin for the Box-Muller transform: moments and KS over 3e6 draws."""
    xs = np.concatenate([orc.normals(1234, step, 100000) for step in range(1, 11)])
    assert xs.shape == (1000000, 3)
    for c in range(3):
        x = xs[:, c]
        assert abs(x.mean()) < 4e-3
        assert abs(x.var() - 1.0) < 6e-3
        assert abs(stats.kurtosis(x, fisher=False) - 3.0) < 2e-2
        assert stats.kstest(x[:200000], "norm").pvalue > 1e-3
    cc = np.corrcoef(xs.T)
    assert np.abs(cc - np.eye(3)).max() < 4e-3
    # different steps / tags give different, uncorrelated streams
    a, b = orc.normals(1234, 1, 50000), orc.normals(1234, 2, 50000)
    assert abs(np.corrcoef(a[:, 0], b[:, 0])[0, 1]) < 2e-2
    assert not np.array_equal(orc.normals(1234, 1, 10, tag=0), orc.normals(1234, 1, 10, tag=2))


def test_uniform_is_uniform_open_interval(orc):
    u = np.array([orc.uniform(99, s) for s in range(1, 200001)])
    assert u.min() > 0.0 and u.max() < 1.0
    assert abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1 / 12) < 1e-3
    assert stats.kstest(u, "uniform").pvalue > 1e-3


def test_initial_momenta_maxwell_boltzmann(orc):
    import lsd_inputs as L
    w = L.make_workload("cfg5", cells=(16, 16, 8))          # 24,576 components: chi^2 rel. std 0.9 %
    p = orc.initial_momenta(w)
    kin_T = (p**2 / (w.mass_amu[:, None] * L.AMU)).mean() / L.K_B       # <p^2/m> = kT per component
    assert abs(kin_T / w.temperature_K - 1.0) < 0.04
