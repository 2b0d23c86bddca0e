"""Pins for the oracle's counter-based hash (R13/R14)."""
import ctypes as C
import glob
import os

import numpy as np
import pytest

import oracle

GOLD = os.path.join(os.path.dirname(__file__), "golden", "philox4x32_10_kat.txt")


def _kat():
    rows = []
    for line in open(GOLD):
        line = line.strip()
        if not line or line.startswith("#"):
            continue
        w = [int(t, 16) for t in line.split()]
        rows.append((w[0:4], w[4:6], w[6:10]))
    return rows


def test_known_answer_vectors():
    rows = _kat()
    assert len(rows) == 3
    for ctr, key, out in rows:
        got = oracle.philox4x32_10(ctr, key)
        assert [int(x) for x in got] == out


def _curand_host():
    cands = glob.glob("/usr/local/cuda/lib64/libcurand.so.10") + glob.glob(
        os.path.join(os.path.dirname(np.__file__), "..", "nvidia", "curand", "lib", "libcurand.so.10"))
    for p in cands:
        try:
            return C.CDLL(p)
        except OSError:
            continue
    return None


def test_curand_host_third_opinion():
    """NVIDIA's HOST generator CURAND_RNG_PHILOX4_32_10 (runs on the CPU, no GPU needed) is an independent
    implementation: with seed s and offset 0 its first four outputs are Philox4x32-10(counter 0, key (s lo, s hi))."""
    L = _curand_host()
    if L is None:
        pytest.skip("libcurand not loadable")
    gen = C.c_void_p()
    if L.curandCreateGeneratorHost(C.byref(gen), 161) != 0:
        pytest.skip("host generator unavailable")
    out = np.zeros(4, dtype=np.uint32)
    for seed in (0, 42, 0x123456789ABCDEF1, 2 ** 64 - 1):
        assert L.curandSetPseudoRandomGeneratorSeed(gen, C.c_ulonglong(seed)) == 0
        assert L.curandSetGeneratorOffset(gen, C.c_ulonglong(0)) == 0
        assert L.curandGenerate(gen, out.ctypes.data_as(C.POINTER(C.c_uint32)), C.c_size_t(4)) == 0
        mine = oracle.philox4x32_10([0, 0, 0, 0], [seed & 0xFFFFFFFF, seed >> 32])
        assert np.array_equal(mine, out)
    L.curandDestroyGenerator(gen)


def test_theta_symmetric_and_keyed():
    t = oracle.dpd_theta(3, 17, 5, 42)
    assert t == oracle.dpd_theta(17, 3, 5, 42)            # keyed on (min tag, max tag)
    assert t != oracle.dpd_theta(3, 17, 6, 42)            # fresh number every step
    assert t != oracle.dpd_theta(3, 17, 5, 43)            # and per seed
    assert t != oracle.dpd_theta(3, 18, 5, 42)
    assert oracle.dpd_theta(3, 17, 5 + 2 ** 32, 42) != t  # high step word enters the counter
    assert oracle.dpd_theta(3, 17, 5, 42 + 2 ** 32) != t  # high seed word enters the key


def test_theta_matches_word0_mapping():
    # theta = sqrt(3) (2u-1), u = (X0 + 0.5) 2^-32 with X0 = word 0 of the hash of (min, max, step, seed)
    x = oracle.philox4x32_10([3, 17, 5, 0], [42, 0])
    u = (int(x[0]) + 0.5) / 2.0 ** 32
    assert oracle.dpd_theta(17, 3, 5, 42) == np.sqrt(3.0) * (2.0 * u - 1.0)


def test_theta_moments():
    """Uniform with zero mean and unit variance (first two moments are what DPD needs)."""
    n = 200_000
    rng = np.random.default_rng(0)
    a = rng.integers(0, 1_000_000, n)
    b = rng.integers(0, 1_000_000, n)
    th = np.array([oracle.dpd_theta(int(x), int(y), 7, 42) for x, y in zip(a, b) if x != y])
    assert abs(th.mean()) < 4 * 1.0 / np.sqrt(len(th))
    assert abs(th.var() - 1.0) < 0.01
    assert th.min() > -np.sqrt(3.0) and th.max() < np.sqrt(3.0)
    # uniformity: chi^2 over 20 bins, 19 dof -> 99.9 % quantile 43.8
    h, _ = np.histogram(th, bins=20, range=(-np.sqrt(3.0), np.sqrt(3.0)))
    chi2 = ((h - len(th) / 20) ** 2 / (len(th) / 20)).sum()
    assert chi2 < 43.8
    # kurtosis of a uniform distribution: <t^4> = 9/5
    assert abs((th ** 4).mean() - 1.8) < 0.03
