"""Pins for the oracle's Philox4x32-10 and director noise (R16).

The core is pinned to a LIBRARY routine: cuRAND's *host* generator CURAND_RNG_PSEUDO_PHILOX4_32_10
(libcurand runs it on the CPU, no GPU needed).  In its default ordering output word i belongs to
block b = i // 4 with subsequence b % 65536 and counter b // 65536 (verified below rather than
assumed), i.e. exactly the (counter word 0 = step, counter word 2 = cell) layout of R16, and a
generator offset of 2**50 words reaches counter word 1 (step high).  Both key words come from the
64-bit seed."""
import ctypes
import os

import numpy as np
import pytest

import oracle

_CURAND = None
for cand in ("/usr/local/cuda/lib64/libcurand.so.10", "libcurand.so.10", "libcurand.so"):
    try:
        _CURAND = ctypes.CDLL(cand)
        break
    except OSError:
        continue


def _curand_host(seed, n_words, offset=0):
    gen = ctypes.c_void_p()
    assert _CURAND.curandCreateGeneratorHost(ctypes.byref(gen), 161) == 0   # PHILOX4_32_10
    assert _CURAND.curandSetPseudoRandomGeneratorSeed(gen, ctypes.c_ulonglong(seed)) == 0
    assert _CURAND.curandSetGeneratorOffset(gen, ctypes.c_ulonglong(offset)) == 0
    out = np.zeros(n_words, dtype=np.uint32)
    assert _CURAND.curandGenerate(gen, ctypes.c_void_p(out.ctypes.data), ctypes.c_size_t(n_words)) == 0
    _CURAND.curandDestroyGenerator(gen)
    return out


needs_curand = pytest.mark.skipif(_CURAND is None, reason="libcurand not found")


@needs_curand
@pytest.mark.parametrize("seed", [7, 0x0123456789ABCDEF, 0xDEADBEEFCAFEF00D])
def test_philox_words_match_curand_host(seed):
    n_sub, n_ctr = 65536, 3
    words = _curand_host(seed, 4 * n_sub * n_ctr).reshape(n_ctr, n_sub, 4)
    for step in range(n_ctr):
        mine = oracle.philox_words(seed, step, 0, n_sub)
        assert np.array_equal(mine, words[step]), f"step {step}"


@needs_curand
def test_philox_high_counter_word_matches_curand_host():
    seed = 0xDEADBEEFCAFEF00D
    for c0, c1, c2 in [(0, 1, 0), (7, 3, 9), (0, 2 ** 13 - 1, 65535)]:
        off = (c1 << 50) + 4 * 65536 * c0 + 4 * c2
        lib_words = _curand_host(seed, 4, offset=off)
        step = (c1 << 32) | c0
        assert np.array_equal(oracle.philox_words(seed, step, c2, 1)[0], lib_words)


def test_philox_is_a_bijection_on_low_counter_bits():
    # distinct counters -> distinct outputs (a dropped round or a constant output would fail)
    w = oracle.philox_words(7, 0, 0, 4096)
    assert len({tuple(r) for r in w.tolist()}) == 4096
    w2 = oracle.philox_words(7, 1, 0, 4096)
    assert not np.array_equal(w, w2)
    assert not np.array_equal(oracle.philox_words(8, 0, 0, 16), w[:16])


def test_noise_formula_from_words():
    """xi = sqrt(-2 ln u1) cos(2 pi u2), u from 52-bit halves (R16), written out with numpy."""
    seed, step = 7, 5
    w = oracle.philox_words(seed, step, 100, 1000).astype(np.uint64)
    a = (w[:, 1] << np.uint64(32)) | w[:, 0]
    b = (w[:, 3] << np.uint64(32)) | w[:, 2]
    u1 = ((a >> np.uint64(12)).astype(np.float64) + 0.5) * 2.0 ** -52
    u2 = ((b >> np.uint64(12)).astype(np.float64) + 0.5) * 2.0 ** -52
    assert (u1 > 0).all() and (u1 < 1).all() and (u2 > 0).all() and (u2 < 1).all()
    xi = np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
    got = oracle.director_noise(seed, step, 100, 1000)
    assert np.allclose(got, xi, rtol=0, atol=1e-14)


def test_noise_is_standard_normal():
    from scipy import stats
    n = 1_000_000
    xi = np.concatenate([oracle.director_noise(7, s, 0, n // 10) for s in range(10)])
    assert abs(xi.mean()) < 4.0 / np.sqrt(n)
    assert abs(xi.var() - 1.0) < 4.0 * np.sqrt(2.0 / n)
    assert abs(stats.skew(xi)) < 0.02 and abs(stats.kurtosis(xi)) < 0.03
    ks = stats.kstest(xi, "norm")
    assert ks.pvalue > 1e-3
    # consecutive steps of the same cell and neighbouring cells of the same step are uncorrelated
    a = oracle.director_noise(7, 0, 0, 100000)
    b = oracle.director_noise(7, 1, 0, 100000)
    assert abs(np.corrcoef(a, b)[0, 1]) < 0.015
    assert abs(np.corrcoef(a[:-1], a[1:])[0, 1]) < 0.015
