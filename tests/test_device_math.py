"""The director update's elementary functions (csrc/avm_math.cuh) against mpmath.

The header compiles as plain C++, so the polynomials, range reductions and constants the CUDA
path uses are checked here on the host (the only difference on the device is the reciprocal seed,
which the Newton steps wash out).  Pins: mpmath at 40 digits; the split constants of ln 2 and
pi/2 against their definitions.
"""
import ctypes
import os
import subprocess

import mpmath
import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def lib(tmp_path_factory):
    so = str(tmp_path_factory.mktemp("devmath") / "libdevmath.so")
    subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-shared", "-fPIC", "-o", so,
                           os.path.join(HERE, "device_math_harness.cpp")])
    L = ctypes.CDLL(so)
    p = ctypes.c_void_p
    L.h_log_unit.argtypes = [ctypes.c_long, p, p]
    L.h_cos_2pi.argtypes = [ctypes.c_long, p, p]
    L.h_sincos_any.argtypes = [ctypes.c_long, p, p, p]
    return L


def _call1(f, x):
    x = np.ascontiguousarray(x, dtype=np.float64)
    out = np.empty_like(x)
    f(len(x), x.ctypes.data, out.ctypes.data)
    return out


def _ulps(got, exact):
    """error of `got` in units of the last place of the exact value (mpmath numbers)."""
    errs = []
    for g, e in zip(got, exact):
        ulp = np.spacing(abs(float(e))) if e != 0 else np.spacing(0.0)
        errs.append(abs(mpmath.mpf(float(g)) - e) / mpmath.mpf(float(ulp)))
    return max(errs)


def _uniforms(rng, n):
    m = rng.integers(0, 2 ** 52, size=n, dtype=np.uint64)
    return (m.astype(np.float64) + 0.5) * 2.0 ** -52


def test_split_constants():
    mpmath.mp.dps = 60
    hi, lo = 6.93147180369123816490e-01, 1.9082149292705877e-10
    assert abs(mpmath.mpf(hi) + mpmath.mpf(lo) - mpmath.log(2)) < mpmath.mpf(2) ** -84
    import struct
    assert struct.unpack("<Q", struct.pack("<d", hi))[0] & ((1 << 21) - 1) == 0     # e * hi exact for |e| < 2^20
    p1, p2, p3 = 1.57079632679489655800e+00, 6.12323399573676603587e-17, -1.49738490485916983294e-33
    assert abs(mpmath.mpf(p1) + mpmath.mpf(p2) + mpmath.mpf(p3) - mpmath.pi / 2) < mpmath.mpf(2) ** -155


def test_log_unit(lib):
    mpmath.mp.dps = 40
    rng = np.random.default_rng(1)
    u = np.concatenate([_uniforms(rng, 4000), [0.5 * 2.0 ** -52, 1.0 - 2.0 ** -53, 0.5, 0.70710678118654746, 0.70710678118654757,
                                               2.0 ** -30, 0.999, 1e-5, 0.25 + 2.0 ** -53]])
    got = _call1(lib.h_log_unit, u)
    exact = [mpmath.log(mpmath.mpf(float(x))) for x in u]
    assert _ulps(got, exact) <= 1.5
    assert np.all(got < 0)


def test_cos_2pi(lib):
    mpmath.mp.dps = 40
    rng = np.random.default_rng(2)
    u = np.concatenate([_uniforms(rng, 4000), [0.5 * 2.0 ** -52, 1.0 - 2.0 ** -53, 0.25 + 2.0 ** -53, 0.75 - 2.0 ** -53,
                                               0.5 + 2.0 ** -53, 0.125 + 2.0 ** -53]])
    got = _call1(lib.h_cos_2pi, u)
    exact = [mpmath.cos(2 * mpmath.pi * mpmath.mpf(float(x))) for x in u]
    # absolute accuracy is what Box-Muller needs (near the zeros of the cosine the ulp shrinks)
    err = max(abs(mpmath.mpf(float(g)) - e) for g, e in zip(got, exact))
    assert err < 2.5e-16
    big = [i for i, e in enumerate(exact) if abs(e) > 0.1]
    assert _ulps(got[big], [exact[i] for i in big]) <= 4.0


@pytest.mark.parametrize("scale", [1.0, 30.0, 1e4, 1e8])
def test_sincos_any(lib, scale):
    mpmath.mp.dps = 50
    rng = np.random.default_rng(3)
    t = np.concatenate([rng.normal(0.0, scale, size=3000), [0.0, 1e-300, -1e-8, np.pi / 4, -np.pi / 4, np.pi / 2, 3 * np.pi / 4,
                                                           np.pi, 1e5 * np.pi, 1.0e9, -1.0e9]])
    s = np.empty_like(t)
    c = np.empty_like(t)
    lib.h_sincos_any(len(t), t.ctypes.data, s.ctypes.data, c.ctypes.data)
    es = [mpmath.sin(mpmath.mpf(float(x))) for x in t]
    ec = [mpmath.cos(mpmath.mpf(float(x))) for x in t]
    assert max(abs(mpmath.mpf(float(g)) - e) for g, e in zip(s, es)) < 2.0e-16
    assert max(abs(mpmath.mpf(float(g)) - e) for g, e in zip(c, ec)) < 2.0e-16
    assert np.allclose(s * s + c * c, 1.0, rtol=0, atol=5e-16)


def test_sincos_fallback_range(lib):
    t = np.array([2.0 ** 31, -3.0e12, 1.0e15])
    s = np.empty_like(t)
    c = np.empty_like(t)
    lib.h_sincos_any(len(t), t.ctypes.data, s.ctypes.data, c.ctypes.data)
    assert np.allclose(s, np.sin(t), atol=1e-15) and np.allclose(c, np.cos(t), atol=1e-15)
