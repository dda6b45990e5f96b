"""Host-side checks of the CUDA library's double-double arithmetic (csrc/dd.cuh, newell_dd.cuh).

The same source that the setup kernels compile for the device is built here with g++
(-DHFFT_DD_HOST_TEST) and compared with mpmath (log, atan, sqrt, div) and with the oracle's
binary128 f and g (Eq.10, Eq.16), including the zero-argument
cases of reading A5.  No GPU needed.
"""
import ctypes
import os
import subprocess

import mpmath as mp
import numpy as np
import pytest

import oracle as O

HERE = os.path.dirname(os.path.abspath(__file__))
mp.mp.dps = 50


@pytest.fixture(scope="module")
def lib(tmp_path_factory):
    so = str(tmp_path_factory.mktemp("dd") / "libddhost.so")
    subprocess.check_call(["g++", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-Wno-unknown-pragmas",
                           "-o", so, os.path.join(HERE, "dd_host_harness.cpp")])
    L = ctypes.CDLL(so)
    dp = ctypes.POINTER(ctypes.c_double)
    L.hfft_test_phi6.argtypes = [dp] * 4
    L.hfft_test_log.argtypes = [dp] * 2
    L.hfft_test_atan.argtypes = [dp] * 2
    L.hfft_test_sqrt_div.argtypes = [dp] * 3
    return L


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _split(v):
    hi = float(v)
    return np.array([hi, float(v - mp.mpf(hi))])


def _join(a, k=0):
    return mp.mpf(float(a[k])) + mp.mpf(float(a[k + 1]))


def test_log_atan_sqrt_div(lib):
    rng = np.random.default_rng(1)
    vals = [mp.mpf(v) for v in (1e-8, 0.3, 0.70710678, 0.99999, 1, 1.0000001, 1.4142, 2, 17.5, 3e9)]
    vals += [mp.mpf(float(v)) * mp.mpf("1.000000000000000000012345") for v in np.exp(rng.uniform(-20, 20, 200))]
    out = np.zeros(4)
    for v in vals:
        a = _split(v)
        lib.hfft_test_log(_p(a), _p(out))
        ref = mp.log(_join(a))
        assert abs(_join(out) - ref) <= 1e-30 * max(abs(ref), mp.mpf(1)), (v, _join(out), ref)
        lib.hfft_test_atan(_p(a), _p(out))
        ref = mp.atan(_join(a))
        assert abs(_join(out) - ref) <= 2e-31, (v,)
        b = _split(mp.mpf(3) / 7 + v)
        lib.hfft_test_sqrt_div(_p(a), _p(b), _p(out))
        assert abs(_join(out, 0) / mp.sqrt(_join(a)) - 1) < 1e-30
        assert abs(_join(out, 2) / (_join(a) / _join(b)) - 1) < 1e-30


def _oracle_six(x, y, z):
    f, g = O.newell_f, O.newell_g
    vals = [f(x, y, z), f(y, x, z), f(z, x, y), g(x, y, z), g(x, z, y), g(y, z, x)]
    return [mp.mpf(h) + mp.mpf(l) for h, l in vals]


PTS = [(2.0, 1.5, 0.7), (0.0, 1.5, 0.7), (2.0, 0.0, 0.7), (2.0, 1.5, 0.0), (0.0, 0.0, 0.7), (0.0, 1.5, 0.0),
       (2.0, 0.0, 0.0), (0.0, 0.0, 0.0), (1.0, 1.0, 1.0), (512.0, 510.0, 0.3), (3.0, 3.0, 0.5), (1e-3, 400.0, 37.1),
       (510.0, 2.0, 55.5)]


@pytest.mark.parametrize("x,y,z", PTS)
def test_phi6_matches_binary128_oracle(lib, x, y, z):
    out = np.zeros(12)
    ax, ay, az = (np.array([v, 0.0]) for v in (x, y, z))
    lib.hfft_test_phi6(_p(ax), _p(ay), _p(az), _p(out))
    ref = _oracle_six(x, y, z)
    scale = max(x, y, z, 1.0) ** 3
    for c in range(6):
        got = _join(out, 2 * c)
        assert abs(got - ref[c]) <= 1e-28 * scale, (c, got, ref[c])
