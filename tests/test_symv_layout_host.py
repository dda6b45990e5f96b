"""Host-side checks of the reciprocity bank's layout (csrc/symv_layout.h, read by coupling_symv.cu and written by
tensor_build.cu): the header is compiled here with g++ and every layer count the kernel accepts is checked for what the
schedule promises -- every unordered layer pair stored exactly once, (i, j) and (j, i) in the same slot with opposite
orientation, slots inside the unit's stream and disjoint, blocks ending on stage boundaries.  No GPU needed."""
import ctypes
import os
import subprocess

import numpy as np
import pytest

HERE = os.path.dirname(os.path.abspath(__file__))


@pytest.fixture(scope="module")
def lib(tmp_path_factory):
    so = str(tmp_path_factory.mktemp("symv") / "libsymvhost.so")
    subprocess.check_call(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-o", so, os.path.join(HERE, "symv_layout_harness.cpp")])
    L = ctypes.CDLL(so)
    lp = ctypes.POINTER(ctypes.c_longlong)
    L.hfft_test_symv_geom.argtypes = [ctypes.c_int, lp]
    L.hfft_test_symv_pos.argtypes = [ctypes.c_int] * 5 + [lp]
    return L


def _geom(lib, nz):
    out = (ctypes.c_longlong * 8)()
    lib.hfft_test_symv_geom(nz, out)
    return dict(zip(("W", "LW", "EPW", "nfull", "half", "NC", "SPE", "pairs"), out))


def _pos(lib, nz, i, j, ent=0, c=0):
    out = (ctypes.c_longlong * 5)()
    lib.hfft_test_symv_pos(nz, i, j, ent, c, out)
    return tuple(out)


@pytest.mark.parametrize("nz", list(range(2, 65)))
def test_every_unordered_pair_is_stored_once(lib, nz):
    g = _geom(lib, nz)
    assert g["W"] == (nz + 3) // 4 and g["LW"] >= g["W"] and g["LW"] & (g["LW"] - 1) == 0 and g["EPW"] * g["LW"] == 16
    assert g["NC"] == 8 * g["nfull"] + 4 * g["half"] + 5
    assert g["NC"] % 4 == 1 and g["SPE"] == (g["NC"] + 3) // 4         # the last 3 KB stage of a unit is a single couple
    # W strips meet round-robin: nfull full steps, one half step if W is even, the diagonal
    assert 2 * g["nfull"] + g["half"] + 1 == g["W"]
    slots = {}
    for i in range(nz):
        for j in range(nz):
            couple, h, strip, transposed, _ = _pos(lib, nz, i, j)
            assert 0 <= couple < g["NC"] and h in (0, 1) and 0 <= strip < g["W"]
            key = (couple, h, strip)
            if i <= j:
                assert key not in slots, "two unordered pairs share a slot"
                slots[key] = (i, j, transposed)
            else:
                # (j, i) was seen first: same slot, the other orientation
                assert slots[key][:2] == (j, i) and slots[key][2] != transposed
            if i == j:
                assert transposed == 0
    assert len(slots) == nz * (nz + 1) // 2
    # what the stream costs: NC couples x 2 pairs x 16 strip-lanes, shared by EPW entries
    assert g["pairs"] == g["NC"] * 32 // g["EPW"] >= nz * (nz + 1) // 2


@pytest.mark.parametrize("nz", [2, 3, 8, 10, 16, 17, 33, 64])
def test_float_offsets_are_disjoint_and_inside_the_unit(lib, nz):
    g = _geom(lib, nz)
    unit_floats = g["NC"] * 192
    seen = set()
    for ent in range(g["EPW"]):
        for i in range(nz):
            for j in range(i, nz):
                for c in range(6):
                    off = _pos(lib, nz, i, j, ent, c)[4]
                    assert 0 <= off < unit_floats and off not in seen
                    seen.add(off)
    assert len(seen) == g["EPW"] * 6 * nz * (nz + 1) // 2


def test_config_sizes(lib):
    # C4 (nz = 64): 16 strips, no padding: 2080 pairs per entry = nz (nz + 1) / 2; C3 (nz = 16): 136
    assert _geom(lib, 64)["pairs"] == 2080 and _geom(lib, 64)["EPW"] == 1
    assert _geom(lib, 16)["pairs"] == 136 and _geom(lib, 16)["EPW"] == 4
