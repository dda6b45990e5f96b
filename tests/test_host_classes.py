"""Host logic of the deduplicated bank (no GPU): hfft_tensor_classes against the definition.

N_ij depends on (dz_i, dz_j, Z_ij = zeta_i - zeta_j) alone (Eq.19 with Eq.5 :52 / Eq.11 :99), so two
pairs share a bank slot exactly when the three agree.  The expected partition is computed here in exact rational
arithmetic; for equal thicknesses the library folds i - j to |i - j| (reciprocity and parity).
"""
import os
import sys
from fractions import Fraction

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


@pytest.fixture(scope="module")
def hb():
    from paper_1910_07054_b200 import build as hbuild
    hbuild.build()
    from paper_1910_07054_b200 import binding
    return binding


def _keys(dz):
    fz = [Fraction(float(v)) for v in dz]
    zeta = [sum(fz[:k], Fraction(0)) for k in range(len(dz))]
    return [[(fz[i], fz[j], zeta[i] - zeta[j]) for j in range(len(dz))] for i in range(len(dz))]


def _check_partition(cls, keys, fold):
    """Same slot <=> same key (after folding Z -> |Z| for equal thicknesses)."""
    nz = len(keys)
    norm = (lambda k: (k[0], k[1], abs(k[2]))) if fold else (lambda k: k)
    slot_of = {}
    for i in range(nz):
        for j in range(nz):
            k = norm(keys[i][j])
            assert slot_of.setdefault(k, cls[i, j]) == cls[i, j], (i, j)
    assert len(set(slot_of.values())) == len(slot_of)          # distinct keys -> distinct slots
    return len(slot_of)


STACKS = [
    [1.0], [1.0, 1.0], [1.0, 2.0], [0.75] * 7, [0.1] * 40, [1.0, 0.5] * 5, [1.0, 0.25, 2.0] * 4,
    [5.0, 1.0, 5.0, 1.0, 3.0], [1.0, 2.0, 0.6], [1.0, 0.8, 0.9, 1.2, 1.0, 2.5], [0.3] * 3 + [0.7] * 3,
]


@pytest.mark.parametrize("dz", STACKS, ids=lambda d: "%dx%g" % (len(d), d[0]))
def test_classes_match_the_definition(hb, dz):
    cls, n, toep = hb.tensor_classes(dz)
    equal = len(dz) > 1 and len(set(dz)) == 1
    assert toep == equal
    assert n == _check_partition(cls, _keys(dz), fold=toep)
    assert sorted(set(cls.ravel())) == list(range(n))
    if toep:
        nz = len(dz)
        assert n == nz and all(cls[i, j] == abs(i - j) for i in range(nz) for j in range(nz))


def test_classes_of_random_stacks_are_all_distinct(hb):
    rng = np.random.default_rng(1)
    dz = np.exp(rng.uniform(np.log(0.3), np.log(3.0), size=24))
    cls, n, toep = hb.tensor_classes(dz)
    assert n == 24 * 24 and not toep
    assert np.array_equal(cls, np.arange(576).reshape(24, 24))


def test_classes_with_inexact_sums(hb):
    """dz = 0.1 is not a binary fraction: the interface coordinates are accumulated in double-double, and pairs with
    the same i - j must still land in one class (tolerance 2^-80 of the stack height)."""
    cls, n, toep = hb.tensor_classes([0.1] * 64)
    assert toep and n == 64


def test_classes_argument_errors(hb):
    L = hb.lib()
    import ctypes
    out = (ctypes.c_int * 4)()
    n, t = ctypes.c_int(), ctypes.c_int()
    dz = (ctypes.c_double * 2)(1.0, -1.0)
    assert L.hfft_tensor_classes(2, dz, out, ctypes.byref(n), ctypes.byref(t)) == hb.EINVAL
    assert L.hfft_tensor_classes(0, dz, out, ctypes.byref(n), ctypes.byref(t)) == hb.EINVAL
    assert L.hfft_tensor_classes(2, None, out, ctypes.byref(n), ctypes.byref(t)) == hb.EINVAL
