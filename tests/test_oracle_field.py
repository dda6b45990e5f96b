"""Pins of the oracle's field tiers (oracle/oracle.py): T0 direct sum (Eq.18) and T1 hybrid (Eq.24).

P8   coarse-graining: for uniform m the volume average of H equals -Ms N_box m with N_box the
     self-term of the bounding box (additivity of Eq.3); cube -> -Ms/3 per axis
P10  the paper's worked example: SAF stack -> t = 3.44 nm (tests/golden/saf_thickness.txt)
P11  T1 == T0 to rounding on C1 and C2 (discrete convolution theorem, Eq.20-24)
     naive-DFT form == numpy FFT form of T1 (library routine)
A12  linearity in per-layer Ms
"""
import os

import numpy as np
import pytest

import oracle as O
from paper_1910_07054_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _relerr(a, b):
    return np.abs(a - b).max() / np.abs(b).max()


def test_T1_equals_T0_on_C1():
    w = W.config(1)
    m = w.m()[0]
    H0 = O.direct_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms)
    H1 = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, dft="naive")
    H2 = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    assert _relerr(H1, H0) < 1e-14
    assert _relerr(H2, H0) < 1e-14
    # demag field opposes the magnetisation on average and is of order Ms
    assert 0.05 * 8e5 < np.abs(H0).max() < 8e5


def test_T1_equals_T0_on_C2_sampled_layers():
    w = W.config(2, "f64")
    m = w.m()[0]
    rng = np.random.default_rng(5)
    layers = [0, 3, 5]
    H1 = O.hybrid_layers(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, layers, dft="fft")
    for t, i in enumerate(layers):
        cells = rng.choice(w.nx * w.ny, size=400, replace=False).astype(np.int32)
        H0 = O.direct_cells(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, i, cells)
        got = H1[t].reshape(3, -1)[:, cells].T
        assert np.abs(got - H0).max() / np.abs(H1).max() < 1e-14


def test_naive_dft_equals_fft_and_batched():
    w = W.small(8, 16, 4, B=3, seed=3)
    m = w.m()
    Hn = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, dft="naive")
    Hf = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    assert Hn.shape == m.shape
    assert _relerr(Hn, Hf) < 1e-14
    for b in range(3):
        H0 = O.direct_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m[b], w.Ms)
        assert _relerr(Hn[b], H0) < 1e-14


def test_linearity_in_per_layer_Ms():
    w = W.small(8, 8, 3, seed=4)
    m = w.m()[0]
    H = O.direct_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms)
    acc = np.zeros_like(H)
    for j in range(w.nz):
        e = np.zeros(w.nz)
        e[j] = 1.0
        acc += w.Ms[j] * O.direct_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, e)
    assert _relerr(acc, H) < 1e-14
    # Ms = None means m already holds M
    Hn = O.direct_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m * w.Ms[None, :, None, None], None)
    assert _relerr(Hn, H) < 1e-15


@pytest.mark.parametrize("nx,ny,dz,dx,dy", [
    (4, 6, [1.0, 2.0, 0.6], 2.0, 1.5),
    (3, 3, [1.5, 1.0, 2.0], 1.5, 1.5),      # 4.5 nm cube -> -Ms/3 per axis
])
def test_coarse_graining_uniform_magnetisation(nx, ny, dz, dx, dy):
    dz = np.array(dz)
    nz = len(dz)
    Ms = 8e5
    box = np.array([nx * dx, ny * dy, dz.sum()])
    hi, lo = O.tensor_point([0, 0, 0], box, box)
    for a in range(3):
        m = np.zeros((3, nz, ny, nx))
        m[a] = 1.0
        for field in (O.direct_field, lambda *args: O.hybrid_field(*args, dft="naive")):
            H = field(nx, ny, nz, dx, dy, dz, m, Ms)
            avg = (H * dz[None, :, None, None]).sum(axis=(1, 2, 3)) / (nx * ny * dz.sum())
            ref = np.zeros(3)
            ref[a] = -Ms * (hi[a] + lo[a])
            assert np.abs(avg - ref).max() < 1e-12 * Ms
    if abs(box[0] - box[1]) < 1e-12 and abs(box[0] - box[2]) < 1e-12:
        assert abs(hi[0] - 1 / 3) < 1e-15


def test_paper_worked_example_saf_thickness():
    """60 nm cylinder, 64 x 64 x 5, layers 5 / 1 / t / 1 / 3 nm, layer 0 +z,
    layer 2 -z; t such that <H_z> over the free layer vanishes is printed as 3.44 nm.
    Reading A14: cell = 60/64 nm, sources = cells whose centre lies inside
    r = 30 nm, equal Ms, average over all 64 x 64 free-layer cells."""
    with open(os.path.join(GOLD, "saf_thickness.txt")) as fh:
        rows = [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]
    t_paper, tol = float(rows[0][0]), float(rows[0][1])

    n = 64
    d = 60.0 / n
    c = (np.arange(n) + 0.5) * d - 30.0
    disc = (c[None, :] ** 2 + c[:, None] ** 2) < 30.0 ** 2
    m = np.zeros((3, 5, n, n))
    m[2, 0][disc] = 1.0
    m[2, 2][disc] = -1.0

    def mean_hz(t):
        dz = np.array([5.0, 1.0, t, 1.0, 3.0])
        H = O.hybrid_layers(n, n, 5, d, d, dz, m, None, [4], dft="fft")
        return H[0, 2].mean()

    # secant iteration (the paper uses Newton; how its derivative is formed is not stated)
    t0, t1 = 5.0, 3.0
    f0, f1 = mean_hz(t0), mean_hz(t1)
    for _ in range(8):
        t2 = t1 - f1 * (t1 - t0) / (f1 - f0)
        t0, f0, t1 = t1, f1, t2
        f1 = mean_hz(t1)
        if abs(f1) < 1e-9:
            break
    assert abs(t1 - t_paper) < tol, t1
    assert round(t1, 2) == t_paper
