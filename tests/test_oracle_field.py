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


@pytest.mark.parametrize("dft", ["naive", "fft"])
def test_hoisted_setup_arguments_do_not_change_the_field(dft):
    """hybrid_layers(rows=, nhat=): tensor rows / tensor spectra computed by the caller beforehand (what bench.py's CPU
    baseline does so that it times the evaluation with the bank pre-built, like the GPU arm) give the same bits as
    the call that computes them itself, and the spectrum they carry is the DFT of the periodic tensor (checked at
    k = 0, where the transform is the plain sum over the offsets)."""
    w = W.small(8, 4, 3, B=2, seed=9)
    m = w.m()
    layers = [2, 0]
    plain = O.hybrid_layers(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, layers, dft=dft)
    rows = {i: O.tensor_row(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, i) for i in layers}
    nhat = {i: O.tensor_spectrum(rows[i], w.nx, w.ny, dft) for i in layers}
    assert nhat[0].shape == (w.nz, 6, 2 * w.ny, 2 * w.nx)
    assert np.abs(nhat[2][:, :, 0, 0] - rows[2].sum(axis=(-1, -2))).max() <= 1e-14 * np.abs(rows[2]).sum(axis=(-1, -2)).max()
    assert np.array_equal(O.hybrid_layers(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, layers, dft=dft, rows=rows), plain)
    assert np.array_equal(O.hybrid_layers(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, layers, dft=dft, nhat=nhat), plain)
    # a partial dictionary falls back to the computation for the missing layer
    assert np.array_equal(O.hybrid_layers(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, layers, dft=dft, nhat={0: nhat[0]}), plain)


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


# ---------------------------------------------------------------- off-diagonal plumbing of T0 / T1
@pytest.mark.parametrize("src,tgt", [((1, 2, 0), (10, 8, 2)), ((9, 1, 2), (0, 7, 0)), ((3, 8, 1), (11, 0, 2))])
def test_single_cell_source_gives_every_field_component_in_another_layer(src, tgt):
    """One cell of layer j magnetised along b = x, y, z in turn; all three components of H in a distant cell of
    another layer i, from T0 (direct_field) and T1 (hybrid_field):

      H_a(target) = - Ms_j N^{ab}_{ij}((a1-b1) dx, (a2-b2) dy) m_b           (Eq.18, one term)

    (a) against hfft_oracle_tensor_point evaluated here at the offset (X, Y, zeta_i - zeta_j) with the symmetric
        3 x 3 tensor written out from its six components (Eq.4) -- pins the component table COMP of
        oracle.py / hfft_oracle.c and the sign and index conventions of the off-diagonal entries, which no
        uniform-magnetisation or zz-only test sees;
    (b) against the point-dipole field of Eq.1-2, H = (3 r (r.mu) - mu r^2) / (4 pi r^5),
        mu = Ms V' m, r from the source centre to the target centre: relative deviation O((cell / r)^2)."""
    nx, ny, nz = 12, 10, 3
    dx, dy = 1.0, 1.2
    dz = np.array([0.7, 1.6, 1.1])
    Ms = np.array([8e5, 1.1e6, 9e5])
    zeta = np.concatenate([[0.0], np.cumsum(dz)])
    (b1, b2, j), (a1, a2, i) = src, tgt
    assert i != j
    X = np.array([(a1 - b1) * dx, (a2 - b2) * dy, zeta[i] - zeta[j]])
    hi, lo = O.tensor_point(X, [dx, dy, dz[i]], [dx, dy, dz[j]])
    n = hi + lo
    xx, yy, zz, xy, xz, yz = n
    N = np.array([[xx, xy, xz], [xy, yy, yz], [xz, yz, zz]])
    assert min(abs(xy), abs(xz), abs(yz)) > 1e-6                 # generic offset: no component vanishes
    # centre-to-centre vector and the dipole tensor (1 / 4 pi) (3 r r^T / r^5 - I / r^3)
    r = X + 0.5 * np.array([0.0, 0.0, dz[i] - dz[j]])
    rn = np.linalg.norm(r)
    dip = (3.0 * np.outer(r, r) / rn**5 - np.eye(3) / rn**3) / (4.0 * np.pi)
    Vp = dx * dy * dz[j]
    for b in range(3):
        m = np.zeros((3, nz, ny, nx))
        m[b, j, b2, b1] = 1.0
        want = -Ms[j] * N[:, b]
        H0 = O.direct_field(nx, ny, nz, dx, dy, dz, m, Ms)
        H1 = O.hybrid_field(nx, ny, nz, dx, dy, dz, m, Ms, dft="fft")
        for H in (H0, H1):
            got = H[:, i, a2, a1]
            assert np.abs(got - want).max() <= 1e-13 * np.abs(Ms[j] * n).max(), (b, got, want)
        # dipole limit: sign and position of every off-diagonal entry, independent of the Newell formulas
        mu = np.zeros(3)
        mu[b] = Ms[j] * Vp
        Hd = dip @ mu
        assert np.abs(H0[:, i, a2, a1] - Hd).max() <= 0.05 * np.abs(Hd).max(), (b, H0[:, i, a2, a1], Hd)
        for a in range(3):
            if abs(Hd[a]) > 0.2 * np.abs(Hd).max():
                assert np.sign(H0[a, i, a2, a1]) == np.sign(Hd[a])
