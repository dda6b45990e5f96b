"""Pins of the oracle's tensor (oracle/hfft_oracle.c) against what the paper and the
mathematics fix -- none of these retype Eq.10/16 or the 64-term sums.

P1  f, g:  parity / symmetry and  d2y d2z f = 1/R (Eq.8),  dx dy d2z g = 1/R (Eq.14)
P2  cube self-term = (1/3,1/3,1/3), off-diagonals 0
P3  trace = 1 (self) / 0 (disjoint)              [Eq.3: laplace(1/r) = -4 pi delta]
P4  prism self-term = Aharoni's closed form (textbook); equal sizes = classical Newell limit
P5  additivity (source / target split), reciprocity, in-plane parity
P6  far field -> point dipole  V'(I - 3 rr^T)/(4 pi r^3)   [Eq.1-2 PAPER.md:29-33]
P7  6-D Gauss-Legendre quadrature of the volume-integral definition Eq.3 for fully unequal cuboids
P9  binary128 really is needed: the fp64 evaluation of the same sums is visibly worse
"""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle as O

mp.mp.dps = 45
rng = np.random.default_rng(1910_07054)


def _split(v):
    hi = float(v)
    return hi, float(v - mp.mpf(hi))


def _f(x, y, z):
    hi, lo = O.newell_f(_split(x), _split(y), _split(z))
    return mp.mpf(hi) + mp.mpf(lo)


def _g(x, y, z):
    hi, lo = O.newell_g(_split(x), _split(y), _split(z))
    return mp.mpf(hi) + mp.mpf(lo)


def _N(X, D, Dp):
    hi, lo = O.tensor_point(X, D, Dp)
    return hi + lo  # fp64 is enough for most pins; hi/lo used where more is needed


PTS = [(0.7, 1.3, 2.1), (2.0, 0.4, 0.9), (5.5, 3.25, 0.125), (0.3, 0.3, 4.0)]


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("x,y,z", PTS)
def test_f_parity_and_symmetry(x, y, z):
    x, y, z = mp.mpf(x), mp.mpf(y), mp.mpf(z)
    v = _f(x, y, z)
    for sx in (1, -1):
        for sy in (1, -1):
            for sz in (1, -1):
                assert abs(_f(sx * x, sy * y, sz * z) - v) <= mp.mpf(10) ** -30 * abs(v)
    # f is symmetric in its last two arguments (the y/z roles of Eq.8 are interchangeable)
    assert abs(_f(x, z, y) - v) <= mp.mpf(10) ** -30 * abs(v)


@pytest.mark.parametrize("x,y,z", PTS)
def test_g_parity_and_symmetry(x, y, z):
    x, y, z = mp.mpf(x), mp.mpf(y), mp.mpf(z)
    v = _g(x, y, z)
    tol = mp.mpf(10) ** -30 * abs(v)
    assert abs(_g(-x, y, z) + v) <= tol      # odd in x
    assert abs(_g(x, -y, z) + v) <= tol      # odd in y
    assert abs(_g(x, y, -z) - v) <= tol      # even in z
    assert abs(_g(y, x, z) - v) <= tol       # x <-> y symmetric (Eq.14)


def _second_diff(fun, h):
    return lambda t: (fun(t + h) - 2 * fun(t) + fun(t - h)) / h ** 2


@pytest.mark.parametrize("x,y,z", PTS)
def test_f_fourth_derivative_is_inverse_distance(x, y, z):
    """Eq.8: F2 is the 4-fold integral of 1/sqrt(X^2+y~^2+z~^2), so
    d^2/dY^2 d^2/dZ^2 f(X,Y,Z) = 1/R."""
    x, y, z = mp.mpf(x), mp.mpf(y), mp.mpf(z)
    h = mp.mpf(10) ** -5
    d = _second_diff(lambda yy: _second_diff(lambda zz: _f(x, yy, zz), h)(z), h)(y)
    R = mp.sqrt(x * x + y * y + z * z)
    assert abs(d * R - 1) < mp.mpf(10) ** -8


@pytest.mark.parametrize("x,y,z", PTS)
def test_g_fourth_derivative_is_inverse_distance(x, y, z):
    """Eq.14: d/dX d/dY d^2/dZ^2 g(X,Y,Z) = 1/R."""
    x, y, z = mp.mpf(x), mp.mpf(y), mp.mpf(z)
    h = mp.mpf(10) ** -5

    def dxy(zz):
        return (_g(x + h, y + h, zz) - _g(x + h, y - h, zz) - _g(x - h, y + h, zz) + _g(x - h, y - h, zz)) / (4 * h * h)

    d = _second_diff(dxy, h)(z)
    R = mp.sqrt(x * x + y * y + z * z)
    assert abs(d * R - 1) < mp.mpf(10) ** -8


def test_f_g_boundary_values_of_the_four_fold_integrals():
    """F2 (Eq.8/9) vanishes when Y = 0 or Z = 0; G2 (Eq.14/15) when X = 0, Y = 0 or Z = 0.
    With Eq.9 / Eq.15 this fixes the terms the derivative test cannot see."""
    x, y, z = mp.mpf("0.9"), mp.mpf("1.7"), mp.mpf("0.6")

    def F2(X, Y, Z):
        return _f(X, Y, Z) - _f(X, 0, Z) - _f(X, Y, 0) + _f(X, 0, 0)

    def G2(X, Y, Z):
        return _g(X, Y, Z) - _g(X, Y, 0)

    assert F2(x, 0, z) == 0 and F2(x, y, 0) == 0
    assert G2(x, y, 0) == 0
    assert abs(G2(0, y, z)) < mp.mpf(10) ** -32 and abs(G2(x, 0, z)) < mp.mpf(10) ** -32
    # and F2 itself against direct 2-D quadrature of its twice-differentiated form:
    # d/dY d/dZ F2 = int_0^Z int_0^Y 1/R
    h = mp.mpf(10) ** -8
    dF = (F2(x, y + h, z + h) - F2(x, y + h, z - h) - F2(x, y - h, z + h) + F2(x, y - h, z - h)) / (4 * h * h)
    ref = mp.quad(lambda a, b: 1 / mp.sqrt(x * x + a * a + b * b), [0, y], [0, z])
    assert abs(dF - ref) < mp.mpf(10) ** -12


# ---------------------------------------------------------------- P2, P3
def test_cube_self_term():
    for s in (1.0, 2.0, 0.37):
        hi, lo = O.tensor_point([0, 0, 0], [s, s, s], [s, s, s])
        v = [mp.mpf(hi[c]) + mp.mpf(lo[c]) for c in range(6)]
        for c in range(3):
            assert abs(v[c] - mp.mpf(1) / 3) < mp.mpf(10) ** -31
        for c in range(3, 6):
            assert abs(v[c]) < mp.mpf(10) ** -31


def test_trace_self_and_disjoint():
    for _ in range(20):
        D = rng.uniform(0.3, 3.0, 3)
        hi, lo = O.tensor_point([0, 0, 0], D, D)
        assert abs(float(sum(mp.mpf(hi[c]) + mp.mpf(lo[c]) for c in range(3)) - 1)) < 1e-30
        Dp = rng.uniform(0.3, 3.0, 3)
        # disjoint: put the target beyond the source along a random axis
        X = rng.uniform(-4, 4, 3)
        ax = rng.integers(3)
        X[ax] = Dp[ax] + rng.uniform(0.0, 2.0)  # touching faces allowed (0.0)
        hi, lo = O.tensor_point(X, D, Dp)
        tr = sum(mp.mpf(hi[c]) + mp.mpf(lo[c]) for c in range(3))
        assert abs(float(tr)) < 1e-29


# ---------------------------------------------------------------- P4
def _aharoni_Dz(a, b, c):
    """Demagnetizing factor along z of a uniformly magnetised 2a x 2b x 2c prism,
    A. Aharoni, J. Appl. Phys. 83, 3432 (1998), Eq.(1) -- textbook closed form."""
    a, b, c = mp.mpf(a), mp.mpf(b), mp.mpf(c)
    r = mp.sqrt(a * a + b * b + c * c)
    ab, bc, ac = mp.sqrt(a * a + b * b), mp.sqrt(b * b + c * c), mp.sqrt(a * a + c * c)
    t = (b * b - c * c) / (2 * b * c) * mp.log((r - a) / (r + a))
    t += (a * a - c * c) / (2 * a * c) * mp.log((r - b) / (r + b))
    t += b / (2 * c) * mp.log((ab + a) / (ab - a))
    t += a / (2 * c) * mp.log((ab + b) / (ab - b))
    t += c / (2 * a) * mp.log((bc - b) / (bc + b))
    t += c / (2 * b) * mp.log((ac - a) / (ac + a))
    t += 2 * mp.atan(a * b / (c * r))
    t += (a ** 3 + b ** 3 - 2 * c ** 3) / (3 * a * b * c)
    t += (a * a + b * b - 2 * c * c) / (3 * a * b * c) * r
    t += c / (a * b) * (ac + bc)
    t -= (ab ** 3 + bc ** 3 + ac ** 3) / (3 * a * b * c)
    return t / mp.pi


def test_prism_self_term_matches_aharoni():
    assert abs(_aharoni_Dz(1, 1, 1) - mp.mpf(1) / 3) < mp.mpf(10) ** -40
    for _ in range(10):
        D = rng.uniform(0.2, 5.0, 3)
        hi, lo = O.tensor_point([0, 0, 0], D, D)
        a, b, c = D / 2
        ref = [_aharoni_Dz(b, c, a), _aharoni_Dz(c, a, b), _aharoni_Dz(a, b, c)]  # x, y, z
        for k in range(3):
            got = mp.mpf(hi[k]) + mp.mpf(lo[k])
            assert abs(got - ref[k]) < mp.mpf(10) ** -29


def test_thin_film_and_rod_limits():
    # thin film: Nzz -> 1 (north_star; SURVEY P8 quotes 0.99514 for 1000x1000x1)
    hi, _ = O.tensor_point([0, 0, 0], [1000, 1000, 1], [1000, 1000, 1])
    assert abs(hi[2] - 0.99514) < 5e-6 and hi[0] < 3e-3 and hi[1] < 3e-3
    hi, _ = O.tensor_point([0, 0, 0], [1, 1, 1000], [1, 1, 1000])
    assert hi[2] < 1e-3 and abs(hi[0] - 0.5) < 1e-3 and abs(hi[1] - 0.5) < 1e-3


def test_equal_sizes_reduce_to_classical_newell_stencil():
    """F2 is adopted from Newell without modification, so for equal sizes the
    4-point pattern (D, 0, D-D', -D') collapses to the classical second difference (1,-2,1):
    N = -(1/(4 pi V)) sum_{a,b,c in {-1,0,1}} w_a w_b w_c f(X+a dx, Y+b dy, Z+c dz), w = (1,-2,1)."""
    D = np.array([1.5, 0.8, 2.2])
    X = np.array([3.0, -1.6, 2.2])
    w = {-1: 1, 0: -2, 1: 1}
    accf = mp.mpf(0)
    accg = mp.mpf(0)
    for a in (-1, 0, 1):
        for b in (-1, 0, 1):
            for c in (-1, 0, 1):
                args = (mp.mpf(X[0]) + a * mp.mpf(D[0]), mp.mpf(X[1]) + b * mp.mpf(D[1]), mp.mpf(X[2]) + c * mp.mpf(D[2]))
                accf += w[a] * w[b] * w[c] * _f(*args)
                accg += w[a] * w[b] * w[c] * _g(*args)
    V = mp.mpf(D[0]) * mp.mpf(D[1]) * mp.mpf(D[2])
    hi, lo = O.tensor_point(X, D, D)
    assert abs(-accf / (4 * mp.pi * V) - (mp.mpf(hi[0]) + mp.mpf(lo[0]))) < mp.mpf(10) ** -30
    assert abs(-accg / (4 * mp.pi * V) - (mp.mpf(hi[3]) + mp.mpf(lo[3]))) < mp.mpf(10) ** -30


# ---------------------------------------------------------------- P5
def test_source_and_target_additivity():
    for _ in range(10):
        D = rng.uniform(0.3, 3.0, 3)
        Dp = rng.uniform(0.3, 3.0, 3)
        X = rng.uniform(-5, 5, 3)
        ax = int(rng.integers(3))
        full = _N(X, D, Dp)
        # split the source along ax into [0,s] and [s,Dp]
        s = Dp[ax] * rng.uniform(0.2, 0.8)
        Dp1, Dp2 = Dp.copy(), Dp.copy()
        Dp1[ax], Dp2[ax] = s, Dp[ax] - s
        X2 = X.copy()
        X2[ax] -= s
        assert np.abs(full - (_N(X, D, Dp1) + _N(X2, D, Dp2))).max() < 1e-16
        # split the target along ax: volume-weighted mean (Eq.2 PAPER.md:33 averages over the target)
        t = D[ax] * rng.uniform(0.2, 0.8)
        D1, D2 = D.copy(), D.copy()
        D1[ax], D2[ax] = t, D[ax] - t
        X3 = X.copy()
        X3[ax] += t
        mix = (t * _N(X, D1, Dp) + (D[ax] - t) * _N(X3, D2, Dp)) / D[ax]
        assert np.abs(full - mix).max() < 1e-16


def test_reciprocity_and_parity():
    sgn_x = np.array([1, 1, 1, -1, -1, 1])
    sgn_y = np.array([1, 1, 1, -1, 1, -1])
    for _ in range(10):
        D = rng.uniform(0.3, 3.0, 3)
        Dp = rng.uniform(0.3, 3.0, 3)
        X = rng.uniform(-5, 5, 3)
        # reciprocity: V N(X; D,D') = V' N(-X; D',D)
        a = np.prod(D) * _N(X, D, Dp)
        b = np.prod(Dp) * _N(-X, Dp, D)
        assert np.abs(a - b).max() < 1e-15 * max(1.0, np.abs(a).max())
    # in-plane parity for layer geometry (equal in-plane sizes): mirror x about the common centre
    for _ in range(10):
        dxy = rng.uniform(0.5, 2.0, 2)
        D = np.array([dxy[0], dxy[1], rng.uniform(0.3, 3)])
        Dp = np.array([dxy[0], dxy[1], rng.uniform(0.3, 3)])
        X = np.array([rng.integers(-4, 5) * dxy[0], rng.integers(-4, 5) * dxy[1], rng.uniform(-4, 4)])
        n0 = _N(X, D, Dp)
        nx_ = _N(X * [-1, 1, 1], D, Dp)
        ny_ = _N(X * [1, -1, 1], D, Dp)
        assert np.abs(nx_ - sgn_x * n0).max() < 1e-17
        assert np.abs(ny_ - sgn_y * n0).max() < 1e-17


def test_eq11_as_printed_breaks_symmetry():
    """Reading A1: with the literal 4th term G(X-dx', Y-dy, Z) N_xy is not odd in Y / not
    symmetric; the oracle's reading gives N_xy(X,Y) = N_yx(X,Y), i.e. the xy entry equals the
    xy entry of the x<->y relabelled problem."""
    D = np.array([1.0, 2.0, 0.7])
    Dp = np.array([1.5, 0.4, 1.1])
    X = np.array([3.0, 1.0, -2.5])
    n = _N(X, D, Dp)
    sw = [1, 0, 2]
    n_sw = _N(X[sw], D[sw], Dp[sw])
    assert abs(n[3] - n_sw[3]) < 1e-18            # N_xy == N_yx
    assert abs(n[4] - n_sw[5]) < 1e-18 and abs(n[0] - n_sw[1]) < 1e-18


# ---------------------------------------------------------------- P6
def test_far_field_is_a_point_dipole():
    D = np.array([2.0, 2.0, 1.3])
    Dp = np.array([2.0, 2.0, 0.6])
    dirs = rng.normal(size=(4, 3))
    prev = None
    for dist in (40.0, 80.0, 160.0):
        worst = 0.0
        for u in dirs:
            u = u / np.linalg.norm(u)
            rc = dist * u                       # centre-to-centre
            X = rc - D / 2 + Dp / 2             # lower-corner offset (reading A8)
            n = _N(X, D, Dp)
            T = np.prod(Dp) * (np.eye(3) - 3 * np.outer(u, u)) / (4 * math.pi * dist ** 3)
            ref = np.array([T[0, 0], T[1, 1], T[2, 2], T[0, 1], T[0, 2], T[1, 2]])
            worst = max(worst, np.abs(n - ref).max() / np.abs(ref).max())
        assert worst < 3.0 * (2.0 / dist) ** 2
        if prev is not None:
            assert worst < prev / 3.0           # O((cell/r)^2) decay
        prev = worst


# ---------------------------------------------------------------- P7
def test_six_dimensional_quadrature_of_the_definition():
    """Eq.3: N = 1/(4 pi tau) int_tau int_tau' grad grad' 1/|r-r'|
    = 1/(4 pi tau) int int (I - 3 rho rho^T/rho^2)/rho^3 for separated cuboids."""
    D = np.array([1.0, 2.0, 0.7])
    Dp = np.array([1.5, 0.4, 1.1])
    X = np.array([3.0, 1.0, -2.5])
    n = 12
    t, w = np.polynomial.legendre.leggauss(n)
    t = 0.5 * (t + 1)
    w = 0.5 * w
    # target points X + t*D, source points t*Dp
    acc = np.zeros(6)
    tx, ty, tz = X[0] + t * D[0], X[1] + t * D[1], X[2] + t * D[2]
    sx, sy, sz = t * Dp[0], t * Dp[1], t * Dp[2]
    rx = (tx[:, None] - sx[None, :]).ravel()
    wx = (w[:, None] * w[None, :]).ravel()
    ry = (ty[:, None] - sy[None, :]).ravel()
    rz = (tz[:, None] - sz[None, :]).ravel()
    RX, RY, RZ = np.meshgrid(rx, ry, rz, indexing="ij")
    W = wx[:, None, None] * wx[None, :, None] * wx[None, None, :]
    r2 = RX ** 2 + RY ** 2 + RZ ** 2
    r5 = r2 ** 2.5
    acc[0] = np.sum(W * (r2 - 3 * RX * RX) / r5)
    acc[1] = np.sum(W * (r2 - 3 * RY * RY) / r5)
    acc[2] = np.sum(W * (r2 - 3 * RZ * RZ) / r5)
    acc[3] = np.sum(W * (-3 * RX * RY) / r5)
    acc[4] = np.sum(W * (-3 * RX * RZ) / r5)
    acc[5] = np.sum(W * (-3 * RY * RZ) / r5)
    # int over both volumes / (4 pi tau):   weights are on the unit cube -> * V * V'
    ref = acc * np.prod(Dp) / (4 * math.pi)
    got = _N(X, D, Dp)
    assert np.abs(got - ref).max() < 1e-12 * np.abs(ref).max() + 1e-15


# ---------------------------------------------------------------- P9
def test_binary128_is_needed():
    """SURVEY finding 2: the 64-term sums cancel catastrophically; the same sums in fp64 are
    orders of magnitude less accurate far from the source."""
    D = np.array([2.0, 2.0, 1.0])
    Dp = np.array([2.0, 2.0, 2.0])
    errs = []
    for p in (4, 32, 250):
        X = np.array([2.0 * p, 2.0 * (p // 2), 1.0])
        hi, _ = O.tensor_point(X, D, Dp)
        errs.append(abs(O.nxx_fp64(X, D, Dp) - hi[0]) / abs(hi[0]))
    assert errs[0] < 1e-9
    assert errs[2] > 1e-6          # fp64 has lost most digits at 250 cells
    assert errs[2] > 100 * errs[0]


# ---------------------------------------------------------------- lattice-memo path of tensor_row
def test_tensor_row_equals_tensor_point_on_every_entry():
    """hfft_oracle_tensor_row (lattice memo: its own parity tables PAR_X / PAR_Y, its own ROLE permutations
    and `shift` logic, a second transcription of PAPER.md:46 and :99 / Eq.5, 11, 19 :150) against
    hfft_oracle_tensor_point (pinned above by quadrature, dipole limit, Aharoni, trace, additivity,
    reciprocity): all six components, every target i and source j, every in-plane offset p, q including
    the negative ones; unequal dz, nx != ny, dx != dy.  Mutations tried against this test:
    a sign on PAR_X[4] or PAR_Y[5], a sign on the memoised g, and exchanging the argument permutations of xz and
    yz in phi_eval all FAIL here.  Permuting ROLE[c] cannot fail anything: the nested sums of Eq.5 x 28 x 27 and
    Eq.11 x 31 x 30 are a product of one four-point stencil per physical axis, so which axis plays which of the
    paper's roles does not change the result (an equivalent mutant, like exchanging a and b in `shift`)."""
    nx, ny, nz = 8, 4, 4
    dx, dy = 1.7, 0.9
    dz = np.array([1.0, 2.3, 0.6, 1.45])
    zeta = np.concatenate([[0.0], np.cumsum(dz)])
    worst = 0.0
    scale = 0.0
    for i in range(nz):
        row = O.tensor_row(nx, ny, nz, dx, dy, dz, i)
        assert row.shape == (nz, 6, 2 * ny - 1, 2 * nx - 1)
        for j in range(nz):
            D, Dp = [dx, dy, dz[i]], [dx, dy, dz[j]]
            for q in range(-(ny - 1), ny):
                for p in range(-(nx - 1), nx):
                    # Z_ij = zeta_i - zeta_j (lower faces, reading A8), formed exactly as the sum of whole layers
                    Z = float(sum(dz[j:i])) if i >= j else -float(sum(dz[i:j]))
                    assert abs(Z - (zeta[i] - zeta[j])) < 1e-15
                    hi, lo = O.tensor_point([p * dx, q * dy, Z], D, Dp)
                    got = row[j, :, q + ny - 1, p + nx - 1]
                    worst = max(worst, float(np.abs(got - (hi + lo)).max()))
                    scale = max(scale, float(np.abs(hi).max()))
    # both paths are binary128 rounded once to fp64; they differ by the rounding of p*dx, of zeta (a few ulp
    # of the arguments) and of the final value
    assert scale > 0.1 and worst <= 1e-15 * max(scale, 1.0), worst


def test_tensor_row_off_diagonal_signs_under_offset_reversal():
    """R4 on the row itself: xy odd in X and Y, xz odd in X / even in Y, yz even in X / odd in Y, diagonals
    even -- read straight from the stored negative offsets (the PAR_X / PAR_Y tables), with values that are
    not small (so a wrong sign cannot hide in rounding)."""
    nx, ny, nz = 6, 5, 3
    dz = np.array([0.8, 1.9, 1.1])
    row = O.tensor_row(nx, ny, nz, 1.3, 1.1, dz, 1)
    cx, cy = nx - 1, ny - 1
    sx = [1, 1, 1, -1, -1, 1]
    sy = [1, 1, 1, -1, 1, -1]
    for j in (0, 2):
        for c in range(6):
            a = row[j, c]
            assert np.abs(a).max() > 1e-4
            assert np.abs(a[:, ::-1] - sx[c] * a).max() <= 1e-16, (j, c)
            assert np.abs(a[::-1, :] - sy[c] * a).max() <= 1e-16, (j, c)
            assert np.abs(a[cy + 1, cx + 2]) > 1e-5      # a generic offset is non-zero for every component
