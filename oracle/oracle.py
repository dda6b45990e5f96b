"""CPU ORACLE (test infrastructure, NOT the product) for arXiv 1910.07054.

Plain fp64 / binary128 restatement of what ``hfft_demag`` must compute, written
from the paper (citations are ``PAPER.md:<line>`` + equation).  It shares no
code with ``paper_1910_07054_b200/`` and never imports it.  Allowed callers:
``tests/``, ``__graft_entry__.smoke()``, ``bench.py`` (``cpu_baseline`` and
``--impl reference``).

Tiers
  tensor   binary128 generalized Newell tensor          (oracle/hfft_oracle.c)
  T0       direct real-space sum, Eq.18 PAPER.md:144    (``direct_*``)
  T1       hybrid: 2-D DFT in-plane + explicit z-sum,   (``hybrid_*``)
           Eq.24; the DFT is the naive O(n^2) matrix form
           (``dft="naive"``) or numpy's FFT as a library step (``dft="fft"``,
           pinned against the naive form in tests/test_oracle_field.py).

Layouts (all fp64, C order):
  m, H : [3][nz][ny][nx]  or batched [B][3][nz][ny][nx]   (x fastest)
  Ms   : None (=1), scalar, or [nz] per-layer (reading A12 in DESIGN.md)
  Nrow : [nz(j)][6][2ny-1][2nx-1], component order xx,yy,zz,xy,xz,yz,
         offset (p,q) stored at [q+ny-1][p+nx-1]
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "hfft_oracle.c")
_SO = os.path.join(_HERE, "libhfft_oracle.so")
_lib = None

# (a,b) -> component index of the symmetric tensor (Eq.4)
COMP = ((0, 3, 4), (3, 1, 5), (4, 5, 2))


def build(force: bool = False) -> str:
    """Compile the C part of the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", _SO, _SRC, "-lquadmath", "-lm"]
        subprocess.check_call(cmd)
    return _SO


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_SO)
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int)
        lib.hfft_oracle_f.argtypes = [dp, dp, dp]
        lib.hfft_oracle_g.argtypes = [dp, dp, dp]
        lib.hfft_oracle_tensor_point.argtypes = [dp, dp, dp, dp, dp]
        lib.hfft_oracle_nxx_fp64.argtypes = [dp, dp, dp]
        lib.hfft_oracle_nxx_fp64.restype = ctypes.c_double
        lib.hfft_oracle_tensor_row.argtypes = [ctypes.c_int] * 3 + [ctypes.c_double] * 2 + [dp, ctypes.c_int, dp]
        lib.hfft_oracle_tensor_row.restype = ctypes.c_int
        lib.hfft_oracle_direct_row.argtypes = [ctypes.c_int] * 3 + [dp, dp, ctypes.c_int, ip, dp]
        lib.hfft_oracle_direct_row.restype = ctypes.c_int
        lib.hfft_oracle_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def threads() -> int:
    return int(_load().hfft_oracle_threads())


def _pairs(v):
    """Accept floats or (hi, lo) pairs -> two fp64 arrays of 3."""
    hi = np.zeros(3)
    lo = np.zeros(3)
    for k, x in enumerate(v):
        if isinstance(x, (tuple, list)):
            hi[k], lo[k] = float(x[0]), float(x[1])
        else:
            hi[k] = float(x)
    return hi, lo


def newell_f(x, y, z):
    """Eq.10 in binary128.  Returns (hi, lo) with hi+lo the value."""
    hi, lo = _pairs((x, y, z))
    out = np.zeros(2)
    _load().hfft_oracle_f(_dptr(hi), _dptr(lo), _dptr(out))
    return float(out[0]), float(out[1])


def newell_g(x, y, z):
    """Eq.16 in binary128.  Returns (hi, lo)."""
    hi, lo = _pairs((x, y, z))
    out = np.zeros(2)
    _load().hfft_oracle_g(_dptr(hi), _dptr(lo), _dptr(out))
    return float(out[0]), float(out[1])


def tensor_point(X, D, Dp):
    """N(X,Y,Z) for a target cuboid of size D offset by X from a source cuboid of size Dp.

    Eq.5 / Eq.11 with Eq.27-28 / Eq.30-31, remaining
    components by permutation.  Returns (hi[6], lo[6]), order
    xx,yy,zz,xy,xz,yz.
    """
    X = np.ascontiguousarray(X, dtype=np.float64)
    D = np.ascontiguousarray(D, dtype=np.float64)
    Dp = np.ascontiguousarray(Dp, dtype=np.float64)
    hi = np.zeros(6)
    lo = np.zeros(6)
    _load().hfft_oracle_tensor_point(_dptr(X), _dptr(D), _dptr(Dp), _dptr(hi), _dptr(lo))
    return hi, lo


def nxx_fp64(X, D, Dp) -> float:
    """N_xx from the same 64 terms evaluated in plain fp64 (pin P9 only)."""
    X = np.ascontiguousarray(X, dtype=np.float64)
    D = np.ascontiguousarray(D, dtype=np.float64)
    Dp = np.ascontiguousarray(Dp, dtype=np.float64)
    return float(_load().hfft_oracle_nxx_fp64(_dptr(X), _dptr(D), _dptr(Dp)))


def tensor_row(nx, ny, nz, dx, dy, dz, i):
    """Eq.19: N_ij(p dx, q dy) for target layer i and every source layer j."""
    dz = np.ascontiguousarray(dz, dtype=np.float64)
    assert dz.shape == (nz,)
    out = np.empty((nz, 6, 2 * ny - 1, 2 * nx - 1), dtype=np.float64)
    rc = _load().hfft_oracle_tensor_row(nx, ny, nz, float(dx), float(dy), _dptr(dz), int(i), _dptr(out))
    if rc != 0:
        raise MemoryError("hfft_oracle_tensor_row")
    return out


def _magnetisation(m, Ms, nz):
    """M = Ms_j m_j (Eq.17; per-layer Ms is reading A12)."""
    m = np.asarray(m, dtype=np.float64)
    if Ms is None:
        return m
    Ms = np.asarray(Ms, dtype=np.float64)
    if Ms.ndim == 0:
        return m * Ms
    assert Ms.shape == (nz,)
    shape = [1] * m.ndim
    shape[-3] = nz
    return m * Ms.reshape(shape)


def direct_cells(nx, ny, nz, dx, dy, dz, m, Ms, i, cells, Nrow=None):
    """T0: Eq.18 direct sum for the listed cells (flat a2*nx+a1) of target layer i.

    m: [3][nz][ny][nx].  Returns [ncells][3].
    """
    M = np.ascontiguousarray(_magnetisation(m, Ms, nz))
    assert M.shape == (3, nz, ny, nx)
    if Nrow is None:
        Nrow = tensor_row(nx, ny, nz, dx, dy, dz, i)
    cells = np.ascontiguousarray(cells, dtype=np.int32)
    H = np.empty((cells.size, 3), dtype=np.float64)
    _load().hfft_oracle_direct_row(nx, ny, nz, _dptr(Nrow), _dptr(M), int(cells.size),
                                   cells.ctypes.data_as(ctypes.POINTER(ctypes.c_int)), _dptr(H))
    return H


def direct_field(nx, ny, nz, dx, dy, dz, m, Ms=None):
    """T0 on the whole grid: H [3][nz][ny][nx].  O((nx ny nz)^2)."""
    H = np.empty((3, nz, ny, nx))
    cells = np.arange(nx * ny, dtype=np.int32)
    for i in range(nz):
        Hi = direct_cells(nx, ny, nz, dx, dy, dz, m, Ms, i, cells)
        H[:, i] = Hi.T.reshape(3, ny, nx)
    return H


def _dft_matrix(N):
    """Unnormalised forward DFT matrix W[k,n] = exp(-2 pi i (k n mod N)/N) (reading A11).

    The phase index is reduced exactly in integers before the trigonometric call.
    """
    k = np.arange(N, dtype=np.int64)
    kn = np.outer(k, k) % N
    ang = -2.0 * np.pi * kn.astype(np.float64) / N
    return np.cos(ang) + 1j * np.sin(ang)


def _pad_kernel(Nrow, nx, ny):
    """Place N(p,q), p in [-(nx-1),nx-1], on the 2nx x 2ny periodic grid at
    (p mod 2nx, q mod 2ny); the unused slots p = nx, q = ny stay 0 (reading A10)."""
    nzj = Nrow.shape[0]
    pad = np.zeros((nzj, 6, 2 * ny, 2 * nx), dtype=np.float64)
    p = np.arange(-(nx - 1), nx)
    q = np.arange(-(ny - 1), ny)
    pad[:, :, (q % (2 * ny))[:, None], (p % (2 * nx))[None, :]] = Nrow
    return pad


def tensor_spectrum(Nrow, nx, ny, dft="naive"):
    """Left factor of Eq.24, F1F2(N_kl) of one target layer: the tensor row placed on the
    2nx x 2ny periodic grid (A10) and transformed in the plane.  Nrow: tensor_row(..., i); returns complex
    [nz][6][2ny][2nx].  These are the lines hybrid_layers runs per target layer, under a name of their own so that a
    caller (bench.py's CPU baseline: "tensor bank pre-built, setup excluded, as for the GPU") can run them once,
    outside its timing, and hand the result back through `nhat=`."""
    pad = _pad_kernel(Nrow, nx, ny)
    if dft == "naive":
        Wx, Wy = _dft_matrix(2 * nx), _dft_matrix(2 * ny)
        return np.einsum("kq,jcqp,np->jckn", Wy, pad, Wx, optimize=True)
    if dft == "fft":
        return np.fft.fft2(pad, axes=(-2, -1))
    raise ValueError(dft)


def hybrid_layers(nx, ny, nz, dx, dy, dz, m, Ms, layers, dft="naive", rows=None, nhat=None):
    """T1: Eq.24 for the listed target layers.

      H_{k,i1,i2,i3} = - sum_l F2^-1 F1^-1 sum_{j3} [ F1F2(N_kl)_{i3-j3} F1F2(M_l)_{j3} ]_{i1,i2}

    with the in-plane transforms taken on the zero-padded 2nx x 2ny grid (A10)
    and the z-sum written out.  m: [3][nz][ny][nx] or [B][3][nz][ny][nx].
    Returns [len(layers)][3][ny][nx] (or [B][len(layers)][3][ny][nx]).
    rows: optional {i: tensor_row(..., i)} of precomputed tensor rows (setup hoisted out, e.g. when
    bench.py times the evaluation without the tensor build); the arithmetic is unchanged.
    nhat: optional {i: tensor_spectrum(rows[i], nx, ny, dft)} of precomputed tensor spectra -- the same hoist one step
    further (the GPU path's hfft_build_tensor covers both); the arithmetic is unchanged.
    """
    M = _magnetisation(m, Ms, nz)
    batched = M.ndim == 5
    if not batched:
        M = M[None]
    B = M.shape[0]
    assert M.shape[1:] == (3, nz, ny, nx)
    if dft == "naive":
        Wx, Wy = _dft_matrix(2 * nx), _dft_matrix(2 * ny)
        # zero padding: only the first nx (ny) columns of W meet non-zero data
        Mhat = np.einsum("kq,bljqp,np->bljkn", Wy[:, :ny], M, Wx[:, :nx], optimize=True)
    elif dft == "fft":
        Mhat = np.fft.fft2(M, s=(2 * ny, 2 * nx), axes=(-2, -1))
    else:
        raise ValueError(dft)
    out = np.empty((B, len(layers), 3, ny, nx))
    for t, i in enumerate(layers):
        if nhat is not None and i in nhat:
            Nhat = nhat[i]
        else:
            Nrow = rows[i] if rows is not None and i in rows else tensor_row(nx, ny, nz, dx, dy, dz, i)
            Nhat = tensor_spectrum(Nrow, nx, ny, dft)
            del Nrow
        for k in range(3):
            Hhat = np.zeros((B, 2 * ny, 2 * nx), dtype=np.complex128)
            for l in range(3):
                # explicit convolution along z: sum over source layers j3
                Hhat -= np.einsum("jkn,bjkn->bkn", Nhat[:, COMP[k][l]], Mhat[:, l], optimize=True)
            if dft == "naive":
                h = np.einsum("qk,bkn,pn->bqp", np.conj(Wy)[:ny, :], Hhat, np.conj(Wx)[:nx, :],
                              optimize=True) / (4.0 * nx * ny)
            else:
                h = np.fft.ifft2(Hhat, axes=(-2, -1))[:, :ny, :nx]
            assert np.abs(h.imag).max() <= 1e-9 * max(np.abs(h.real).max(), 1e-300)
            out[:, t, k] = h.real
    return out if batched else out[0]


def hybrid_field(nx, ny, nz, dx, dy, dz, m, Ms=None, dft="naive"):
    """T1 on every layer: H in the layout of m."""
    H = hybrid_layers(nx, ny, nz, dx, dy, dz, m, Ms, list(range(nz)), dft=dft)
    # [.., layer, comp, y, x] -> [.., comp, layer, y, x]
    return np.swapaxes(H, -4, -3).copy()
