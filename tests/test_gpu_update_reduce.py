"""SURVEY 8f-1 / 8f-3 on the GPU: hfft_update_dz (partial tensor rebuild), the fused <H> and m.H
reductions of S5, and the paper's thickness-optimisation example driven through the C ABI.  -m gpu.

Every expected value comes from the oracle (or from a fresh full build of the same library for the
"partial rebuild == full rebuild" property, which is bit-exact by construction of the method:
N_ij depends on (dz_i, dz_j, zeta_i - zeta_j) only, Eq.19).
"""
import os

import numpy as np
import pytest

import oracle as O
from paper_1910_07054_b200 import workloads as W

pytestmark = pytest.mark.gpu
GOLD = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
TOL = {"f32": 2e-6, "f64": 1e-12}


@pytest.fixture(scope="module")
def hb():
    import torch
    from paper_1910_07054_b200 import binding
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    binding.lib()
    return binding


def _relerr(a, b):
    return float(np.abs(a - b).max() / np.abs(b).max())


def _bank(hb, plan):
    nz = plan.nz
    return np.stack([[[hb.read_bank(plan.handle, i, j, c) for c in range(6)] for j in range(nz)] for i in range(nz)])


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("k", [0, 2, 4])
def test_update_dz_equals_full_rebuild(hb, prec, k):
    """The pairs update_dz leaves alone are exactly the ones whose tensor does not change, and the
    ones it rebuilds get the same arithmetic as a full build: banks agree bit for bit."""
    w = W.small(16, 32, 5, precision=prec, seed=77)
    dz2 = w.dz.copy()
    dz2[k] = 1.7 * w.dz[k] + 0.123
    a = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec)
    a.build_tensor()
    before = _bank(hb, a)
    a.update_dz(k, dz2[k])
    b = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, dz2, prec)
    b.build_tensor()
    got, want = _bank(hb, a), _bank(hb, b)
    assert np.array_equal(got, want)
    # pairs on one side of layer k are untouched (and really did not need rebuilding)
    for i in range(w.nz):
        for j in range(w.nz):
            if (i < k and j < k) or (i > k and j > k):
                assert np.array_equal(before[i, j], want[i, j])
    assert not np.array_equal(before[k, k], want[k, k])
    # and the field after the update matches the oracle on the new geometry
    import torch
    m = w.m_rounded()
    dt = torch.float32 if prec == "f32" else torch.float64
    H = a.demag(torch.from_numpy(m).to(dt).cuda(), w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, dz2, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL[prec]
    a.close()
    b.close()


@pytest.mark.parametrize("prec,nz,mir", [("f32", 10, 3), ("f64", 6, 2)])
@pytest.mark.parametrize("k", [0, 3, -1])
def test_update_dz_partial_rebuild_under_reciprocity_storage(hb, prec, nz, mir, k):
    """Reciprocity storage (one stored orientation S_pq = dz_p R_pq per unordered pair; the symmetric-matvec layout in
    fp32, the pair table in fp64): hfft_update_dz rewrites only the pairs that have layer k between or at their two
    layers and leaves the other blocks -- and the layout's zero padding -- alone.  The bank, read back pair by pair in
    both orientations, equals that of a fresh build bit for bit, and the field matches the oracle."""
    import torch
    k = k % nz
    w = W.small(16, 8, nz, precision=prec, seed=31)
    kw = dict(dedup=0, mirror=2, recip=1)
    dz2 = w.dz.copy()
    dz2[k] = 0.55 * w.dz[k] + 0.2
    a = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec, **kw)
    assert a.info.mirror == mir
    a.build_tensor()
    a.update_dz(k, dz2[k])
    b = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, dz2, prec, **kw)
    b.build_tensor()
    assert np.array_equal(_bank(hb, a), _bank(hb, b))
    m = w.m_rounded()
    dt = torch.float32 if prec == "f32" else torch.float64
    H = a.demag(torch.from_numpy(m).to(dt).cuda(), w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, dz2, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL[prec]
    a.close()
    b.close()


def test_update_dz_errors(hb):
    w = W.small(8, 8, 3, precision="f64", seed=3)
    p = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, "f64")
    with pytest.raises(hb.HfftError) as e:
        p.update_dz(1, 2.0)
    assert e.value.status == hb.ESTATE
    p.build_tensor()
    for k, dz in [(-1, 1.0), (3, 1.0), (1, 0.0), (1, -2.0), (1, float("nan")), (1, float("inf"))]:
        with pytest.raises(hb.HfftError) as e:
            p.update_dz(k, dz)
        assert e.value.status == hb.EINVAL
    p.close()


@pytest.mark.parametrize("nx,ny,nz,B,prec", [(16, 16, 3, 1, "f64"), (64, 32, 4, 3, "f64"), (32, 64, 5, 2, "f32"),
                                             (256, 256, 2, 1, "f32"), (4, 2, 2, 2, "f64")])
def test_fused_reductions_match_oracle(hb, nx, ny, nz, B, prec):
    """sums[b][c][i] = (sum_cells h_c, sum_cells m_c h_c) against the same sums of the oracle's field;
    the field itself is unchanged by switching the reductions on."""
    import torch
    w = W.small(nx, ny, nz, precision=prec, B=B, seed=11 + nx + ny)
    m = w.m_rounded()
    dt = torch.float32 if prec == "f32" else torch.float64
    md = torch.from_numpy(m).to(dt).cuda()
    plan = hb.Plan(nx, ny, nz, w.dx, w.dy, w.dz, prec, batch=B)
    plan.build_tensor()
    H0 = plan.demag(md, w.Ms).double().cpu().numpy()
    sums = plan.set_reduction(True)
    for _ in range(2):                      # zeroed on every call, not accumulated across calls
        H1 = plan.demag(md, w.Ms).double().cpu().numpy()
    assert np.array_equal(H0, H1)
    got = sums.cpu().numpy()
    ref = O.hybrid_field(nx, ny, nz, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    want = np.stack([ref.sum(axis=(-1, -2)), (ref * m).sum(axis=(-1, -2))], axis=-1)
    scale = np.abs(ref).max() * nx * ny
    assert np.abs(got - want).max() <= TOL[prec] * scale
    # energy in the paper's units: E = -(mu0/2) sum_i V_i Ms_i sum_c sum_cells m_c h_c  (Eq.1-2)
    mu0 = 4e-7 * np.pi
    vol = w.dx * w.dy * w.dz * 1e-27
    E_got = -0.5 * mu0 * (got[..., 1] * (vol * w.Ms)[None, None, :]).sum(axis=(1, 2))
    E_ref = -0.5 * mu0 * (want[..., 1] * (vol * w.Ms)[None, None, :]).sum(axis=(1, 2))
    assert np.all(E_got > 0)                # demagnetization energy is positive definite
    assert np.abs(E_got - E_ref).max() <= 10 * TOL[prec] * np.abs(E_ref).max()
    plan.set_reduction(False)
    H2 = plan.demag(md, w.Ms).double().cpu().numpy()
    assert np.array_equal(H0, H2)
    plan.close()


def test_paper_thickness_optimisation_on_gpu(hb):
    """PAPER.md:205-211 through the C ABI: update_dz + fused <H_z> reduction, Newton iteration on the
    thickness t of the second SAF layer -> 3.44 nm (tests/golden/saf_thickness.txt) in <= 7 steps
    (SURVEY 8f-1 acceptance).  The derivative is a finite difference, as the paper leaves it open."""
    import torch
    with open(os.path.join(GOLD, "saf_thickness.txt")) as fh:
        rows = [ln.split() for ln in fh if ln.strip() and not ln.startswith("#")]
    t_paper, tol = float(rows[0][0]), float(rows[0][1])
    n = 64
    d = 60.0 / n
    c = (np.arange(n) + 0.5) * d - 30.0
    disc = (c[None, :] ** 2 + c[:, None] ** 2) < 30.0 ** 2
    m = np.zeros((1, 3, 5, n, n))
    m[0, 2, 0][disc] = 1.0
    m[0, 2, 2][disc] = -1.0
    md = torch.from_numpy(m).cuda()
    plan = hb.Plan(n, n, 5, d, d, np.array([5.0, 1.0, 5.0, 1.0, 3.0]), "f64")
    plan.build_tensor()
    sums = plan.set_reduction(True)

    def mean_hz(t):
        plan.update_dz(2, t)
        plan.demag(md, None)
        return float(sums[0, 2, 4, 0].item()) / (n * n)

    t, steps = 5.0, 0
    f = mean_hz(t)
    while steps < 7:
        eps = 1e-4
        df = (mean_hz(t + eps) - f) / eps
        t -= f / df
        f = mean_hz(t)
        steps += 1
        if abs(f) < 1e-10:
            break
    assert abs(f) < 1e-10 and steps <= 7
    assert abs(t - t_paper) < tol and round(t, 2) == t_paper
    # the oracle agrees that this t zeroes the average field
    dz = np.array([5.0, 1.0, t, 1.0, 3.0])
    Href = O.hybrid_layers(n, n, 5, d, d, dz, m[0], None, [4], dft="fft")
    assert abs(Href[0, 2].mean()) < 1e-9
    plan.close()


def test_pipelined_host_path_matches_plain_host_path(hb):
    """hfft_demag_host_async / hfft_host_join: several evaluations in flight over two staging slots give,
    in call order, exactly the fields of hfft_demag_host; one of them is checked against the oracle."""
    import torch
    w = W.small(32, 16, 4, precision="f32", B=2, seed=8)
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, "f32", batch=2)
    plan.build_tensor()
    rng = np.random.default_rng(5)
    ms, want, got = [], [], []
    for t in range(5):
        m = rng.normal(size=(2, 3, w.nz, w.ny, w.nx))
        m /= np.sqrt((m ** 2).sum(axis=1, keepdims=True))
        ms.append(torch.from_numpy(m).float().pin_memory())
    for m in ms:
        want.append(plan.demag_host(m, w.Ms))     # a fresh pinned buffer per call
    torch.cuda.synchronize()
    for m in ms:                                     # five calls back to back, nothing synchronised in between
        got.append(plan.demag_host_async(m, w.Ms))
    # until the join, nothing may rewrite the bank or the spectra the pipeline's own streams are still using
    for call in (lambda: plan.update_dz(1, 2.0), lambda: plan.update_dz_static(1, 2.0), plan.build_tensor):
        with pytest.raises(hb.HfftError) as e:
            call()
        assert e.value.status == hb.ESTATE and "hfft_host_join" in str(e.value)
    plan.host_join()
    torch.cuda.synchronize()
    for a, b in zip(got, want):
        assert torch.equal(a, b)
    m3 = ms[3].double().numpy()
    ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m3, w.Ms, dft="fft")
    assert _relerr(got[3].double().numpy(), ref) <= TOL["f32"]
    # join with nothing outstanding, and errors
    plan.host_join()
    with pytest.raises(hb.HfftError) as e:
        hb.demag_host_async(plan.handle, 0, None, 0)
    assert e.value.status == hb.EINVAL
    plan.close()


@pytest.mark.parametrize("kw", [dict(), dict(dedup=0, mirror=2), dict(dedup=3)])
def test_demag_is_capturable_in_a_cuda_graph(hb, kw):
    """hfft.h: hfft_demag only enqueues kernels (no synchronisation, no allocation) -- so a CUDA graph can capture it;
    replays with new data in the captured buffers give the fields of direct calls."""
    import torch
    dz = np.full(16, 0.5) if kw.get("dedup") == 3 else None
    w = W.small(32, 16, 16 if dz is not None else 4, precision="f32", seed=61, dz=dz)
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, "f32", **kw)
    plan.build_tensor()
    m = torch.from_numpy(w.m_rounded()).float().cuda()
    h = torch.empty_like(m)
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):
        plan.demag(m, w.Ms, h)                       # warm-up outside the capture (function attributes, occupancy caches)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        plan.demag(m, w.Ms, h)
    rng = np.random.default_rng(3)
    for _ in range(3):
        mm = rng.normal(size=tuple(m.shape))
        mm /= np.sqrt((mm ** 2).sum(axis=1, keepdims=True))
        m.copy_(torch.from_numpy(mm).float())
        g.replay()
        torch.cuda.synchronize()
        got = h.clone()
        want = plan.demag(m, w.Ms)
        torch.cuda.synchronize()
        assert torch.equal(got, want)
    plan.close()
