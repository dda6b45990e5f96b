"""ky-mirror storage of the bank (hfft_plan_set_mirror) against the oracle through the C ABI.  -m gpu.

The spectra of xx, yy, zz, xz are even in ky, those of xy, yz odd, so ky and 2ny - ky share one bank entry; S2 / S4
keep each pair in adjacent spectrum slots.  mode 2 forces the storage on small grids (ragged tiles, tiny ny)."""
import numpy as np
import pytest

import oracle as O
from paper_1910_07054_b200 import workloads as W

pytestmark = pytest.mark.gpu
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


SHAPES = [(16, 16, 3, 1), (8, 2, 2, 1), (2, 4, 1, 1), (32, 8, 5, 2), (4, 64, 4, 1), (64, 32, 17, 1), (128, 16, 2, 3)]


@pytest.mark.parametrize("nx,ny,nz,B", SHAPES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_mirror_storage_vs_oracle(hb, nx, ny, nz, B, prec):
    import torch
    w = W.small(nx, ny, nz, precision=prec, B=B, seed=900 + nx + 3 * ny + 7 * nz)
    m = w.m_rounded()
    plan = hb.Plan(nx, ny, nz, w.dx, w.dy, w.dz, prec, batch=B, dedup=0, mirror=2)
    plan.build_tensor()
    info = hb.plan_info(plan.handle)
    batched_kernel = B > 1 and 6 * nz * (4 if prec == "f32" else 8) <= 384      # register-bank kernel keeps its layout
    assert info.mirror == (0 if batched_kernel else 1)
    if info.mirror:
        s = 4 if prec == "f32" else 8
        assert info.n_k_padded >= (nx + 1) * (2 * ny + 2)
        assert info.bank_bytes == 6 * nz * nz * (info.n_k_padded // 2) * s
    dt = torch.float32 if prec == "f32" else torch.float64
    md = torch.from_numpy(m).to(dt).cuda()
    for _ in range(2):                                   # second call: the dummy slots still hold zeros
        H = plan.demag(md, w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(nx, ny, nz, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL[prec]
    if nx * ny * nz <= 2048:
        ref0 = O.direct_field(nx, ny, nz, w.dx, w.dy, w.dz, m[0], w.Ms)          # the definition, Eq.18
        assert _relerr(H[0], ref0) <= TOL[prec]
    plan.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_mirror_bank_reads_back_like_the_plain_bank(hb, prec):
    """hfft_read_bank reconstructs every wavevector from the half bank (signs of xy, yz for ky > ny included)."""
    w = W.small(16, 8, 3, precision=prec, seed=12)
    a = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec, dedup=0, mirror=0)
    b = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec, dedup=0, mirror=2)
    a.build_tensor()
    b.build_tensor()
    assert hb.plan_info(a.handle).mirror == 0 and hb.plan_info(b.handle).mirror == 1
    worst = 0.0
    for i in range(3):
        for j in range(3):
            for c in range(6):
                x, y = hb.read_bank(a.handle, i, j, c), hb.read_bank(b.handle, i, j, c)
                worst = max(worst, np.abs(x - y).max() / max(np.abs(x).max(), 1e-30))
    assert worst <= (1e-6 if prec == "f32" else 1e-12)    # mirrored entries agree to the rounding of the fp64 FFT
    a.close()
    b.close()


def test_mirror_with_update_dz_and_reductions(hb):
    import torch
    w = W.small(32, 16, 4, precision="f64", seed=33)
    dz2 = w.dz.copy()
    dz2[1] = 2.25
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, "f64", dedup=0, mirror=2)
    plan.build_tensor()
    plan.update_dz(1, 2.25)
    sums = plan.set_reduction(True)
    m = w.m_rounded()
    H = plan.demag(torch.from_numpy(m).cuda(), w.Ms).cpu().numpy()
    ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, dz2, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL["f64"]
    assert np.abs(sums.cpu().numpy()[..., 0] - ref.sum(axis=(-1, -2))).max() <= 1e-10 * np.abs(ref).max() * w.nx * w.ny
    plan.close()


def test_mirror_errors_and_automatic_mode(hb):
    p = hb.Plan(16, 16, 3, 1.0, 1.0, np.array([1.0, 2.0, 0.5]), "f32")
    assert hb.plan_info(p.handle).mirror == 0            # small grid: narrow tiles, plain storage
    with pytest.raises(hb.HfftError) as e:
        hb.plan_set_mirror(p.handle, 3)
    assert e.value.status == hb.EINVAL
    with pytest.raises(hb.HfftError) as e:
        hb.plan_set_mirror(p.handle, 0)
    assert e.value.status == hb.ESTATE
    p.close()
    q = hb.Plan(256, 256, 4, 2.0, 2.0, np.array([1.0, 2.0, 0.5, 0.7]), "f32", torch_buffers=False)
    assert hb.plan_info(q.handle).mirror == 1            # large grid: automatic
    q.close()


def test_mirror_many_layers_one_cta_per_sm(hb):
    """fp32, nz = 80: the M^ tile (120 KB) leaves room for one CTA per SM, which then runs 32 warps."""
    import torch
    nz = 80
    w = W.small(8, 8, nz, precision="f32", seed=80)
    m = w.m_rounded()
    plan = hb.Plan(w.nx, w.ny, nz, w.dx, w.dy, w.dz, "f32", dedup=0, mirror=2)
    plan.build_tensor()
    assert hb.plan_info(plan.handle).mirror == 1
    H = plan.demag(torch.from_numpy(m).float().cuda(), w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(w.nx, w.ny, nz, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL["f32"]
    plan.close()


# ---- reciprocity storage on top (hfft_plan_set_recip): S_pq = dz_p R_pq kept for p <= q only ----
@pytest.mark.parametrize("nx,ny,nz,B", [(16, 16, 3, 1), (8, 2, 2, 1), (32, 8, 5, 2), (4, 64, 4, 1), (64, 32, 17, 1),
                                        (16, 8, 33, 1), (8, 8, 80, 1)])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_reciprocity_storage_vs_oracle(hb, nx, ny, nz, B, prec):
    import torch
    w = W.small(nx, ny, nz, precision=prec, B=B, seed=1900 + nx + 3 * ny + 7 * nz)
    m = w.m_rounded()
    plan = hb.Plan(nx, ny, nz, w.dx, w.dy, w.dz, prec, batch=B, dedup=0, mirror=2, recip=1)
    plan.build_tensor()
    info = hb.plan_info(plan.handle)
    batched_kernel = B > 1 and 6 * nz * (4 if prec == "f32" else 8) <= 384
    too_many_layers = 3 * nz * 64 * (8 if prec == "f32" else 16) > 200 * 1024      # the M^ tile must fit shared memory
    symv = prec == "f32" and nz <= 64                       # fp32, at most 16 strips of 4 layers: the symv layout
    assert info.mirror == (0 if batched_kernel or too_many_layers else (3 if symv else 2))
    if info.mirror == 2:
        assert info.bank_bytes == 6 * (nz * (nz + 1) // 2) * (info.n_k_padded // 2) * (4 if prec == "f32" else 8)
    if info.mirror == 3:
        assert info.bank_bytes == (info.n_k_padded // info.tile_k) * 8 * _symv_couples(nz) * 768
    dt = torch.float32 if prec == "f32" else torch.float64
    H = plan.demag(torch.from_numpy(m).to(dt).cuda(), w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(nx, ny, nz, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL[prec]
    if nx * ny * nz <= 2048:
        ref0 = O.direct_field(nx, ny, nz, w.dx, w.dy, w.dz, m[0], w.Ms)
        assert _relerr(H[0], ref0) <= TOL[prec]
    plan.close()


def _symv_couples(nz):
    """Couples (two stored layer pairs for each of 16 strip-lanes, 768 bytes) in a warp-unit's stream: symv_layout.h."""
    W = (nz + 3) // 4
    return 8 * ((W - 1) // 2) + 4 * (1 if W >= 2 and W % 2 == 0 else 0) + 5


@pytest.mark.parametrize("nx,ny,nz,B", [(8, 8, 2, 1), (16, 4, 4, 1), (8, 16, 5, 1), (16, 16, 8, 1), (8, 8, 9, 1),
                                        (4, 16, 12, 1), (16, 8, 16, 1), (8, 4, 17, 1), (8, 8, 24, 1), (4, 8, 27, 2),
                                        (8, 8, 32, 1), (4, 4, 33, 1), (8, 4, 48, 1), (4, 8, 61, 1), (8, 8, 64, 1),
                                        (64, 32, 20, 1), (32, 16, 40, 3)])
def test_symv_reciprocity_kernel_vs_oracle(hb, nx, ny, nz, B):
    """coupling_symv_kernel (fp32 reciprocity bank, every block used for both of its layer pairs): every strip count
    W = 1..16, odd and even (with and without the half block), layer counts that are not multiples of 4 (padding
    rows), idle strip-lanes (W not a power of two), several entries per warp, ragged last tile, batches."""
    import torch
    w = W.small(nx, ny, nz, precision="f32", B=B, seed=2900 + nx + 3 * ny + 7 * nz)
    m = w.m_rounded()
    plan = hb.Plan(nx, ny, nz, w.dx, w.dy, w.dz, "f32", batch=B, dedup=0, mirror=2, recip=1)
    plan.build_tensor()
    info = hb.plan_info(plan.handle)
    assert info.mirror == 3
    md = torch.from_numpy(m).float().cuda()
    for _ in range(2):                                   # second call: padding and dummy slots still hold zeros
        H = plan.demag(md, w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(nx, ny, nz, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL["f32"]
    if nx * ny * nz <= 2048:
        ref0 = O.direct_field(nx, ny, nz, w.dx, w.dy, w.dz, m[0], w.Ms)          # the definition, Eq.18
        assert _relerr(H[0], ref0) <= TOL["f32"]
    plan.close()


def test_symv_bank_reads_back_like_the_plain_bank(hb):
    """hfft_read_bank through the symv layout: every ordered pair (stored orientation or its transpose) of a stack
    with a half block (W = 2) and one with full blocks and idle strip-lanes (W = 5)."""
    for nz in (7, 18):
        w = W.small(16, 8, nz, precision="f32", seed=14 + nz)
        a = hb.Plan(w.nx, w.ny, nz, w.dx, w.dy, w.dz, "f32", dedup=0, mirror=0)
        b = hb.Plan(w.nx, w.ny, nz, w.dx, w.dy, w.dz, "f32", dedup=0, mirror=2, recip=1)
        a.build_tensor()
        b.build_tensor()
        assert hb.plan_info(b.handle).mirror == 3
        worst = 0.0
        for i in range(nz):
            for j in range(nz):
                for c in range(6):
                    x, y = hb.read_bank(a.handle, i, j, c), hb.read_bank(b.handle, i, j, c)
                    worst = max(worst, np.abs(x - y).max() / max(np.abs(x).max(), 1e-30))
        assert worst <= 2e-6, (nz, worst)
        a.close()
        b.close()


def test_symv_with_update_dz_and_reductions(hb):
    import torch
    w = W.small(32, 16, 9, precision="f32", seed=36)
    dz2 = w.dz.copy()
    dz2[4] = 0.9
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, "f32", dedup=0, mirror=2, recip=1)
    plan.build_tensor()
    assert hb.plan_info(plan.handle).mirror == 3
    plan.update_dz(4, 0.9)
    sums = plan.set_reduction(True)
    m = w.m_rounded()
    H = plan.demag(torch.from_numpy(m).float().cuda(), w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, dz2, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL["f32"]
    assert np.abs(sums.cpu().numpy()[..., 0] - ref.sum(axis=(-1, -2))).max() <= 2e-6 * np.abs(ref).max() * w.nx * w.ny
    plan.close()


def test_symv_automatic_mode(hb):
    """Default plans: the symv bank is chosen where the mirror storage is and it streams at least 30 % fewer bytes."""
    for nz, want in ((16, 3), (64, 3), (8, 3), (3, 1), (4, 1), (20, 1)):
        q = hb.Plan(256, 256, nz, 2.0, 2.0, np.exp(np.linspace(-0.5, 0.7, nz)), "f32", torch_buffers=False)
        assert hb.plan_info(q.handle).mirror == want, (nz, hb.plan_info(q.handle).mirror)
        q.close()
    q = hb.Plan(256, 256, 16, 2.0, 2.0, np.exp(np.linspace(-0.5, 0.7, 16)), "f64", torch_buffers=False)
    assert hb.plan_info(q.handle).mirror == 1            # fp64: mirror storage only
    q.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_reciprocity_bank_reads_back_like_the_plain_bank(hb, prec):
    """Every ordered pair, read through the half bank (transpose sign and 1/dz_i included), equals the plain entry:
    this is reciprocity R3, dz_i N_ij(X, Y) = dz_j N_ji(-X, -Y), checked on the device-built tensors."""
    w = W.small(16, 8, 4, precision=prec, seed=14)
    a = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec, dedup=0, mirror=0)
    b = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec, dedup=0, mirror=2, recip=1)
    a.build_tensor()
    b.build_tensor()
    assert hb.plan_info(b.handle).mirror == (3 if prec == "f32" else 2)
    worst = 0.0
    for i in range(4):
        for j in range(4):
            for c in range(6):
                x, y = hb.read_bank(a.handle, i, j, c), hb.read_bank(b.handle, i, j, c)
                worst = max(worst, np.abs(x - y).max() / max(np.abs(x).max(), 1e-30))
    assert worst <= (2e-6 if prec == "f32" else 1e-12)
    a.close()
    b.close()


def test_reciprocity_with_update_dz(hb):
    import torch
    w = W.small(32, 16, 4, precision="f64", seed=35)
    dz2 = w.dz.copy()
    dz2[2] = 0.9
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, "f64", dedup=0, mirror=2, recip=1)
    plan.build_tensor()
    plan.update_dz(2, 0.9)
    m = w.m_rounded()
    H = plan.demag(torch.from_numpy(m).cuda(), w.Ms).cpu().numpy()
    ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, dz2, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL["f64"]
    plan.close()


@pytest.mark.parametrize("prec,nx,ny", [("f64", 128, 128), ("f32", 256, 128), ("f32", 128, 256)])
def test_mirror_automatic_mode_on_mid_size_grids(hb, prec, nx, ny):
    """Grids large enough for the automatic choice (no forcing): the mirror storage is what a default plan uses."""
    import torch
    w = W.small(nx, ny, 3, precision=prec, seed=5 + nx)
    m = w.m_rounded()
    plan = hb.Plan(nx, ny, 3, w.dx, w.dy, w.dz, prec)
    plan.build_tensor()
    assert hb.plan_info(plan.handle).mirror == 1 and hb.plan_info(plan.handle).tile_k == 64
    dt = torch.float32 if prec == "f32" else torch.float64
    H = plan.demag(torch.from_numpy(m).to(dt).cuda(), w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(nx, ny, 3, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL[prec]
    plan.close()


def test_storage_variants_agree_on_random_shapes(hb):
    """Plain, mirror, mirror + reciprocity and class-indexed banks are storages of the same tensor: on 40 seeded random
    shapes (ragged tiles, tiny and odd layer counts, batches) their fields agree to rounding order."""
    import torch
    rng = np.random.default_rng(20240607)
    torch.manual_seed(20240607)
    done = 0
    while done < 40:
        nx, ny = int(rng.choice([2, 4, 8, 16, 32, 64, 128])), int(rng.choice([2, 4, 8, 16, 32, 64]))
        nz, B = int(rng.integers(1, 41)), int(rng.choice([1, 1, 2, 3]))
        prec = str(rng.choice(["f32", "f64"]))
        if nx * ny * nz * B > 4e5:
            continue
        done += 1
        dz = np.exp(rng.uniform(np.log(0.3), np.log(3.0), size=nz))
        Ms = 8e5 * (0.5 + rng.uniform(size=nz))
        dt = torch.float32 if prec == "f32" else torch.float64
        m = torch.randn(B, 3, nz, ny, nx, device="cuda", dtype=dt)
        m /= m.norm(dim=1, keepdim=True)
        fields = {}
        for name, kw in [("plain", dict(dedup=0, mirror=0)), ("mirror", dict(dedup=0, mirror=2, recip=0)),
                         ("recip", dict(dedup=0, mirror=2, recip=1)), ("classes", dict(dedup=2, mirror=0))]:
            plan = hb.Plan(nx, ny, nz, 2.0, 1.5, dz, prec, batch=B, **kw)
            plan.build_tensor()
            fields[name] = plan.demag(m, Ms).double().cpu().numpy()
            plan.close()
        ref = fields["plain"]
        assert np.isfinite(ref).all()
        for name, H in fields.items():
            assert _relerr(H, ref) <= (1e-6 if prec == "f32" else 1e-13), (name, nx, ny, nz, B, prec)
