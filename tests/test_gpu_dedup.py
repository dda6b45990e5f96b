"""SURVEY 8f-2 on the GPU: deduplicated tensor bank (hfft_plan_set_dedup) -- tensor classes, the
shared-memory class kernel (generic and Toeplitz window) and the class-indexed streaming kernel,
all against the CPU oracle through the C ABI.  -m gpu.
"""
from fractions import Fraction

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


def _field(hb, w, m, dedup, batch=1):
    import torch
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.precision, batch=batch, dedup=dedup)
    plan.build_tensor()
    dt = torch.float32 if w.precision == "f32" else torch.float64
    H = plan.demag(torch.from_numpy(m).to(dt).cuda(), w.Ms).double().cpu().numpy()
    return plan, H


def _expected_classes(dz):
    """Distinct (dz_i, dz_j, zeta_i - zeta_j) in exact rational arithmetic (Eq.19)."""
    fz = [Fraction(float(v)) for v in dz]
    zeta = [sum(fz[:k], Fraction(0)) for k in range(len(dz))]
    return len({(fz[i], fz[j], zeta[i] - zeta[j]) for i in range(len(dz)) for j in range(len(dz))})


# dz exactly representable so that "equal Z" is an exact statement
STACKS = {
    "equal5": [1.0] * 5,
    "equal8": [0.75] * 8,
    "equal12": [1.5] * 12,
    "equal33": [0.5] * 33,                       # Toeplitz window, ragged last warp (33 = 4*8 + 1)
    "equal70": [0.25] * 70,                      # one CTA per SM (more than 64 layers); fp64: 18 warps
    "period2x4": [1.0, 0.5] * 4,                 # [A/B]x4 multilayer: generic classes
    "period3x6": [1.0, 0.25, 2.0] * 6,           # 18 layers: generic classes, 4 targets per warp
    "saf": [5.0, 1.0, 5.0, 1.0, 3.0],            # one coincidence only: automatic mode leaves it off
}


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("stack", list(STACKS))
def test_dedup_field_matches_oracle(hb, stack, prec):
    dz = np.array(STACKS[stack])
    nz = len(dz)
    w = W.small(16, 8, nz, precision=prec, seed=31 + nz, dz=dz)
    m = w.m_rounded()
    plan, H = _field(hb, w, m, dedup=2)
    info = hb.plan_info(plan.handle)
    if stack.startswith("equal"):
        # 2nz-1 distinct tensors, folded to |i-j| (N_ji = N_ij up to the sign of xz, yz)
        assert _expected_classes(dz) == 2 * nz - 1 and info.n_classes == nz
        assert info.dedup == (3 if nz <= 64 or prec == "f32" else 1)
    else:
        assert info.n_classes == _expected_classes(dz) and info.dedup == 2
    assert info.bank_bytes == 6 * info.n_classes * info.n_k_padded * (4 if prec == "f32" else 8)
    ref = O.hybrid_field(w.nx, w.ny, nz, w.dx, w.dy, dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL[prec]
    # automatic mode: on iff at most half of the pairs carry their own tensor
    auto = hb.Plan(w.nx, w.ny, nz, w.dx, w.dy, dz, prec)
    assert (hb.plan_info(auto.handle).dedup != 0) == (2 * info.n_classes <= nz * nz)
    if stack.startswith("equal"):
        # the folded bank reproduces the plain bank pair by pair (signs of xz, yz for i < j included)
        plain = hb.Plan(w.nx, w.ny, nz, w.dx, w.dy, dz, prec, dedup=0)
        plain.build_tensor()
        for (i, j) in [(0, nz - 1), (nz - 1, 0), (1, 3), (3, 1), (2, 2)]:
            for c in range(6):
                x, y = hb.read_bank(plain.handle, i, j, c), hb.read_bank(plan.handle, i, j, c)
                assert np.abs(x - y).max() <= 1e-13 * max(np.abs(x).max(), 1e-30)
        plain.close()
    auto.close()
    plan.close()


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_dedup_bank_equals_plain_bank(hb, prec):
    """Every pair reads, through its class, the tensor it would have had in the plain bank."""
    dz = np.array([1.0, 0.5, 1.0, 0.5, 1.0, 2.0])
    w = W.small(8, 16, 6, precision=prec, seed=9, dz=dz)
    a = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, dz, prec, dedup=0)
    b = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, dz, prec, dedup=2)
    a.build_tensor()
    b.build_tensor()
    assert hb.plan_info(b.handle).n_classes == _expected_classes(dz) < 36
    for i in range(6):
        for j in range(6):
            for c in range(6):
                x, y = hb.read_bank(a.handle, i, j, c), hb.read_bank(b.handle, i, j, c)
                assert np.abs(x - y).max() <= 1e-13 * max(np.abs(x).max(), 1e-30)
    a.close()
    b.close()


def test_dedup_on_a_stack_without_duplicates(hb):
    """mode 2 with nz^2 classes: same field as the plain bank (generic class kernel, no savings)."""
    w = W.small(32, 16, 9, precision="f32", seed=4)
    m = w.m_rounded()
    p0, H0 = _field(hb, w, m, dedup=0)
    p2, H2 = _field(hb, w, m, dedup=2)
    assert hb.plan_info(p2.handle).n_classes == 81 and hb.plan_info(p2.handle).dedup == 2
    ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m, w.Ms, dft="fft")
    assert _relerr(H0, ref) <= TOL["f32"] and _relerr(H2, ref) <= TOL["f32"]
    assert _relerr(H2, H0) <= 1e-6
    p0.close()
    p2.close()


@pytest.mark.parametrize("prec,nz", [("f64", 80), ("f32", 100)])
def test_dedup_streaming_kernel_when_the_tile_does_not_fit(hb, prec, nz):
    """Equal thicknesses with too many layers for the shared-memory kernel: class-indexed streaming kernel."""
    dz = np.full(nz, 0.5)
    w = W.small(8, 8, nz, precision=prec, seed=nz, dz=dz)
    m = w.m_rounded()
    plan, H = _field(hb, w, m, dedup=2)
    info = hb.plan_info(plan.handle)
    assert info.dedup == 1 and info.n_classes == nz
    ref = O.hybrid_field(w.nx, w.ny, nz, w.dx, w.dy, dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL[prec]
    plan.close()


@pytest.mark.parametrize("stack", ["equal12", "period2x4"])
def test_dedup_batched(hb, stack):
    dz = np.array(STACKS[stack])
    w = W.small(16, 16, len(dz), precision="f32", B=3, seed=21, dz=dz)
    m = w.m_rounded()
    plan, H = _field(hb, w, m, dedup=1, batch=3)
    assert hb.plan_info(plan.handle).dedup >= 2
    ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL["f32"]
    plan.close()


def test_dedup_errors(hb):
    dz = np.ones(6)
    p = hb.Plan(8, 8, 6, 1.0, 1.0, dz, "f64")
    with pytest.raises(hb.HfftError) as e:
        hb.plan_set_dedup(p.handle, 4)
    assert e.value.status == hb.EINVAL
    with pytest.raises(hb.HfftError) as e:          # buffers already handed over: sizes are fixed
        hb.plan_set_dedup(p.handle, 0)
    assert e.value.status == hb.ESTATE
    p.build_tensor()
    assert hb.plan_info(p.handle).dedup == 3
    with pytest.raises(hb.HfftError) as e:
        p.update_dz(2, 1.5)
    assert e.value.status == hb.EUNSUPPORTED
    p.close()
    q = hb.Plan(8, 8, 6, 1.0, 1.0, dz, "f64", dedup=0)
    q.build_tensor()
    q.update_dz(2, 1.5)                              # allowed on the plain bank
    q.close()


# ---- z-FFT mode (mode 3): the equidistant 3-D FFT method of PAPER.md:182 Eq.25 as stage S3 ----
ZFFT_NZ = [2, 3, 4, 5, 8, 12, 16, 17, 32, 33, 64, 70, 128]


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("nz", ZFFT_NZ)
def test_zfft_field_matches_oracle(hb, nz, prec):
    if prec == "f64" and nz > 32:
        pytest.skip("fp64 z-FFT kernel: Lz <= 64")
    dz = np.full(nz, 0.75)
    nx, ny = (16, 8) if nz <= 33 else (8, 8)
    w = W.small(nx, ny, nz, precision=prec, seed=400 + nz, dz=dz)
    m = w.m_rounded()
    plan, H = _field(hb, w, m, dedup=3)
    info = hb.plan_info(plan.handle)
    lz = 1
    while lz < 2 * nz:
        lz *= 2
    assert info.dedup == 4
    # S(k, Lz - kz) = +- S(k, kz): only kz = 0 .. Lz / 2 is stored (coupling_zfft.cu)
    assert info.bank_bytes == 6 * (lz // 2 + 1) * info.n_k_padded * (4 if prec == "f32" else 8)
    ref = O.hybrid_field(nx, ny, nz, w.dx, w.dy, dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL[prec]
    if nx * ny * nz <= 2048:
        ref0 = O.direct_field(nx, ny, nz, w.dx, w.dy, dz, m[0], w.Ms)     # the definition, Eq.18
        assert _relerr(H[0], ref0) <= TOL[prec]
    # automatic mode picks the z-FFT from 16 equal layers on
    auto = hb.Plan(nx, ny, nz, w.dx, w.dy, dz, prec)
    assert (hb.plan_info(auto.handle).dedup == 4) == (nz >= 16)
    auto.close()
    plan.close()


def test_zfft_batched_and_reductions(hb):
    import torch
    nz, B = 16, 3
    dz = np.full(nz, 1.25)
    w = W.small(32, 16, nz, precision="f32", B=B, seed=77, dz=dz)
    m = w.m_rounded()
    plan = hb.Plan(w.nx, w.ny, nz, w.dx, w.dy, dz, "f32", batch=B, dedup=3)
    plan.build_tensor()
    sums = plan.set_reduction(True)
    H = plan.demag(torch.from_numpy(m).float().cuda(), w.Ms).double().cpu().numpy()
    ref = O.hybrid_field(w.nx, w.ny, nz, w.dx, w.dy, dz, m, w.Ms, dft="fft")
    assert _relerr(H, ref) <= TOL["f32"]
    got = sums.cpu().numpy()[..., 0]
    assert np.abs(got - ref.sum(axis=(-1, -2))).max() <= TOL["f32"] * np.abs(ref).max() * w.nx * w.ny
    plan.close()


def test_zfft_errors(hb):
    p = hb.Plan(8, 8, 4, 1.0, 1.0, np.array([1.0, 2.0, 1.0, 1.0]), "f32", torch_buffers=False)
    with pytest.raises(hb.HfftError) as e:          # unequal thicknesses
        hb.plan_set_dedup(p.handle, 3)
    assert e.value.status == hb.EUNSUPPORTED
    p.close()
    q = hb.Plan(8, 8, 40, 1.0, 1.0, np.ones(40), "f64", torch_buffers=False)
    with pytest.raises(hb.HfftError) as e:          # fp64: Lz <= 64
        hb.plan_set_dedup(q.handle, 3)
    assert e.value.status == hb.EUNSUPPORTED
    q.close()
    r = hb.Plan(8, 8, 4, 1.0, 1.0, np.ones(4), "f64", dedup=3)
    r.build_tensor()
    with pytest.raises(hb.HfftError) as e:
        hb.read_bank(r.handle, 0, 0, 0)
    assert e.value.status == hb.EUNSUPPORTED
    with pytest.raises(hb.HfftError) as e:
        r.update_dz(1, 2.0)
    assert e.value.status == hb.EUNSUPPORTED
    r.close()


@pytest.mark.parametrize("case", ["plain", "batched", "classes", "toeplitz", "zfft", "plain_f64"])
def test_repeated_calls_are_bitwise_identical(hb, case):
    """No kernel of the path uses atomics or an order that depends on scheduling (the fused reductions, off here, are
    the one exception), so repeated evaluations must agree bit for bit; a shared-memory race in the exchange or
    staging buffers would show up here (compute-sanitizer is not available on the GPU pool)."""
    import torch
    cfg = {
        "plain": dict(nx=64, ny=128, dz=None, nz=7, B=1, prec="f32", dedup=0),
        "batched": dict(nx=128, ny=64, dz=None, nz=5, B=4, prec="f32", dedup=0),
        "classes": dict(nx=64, ny=64, dz=[1.0, 0.5] * 8, nz=16, B=1, prec="f32", dedup=2),
        "toeplitz": dict(nx=64, ny=64, dz=[0.5] * 40, nz=40, B=2, prec="f32", dedup=2),
        "zfft": dict(nx=64, ny=64, dz=[0.5] * 40, nz=40, B=2, prec="f32", dedup=3),
        "plain_f64": dict(nx=32, ny=64, dz=None, nz=6, B=1, prec="f64", dedup=0),
    }[case]
    w = W.small(cfg["nx"], cfg["ny"], cfg["nz"], precision=cfg["prec"], B=cfg["B"], seed=17,
                dz=None if cfg["dz"] is None else np.array(cfg["dz"]))
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, cfg["prec"], batch=cfg["B"], dedup=cfg["dedup"])
    plan.build_tensor()
    dt = torch.float32 if cfg["prec"] == "f32" else torch.float64
    m = torch.from_numpy(w.m_rounded()).to(dt).cuda()
    first = plan.demag(m, w.Ms).clone()
    assert bool(torch.isfinite(first).all())
    for _ in range(25):
        assert torch.equal(plan.demag(m, w.Ms), first)
    plan.close()


def test_automatic_mode_takes_a_class_path_only_where_it_was_measured_faster(hb):
    """hfft_api.cu plan_sizes (numbers in profiles/r02_scaling_nz.md): on a large grid a repeating, non-equidistant stack
    keeps the reciprocity / ky-mirror bank from 16 layers on (the generic class kernel and the class-indexed streaming
    fallback lose to it); equal thicknesses always take the Toeplitz window kernel or the z-FFT; small grids, where the
    mirror storage does not apply, deduplicate as before."""
    def info(nx, ny, dz):
        plan = hb.plan_create(nx, ny, len(dz), 2.0, 2.0, np.asarray(dz, float), hb.F32)
        i = hb.plan_info(plan)
        hb.lib().hfft_destroy(plan)
        return i
    alt = lambda nz: [1.0, 2.5] * (nz // 2)
    for nz in (16, 32, 64):
        i = info(256, 256, alt(nz))
        assert (i.dedup, i.mirror) == (0, 3), nz          # symv layout of the reciprocity bank
    i = info(256, 256, alt(96))
    assert (i.dedup, i.mirror) == (0, 1)                  # ky-mirror bank (symv: nz <= 64)
    i = info(256, 256, alt(8))
    assert i.dedup == 2                                   # generic class kernel, few layers
    i = info(256, 256, alt(160))
    assert i.dedup == 1 and i.mirror == 0                 # mirror storage does not fit: class-indexed stream
    assert info(256, 256, [1.0] * 8).dedup == 3           # Toeplitz window
    assert info(256, 256, [1.0] * 64).dedup == 4          # z-FFT
    assert info(256, 256, [1.0] * 128).dedup == 4
    assert info(32, 32, alt(16)).dedup in (1, 2)          # small grid: deduplicated as before
