"""The fused S2 + S3 + S4 kernel (hfft_plan_set_fusion; fused_ycy.cu) against the CPU oracle and against the staged path.
-m gpu.  Fusion mode 2 forces the kernel wherever its column fits shared memory; mode 0 gives the five-kernel path."""
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


def _field(hb, w, m, **kw):
    import torch
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.precision, batch=m.shape[0], **kw)
    plan.build_tensor()
    dt = torch.float32 if w.precision == "f32" else torch.float64
    h = plan.demag(torch.from_numpy(m).to(dt).cuda(), w.Ms)
    torch.cuda.synchronize()
    H = h.double().cpu().numpy()
    info = hb.plan_info(plan.handle)
    plan.close()
    return H, info


SHAPES = [
    # nx, ny, nz, B: tiny, ragged, rows narrower and wider than a warp, several row passes, nz beyond one round of warps
    (2, 2, 1, 1), (4, 2, 3, 2), (8, 32, 5, 1), (32, 8, 2, 3), (16, 16, 7, 1), (64, 64, 6, 1), (16, 128, 3, 1),
    (32, 256, 2, 1), (16, 16, 20, 1),
]


@pytest.mark.parametrize("nx,ny,nz,B", SHAPES)
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_fused_kernel_vs_oracle_and_staged_path(hb, nx, ny, nz, B, prec):
    w = W.small(nx, ny, nz, precision=prec, B=B, seed=900 + nx + 3 * ny + 7 * nz)
    m = w.m_rounded()
    Hf, info_f = _field(hb, w, m, fusion=2, dedup=0)
    Hs, info_s = _field(hb, w, m, fusion=0, dedup=0)
    assert info_f.fused == 1 and info_f.launches_per_demag == 3
    assert info_s.fused == 0 and info_s.launches_per_demag == 5
    ref = np.stack([O.hybrid_field(nx, ny, nz, w.dx, w.dy, w.dz, m[b], w.Ms, dft="fft") for b in range(B)])
    scale = np.abs(ref).max()
    assert np.abs(Hf - ref).max() / scale <= TOL[prec]
    assert np.abs(Hs - ref).max() / scale <= TOL[prec]
    # same bank, same transforms, same order of the sum over source layers
    assert np.abs(Hf - Hs).max() / scale <= (1e-6 if prec == "f32" else 1e-13)


def test_automatic_mode_fuses_the_small_configs_only(hb):
    # config 2 in fp64: the column's bank slice (221 KB) does not fit shared memory next to the spectra -> staged path
    for cfg, want in ((W.config(1), 1), (W.config(2), 1), (W.config(2, "f64"), 0), (W.config(3), 0)):
        plan = hb.plan_create(cfg.nx, cfg.ny, cfg.nz, cfg.dx, cfg.dy, cfg.dz, hb.F32 if cfg.precision == "f32" else hb.F64)
        info = hb.plan_info(plan)
        assert info.fused == want, cfg.name
        hb.lib().hfft_destroy(plan)


def test_fusion_mode_is_refused_after_build_and_for_bad_values(hb):
    w = W.small(8, 8, 2, precision="f32")
    plan = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, "f32")
    with pytest.raises(hb.HfftError) as e:
        hb.plan_set_fusion(plan.handle, 3)
    assert e.value.status == hb.EINVAL
    with pytest.raises(hb.HfftError) as e:
        hb.plan_set_fusion(plan.handle, 0)          # Plan() has called hfft_plan_set_buffers
    assert e.value.status == hb.ESTATE
    plan.close()


def test_config2_through_the_fused_path_full_grid(hb):
    for variant, kw in (("", {}), ("f64", dict(fusion=2))):
        w = W.config(2, variant)
        m = w.m_rounded()
        H, info = _field(hb, w, m, **kw)
        assert info.fused == 1
        ref = O.hybrid_field(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, m[0], w.Ms, dft="fft")
        assert np.abs(H[0] - ref).max() / np.abs(ref).max() <= TOL[w.precision]
