"""hfft_update_dz_static: the thickness update for callers that cannot allocate device memory.  -m gpu.

Some users of this library cannot call cudaMalloc while they run: programs that gave the whole GPU to a memory pool of
their own at start-up (cudaMalloc then reports "out of memory"), optimisation and real-time loops that cannot take the
device-wide synchronisation and the driver lock that cudaMalloc / cudaFree bring, and host threads that work while
another thread records a CUDA graph in the global capture mode.  hfft_update_dz allocates and frees its scratch on
every call; hfft_update_dz_static (include/hfft.h) does the same rebuild with the scratch in a fixed 32 MiB array of the
library's device image.  The array is shared by all plans and keeps the previous call's contents, so this file checks
what such a caller relies on:

  - the bank after the static call equals, bit for bit, the bank after hfft_update_dz (the comparison the existing
    update tests use, tests/test_gpu_update_reduce.py), and the field computed from it is the same array -- on TWO
    calls in a row, with a call on a plan of another shape in between, so that the second call starts from an array
    full of foreign intermediates;
  - a plan that needs more than the 32 MiB is refused with HFFT_EUNSUPPORTED and is left untouched.

The file is named so that pytest collects it last: `pytest -x` stops at the first failure, and a failure here must not
hide the parity tests.  It makes no assumption about what ran before it in the process (the first static call on the
device does the one-time address look-up whether or not other tests ran).
"""
import numpy as np
import pytest

from paper_1910_07054_b200 import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hb():
    import torch
    from paper_1910_07054_b200 import binding
    assert torch.cuda.is_available(), "gpu tests need a CUDA device"
    binding.lib()
    return binding


def _bank(hb, plan):
    nz = plan.nz
    return np.stack([[[hb.read_bank(plan.handle, i, j, c) for c in range(6)] for j in range(nz)] for i in range(nz)])


def _field(plan, w, prec):
    import torch
    dt = torch.float32 if prec == "f32" else torch.float64
    return plan.demag(torch.from_numpy(w.m_rounded()).to(dt).cuda(), w.Ms).double().cpu().numpy()


# plain bank in both precisions, and the reciprocity bank of the symmetric-matvec kernel (fp32): there the update
# rebuilds the whole bank and refreshes the 1/dz table, the other branch of the entry point
CASES = [("f64", 16, 32, 5, {}), ("f32", 16, 32, 5, {}), ("f32", 16, 8, 10, dict(dedup=0, mirror=2, recip=1))]


@pytest.mark.parametrize("prec,nx,ny,nz,kw", CASES)
def test_static_update_equals_allocating_update_twice_in_a_row(hb, prec, nx, ny, nz, kw):
    w = W.small(nx, ny, nz, precision=prec, seed=77)
    ref = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec, **kw)    # the existing path: hfft_update_dz
    sta = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, prec, **kw)    # the new one
    ref.build_tensor()
    sta.build_tensor()
    assert sta.info.setup_scratch_bytes <= hb.STATIC_SCRATCH_BYTES
    # a plan of another shape that uses the shared array between the two calls
    wo = W.small(32, 16, 3, precision="f64", seed=5)
    other = hb.Plan(wo.nx, wo.ny, wo.nz, wo.dx, wo.dy, wo.dz, "f64")
    other.build_tensor()
    start = _bank(hb, sta)
    assert np.array_equal(start, _bank(hb, ref))
    # call 1 grows layer 2; call 2 shrinks layer 0 (fewer pairs change than in call 1: stale data stay in the array)
    for call, (k, dz_new) in enumerate([(2, 1.7 * w.dz[2] + 0.123), (0, 0.61 * w.dz[0])]):
        ref.update_dz(k, dz_new)
        sta.update_dz_static(k, dz_new)
        got, want = _bank(hb, sta), _bank(hb, ref)
        assert np.array_equal(got, want), "call %d: banks differ" % (call + 1)
        assert not np.array_equal(got[k, k], start[k, k])            # the update did happen
        assert np.array_equal(_field(sta, w, prec), _field(ref, w, prec)), "call %d: fields differ" % (call + 1)
        if call == 0:
            other.update_dz_static(1, 2.5 * wo.dz[1])
    # the plan in between got the right bank as well
    dzo = wo.dz.copy()
    dzo[1] = 2.5 * wo.dz[1]
    fresh = hb.Plan(wo.nx, wo.ny, wo.nz, wo.dx, wo.dy, dzo, "f64")
    fresh.build_tensor()
    assert np.array_equal(_bank(hb, other), _bank(hb, fresh))
    for p in (ref, sta, other, fresh):
        p.close()


def test_static_update_refuses_plans_beyond_the_fixed_array(hb):
    w = W.small(128, 128, 4, precision="f32", seed=3)
    p = hb.Plan(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, "f32", dedup=0, mirror=0, recip=0)
    p.build_tensor()
    assert p.info.setup_scratch_bytes > hb.STATIC_SCRATCH_BYTES
    before = hb.read_bank(p.handle, 1, 2, 0)
    with pytest.raises(hb.HfftError) as e:
        p.update_dz_static(1, 2.0 * w.dz[1])
    assert e.value.status == hb.EUNSUPPORTED
    assert str(p.info.setup_scratch_bytes) in str(e.value) and str(hb.STATIC_SCRATCH_BYTES) in str(e.value)
    assert hb.plan_info(p.handle).built == 1                                       # untouched: still usable, bank unchanged
    assert np.array_equal(hb.read_bank(p.handle, 1, 2, 0), before)
    # argument errors as in hfft_update_dz
    for k, dz in [(-1, 1.0), (4, 1.0), (1, 0.0), (1, float("nan"))]:
        with pytest.raises(hb.HfftError) as e:
            p.update_dz_static(k, dz)
        assert e.value.status == hb.EINVAL
    p.close()
