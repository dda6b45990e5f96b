"""Thin ctypes binding over the C-ABI library libhfft.so (include/hfft.h).

Argument marshalling only: every step of the method runs in the CUDA kernels behind the C calls.
The functions carry the names of the C entry points without the ``hfft_`` prefix.  PyTorch is
used for device memory and streams only (``Plan`` below); there is no CPU path: if the library
or a CUDA device is missing, loading / plan creation fails loudly.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libhfft.so")

F32, F64 = 0, 1
OK, EINVAL, ENOMEM, ECUDA, ESTATE, EUNSUPPORTED = range(6)
STATUS_NAMES = ["HFFT_OK", "HFFT_EINVAL", "HFFT_ENOMEM", "HFFT_ECUDA", "HFFT_ESTATE", "HFFT_EUNSUPPORTED"]
NUM_STAGES = 5
STAGE_NAMES = ["fftx_fwd", "ffty_fwd", "coupling", "iffty", "ifftx"]
MAX_NZ = 256
STATIC_SCRATCH_BYTES = 32 * 1024 * 1024

# every symbol include/hfft.h declares
EXPORTS = ["hfft_plan_create", "hfft_plan_set_batch", "hfft_plan_set_dedup", "hfft_plan_set_mirror", "hfft_plan_set_recip", "hfft_plan_set_fusion",
           "hfft_tensor_classes", "hfft_plan_info", "hfft_bank_bytes", "hfft_workspace_bytes", "hfft_plan_set_buffers",
           "hfft_build_tensor", "hfft_demag", "hfft_demag_host", "hfft_demag_host_async", "hfft_host_join", "hfft_update_dz", "hfft_update_dz_static", "hfft_plan_set_reduction",
           "hfft_profile_enable", "hfft_profile_read",
           "hfft_read_bank", "hfft_destroy", "hfft_last_error", "hfft_version"]


class Info(ctypes.Structure):
    _fields_ = [("nx", ctypes.c_int), ("ny", ctypes.c_int), ("nz", ctypes.c_int), ("batch", ctypes.c_int),
                ("precision", ctypes.c_int), ("tile_k", ctypes.c_int),
                ("n_k", ctypes.c_longlong), ("n_k_padded", ctypes.c_longlong),
                ("bank_bytes", ctypes.c_size_t), ("workspace_bytes", ctypes.c_size_t),
                ("setup_scratch_bytes", ctypes.c_size_t),
                ("launches_per_demag", ctypes.c_int), ("built", ctypes.c_int),
                ("n_classes", ctypes.c_int), ("mirror", ctypes.c_int), ("dedup", ctypes.c_int), ("fused", ctypes.c_int)]


class HfftError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (STATUS_NAMES[status] if 0 <= status < 6 else status, msg))
        self.status = status


_lib = None


def lib():
    """Load libhfft.so.  Raises if it has not been built (python -m paper_1910_07054_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise FileNotFoundError(
                LIB_PATH + " is missing: build it with `python -m paper_1910_07054_b200.build` "
                "(there is no CPU fallback)")
        L = ctypes.CDLL(LIB_PATH)
        vp, dp, ip = ctypes.c_void_p, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_int)
        L.hfft_plan_create.argtypes = [ctypes.POINTER(vp), ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                       ctypes.c_double, ctypes.c_double, dp, ctypes.c_int]
        L.hfft_plan_set_batch.argtypes = [vp, ctypes.c_int]
        L.hfft_plan_set_dedup.argtypes = [vp, ctypes.c_int]
        L.hfft_plan_set_mirror.argtypes = [vp, ctypes.c_int]
        L.hfft_plan_set_recip.argtypes = [vp, ctypes.c_int]
        L.hfft_plan_set_fusion.argtypes = [vp, ctypes.c_int]
        L.hfft_tensor_classes.argtypes = [ctypes.c_int, dp, ip, ip, ip]
        L.hfft_plan_info.argtypes = [vp, ctypes.POINTER(Info)]
        L.hfft_bank_bytes.argtypes = [vp]
        L.hfft_workspace_bytes.argtypes = [vp]
        L.hfft_plan_set_buffers.argtypes = [vp, vp, vp]
        L.hfft_build_tensor.argtypes = [vp, vp]
        L.hfft_demag.argtypes = [vp, vp, dp, vp, vp]
        L.hfft_demag_host.argtypes = [vp, vp, dp, vp, vp]
        L.hfft_demag_host_async.argtypes = [vp, vp, dp, vp, vp]
        L.hfft_host_join.argtypes = [vp, vp]
        L.hfft_update_dz.argtypes = [vp, ctypes.c_int, ctypes.c_double, vp]
        L.hfft_update_dz_static.argtypes = [vp, ctypes.c_int, ctypes.c_double, vp]
        L.hfft_plan_set_reduction.argtypes = [vp, vp]
        L.hfft_profile_enable.argtypes = [vp, ctypes.c_int]
        L.hfft_profile_read.argtypes = [vp, dp, ip]
        L.hfft_read_bank.argtypes = [vp, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp]
        L.hfft_destroy.argtypes = [vp]
        L.hfft_last_error.argtypes = [vp]
        L.hfft_last_error.restype = ctypes.c_char_p
        L.hfft_version.restype = ctypes.c_char_p
        for name in EXPORTS:
            if name not in ("hfft_last_error", "hfft_version", "hfft_bank_bytes", "hfft_workspace_bytes"):
                getattr(L, name).restype = ctypes.c_int
        L.hfft_bank_bytes.restype = ctypes.c_size_t
        L.hfft_workspace_bytes.restype = ctypes.c_size_t
        _lib = L
    return _lib


def _check(status, plan=None):
    if status != OK:
        raise HfftError(status, last_error(plan))


def _dptr(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def version() -> str:
    return lib().hfft_version().decode()


def last_error(plan=None) -> str:
    return lib().hfft_last_error(plan).decode()


def plan_create(nx, ny, nz, dx, dy, dz, precision):
    dz = np.ascontiguousarray(dz, dtype=np.float64)
    if dz.shape != (nz,):
        raise ValueError("dz must have nz entries")
    out = ctypes.c_void_p()
    _check(lib().hfft_plan_create(ctypes.byref(out), int(nx), int(ny), int(nz), float(dx), float(dy), _dptr(dz),
                                  int(precision)))
    return out


def plan_set_batch(plan, batch):
    _check(lib().hfft_plan_set_batch(plan, int(batch)), plan)


def plan_set_dedup(plan, mode):
    """0 off, 1 automatic (default), 2 on, 3 z-FFT method (equal thicknesses; Eq.25)."""
    _check(lib().hfft_plan_set_dedup(plan, int(mode)), plan)


def bank_bytes(plan) -> int:
    return int(lib().hfft_bank_bytes(plan))


def workspace_bytes(plan) -> int:
    return int(lib().hfft_workspace_bytes(plan))


def plan_set_mirror(plan, on):
    _check(lib().hfft_plan_set_mirror(plan, int(on)), plan)


def plan_set_fusion(plan, mode):
    """0 off, 1 automatic (default: small grids), 2 wherever the fused S2+S3+S4 kernel fits."""
    _check(lib().hfft_plan_set_fusion(plan, int(mode)), plan)


def plan_set_recip(plan, on):
    _check(lib().hfft_plan_set_recip(plan, int(on)), plan)


def tensor_classes(dz):
    """Host-only: (cls [nz][nz] int array, n_classes, toeplitz) of a stack of thicknesses dz."""
    dz = np.ascontiguousarray(dz, dtype=np.float64)
    nz = dz.shape[0]
    cls = np.zeros(max(nz * nz, 1), dtype=np.int32)
    n, t = ctypes.c_int(), ctypes.c_int()
    _check(lib().hfft_tensor_classes(nz, _dptr(dz), cls.ctypes.data_as(ctypes.POINTER(ctypes.c_int)),
                                     ctypes.byref(n), ctypes.byref(t)))
    return cls[:nz * nz].reshape(nz, nz), n.value, bool(t.value)


def plan_info(plan) -> Info:
    info = Info()
    _check(lib().hfft_plan_info(plan, ctypes.byref(info)), plan)
    return info


def plan_set_buffers(plan, bank_ptr, workspace_ptr):
    _check(lib().hfft_plan_set_buffers(plan, ctypes.c_void_p(bank_ptr), ctypes.c_void_p(workspace_ptr)), plan)


def build_tensor(plan, stream=0):
    _check(lib().hfft_build_tensor(plan, ctypes.c_void_p(stream)), plan)


def _ms(Ms, nz):
    if Ms is None:
        return None, None
    a = np.ascontiguousarray(np.broadcast_to(np.asarray(Ms, dtype=np.float64), (nz,)))
    return a, _dptr(a)


def demag(plan, m_ptr, Ms, h_ptr, stream=0, nz=None):
    """m_ptr, h_ptr: device addresses (int).  Ms: None, scalar or [nz] host values."""
    if Ms is not None and nz is None:
        nz = plan_info(plan).nz
    keep, p = _ms(Ms, nz)
    _check(lib().hfft_demag(plan, ctypes.c_void_p(m_ptr), p, ctypes.c_void_p(h_ptr), ctypes.c_void_p(stream)), plan)


def demag_host(plan, m_host_ptr, Ms, h_host_ptr, stream=0, nz=None):
    if Ms is not None and nz is None:
        nz = plan_info(plan).nz
    keep, p = _ms(Ms, nz)
    _check(lib().hfft_demag_host(plan, ctypes.c_void_p(m_host_ptr), p, ctypes.c_void_p(h_host_ptr),
                                 ctypes.c_void_p(stream)), plan)


def demag_host_async(plan, m_host_ptr, Ms, h_host_ptr, stream=0, nz=None):
    if Ms is not None and nz is None:
        nz = plan_info(plan).nz
    keep, p = _ms(Ms, nz)
    _check(lib().hfft_demag_host_async(plan, ctypes.c_void_p(m_host_ptr), p, ctypes.c_void_p(h_host_ptr),
                                       ctypes.c_void_p(stream)), plan)


def host_join(plan, stream=0):
    _check(lib().hfft_host_join(plan, ctypes.c_void_p(stream)), plan)


def update_dz(plan, k, dz_new, stream=0):
    _check(lib().hfft_update_dz(plan, int(k), float(dz_new), ctypes.c_void_p(stream)), plan)


def update_dz_static(plan, k, dz_new, stream=0):
    """hfft_update_dz_static: the same rebuild with its scratch in the library's fixed 32 MiB device array
    (STATIC_SCRATCH_BYTES) instead of cudaMalloc / cudaFree -- for callers that must not allocate."""
    _check(lib().hfft_update_dz_static(plan, int(k), float(dz_new), ctypes.c_void_p(stream)), plan)


def plan_set_reduction(plan, sums_ptr):
    """sums_ptr: device address of B*3*nz*2 doubles, or 0 / None to switch the reductions off."""
    _check(lib().hfft_plan_set_reduction(plan, ctypes.c_void_p(sums_ptr or None)), plan)


def profile_enable(plan, on=True):
    _check(lib().hfft_profile_enable(plan, 1 if on else 0), plan)


def profile_read(plan):
    ms = np.zeros(NUM_STAGES)
    calls = ctypes.c_int()
    _check(lib().hfft_profile_read(plan, _dptr(ms), ctypes.byref(calls)), plan)
    return ms, calls.value


def read_bank(plan, i, j, c, n_k=None):
    if n_k is None:
        n_k = plan_info(plan).n_k
    out = np.empty(n_k, dtype=np.float64)
    _check(lib().hfft_read_bank(plan, int(i), int(j), int(c), _dptr(out)), plan)
    return out


def destroy(plan):
    if plan:
        _check(lib().hfft_destroy(plan))


class Plan:
    """Convenience owner: plan + torch-allocated bank / workspace on the current CUDA device."""

    def __init__(self, nx, ny, nz, dx, dy, dz, precision="f32", batch=1, torch_buffers=True, dedup=None, mirror=None, recip=None, fusion=None):
        import torch

        if not torch.cuda.is_available():
            raise RuntimeError("hfft needs a CUDA device (there is no CPU path)")
        self.torch = torch
        self.precision = F32 if precision in ("f32", F32) else F64
        self.dtype = torch.float32 if self.precision == F32 else torch.float64
        self.handle = plan_create(nx, ny, nz, dx, dy, dz, self.precision)
        self.nx, self.ny, self.nz, self.batch = nx, ny, nz, batch
        if batch != 1:
            plan_set_batch(self.handle, batch)
        if dedup is not None:
            plan_set_dedup(self.handle, dedup)
        if mirror is not None:
            plan_set_mirror(self.handle, mirror)
        if recip is not None:
            plan_set_recip(self.handle, recip)
        if fusion is not None:
            plan_set_fusion(self.handle, fusion)
        self.info = plan_info(self.handle)
        self._bank = self._ws = None
        if torch_buffers:
            self._bank = torch.empty(self.info.bank_bytes + 256, dtype=torch.uint8, device="cuda")
            self._ws = torch.empty(self.info.workspace_bytes + 256, dtype=torch.uint8, device="cuda")
            al = lambda t: (t.data_ptr() + 255) & ~255
            plan_set_buffers(self.handle, al(self._bank), al(self._ws))
        self.shape = (batch, 3, nz, ny, nx)

    def _stream(self):
        return self.torch.cuda.current_stream().cuda_stream

    def build_tensor(self):
        build_tensor(self.handle, self._stream())
        self.info = plan_info(self.handle)

    def demag(self, m, Ms=None, h=None):
        """m: CUDA tensor [B][3][nz][ny][nx] (or without B if batch == 1) of the plan dtype."""
        t = self.torch
        assert m.is_cuda and m.dtype == self.dtype and m.is_contiguous()
        assert m.numel() == int(np.prod(self.shape))
        if h is None:
            h = t.empty_like(m)
        demag(self.handle, m.data_ptr(), Ms, h.data_ptr(), self._stream(), nz=self.nz)
        return h

    def demag_host(self, m_host, Ms=None, h_host=None):
        """m_host: pinned CPU tensor; returns a pinned CPU tensor (asynchronous on the current stream)."""
        t = self.torch
        assert not m_host.is_cuda and m_host.dtype == self.dtype and m_host.is_contiguous()
        if h_host is None:
            h_host = t.empty_like(m_host).pin_memory()
        demag_host(self.handle, m_host.data_ptr(), Ms, h_host.data_ptr(), self._stream(), nz=self.nz)
        return h_host

    def demag_host_async(self, m_host, Ms=None, h_host=None):
        """Pipelined host path: returns at once; h_host is valid after host_join() + a stream synchronisation."""
        t = self.torch
        assert not m_host.is_cuda and m_host.dtype == self.dtype and m_host.is_contiguous()
        if h_host is None:
            h_host = t.empty_like(m_host).pin_memory()
        demag_host_async(self.handle, m_host.data_ptr(), Ms, h_host.data_ptr(), self._stream(), nz=self.nz)
        return h_host

    def host_join(self):
        host_join(self.handle, self._stream())

    def update_dz(self, k, dz_new):
        update_dz(self.handle, k, dz_new, self._stream())

    def update_dz_static(self, k, dz_new):
        update_dz_static(self.handle, k, dz_new, self._stream())

    def set_reduction(self, on=True):
        """Returns the device tensor [B][3][nz][2] = (sum of h_c, sum of m_c h_c) per plane that every
        following demag call fills (None when switched off)."""
        t = self.torch
        self.sums = t.zeros((self.batch, 3, self.nz, 2), dtype=t.float64, device="cuda") if on else None
        plan_set_reduction(self.handle, self.sums.data_ptr() if on else 0)
        return self.sums

    def close(self):
        if self.handle:
            destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
