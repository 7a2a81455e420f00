"""Thin ctypes binding of libfdas.so (include/fdas.h): argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; PyTorch is used for
device memory and streams. There is no CPU fallback: a missing library raises.
Function names mirror the C ABI (`fdas_plan_create`, `fdas_spectrum`, ...); `Plan`
is a small convenience wrapper that owns the device buffers.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfdas.so")

FDAS_OK, FDAS_E_INVALID, FDAS_E_STATE, FDAS_E_WORKSPACE, FDAS_E_CUDA, FDAS_E_NOMEM = 0, -1, -2, -3, -4, -5
FDAS_OPT_INTERBIN, FDAS_OPT_MAX_BATCH, FDAS_OPT_QUAD_POINTS = 1, 2, 3
FDAS_OPT_TUNE_SCALAR, FDAS_OPT_TUNE_T_CHUNKS, FDAS_OPT_TUNE_HS_SECTORS, FDAS_OPT_TUNE_HS_ROWS, FDAS_OPT_TUNE_HS_VARIANT, FDAS_OPT_TUNE_SPEC_GENERIC, FDAS_OPT_TUNE_STAGE_TEMPLATES, FDAS_OPT_TUNE_SPEC_SELFTEST = 101, 102, 103, 104, 105, 106, 107, 108
FDAS_STATUS_COPY_TIMEOUT, FDAS_STATUS_TMA_FALLBACK = 1, 2

CAND_DTYPE = np.dtype([("col", "<i4"), ("zi", "<i2"), ("nharm", "<i2"), ("power", "<f4")])
assert CAND_DTYPE.itemsize == 12

EXPORTS = ["fdas_set_device", "fdas_plan_create", "fdas_plan_set_option", "fdas_plan_info",
           "fdas_build_templates", "fdas_plan_status", "fdas_get_templates", "fdas_spectrum", "fdas_correlate",
           "fdas_harmsum", "fdas_candidates", "fdas_resample", "fdas_search_host", "fdas_threshold", "fdas_measure_fp32_tflops", "fdas_measure_l2_gbs", "fdas_kernel_occupancy",
           "fdas_plan_destroy", "fdas_strerror"]


class FdasInfo(C.Structure):
    _fields_ = [("n_samples", C.c_int64), ("n_bins", C.c_int64), ("n_cols", C.c_int64),
                ("bin0", C.c_int32), ("n_z", C.c_int32), ("n_templates", C.c_int32), ("width", C.c_int32),
                ("seg_len", C.c_int32), ("step", C.c_int32), ("n_seg", C.c_int32), ("interbin", C.c_int32),
                ("z_max", C.c_double), ("dz", C.c_double), ("workspace_bytes", C.c_size_t)]


class FdasError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__("%s failed: %d (%s)" % (where, code, lib().fdas_strerror(code).decode()))


_lib = None


def lib():
    """Load libfdas.so (raises if it has not been built: there is no fallback path)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError("libfdas.so not built: run `python -m paper_1511_07343_b200.build` "
                              "(or __graft_entry__.build()); the CUDA library is required")
        L = C.CDLL(LIB_PATH)
        vp, i32, i64, u32, f32, f64 = C.c_void_p, C.c_int32, C.c_int64, C.c_uint32, C.c_float, C.c_double
        L.fdas_set_device.argtypes = [i32]
        L.fdas_plan_create.argtypes = [C.POINTER(vp), i64, f64, f64, i32, i32]
        L.fdas_plan_set_option.argtypes = [vp, i32, i64]
        L.fdas_plan_info.argtypes = [vp, C.POINTER(FdasInfo)]
        L.fdas_build_templates.argtypes = [vp, vp]
        L.fdas_plan_status.argtypes = [vp, C.POINTER(u32)]
        L.fdas_get_templates.argtypes = [vp, vp]
        L.fdas_spectrum.argtypes = [vp, vp, i32, vp, vp, vp, vp]
        L.fdas_correlate.argtypes = [vp, vp, i32, vp, f32, vp, vp, u32, vp, vp]
        L.fdas_harmsum.argtypes = [vp, vp, i32, vp, vp, vp, u32, vp]
        L.fdas_candidates.argtypes = [vp, vp, f32, vp, vp, u32, vp]
        L.fdas_resample.argtypes = [vp, vp, f64, vp, vp]
        L.fdas_search_host.argtypes = [vp, vp, i32, i32, vp, vp, vp, u32, vp]
        L.fdas_measure_fp32_tflops.argtypes = [C.POINTER(f64), C.POINTER(f64), i32, vp]
        L.fdas_measure_l2_gbs.argtypes = [C.POINTER(f64), C.c_size_t, vp]
        L.fdas_kernel_occupancy.argtypes = [C.c_char_p, C.POINTER(i32), C.POINTER(i32), C.POINTER(i32)]
        L.fdas_threshold.argtypes = [i32, f64]
        L.fdas_threshold.restype = f64
        L.fdas_plan_destroy.argtypes = [vp]
        L.fdas_strerror.argtypes = [C.c_int]
        L.fdas_strerror.restype = C.c_char_p
        for n in EXPORTS:
            if n not in ("fdas_threshold", "fdas_strerror"):
                getattr(L, n).restype = C.c_int
        _lib = L
    return _lib


def _check(code, where):
    if code != FDAS_OK:
        raise FdasError(code, where)


def _dptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else None


def _require(t, name, numel, dtypes, device=None, allow_none=False):
    """A device buffer handed to the C ABI: the library cannot know sizes or types, so a wrong tensor would
    become an out-of-bounds access on the GPU.  Raise here instead (torch tensors only; anything else that
    offers data_ptr() -- a test double -- is the caller's responsibility)."""
    if t is None:
        if allow_none:
            return
        raise ValueError("%s is required" % name)
    if not isinstance(t, torch.Tensor):
        return
    if not t.is_cuda:
        raise ValueError("%s must be a CUDA tensor (got %s)" % (name, t.device))
    if device is not None and t.device != device:
        raise ValueError("%s is on %s, the plan on %s" % (name, t.device, device))
    if t.dtype not in dtypes:
        raise ValueError("%s has dtype %s, expected one of %s" % (name, t.dtype, dtypes))
    if not t.is_contiguous():
        raise ValueError("%s must be contiguous" % name)
    if t.numel() < numel:
        raise ValueError("%s has %d elements, the call needs %d" % (name, t.numel(), numel))


_F32 = (torch.float32,)
_I32 = (torch.int32, torch.uint32) if hasattr(torch, "uint32") else (torch.int32,)
_U8 = (torch.uint8,)


def _stream(stream=None):
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


# --------------------------------------------------------------------------- C-ABI mirrors
def fdas_set_device(device: int):
    _check(lib().fdas_set_device(int(device)), "fdas_set_device")


def fdas_plan_create(n_samples, z_max, dz, template_width, segment_len):
    h = C.c_void_p()
    _check(lib().fdas_plan_create(C.byref(h), int(n_samples), float(z_max), float(dz),
                                  int(template_width), int(segment_len)), "fdas_plan_create")
    return h


def fdas_plan_set_option(plan, key, value):
    _check(lib().fdas_plan_set_option(plan, int(key), int(value)), "fdas_plan_set_option")


def fdas_plan_info(plan) -> FdasInfo:
    info = FdasInfo()
    _check(lib().fdas_plan_info(plan, C.byref(info)), "fdas_plan_info")
    return info


def fdas_build_templates(plan, stream=None):
    _check(lib().fdas_build_templates(plan, _stream(stream)), "fdas_build_templates")


def fdas_plan_status(plan) -> int:
    out = C.c_uint32()
    _check(lib().fdas_plan_status(plan, C.byref(out)), "fdas_plan_status")
    return out.value


def fdas_get_templates(plan) -> np.ndarray:
    info = fdas_plan_info(plan)
    out = np.empty((info.n_templates, info.width, 2), dtype=np.float32)
    _check(lib().fdas_get_templates(plan, out.ctypes.data_as(C.c_void_p)), "fdas_get_templates")
    return out[..., 0] + 1j * out[..., 1]


def fdas_spectrum(plan, d_series, n_batch, d_spectrum, d_meanpow, d_workspace, stream=None):
    info = fdas_plan_info(plan)
    _require(d_series, "d_series", n_batch * info.n_samples, _F32)
    _require(d_spectrum, "d_spectrum", n_batch * info.n_bins * 2, _F32)
    _require(d_meanpow, "d_meanpow", n_batch, _F32, allow_none=True)
    _require(d_workspace, "d_workspace", info.workspace_bytes, _U8)
    _check(lib().fdas_spectrum(plan, _dptr(d_series), int(n_batch), _dptr(d_spectrum), _dptr(d_meanpow),
                               _dptr(d_workspace), _stream(stream)), "fdas_spectrum")


def fdas_correlate(plan, d_spectrum, n_batch, d_plane, threshold, d_cands, d_counts, capacity,
                   d_workspace=None, stream=None):
    info = fdas_plan_info(plan)
    _require(d_spectrum, "d_spectrum", n_batch * info.n_bins * 2, _F32)
    _require(d_plane, "d_plane", n_batch * info.n_z * info.n_cols, _F32, allow_none=True)
    _require(d_cands, "d_cands", n_batch * int(capacity) * 3, _I32, allow_none=True)
    _require(d_counts, "d_counts", n_batch, _I32, allow_none=d_cands is None)
    _check(lib().fdas_correlate(plan, _dptr(d_spectrum), int(n_batch), _dptr(d_plane), float(threshold),
                                _dptr(d_cands), _dptr(d_counts), int(capacity), _dptr(d_workspace),
                                _stream(stream)), "fdas_correlate")


def fdas_harmsum(plan, d_plane, max_harm, thresholds, d_cands, d_count, capacity, stream=None):
    thr = np.ascontiguousarray(thresholds, dtype=np.float32)
    info = fdas_plan_info(plan)
    if thr.size < int(max_harm).bit_length():
        raise ValueError("fdas_harmsum needs log2(max_harm)+1 thresholds")
    _require(d_plane, "d_plane", info.n_z * info.n_cols, _F32)
    _require(d_cands, "d_cands", int(capacity) * 3, _I32)
    _require(d_count, "d_count", 1, _I32)
    _check(lib().fdas_harmsum(plan, _dptr(d_plane), int(max_harm), thr.ctypes.data_as(C.c_void_p),
                              _dptr(d_cands), _dptr(d_count), int(capacity), _stream(stream)), "fdas_harmsum")


def fdas_candidates(plan, d_plane, threshold, d_cands, d_count, capacity, stream=None):
    info = fdas_plan_info(plan)
    _require(d_plane, "d_plane", info.n_z * info.n_cols, _F32)
    _require(d_cands, "d_cands", int(capacity) * 3, _I32)
    _require(d_count, "d_count", 1, _I32)
    _check(lib().fdas_candidates(plan, _dptr(d_plane), float(threshold), _dptr(d_cands), _dptr(d_count),
                                 int(capacity), _stream(stream)), "fdas_candidates")


def fdas_resample(plan, d_series, beta, d_out, stream=None):
    info = fdas_plan_info(plan)
    _require(d_series, "d_series", info.n_samples, _F32)
    _require(d_out, "d_out", info.n_samples, _F32)
    _check(lib().fdas_resample(plan, _dptr(d_series), float(beta), _dptr(d_out), _stream(stream)), "fdas_resample")


def fdas_search_host(plan, h_series: np.ndarray, max_harm, thresholds, capacity, h_cands=None, h_counts=None,
                     stream=None):
    """Host-buffer path: h_series float32[n_batch, N] (numpy, or a pinned torch CPU tensor for truly
    asynchronous copies); h_cands [n_batch, capacity] 12-byte records and h_counts [n_batch] uint32, numpy
    or pinned torch CPU tensors (int32[n_batch, capacity, 3] / int32[n_batch])."""
    if isinstance(h_series, torch.Tensor):
        ptr, n_batch = h_series.data_ptr(), (h_series.shape[0] if h_series.dim() == 2 else 1)
    else:
        h_series = np.ascontiguousarray(h_series, dtype=np.float32)
        ptr, n_batch = h_series.ctypes.data, (h_series.shape[0] if h_series.ndim == 2 else 1)
    thr = np.ascontiguousarray(thresholds, dtype=np.float32)
    if h_cands is None:
        h_cands = np.zeros((n_batch, capacity), dtype=CAND_DTYPE)
    if h_counts is None:
        h_counts = np.zeros(n_batch, dtype=np.uint32)
    hptr = lambda a: C.c_void_p(a.data_ptr()) if isinstance(a, torch.Tensor) else a.ctypes.data_as(C.c_void_p)
    _check(lib().fdas_search_host(plan, C.c_void_p(ptr), int(n_batch), int(max_harm),
                                  thr.ctypes.data_as(C.c_void_p), hptr(h_cands), hptr(h_counts), int(capacity),
                                  _stream(stream)),
           "fdas_search_host")
    return h_cands, h_counts


def fdas_threshold(n_harm: int, pfa: float = 1e-6) -> float:
    return lib().fdas_threshold(int(n_harm), float(pfa))


def fdas_measure_fp32_tflops(stream=None, packed=False):
    """(TFLOP/s, ms) of the FFMA-chain microbenchmark on the current device (packed: FFMA2 chains)."""
    tf, ms = C.c_double(), C.c_double()
    _check(lib().fdas_measure_fp32_tflops(C.byref(tf), C.byref(ms), 1 if packed else 0, _stream(stream)),
           "fdas_measure_fp32_tflops")
    return tf.value, ms.value


def fdas_measure_l2_gbs(nbytes=32 << 20, stream=None):
    """L2 -> SM read bandwidth (GB/s) of the current device for an L2-resident buffer of `nbytes`."""
    out = C.c_double()
    _check(lib().fdas_measure_l2_gbs(C.byref(out), int(nbytes), _stream(stream)), "fdas_measure_l2_gbs")
    return out.value


OCCUPANCY_KERNELS = ("spec_pass_a", "spec_pass_b", "spec_pass_c", "correlate", "correlate_fused", "correlate_staged", "harmsum")


def fdas_kernel_occupancy(kernel: str):
    """(resident CTAs per SM, registers per thread, shared memory per CTA) of a kernel family's configs[2] instance."""
    a, b, c = C.c_int32(), C.c_int32(), C.c_int32()
    _check(lib().fdas_kernel_occupancy(kernel.encode(), C.byref(a), C.byref(b), C.byref(c)), "fdas_kernel_occupancy")
    return a.value, b.value, c.value


def fdas_plan_destroy(plan):
    _check(lib().fdas_plan_destroy(plan), "fdas_plan_destroy")


def thresholds(max_harm: int, pfa: float = 1e-6) -> np.ndarray:
    return np.array([fdas_threshold(1 << s, pfa) for s in range(int(max_harm).bit_length())], dtype=np.float64)


# --------------------------------------------------------------------------- convenience
class Plan:
    """Owns an fdas_plan handle plus the torch device buffers the hot calls need."""

    def __init__(self, n_samples, z_max, dz, template_width, segment_len, interbin=0, max_batch=1,
                 quad_points=None, device=None, options=()):
        if not torch.cuda.is_available():
            raise RuntimeError("paper_1511_07343_b200 needs a CUDA device (no CPU fallback)")
        self.device = torch.device("cuda", torch.cuda.current_device() if device is None else device)
        fdas_set_device(self.device.index)
        self.handle = fdas_plan_create(n_samples, z_max, dz, template_width, segment_len)
        if interbin:
            fdas_plan_set_option(self.handle, FDAS_OPT_INTERBIN, 1)
        if max_batch != 1:
            fdas_plan_set_option(self.handle, FDAS_OPT_MAX_BATCH, max_batch)
        if quad_points:
            fdas_plan_set_option(self.handle, FDAS_OPT_QUAD_POINTS, quad_points)
        for key, value in options:                       # tuning keys that must be set before the build
            fdas_plan_set_option(self.handle, key, value)
        self.info = fdas_plan_info(self.handle)
        self.max_batch = max_batch
        fdas_build_templates(self.handle)
        self.workspace = torch.empty(self.info.workspace_bytes, dtype=torch.uint8, device=self.device)

    def status(self):
        """Device status word (0 = fine); synchronises the device first."""
        torch.cuda.synchronize(self.device)
        return fdas_plan_status(self.handle)

    def close(self):
        if self.handle is not None:
            fdas_plan_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # buffers
    def empty_spectrum(self, n_batch=1):
        return torch.empty((n_batch, self.info.n_bins, 2), dtype=torch.float32, device=self.device)

    def empty_plane(self, n_batch=1):
        return torch.empty((n_batch, self.info.n_z, self.info.n_cols), dtype=torch.float32, device=self.device)

    def empty_cands(self, capacity, n_batch=1):
        return (torch.zeros((n_batch, capacity, 3), dtype=torch.int32, device=self.device),
                torch.zeros(n_batch, dtype=torch.int32, device=self.device))

    # calls
    def spectrum(self, d_series, d_spectrum=None, d_meanpow=None, stream=None):
        if d_series.dim() not in (1, 2) or d_series.shape[-1] != self.info.n_samples:
            raise ValueError("d_series must be float32[n_samples] or [n_batch, n_samples], got %s" % (tuple(d_series.shape),))
        n_batch = d_series.shape[0] if d_series.dim() == 2 else 1
        if n_batch > self.max_batch:
            raise ValueError("n_batch %d exceeds the plan's MAX_BATCH %d (sizes the workspace)" % (n_batch, self.max_batch))
        if d_spectrum is None:
            d_spectrum = self.empty_spectrum(n_batch)
        if d_meanpow is None:
            d_meanpow = torch.empty(n_batch, dtype=torch.float32, device=self.device)
        fdas_spectrum(self.handle, d_series, n_batch, d_spectrum, d_meanpow, self.workspace, stream)
        return d_spectrum, d_meanpow

    def correlate(self, d_spectrum, d_plane=None, threshold=0.0, cands=None, capacity=0, stream=None):
        if d_spectrum.dim() != 3 or tuple(d_spectrum.shape[1:]) != (self.info.n_bins, 2):
            raise ValueError("d_spectrum must be float32[n_batch, n_bins, 2], got %s" % (tuple(d_spectrum.shape),))
        n_batch = d_spectrum.shape[0]
        d_c, d_n = cands if cands is not None else (None, None)
        fdas_correlate(self.handle, d_spectrum, n_batch, d_plane, threshold, d_c, d_n, capacity, None, stream)

    def harmsum(self, d_plane, max_harm, thr, cands, capacity, stream=None):
        fdas_harmsum(self.handle, d_plane, max_harm, thr, cands[0], cands[1], capacity, stream)

    def candidates(self, d_plane, threshold, cands, capacity, stream=None):
        fdas_candidates(self.handle, d_plane, threshold, cands[0], cands[1], capacity, stream)

    def resample(self, d_series, beta, d_out=None, stream=None):
        if d_out is None:
            d_out = torch.empty_like(d_series)
        fdas_resample(self.handle, d_series, beta, d_out, stream)
        return d_out

    def search_host(self, h_series, max_harm, thr, capacity, h_cands=None, h_counts=None, stream=None):
        return fdas_search_host(self.handle, h_series, max_harm, thr, capacity, h_cands, h_counts, stream)


def cands_to_numpy(d_cands, d_counts, b=0) -> np.ndarray:
    """Device candidate buffer (int32[n_batch, cap, 3] view of 12-byte records) -> structured array."""
    n = int(d_counts[b].item())
    cap = d_cands.shape[1]
    if n > cap:
        raise OverflowError("candidate capacity %d < %d found" % (cap, n))
    raw = d_cands[b, :n].contiguous().cpu().numpy()
    return raw.view(CAND_DTYPE).reshape(-1)
