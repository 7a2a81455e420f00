"""fp64 CPU oracle for the FDAS hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes/numpy wrapper over `fdas_oracle.c` (see that file's header for the
paper passages each function follows).  Only `tests/`, `__graft_entry__.smoke()`
and `bench.py`'s `cpu_baseline` / `--impl reference` legs may import this
package; nothing under `paper_1511_07343_b200/` does, and this package imports
nothing from there.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fdas_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
CFLAGS = ["-O2", "-march=x86-64-v3", "-fopenmp", "-shared", "-fPIC", "-Wall"]

CAND_DTYPE = np.dtype([("col", "<i4"), ("zi", "<i2"), ("nharm", "<i2"), ("power", "<f8")], align=True)


def build(force: bool = False) -> str:
    """Compile fdas_oracle.c with gcc if the shared object is missing or stale."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *CFLAGS, "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        p = C.c_void_p
        L.ofdas_fft.argtypes = [p, C.c_int64, C.c_int]
        L.ofdas_fft.restype = C.c_int
        L.ofdas_dft_direct.argtypes = [p, p, C.c_int64, C.c_int]
        L.ofdas_dft_direct.restype = None
        L.ofdas_spectrum.argtypes = [p, C.c_int64, p, C.POINTER(C.c_double), p]
        L.ofdas_spectrum.restype = C.c_int
        L.ofdas_response.argtypes = [C.c_double, C.c_double, C.c_int64, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.ofdas_response.restype = None
        L.ofdas_templates.argtypes = [C.c_double, C.c_double, C.c_int32, C.c_int32, C.c_int64, p]
        L.ofdas_templates.restype = C.c_int
        L.ofdas_correlate_direct.argtypes = [p, C.c_int64, p, C.c_int32, C.c_int32, C.c_int32, C.c_int64, C.c_int64, p]
        L.ofdas_correlate_direct.restype = None
        L.ofdas_correlate_fft.argtypes = [p, C.c_int64, p, C.c_int32, C.c_int32, C.c_int32, C.c_int32, C.c_int32, p]
        L.ofdas_correlate_fft.restype = C.c_int
        L.ofdas_candidates.argtypes = [p, C.c_int32, C.c_int64, C.c_double, p, C.c_int64]
        L.ofdas_candidates.restype = C.c_int64
        L.ofdas_harmsum.argtypes = [p, C.c_int32, C.c_int64, C.c_int32, C.c_int32, p, p, C.c_int64, p]
        L.ofdas_harmsum.restype = C.c_int64
        L.ofdas_resample.argtypes = [p, C.c_int64, C.c_double, p]
        L.ofdas_resample.restype = C.c_int
        L.ofdas_gamma_q.argtypes = [C.c_int32, C.c_double]
        L.ofdas_gamma_q.restype = C.c_double
        L.ofdas_threshold.argtypes = [C.c_int32, C.c_double]
        L.ofdas_threshold.restype = C.c_double
        _lib = L
    return _lib


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def n_threads() -> int:
    """Threads the OpenMP regions use (OMP_NUM_THREADS or the host core count)."""
    v = os.environ.get("OMP_NUM_THREADS")
    return int(v) if v else (os.cpu_count() or 1)


def fft(a, sign: int = -1) -> np.ndarray:
    """Own radix-2 fp64 FFT (sign -1 forward, +1 unnormalised inverse)."""
    out = np.ascontiguousarray(a, dtype=np.complex128).copy()
    rc = lib().ofdas_fft(_ptr(out), out.size, sign)
    if rc:
        raise ValueError("ofdas_fft: length must be a power of two")
    return out


def dft_direct(a, sign: int = -1) -> np.ndarray:
    x = np.ascontiguousarray(a, dtype=np.complex128)
    out = np.empty_like(x)
    lib().ofdas_dft_direct(_ptr(x), _ptr(out), x.size, sign)
    return out


def spectrum(x, return_raw: bool = False):
    """O1: float32 series -> (S complex128[N/2] for bins 1..N/2, mu) [+ raw F[0..N/2]]."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    N = x.size
    S = np.empty(N // 2, dtype=np.complex128)
    raw = np.empty(N // 2 + 1, dtype=np.complex128) if return_raw else None
    mu = C.c_double()
    rc = lib().ofdas_spectrum(_ptr(x), N, _ptr(S), C.byref(mu), _ptr(raw) if return_raw else None)
    if rc:
        raise ValueError("ofdas_spectrum failed (%d)" % rc)
    return (S, mu.value, raw) if return_raw else (S, mu.value)


def response(z: float, d: float, n_t: int = 1 << 17) -> complex:
    """O2: R_z(d) by mid-point sampled chirp DFT with n_t samples."""
    re, im = C.c_double(), C.c_double()
    lib().ofdas_response(float(z), float(d), int(n_t), C.byref(re), C.byref(im))
    return complex(re.value, im.value)


def n_z_of(z_max: float, dz: float) -> int:
    return int(round(2.0 * z_max / dz)) + 1


def templates(z_max: float, dz: float, m: int, interbin: int = 0, n_t: int = 1 << 17) -> np.ndarray:
    """O3: complex128[n_z*(1+interbin), m], row t = zi*(1+interbin)+s."""
    nt = n_z_of(z_max, dz) * (2 if interbin else 1)
    T = np.empty((nt, m), dtype=np.complex128)
    lib().ofdas_templates(float(z_max), float(dz), int(m), int(bool(interbin)), int(n_t), _ptr(T))
    return T


def correlate_direct(S, T, interbin: int = 0, c0: int = 0, nc: int | None = None) -> np.ndarray:
    """O4: Eq. (1) direct sum for bins [c0, c0+nc) -> float64[n_z, nc*(1+interbin)]."""
    S = np.ascontiguousarray(S, dtype=np.complex128)
    T = np.ascontiguousarray(T, dtype=np.complex128)
    nset = 2 if interbin else 1
    n_z, m = T.shape[0] // nset, T.shape[1]
    if nc is None:
        nc = S.size - c0
    P = np.empty((n_z, nc * nset), dtype=np.float64)
    lib().ofdas_correlate_direct(_ptr(S), S.size, _ptr(T), n_z, m, int(bool(interbin)), int(c0), int(nc), _ptr(P))
    return P


def correlate_fft(S, T, L: int, interbin: int = 0, step: int | None = None) -> np.ndarray:
    """O7: overlap-save FFT correlation, full plane float64[n_z, n_bins*(1+interbin)]."""
    S = np.ascontiguousarray(S, dtype=np.complex128)
    T = np.ascontiguousarray(T, dtype=np.complex128)
    nset = 2 if interbin else 1
    n_z, m = T.shape[0] // nset, T.shape[1]
    if step is None:
        step = L - m
    P = np.empty((n_z, S.size * nset), dtype=np.float64)
    rc = lib().ofdas_correlate_fft(_ptr(S), S.size, _ptr(T), n_z, m, int(bool(interbin)), int(L), int(step), _ptr(P))
    if rc:
        raise ValueError("ofdas_correlate_fft failed (%d)" % rc)
    return P


def candidates(P, thr: float, cap: int = 1 << 22) -> np.ndarray:
    """O5: structured array of cells with P > thr (nharm = 1)."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    out = np.zeros(cap, dtype=CAND_DTYPE)
    n = lib().ofdas_candidates(_ptr(P), P.shape[0], P.shape[1], float(thr), _ptr(out), cap)
    if n > cap:
        raise OverflowError("oracle candidate capacity %d < %d" % (cap, n))
    return out[:n]


def harmsum(P, max_harm: int, thresholds, bin0: int = 1, cap: int = 1 << 23, return_sums: bool = False):
    """O6: (candidates[, S planes float64[n_stage, n_z, n_cols]])."""
    P = np.ascontiguousarray(P, dtype=np.float64)
    thr = np.ascontiguousarray(thresholds, dtype=np.float64)
    n_stage = int(max_harm).bit_length()
    assert thr.size >= n_stage
    out = np.zeros(cap, dtype=CAND_DTYPE)
    S = np.empty((n_stage,) + P.shape, dtype=np.float64) if return_sums else None
    n = lib().ofdas_harmsum(_ptr(P), P.shape[0], P.shape[1], int(bin0), int(max_harm), _ptr(thr), _ptr(out), cap,
                            _ptr(S) if return_sums else None)
    if n > cap:
        raise OverflowError("oracle candidate capacity %d < %d" % (cap, n))
    return (out[:n], S) if return_sums else out[:n]


def resample(x, beta: float) -> np.ndarray:
    """Time-domain acceleration trial (G23): nearest-sample resampling that undoes
    the time offset beta (u^2 - u)."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    y = np.empty_like(x)
    rc = lib().ofdas_resample(_ptr(x), x.size, C.c_double(beta), _ptr(y))
    if rc:
        raise ValueError("ofdas_resample failed (%d)" % rc)
    return y


def gamma_q(H: int, T: float) -> float:
    return lib().ofdas_gamma_q(int(H), float(T))


def threshold(H: int, pfa: float = 1e-6) -> float:
    return lib().ofdas_threshold(int(H), float(pfa))


def thresholds(max_harm: int, pfa: float = 1e-6) -> np.ndarray:
    return np.array([threshold(1 << s, pfa) for s in range(int(max_harm).bit_length())])
