"""Drive the product's ctypes binding against libfdas_emu.so (the kernels compiled for the host, see
README.md) with guard-paged buffers standing in for device memory.  TEST INFRASTRUCTURE ONLY."""
import ctypes as C
import os
import sys

import numpy as np

ROOT = os.path.abspath(os.path.join(os.path.dirname(__file__), "..", ".."))
sys.path.insert(0, ROOT)
from paper_1511_07343_b200 import fdas  # noqa: E402

try:
    from . import build as _build
except ImportError:
    import build as _build

# a private copy of the binding module, so that the real one (bound to libfdas.so) is left untouched
import importlib.util as _ilu  # noqa: E402
_spec = _ilu.spec_from_file_location("fdas_emulated_binding", fdas.__file__)
fdas = _ilu.module_from_spec(_spec)
_spec.loader.exec_module(fdas)
fdas.LIB_PATH = _build.build()
fdas._stream = lambda stream=None: None
L = fdas.lib()
L.emu_malloc.restype = C.c_void_p
L.emu_malloc.argtypes = [C.c_size_t]
L.emu_free.argtypes = [C.c_void_p]
L.emu_launch_count.restype = C.c_long


class DevBuf:
    """Guard-paged 'device' array."""

    def __init__(self, shape, dtype):
        self.shape = tuple(int(s) for s in np.atleast_1d(shape))
        self.dtype = np.dtype(dtype)
        self.nbytes = int(np.prod(self.shape)) * self.dtype.itemsize
        self.ptr = L.emu_malloc(max(self.nbytes, 1))
        assert self.ptr

    def data_ptr(self):
        return self.ptr

    def np(self):
        buf = (C.c_char * self.nbytes).from_address(self.ptr)
        return np.frombuffer(buf, dtype=self.dtype).reshape(self.shape)

    def set(self, a):
        self.np()[...] = np.asarray(a, dtype=self.dtype).reshape(self.shape)
        return self

    def free(self):
        if self.ptr and L is not None:
            L.emu_free(self.ptr)
            self.ptr = None

    def __del__(self):
        self.free()


def to_dev(a):
    a = np.ascontiguousarray(a)
    return DevBuf(a.shape, a.dtype).set(a)


class Plan:
    def __init__(self, n_samples, z_max, dz, width, seg_len, interbin=0, max_batch=1, quad_points=None, options=()):
        self.handle = fdas.fdas_plan_create(n_samples, z_max, dz, width, seg_len)
        for key, value in options:
            fdas.fdas_plan_set_option(self.handle, key, value)
        if interbin:
            fdas.fdas_plan_set_option(self.handle, fdas.FDAS_OPT_INTERBIN, 1)
        if max_batch != 1:
            fdas.fdas_plan_set_option(self.handle, fdas.FDAS_OPT_MAX_BATCH, max_batch)
        if quad_points:
            fdas.fdas_plan_set_option(self.handle, fdas.FDAS_OPT_QUAD_POINTS, quad_points)
        self.info = fdas.fdas_plan_info(self.handle)
        fdas.fdas_build_templates(self.handle)
        self.workspace = DevBuf(self.info.workspace_bytes, np.uint8)

    def spectrum(self, x):
        x = np.atleast_2d(x).astype(np.float32)
        nb = x.shape[0]
        d_x = to_dev(x)
        d_S = DevBuf((nb, self.info.n_bins, 2), np.float32)
        d_mu = DevBuf(nb, np.float32)
        fdas.fdas_spectrum(self.handle, d_x, nb, d_S, d_mu, self.workspace)
        return d_S, d_mu

    def correlate(self, d_S, plane=True, thr=None, cap=0):
        nb = d_S.shape[0]
        d_P = DevBuf((nb, self.info.n_z, self.info.n_cols), np.float32) if plane else None
        d_c = DevBuf((nb, cap), fdas.CAND_DTYPE) if thr is not None else None
        d_n = DevBuf(nb, np.uint32) if thr is not None else None
        fdas.fdas_correlate(self.handle, d_S, nb, d_P, thr or 0.0, d_c, d_n, cap)
        return d_P, d_c, d_n

    def harmsum(self, d_P, max_harm, thr, cap):
        d_c = DevBuf(cap, fdas.CAND_DTYPE)
        d_n = DevBuf(1, np.uint32)
        fdas.fdas_harmsum(self.handle, d_P, max_harm, thr, d_c, d_n, cap)
        n = int(d_n.np()[0])
        return d_c.np()[:min(n, cap)].copy(), n

    def resample(self, x, beta):
        d_x = to_dev(np.asarray(x, np.float32))
        d_y = DevBuf(d_x.shape, np.float32)
        fdas.fdas_resample(self.handle, d_x, beta, d_y)
        return d_y.np().copy()

    def candidates(self, d_P, thr, cap):
        d_c = DevBuf(cap, fdas.CAND_DTYPE)
        d_n = DevBuf(1, np.uint32)
        fdas.fdas_candidates(self.handle, d_P, thr, d_c, d_n, cap)
        n = int(d_n.np()[0])
        return d_c.np()[:min(n, cap)].copy(), n

    def close(self):
        fdas.fdas_plan_destroy(self.handle)
