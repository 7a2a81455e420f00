"""CPU-side checks of the C-ABI boundary: the library loads, exports every symbol that
include/fdas.h declares, validates arguments, and its host-only logic (sizes, thresholds)
is right.  No kernel is launched here."""
import ctypes as C
import math
import os
import re

import numpy as np
import pytest

from paper_1511_07343_b200 import build as fdas_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def fdas():
    fdas_build.build()
    from paper_1511_07343_b200 import fdas as m
    m.lib()
    return m


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "fdas.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(fdas_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(fdas):
    names = declared_symbols()
    assert len(names) >= 14
    lib = C.CDLL(fdas.LIB_PATH)
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(fdas.EXPORTS) == names          # the binding mirrors the header one to one


def test_plan_sizes_match_survey_table(fdas):
    # SURVEY.md §8 size table
    for (N, zmax, m, L, ib), (n_z, n_t, n_seg) in {
        (1 << 17, 20, 64, 1024, 0): (21, 21, 69),
        (1 << 20, 100, 256, 2048, 1): (101, 202, 293),
        (1 << 23, 84, 256, 2048, 0): (85, 85, 2341),
    }.items():
        h = fdas.fdas_plan_create(N, zmax, 2.0, m, L)
        if ib:
            fdas.fdas_plan_set_option(h, fdas.FDAS_OPT_INTERBIN, 1)
        i = fdas.fdas_plan_info(h)
        assert (i.n_z, i.n_templates, i.n_seg) == (n_z, n_t, n_seg)
        assert i.n_bins == N // 2 and i.n_cols == (N // 2) * (1 + ib) and i.bin0 == 1
        assert i.step == L - m and i.workspace_bytes >= (N // 2) * 8
        fdas.fdas_plan_destroy(h)


@pytest.mark.parametrize("args", [
    (1000, 20, 2, 64, 1024),          # N not a power of two
    (1024, 20, 2, 64, 1024),          # N < 2L
    (1 << 17, 20, 2, 64, 1000),       # L unsupported
    (1 << 17, 20, 2, 63, 1024),       # m odd
    (1 << 17, 20, 2, 1024, 1024),     # m > L/2
    (1 << 17, 21, 2, 64, 1024),       # z_max/dz not an integer
    (1 << 17, 20, 0, 64, 1024),       # dz = 0
    (1 << 17, -2, 2, 64, 1024),       # z_max < 0
])
def test_plan_create_rejects_bad_arguments(fdas, args):
    with pytest.raises(fdas.FdasError) as e:
        fdas.fdas_plan_create(*args)
    assert e.value.code == fdas.FDAS_E_INVALID


def test_state_and_argument_errors_without_gpu(fdas):
    h = fdas.fdas_plan_create(1 << 17, 20, 2, 64, 1024)
    lib = fdas.lib()
    assert lib.fdas_plan_set_option(h, 99, 1) == fdas.FDAS_E_INVALID
    assert lib.fdas_plan_set_option(h, fdas.FDAS_OPT_INTERBIN, 2) == fdas.FDAS_E_INVALID
    assert lib.fdas_get_templates(h, None) == fdas.FDAS_E_INVALID
    buf = np.zeros(4, np.float32)
    assert lib.fdas_get_templates(h, buf.ctypes.data_as(C.c_void_p)) == fdas.FDAS_E_STATE
    # correlate before build -> state error; NULL outputs -> invalid
    one = C.c_void_p(256)
    assert lib.fdas_correlate(h, one, 1, None, 0.0, None, None, 0, None, None) == fdas.FDAS_E_INVALID
    assert lib.fdas_correlate(h, one, 1, one, 0.0, None, None, 0, None, None) == fdas.FDAS_E_STATE
    assert lib.fdas_spectrum(h, one, 1, one, None, None, None) == fdas.FDAS_E_WORKSPACE
    assert lib.fdas_spectrum(h, one, 1, one, None, C.c_void_p(8), None) == fdas.FDAS_E_WORKSPACE
    assert lib.fdas_spectrum(h, one, 2, one, None, one, None) == fdas.FDAS_E_INVALID      # n_batch > MAX_BATCH
    # misaligned device pointers are refused before anything is launched (include/fdas.h, Conventions)
    odd4, odd8 = C.c_void_p(260), C.c_void_p(264)
    assert lib.fdas_spectrum(h, odd4, 1, one, None, one, None) == fdas.FDAS_E_INVALID
    assert lib.fdas_spectrum(h, one, 1, odd4, None, one, None) == fdas.FDAS_E_INVALID
    assert lib.fdas_correlate(h, odd4, 1, one, 0.0, None, None, 0, None, None) == fdas.FDAS_E_INVALID
    assert lib.fdas_correlate(h, one, 1, odd8, 0.0, None, None, 0, None, None) == fdas.FDAS_E_INVALID
    assert lib.fdas_candidates(h, C.c_void_p(258), 1.0, one, one, 1, None) == fdas.FDAS_E_INVALID
    thr = np.ones(5, np.float32)
    assert lib.fdas_harmsum(h, one, 3, thr.ctypes.data_as(C.c_void_p), one, one, 1, None) == fdas.FDAS_E_INVALID
    assert b"invalid" in lib.fdas_strerror(fdas.FDAS_E_INVALID)
    assert lib.fdas_plan_destroy(None) == fdas.FDAS_E_INVALID
    fdas.fdas_plan_destroy(h)
    # harmonic sum is defined on integer-bin planes only (reading G16)
    h = fdas.fdas_plan_create(1 << 17, 20, 2, 64, 1024)
    fdas.fdas_plan_set_option(h, fdas.FDAS_OPT_INTERBIN, 1)
    assert lib.fdas_harmsum(h, one, 2, thr.ctypes.data_as(C.c_void_p), one, one, 1, None) == fdas.FDAS_E_INVALID
    fdas.fdas_plan_destroy(h)


def test_binding_refuses_wrong_tensors_before_calling_the_library(fdas):
    """the C ABI cannot know buffer sizes, so the Python mirrors check device, dtype,
    contiguity and element count and raise instead of launching on a wrong buffer."""
    import torch
    h = fdas.fdas_plan_create(1 << 12, 4, 2, 16, 256)
    info = fdas.fdas_plan_info(h)
    cpu_series = torch.zeros(1 << 12)
    with pytest.raises(ValueError, match="CUDA tensor"):
        fdas.fdas_spectrum(h, cpu_series, 1, cpu_series, None, cpu_series)
    with pytest.raises(ValueError, match="CUDA tensor"):
        fdas.fdas_correlate(h, torch.zeros((1, info.n_bins, 2)), 1, None, 0.0, None, None, 0)
    with pytest.raises(ValueError, match="thresholds"):
        fdas.fdas_harmsum(h, cpu_series, 16, np.ones(2), cpu_series, cpu_series, 4)
    # the size / dtype / layout rules themselves (a meta tensor stands in for a CUDA one: no GPU here)
    class FakeCuda(torch.Tensor):
        is_cuda = True
    def fake(*shape, dtype=torch.float32):
        return torch.zeros(shape, dtype=dtype).as_subclass(FakeCuda)
    with pytest.raises(ValueError, match="elements"):
        fdas._require(fake(10), "d_plane", 11, fdas._F32)
    with pytest.raises(ValueError, match="dtype"):
        fdas._require(fake(10, dtype=torch.float64), "d_plane", 10, fdas._F32)
    with pytest.raises(ValueError, match="contiguous"):
        fdas._require(fake(10, 2)[:, 0], "d_plane", 10, fdas._F32)
    fdas._require(fake(10), "d_plane", 10, fdas._F32)
    fdas._require(None, "d_meanpow", 1, fdas._F32, allow_none=True)
    with pytest.raises(ValueError, match="required"):
        fdas._require(None, "d_plane", 1, fdas._F32)
    fdas.fdas_plan_destroy(h)


def test_tuning_keys_and_size_limit(fdas):
    lib = fdas.lib()
    h = fdas.fdas_plan_create(1 << 12, 4, 2, 16, 256)
    for key, bad in ((fdas.FDAS_OPT_TUNE_SCALAR, 2), (fdas.FDAS_OPT_TUNE_T_CHUNKS, -1), (fdas.FDAS_OPT_TUNE_HS_SECTORS, 65),
                     (fdas.FDAS_OPT_TUNE_HS_ROWS, 9), (fdas.FDAS_OPT_TUNE_HS_VARIANT, 2)):
        assert lib.fdas_plan_set_option(h, key, bad) == fdas.FDAS_E_INVALID
        assert lib.fdas_plan_set_option(h, key, 1) == fdas.FDAS_OK
        assert lib.fdas_plan_set_option(h, key, 0) == fdas.FDAS_OK
    fdas.fdas_plan_destroy(h)
    # include/fdas.h: n_samples <= 2^25
    hh = C.c_void_p()
    assert lib.fdas_plan_create(C.byref(hh), 1 << 25, 2.0, 2.0, 256, 2048) == fdas.FDAS_OK
    fdas.fdas_plan_destroy(hh)
    assert lib.fdas_plan_create(C.byref(hh), 1 << 26, 2.0, 2.0, 256, 2048) == fdas.FDAS_E_INVALID
    assert "2^25" in open(os.path.join(ROOT, "include", "fdas.h")).read()


def test_thresholds_host_logic(fdas, golden):
    for H, T in golden("thresholds.txt"):
        assert fdas.fdas_threshold(int(H), 1e-6) == pytest.approx(T, abs=2e-9)
    assert fdas.fdas_threshold(1, 1e-3) == pytest.approx(-math.log(1e-3), abs=1e-12)
    assert math.isnan(fdas.fdas_threshold(0, 1e-6)) and math.isnan(fdas.fdas_threshold(2, 1.5))


def test_candidate_record_is_12_bytes(fdas):
    assert fdas.CAND_DTYPE.itemsize == 12
    assert fdas.CAND_DTYPE.fields["zi"][1] == 4 and fdas.CAND_DTYPE.fields["power"][1] == 8


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1511_07343_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "liboracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1511_07343_b200 import" not in txt and "libfdas" not in txt, f
