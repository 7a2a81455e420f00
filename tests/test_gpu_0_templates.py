"""GPU parity, row a0: template bank (k_gen_taps, k_template_spectrum, k_permute_templates_2048) (see tests/gpu_common.py for the tolerances and the order of the session)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1511_07343_b200 import synth
from gpu_common import assert_cand_parity, assert_power_parity, cand_set, make_plan, run_gpu_plane  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("idx", [0, 1, 2])
def test_templates_match_oracle(fdas, idx):
    cfg = synth.config(idx)
    plan = make_plan(fdas, cfg)
    T_gpu = fdas.fdas_get_templates(plan.handle)
    T_ref = oracle.templates(cfg.z_max, cfg.dz, cfg.width, cfg.interbin)
    assert T_gpu.shape == T_ref.shape
    assert np.max(np.abs(T_gpu - T_ref)) <= 1e-6


def test_fp32_peak_microbenchmark_is_sane(fdas):
    """fdas_measure_fp32_tflops: a B200 must land between a quarter of and slightly above the nominal
    148 SM x 128 lanes x 2 x 1.965 GHz = 74.4 TFLOP/s."""
    tf, ms = fdas.fdas_measure_fp32_tflops()
    assert 18.0 < tf < 85.0 and ms > 0.0
    l2 = fdas.fdas_measure_l2_gbs()                                      # L2 -> SM: above the HBM copy rate, below 40 TB/s
    assert 3.0e3 < l2 < 4.0e4
    tf2, _ = fdas.fdas_measure_fp32_tflops(packed=True)               # FFMA2 chains: same lanes, half the issue slots
    assert 18.0 < tf2 < 170.0


def test_occupancy_matches_the_design(fdas):
    """3 CTAs/SM for the three spectrum passes and the fused segment kernel, 1 for the staged
    variant (384 threads), 3 CTAs of 4 warps for the harmonic sum -- from the occupancy API, not by hand."""
    occ = {k: fdas.fdas_kernel_occupancy(k) for k in fdas.OCCUPANCY_KERNELS}
    print(occ)
    for k in ("spec_pass_a", "spec_pass_b", "spec_pass_c", "correlate", "correlate_fused", "harmsum"):
        assert occ[k][0] >= 3, (k, occ[k])
    assert occ["correlate_staged"][0] == 1 and occ["correlate"][1] <= 168
