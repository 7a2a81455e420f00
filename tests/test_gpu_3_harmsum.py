"""GPU parity, rows a7, a8: harmonic sum and candidate compaction at small sizes (see tests/gpu_common.py for the tolerances and the order of the session)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1511_07343_b200 import synth
from gpu_common import assert_cand_parity, assert_power_parity, cand_set, make_plan, run_gpu_plane  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("max_harm", [1, 2, 4, 8, 16])
def test_harmsum_random_plane(fdas, max_harm):
    N = 1 << 13
    plan = fdas.Plan(N, 8.0, 2.0, 16, 256)
    n_z, n_cols = plan.info.n_z, plan.info.n_cols
    rng = np.random.default_rng(77)
    P = rng.exponential(1.0, size=(n_z, n_cols)).astype(np.float32)
    P[4, 1000] = 40.0; P[6, 2001] = 35.0; P[1, 7] = 50.0
    thr = oracle.thresholds(max_harm, 1e-3)
    cands = plan.empty_cands(1 << 18)
    plan.harmsum(torch.from_numpy(P).cuda(), max_harm, thr, cands, 1 << 18)
    c_gpu = fdas.cands_to_numpy(*cands)
    c_ref = oracle.harmsum(P.astype(np.float64), max_harm, thr, bin0=1)
    assert len(c_ref) > 20
    thr32 = thr.astype(np.float32)
    assert_cand_parity(c_gpu, c_ref, lambda h: float(thr32[int(h).bit_length() - 1]))


def test_pulse_train_is_found_by_the_harmonic_sum(fdas):
    """Multi-harmonic workload for row a7: eight harmonics of a fundamental at bin
    250, z0 = 1, in N(0,1) noise; candidates as the oracle's, and the most significant one is the
    8-harmonic sum labelled by the top harmonic (8 r0, 8 z0)."""
    N, r0, z0, nh = 1 << 14, 250, 1, 8
    x = synth.make_series(N, 4711, synth.pulse_train(0.055, r0, z0, nh, phi=0.4))
    plan = fdas.Plan(N, 8.0, 1.0, 64, 2048)
    d_P, _ = run_gpu_plane(fdas, plan, x)
    thr = oracle.thresholds(16, 1e-5)
    cands = plan.empty_cands(1 << 14)
    plan.harmsum(d_P, 16, thr, cands, 1 << 14)
    c = fdas.cands_to_numpy(*cands)
    S, _ = oracle.spectrum(x)
    c_ref = oracle.harmsum(oracle.correlate_direct(S, oracle.templates(8.0, 1.0, 64)), 16, thr, bin0=1)
    thr32 = thr.astype(np.float32)
    assert_cand_parity(c, c_ref, lambda h: float(thr32[int(h).bit_length() - 1]))
    best = min(c, key=lambda r: oracle.gamma_q(int(r["nharm"]), float(r["power"])))
    assert (int(best["nharm"]), int(best["col"]), int(best["zi"])) == (8, r0 * nh - 1, 8 + z0 * nh)


def test_kernel_variants_agree(fdas):
    """The tuning keys (FDAS_OPT_TUNE_*): packed f32x2 butterflies give the scalar ones' plane bit for bit, the
    template chunking does not matter, the harmonic sum does not depend on its sector count or tile shape."""
    cfg = synth.small_config(1 << 16, 40.0, 2.0, 256, 2048, n_sig=2, index=7, amp=0.1)
    plan = make_plan(fdas, cfg)
    d_S, _ = plan.spectrum(torch.from_numpy(cfg.series()).cuda().view(1, -1))
    planes = {}
    for name, opts in (("packed", {}), ("scalar", {fdas.FDAS_OPT_TUNE_SCALAR: 1}), ("two_chunks", {fdas.FDAS_OPT_TUNE_T_CHUNKS: 2})):
        for k, v in opts.items():
            fdas.fdas_plan_set_option(plan.handle, k, v)
        try:
            d_P = plan.empty_plane(1)
            plan.correlate(d_S, d_P)
            planes[name] = d_P[0].cpu().numpy()
        finally:
            for k in opts:
                fdas.fdas_plan_set_option(plan.handle, k, 0)
    assert np.array_equal(planes["packed"], planes["scalar"])
    assert np.array_equal(planes["packed"], planes["two_chunks"])
    thr = oracle.thresholds(16, 1e-4)
    d_P = torch.from_numpy(planes["packed"]).cuda()
    lists = []
    for opts in ({fdas.FDAS_OPT_TUNE_HS_SECTORS: 1}, {}, {fdas.FDAS_OPT_TUNE_HS_SECTORS: 32}, {fdas.FDAS_OPT_TUNE_HS_VARIANT: 1}):
        for k, v in opts.items():
            fdas.fdas_plan_set_option(plan.handle, k, v)
        try:
            cands = plan.empty_cands(1 << 18)
            plan.harmsum(d_P, 16, thr, cands, 1 << 18)
            c = fdas.cands_to_numpy(*cands)
        finally:
            for k in opts:
                fdas.fdas_plan_set_option(plan.handle, k, 0)
        lists.append(sorted((int(r["nharm"]), int(r["zi"]), int(r["col"]), float(r["power"])) for r in c))
    assert all(l == lists[0] for l in lists) and len(lists[0]) > 0
