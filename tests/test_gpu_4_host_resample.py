"""GPU parity, host-buffer path and the time-domain trial at small sizes (see tests/gpu_common.py for the tolerances and the order of the session)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1511_07343_b200 import synth
from gpu_common import assert_cand_parity, assert_power_parity, cand_set, make_plan, run_gpu_plane  # noqa: F401

pytestmark = pytest.mark.gpu


def test_search_host_matches_device_calls(fdas):
    cfg = synth.config(0)
    x = cfg.series()
    plan = make_plan(fdas, cfg)
    thr = fdas.thresholds(8)
    h_c, h_n = plan.search_host(x.reshape(1, -1), 8, thr, 1 << 16)
    d_P, _ = run_gpu_plane(fdas, plan, x)
    cands = plan.empty_cands(1 << 16)
    plan.harmsum(d_P, 8, thr, cands, 1 << 16)
    ref = fdas.cands_to_numpy(*cands)
    assert int(h_n[0]) == len(ref) and cand_set(h_c[0, :len(ref)]) == cand_set(ref)
    # fused threshold mode (max_harm = 0)
    h_c, h_n = plan.search_host(x.reshape(1, -1), 0, np.array([20.0]), 1 << 12)
    S, _ = oracle.spectrum(x)
    c_ref = oracle.candidates(oracle.correlate_direct(S, oracle.templates(cfg.z_max, cfg.dz, cfg.width)), 20.0)
    assert_cand_parity(h_c[0, :int(h_n[0])], c_ref, lambda h: 20.0)


@pytest.mark.parametrize("log2n,beta", [(13, 0.0), (13, -0.3), (17, 0.004), (23, 1.0e-5), (23, 0.49)])
def test_resample_is_bit_exact(fdas, log2n, beta):
    """fdas_resample (G23): the chosen sample index is decided in fp64 with separately
    rounded operations on both sides, so the output is identical bit for bit."""
    N = 1 << log2n
    x = synth.make_series(N, 31 + log2n)
    plan = fdas.Plan(N, 0.0, 2.0, 2, 2048)
    y = plan.resample(torch.from_numpy(x).cuda(), beta).cpu().numpy()
    assert np.array_equal(y, oracle.resample(x, beta))


def test_time_domain_trial_end_to_end(fdas):
    """Resample at beta = z/(2 r0), spectrum, |S|^2 through the z_max = 0 plan (one delta template), candidates:
    the accelerated sinusoid comes back as a tone at r0; the FDAS plane of the raw series agrees on (r0, z)."""
    N, r0, z = 1 << 17, 10000, 8.0
    x = synth.make_series(N, 32, [synth.Signal(0.06, r0, z, 0.3)])
    plan0 = fdas.Plan(N, 0.0, 2.0, 2, 2048)
    d_y = plan0.resample(torch.from_numpy(x).cuda(), z / (2.0 * r0))
    d_P, c = run_gpu_plane(fdas, plan0, d_y.cpu().numpy(), thr=40.0)
    S_ref, _ = oracle.spectrum(oracle.resample(x, z / (2.0 * r0)))
    assert_power_parity(d_P[0].cpu().numpy(), np.abs(S_ref) ** 2)
    assert len(c) >= 1 and int(c[np.argmax(c["power"])]["col"]) == r0 - 1
    plan = fdas.Plan(N, 20.0, 2.0, 64, 1024)
    d_Pf, _ = run_gpu_plane(fdas, plan, x)
    zi, col = np.unravel_index(int(torch.argmax(d_Pf)), d_Pf.shape)
    assert (-20 + 2 * zi, col) == (8, r0 - 1)
    assert float(d_Pf.max()) == pytest.approx(float(d_P.max()), rel=0.15)
