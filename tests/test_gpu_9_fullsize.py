"""GPU parity, BASELINE.json configs[1..4] and the maximum series length at FULL size, in the launch configuration bench.py times (see tests/gpu_common.py for the tolerances and the order of the session)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1511_07343_b200 import synth
from gpu_common import assert_cand_parity, assert_power_parity, cand_set, make_plan, run_gpu_plane  # noqa: F401

pytestmark = pytest.mark.gpu


def full_plane_check(fdas, cfg, windows_seed):
    """GPU plane at full size vs (i) the O7 overlap-save oracle on the whole plane and (ii) the
    Eq. (1) direct sum (O4) on three seeded 2048-column windows x all z.  Returns (plan, d_P, P_ref)."""
    x = cfg.series()
    plan = make_plan(fdas, cfg)
    d_P, _ = run_gpu_plane(fdas, plan, x)
    S, _ = oracle.spectrum(x)
    T = oracle.templates(cfg.z_max, cfg.dz, cfg.width, cfg.interbin)
    P_ref = oracle.correlate_fft(S, T, cfg.seg_len, interbin=cfg.interbin)
    pmax = float(P_ref.max())
    nset = 1 + cfg.interbin
    rng = np.random.default_rng(windows_seed)
    starts = [0, cfg.n_bins - 2048] + [int(v) for v in rng.integers(0, cfg.n_bins - 2048, 2)]
    for c0 in starts:
        Pd = oracle.correlate_direct(S, T, interbin=cfg.interbin, c0=c0, nc=2048)
        ref_w = P_ref[:, c0 * nset:(c0 + 2048) * nset]
        assert np.max(np.abs(Pd - ref_w)) <= 1e-10 * pmax                 # O7 admitted against O4 here too
        assert_power_parity(d_P[:, c0 * nset:(c0 + 2048) * nset].cpu().numpy(), Pd, pmax)
    for zi in range(P_ref.shape[0]):                                       # whole plane, row by row
        assert_power_parity(d_P[zi].cpu().numpy(), P_ref[zi], pmax)
    return plan, d_P, P_ref


def test_config1_interbinned_plane(fdas):
    cfg = synth.config(1)
    plan, d_P, P_ref = full_plane_check(fdas, cfg, 101)
    assert d_P.shape == (101, 1 << 20)
    # each injected signal is recovered near its (r0, z): local maximum within +-2 bins, +-1 z step
    for sg in cfg.signals[0]:
        col = int(round((sg.r0 - 1) * 2)); zi = int(round((sg.z + cfg.z_max) / cfg.dz))
        win = P_ref[max(0, zi - 1):zi + 2, col - 4:col + 5]
        assert win.max() > 0.5 * (sg.amp ** 2 * cfg.n_samples / 4)


def test_config2_ska_plane_and_config4_harmsum(fdas):
    cfg = synth.config(2)
    plan, d_P, P_ref = full_plane_check(fdas, cfg, 202)
    assert d_P.shape == (85, 1 << 22)
    # config 4: harmonic sums over 1..16 harmonics, thresholds for pfa 1e-6 per stage
    thr = oracle.thresholds(16)
    assert np.allclose(thr, fdas.thresholds(16), rtol=0, atol=1e-9)
    cap = 1 << 22
    cands = plan.empty_cands(cap)
    plan.harmsum(d_P, 16, thr, cands, cap)
    c_gpu = fdas.cands_to_numpy(*cands)
    c_ref = oracle.harmsum(P_ref, 16, thr, bin0=1)
    assert len(c_ref) > 1000
    thr32 = thr.astype(np.float32)
    assert_cand_parity(c_gpu, c_ref, lambda h: float(thr32[int(h).bit_length() - 1]))
    # the kernel alone: GPU harmonic sum of the fp32-rounded ORACLE plane vs the oracle on the same values
    P32 = P_ref.astype(np.float32)
    c2 = plan.empty_cands(cap)
    plan.harmsum(torch.from_numpy(P32).cuda(), 16, thr, c2, cap)
    c_ref32 = oracle.harmsum(P32.astype(np.float64), 16, thr, bin0=1)
    assert_cand_parity(fdas.cands_to_numpy(*c2), c_ref32, lambda h: float(thr32[int(h).bit_length() - 1]))


def test_config3_fused_batch(fdas):
    """Streaming batch (configs[3]) at full series length with a reduced batch of 3 DM trials
    (one carries a signal), plane not stored; plus a 64-DM batch at 2^14 samples."""
    cfg = synth.config(3, n_dm=3)
    xs = np.stack([cfg.series(d) for d in range(cfg.n_dm)])
    plan = make_plan(fdas, cfg, max_batch=3)
    d_S, _ = plan.spectrum(torch.from_numpy(xs).cuda())
    cap = 1 << 16
    cands = plan.empty_cands(cap, n_batch=3)
    plan.correlate(d_S, None, threshold=cfg.threshold, cands=cands, capacity=cap)
    T = oracle.templates(cfg.z_max, cfg.dz, cfg.width)
    n_with_signal = 0
    for d in range(cfg.n_dm):
        S, _ = oracle.spectrum(xs[d])
        P_ref = oracle.correlate_fft(S, T, cfg.seg_len)
        c_ref = oracle.candidates(P_ref, cfg.threshold)
        assert_cand_parity(fdas.cands_to_numpy(cands[0], cands[1], d), c_ref, lambda h: cfg.threshold)
        n_with_signal += len(c_ref) > 0 and len(cfg.signals[d]) > 0
    assert n_with_signal == 1
    small = synth.small_config(1 << 14, 16.0, 2.0, 64, 2048, n_dm=64, n_sig=1, index=33, amp=0.3)
    xs = np.stack([small.series(d) for d in range(64)])
    plan = make_plan(fdas, small, max_batch=64)
    d_S, _ = plan.spectrum(torch.from_numpy(xs).cuda())
    cands = plan.empty_cands(1 << 12, n_batch=64)
    plan.correlate(d_S, None, threshold=15.0, cands=cands, capacity=1 << 12)
    T = oracle.templates(16.0, 2.0, 64)
    for d in range(64):
        S, _ = oracle.spectrum(xs[d])
        c_ref = oracle.candidates(oracle.correlate_direct(S, T), 15.0)
        assert_cand_parity(fdas.cands_to_numpy(cands[0], cands[1], d), c_ref, lambda h: 15.0)


def test_maximum_series_length(fdas):
    """The largest series the plan accepts (2^25 samples; 2^24 columns per row): index arithmetic at its
    limits (k h, plane indices, twiddle phases), 3 templates to keep the oracle's share small."""
    N = 1 << 25
    x = synth.make_series(N, 77, [synth.Signal(0.02, 9.0e6 + 0.25, 1.5, 0.3), synth.Signal(0.02, 1.6e7 - 3.5, -2.0, 1.0)])
    plan = fdas.Plan(N, 2.0, 2.0, 256, 2048)
    d_P, c_gpu = run_gpu_plane(fdas, plan, x, thr=30.0)
    S, _ = oracle.spectrum(x)
    T = oracle.templates(2.0, 2.0, 256)
    P_ref = oracle.correlate_fft(S, T, 2048)
    pmax = float(P_ref.max())
    for c0 in (0, (1 << 24) - 2048, 9_000_000 - 1024):
        Pd = oracle.correlate_direct(S, T, c0=c0, nc=2048)
        assert np.max(np.abs(Pd - P_ref[:, c0:c0 + 2048])) <= 1e-10 * pmax
    for zi in range(3):
        assert_power_parity(d_P[zi].cpu().numpy(), P_ref[zi], pmax)
    assert_cand_parity(c_gpu, oracle.candidates(P_ref, 30.0), lambda h: 30.0)
    thr = oracle.thresholds(16)
    cands = plan.empty_cands(1 << 20)
    plan.harmsum(d_P, 16, thr, cands, 1 << 20)
    thr32 = thr.astype(np.float32)
    assert_cand_parity(fdas.cands_to_numpy(*cands), oracle.harmsum(P_ref, 16, thr, bin0=1),
                       lambda h: float(thr32[int(h).bit_length() - 1]))
