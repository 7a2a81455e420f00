"""GPU parity: the CUDA path (through the C ABI) against the fp64 oracle, element by element
on the same seeded inputs.  Tolerances are BASELINE.json north_star's:
  power:  |P_gpu - P_ref| <= 1e-4*max(P_ref) + 1e-5*P_ref
  candidate (col, zi, nharm) sets identical except entries within 1e-4 relative of the threshold.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1511_07343_b200 import synth

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def fdas():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1511_07343_b200 import fdas as m
    m.lib()
    return m


def assert_power_parity(P_gpu, P_ref, pmax=None):
    P_ref = np.asarray(P_ref, dtype=np.float64)
    pmax = float(P_ref.max()) if pmax is None else pmax
    err = np.abs(np.asarray(P_gpu, dtype=np.float64) - P_ref)
    tol = 1e-4 * pmax + 1e-5 * P_ref
    bad = err > tol
    assert not bad.any(), "max err %.3e (tol %.3e) at %s" % (err.max(), tol.flat[err.argmax()],
                                                           np.unravel_index(err.argmax(), err.shape))
    return float(err.max())


def cand_set(c):
    return {(int(r["nharm"]), int(r["zi"]), int(r["col"])) for r in c}


def assert_cand_parity(c_gpu, c_ref, thr_of_nharm, val_ref=None):
    """Sets equal except entries whose (reference) power is within 1e-4 relative of the threshold."""
    g, r = cand_set(c_gpu), cand_set(c_ref)
    assert len(c_gpu) == len(g), "duplicate candidates"
    pw_ref = {(int(x["nharm"]), int(x["zi"]), int(x["col"])): float(x["power"]) for x in c_ref}
    pw_gpu = {(int(x["nharm"]), int(x["zi"]), int(x["col"])): float(x["power"]) for x in c_gpu}
    for key in g ^ r:
        p = pw_ref.get(key, pw_gpu.get(key))
        T = thr_of_nharm(key[0])
        assert abs(p - T) <= 1e-4 * T, "candidate mismatch %s power %g thr %g" % (key, p, T)
    pmax = max(pw_ref.values()) if pw_ref else 1.0
    for key in g & r:
        assert abs(pw_gpu[key] - pw_ref[key]) <= 1e-4 * pmax + 1e-5 * pw_ref[key]


def make_plan(fdas, cfg, max_batch=1):
    return fdas.Plan(cfg.n_samples, cfg.z_max, cfg.dz, cfg.width, cfg.seg_len, interbin=cfg.interbin,
                     max_batch=max_batch)


# ------------------------------------------------------------------ templates (row a0)
@pytest.mark.parametrize("idx", [0, 1, 2])
def test_templates_match_oracle(fdas, idx):
    cfg = synth.config(idx)
    plan = make_plan(fdas, cfg)
    T_gpu = fdas.fdas_get_templates(plan.handle)
    T_ref = oracle.templates(cfg.z_max, cfg.dz, cfg.width, cfg.interbin)
    assert T_gpu.shape == T_ref.shape
    assert np.max(np.abs(T_gpu - T_ref)) <= 1e-6


# ------------------------------------------------------------------ spectrum (row a1)
@pytest.mark.parametrize("log2n", [9, 10, 12, 13, 17, 20])
def test_spectrum_matches_oracle(fdas, log2n):
    N = 1 << log2n
    L = 256
    x = synth.make_series(N, 4242 + log2n, [synth.Signal(0.2, N / 8 + 0.3, 2.0, 0.5)])
    x[: N // 2] += 3.0                                   # non-zero mean and a step: exercises the Parseval path
    plan = fdas.Plan(N, 4.0, 2.0, 16, L)
    d_x = torch.from_numpy(x).cuda()
    d_S, d_mu = plan.spectrum(d_x.view(1, -1))
    S_gpu = d_S.cpu().numpy()[0]
    S_gpu = S_gpu[:, 0] + 1j * S_gpu[:, 1]
    S_ref, mu = oracle.spectrum(x)
    assert float(d_mu[0]) == pytest.approx(mu, rel=2e-6)
    scale = np.sqrt(np.mean(np.abs(S_ref) ** 2))         # = 1
    assert np.max(np.abs(S_gpu - S_ref)) <= 3e-6 * np.max(np.abs(S_ref)) + 2e-5 * scale


def test_spectrum_batched(fdas):
    N = 1 << 14
    xs = np.stack([synth.make_series(N, 900 + b) * (1.0 + b) for b in range(3)])
    plan = fdas.Plan(N, 4.0, 2.0, 16, 256, max_batch=3)
    d_S, d_mu = plan.spectrum(torch.from_numpy(xs).cuda())
    for b in range(3):
        S_ref, mu = oracle.spectrum(xs[b])
        S = d_S[b].cpu().numpy()
        assert np.max(np.abs(S[:, 0] + 1j * S[:, 1] - S_ref)) < 2e-5
        assert float(d_mu[b]) == pytest.approx(mu, rel=2e-6)


def test_all_zero_series(fdas):
    """Degenerate input (G22): zero spectrum, zero plane, no candidates, nothing NaN."""
    N = 1 << 13
    plan = fdas.Plan(N, 4.0, 2.0, 64, 2048)
    d_S, d_mu = plan.spectrum(torch.zeros((1, N), device="cuda"))
    assert float(d_mu[0]) == 0.0 and not bool(d_S.any())
    d_P = plan.empty_plane(1)
    cands = plan.empty_cands(16)
    plan.correlate(d_S, d_P, threshold=0.5, cands=cands, capacity=16)
    assert not bool(d_P.any()) and int(cands[1][0]) == 0
    hs = plan.empty_cands(16)
    plan.harmsum(d_P[0], 16, fdas.thresholds(16), hs, 16)
    assert int(hs[1][0]) == 0


# ------------------------------------------------------------------ correlate (rows a2-a6)
def run_gpu_plane(fdas, plan, x, thr=None, cap=1 << 16):
    d_x = torch.from_numpy(np.ascontiguousarray(x)).cuda().view(1, -1)
    d_S, _ = plan.spectrum(d_x)
    d_P = plan.empty_plane(1)
    cands = plan.empty_cands(cap) if thr is not None else None
    plan.correlate(d_S, d_P, threshold=thr or 0.0, cands=cands, capacity=cap if thr is not None else 0)
    torch.cuda.synchronize()
    c = fdas.cands_to_numpy(*cands) if thr is not None else None
    return d_P[0], c


def test_config0_plane_and_candidates(fdas):
    cfg = synth.config(0)
    x = cfg.series()
    plan = make_plan(fdas, cfg)
    d_P, c_gpu = run_gpu_plane(fdas, plan, x, thr=cfg.threshold)
    S, mu = oracle.spectrum(x)
    T = oracle.templates(cfg.z_max, cfg.dz, cfg.width)
    P_ref = oracle.correlate_direct(S, T)                 # Eq. (1), the definition
    assert_power_parity(d_P.cpu().numpy(), P_ref)
    c_ref = oracle.candidates(P_ref, cfg.threshold)
    assert len(c_ref) >= 3
    assert_cand_parity(c_gpu, c_ref, lambda h: cfg.threshold)
    # the injected signal peaks at its (r0, z): bin 10000, z = 8 (north_star)
    zi, col = np.unravel_index(int(torch.argmax(d_P)), d_P.shape)
    assert (-20 + 2 * zi, col + 1) == (8, 10000)


@pytest.mark.parametrize("N,zmax,m,L,ib", [
    (1 << 12, 6.0, 16, 256, 0), (1 << 12, 6.0, 16, 256, 1), (1 << 14, 10.0, 64, 512, 1),
    (1 << 13, 8.0, 128, 256, 0), (1 << 15, 12.0, 32, 4096, 1), (1 << 14, 0.0, 2, 1024, 0),
    (1 << 13, 8.0, 64, 2048, 1),
])
def test_small_configs_vs_direct_sum(fdas, N, zmax, m, L, ib):
    cfg = synth.small_config(N, zmax, 2.0, m, L, interbin=ib, index=20 + ib)
    x = cfg.series()
    plan = make_plan(fdas, cfg)
    d_P, c_gpu = run_gpu_plane(fdas, plan, x, thr=12.0)
    S, _ = oracle.spectrum(x)
    T = oracle.templates(zmax, 2.0, m, ib)
    P_ref = oracle.correlate_direct(S, T, interbin=ib)
    assert_power_parity(d_P.cpu().numpy(), P_ref)
    assert_cand_parity(c_gpu, oracle.candidates(P_ref, 12.0), lambda h: 12.0)


def test_fused_mode_and_overflow_count(fdas):
    cfg = synth.config(0)
    x = cfg.series()
    plan = make_plan(fdas, cfg)
    d_S, _ = plan.spectrum(torch.from_numpy(x).cuda().view(1, -1))
    cands = plan.empty_cands(1 << 16)
    plan.correlate(d_S, None, threshold=8.0, cands=cands, capacity=1 << 16)       # plane not stored
    c_fused = fdas.cands_to_numpy(*cands)
    d_P = plan.empty_plane(1)
    plan.correlate(d_S, d_P)
    c2 = plan.empty_cands(1 << 16)
    plan.candidates(d_P[0], 8.0, c2, 1 << 16)                                      # fdas_candidates on the stored plane
    c_plane = fdas.cands_to_numpy(*c2)
    assert cand_set(c_fused) == cand_set(c_plane) and len(c_fused) > 100
    P = d_P[0].cpu().numpy()
    assert len(c_fused) == int((P > 8.0).sum())
    for r in c_fused[:50]:
        assert P[r["zi"], r["col"]] == r["power"]
    # overflow: the count is the true number, only `capacity` records are written
    small = plan.empty_cands(16)
    plan.correlate(d_S, None, threshold=8.0, cands=small, capacity=16)
    assert int(small[1][0]) == len(c_fused)


# ------------------------------------------------------------------ harmonic sum (rows a7, a8)
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


# ------------------------------------------------------------------ full-size configs (BASELINE.json configs[1..4])
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


def test_kernel_variants_agree(fdas):
    """The variants kept for tuning (FDAS_* switches, read at every call): packed f32x2 butterflies give the
    scalar ones' plane bit for bit, v1 agrees to rounding, the harmonic sum does not depend on its sector count."""
    import os
    cfg = synth.small_config(1 << 16, 40.0, 2.0, 256, 2048, n_sig=2, index=7, amp=0.1)
    plan = make_plan(fdas, cfg)
    d_S, _ = plan.spectrum(torch.from_numpy(cfg.series()).cuda().view(1, -1))
    planes = {}
    for name, env in (("packed", {}), ("scalar", {"FDAS_CORRELATE_SCALAR": "1"}), ("v1", {"FDAS_CORRELATE_V1": "1"})):
        os.environ.update(env)
        try:
            d_P = plan.empty_plane(1)
            plan.correlate(d_S, d_P)
            planes[name] = d_P[0].cpu().numpy()
        finally:
            for k in env:
                os.environ.pop(k)
    assert np.array_equal(planes["packed"], planes["scalar"])
    assert np.max(np.abs(planes["v1"] - planes["packed"])) <= 2e-5 * planes["packed"].max()
    thr = oracle.thresholds(16, 1e-4)
    d_P = torch.from_numpy(planes["packed"]).cuda()
    lists = []
    for env in ({"FDAS_HS_SECTORS": "1"}, {}, {"FDAS_HS_SECTORS": "32"}, {"FDAS_HS_VARIANT": "1"}):
        os.environ.update(env)
        try:
            cands = plan.empty_cands(1 << 18)
            plan.harmsum(d_P, 16, thr, cands, 1 << 18)
            c = fdas.cands_to_numpy(*cands)
        finally:
            for k in env:
                os.environ.pop(k)
        lists.append(sorted((int(r["nharm"]), int(r["zi"]), int(r["col"]), float(r["power"])) for r in c))
    assert all(l == lists[0] for l in lists) and len(lists[0]) > 0


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


def test_fp32_peak_microbenchmark_is_sane(fdas):
    """fdas_measure_fp32_tflops: a B200 must land between a quarter of and slightly above the nominal
    148 SM x 128 lanes x 2 x 1.965 GHz = 74.4 TFLOP/s."""
    tf, ms = fdas.fdas_measure_fp32_tflops()
    assert 18.0 < tf < 85.0 and ms > 0.0
    tf2, _ = fdas.fdas_measure_fp32_tflops(packed=True)               # FFMA2 chains: same lanes, half the issue slots
    assert 18.0 < tf2 < 170.0
