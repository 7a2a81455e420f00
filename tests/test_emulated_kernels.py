"""The CUDA kernels, run on the CPU: `tests/emu` compiles paper_1511_07343_b200/csrc/*.cu as host C++
(one fibre per CUDA thread, real __syncthreads/__syncwarp semantics, guard pages around every "device"
buffer and shared-memory array) and this file drives them through the product's own ctypes binding
and compares with the fp64 oracle, exactly as tests/test_gpu_parity.py does on the B200.

What this adds to the `-m gpu` tests: it runs where there is no GPU, and an out-of-bounds or
misaligned access, a barrier reached by only part of a CTA, or a dependence on the order in which
the threads of a CTA run (a missing barrier) fails here with the kernel, block and thread named,
instead of raising an Xid on the GPU box.  It says nothing about speed.
Test infrastructure only: nothing under paper_1511_07343_b200/ knows about it (tests/emu/README.md).
"""
import os
import sys

import numpy as np
import pytest

import oracle
from paper_1511_07343_b200 import synth

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from emu import harness as E  # noqa: E402

fdas = E.fdas
ROOT_DIR = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(params=[("end", "fwd"), ("start", "rev"), ("end", "rand7")],
                ids=["guard-after", "guard-before-reversed", "guard-after-random-order"])
def emu(request):
    """Buffer placement against the trailing / leading guard page; thread order within a CTA forward / reversed /
    pseudo-random."""
    os.environ["EMU_ALIGN"], os.environ["EMU_ORDER"] = request.param
    yield E
    os.environ.pop("EMU_ALIGN"), os.environ.pop("EMU_ORDER")


def power_ok(P_gpu, P_ref):
    P_ref = np.asarray(P_ref, np.float64)
    err = np.abs(np.asarray(P_gpu, np.float64) - P_ref)
    assert not (err > 1e-4 * P_ref.max() + 1e-5 * P_ref).any(), err.max()


def cset(c):
    return {(int(r["nharm"]), int(r["zi"]), int(r["col"])) for r in c}


def cand_ok(c_gpu, c_ref, thr_of):
    g, r = cset(c_gpu), cset(c_ref)
    assert len(c_gpu) == len(g), "duplicate candidates"
    pw = {(int(x["nharm"]), int(x["zi"]), int(x["col"])): float(x["power"]) for x in list(c_gpu) + list(c_ref)}
    for k in g ^ r:
        assert abs(pw[k] - thr_of(k[0])) <= 1e-4 * thr_of(k[0]), k


# 2^9, 2^10, 2^12: the generic kernels; 2^13 .. 2^17: two TMA-staged passes (factors 64x64 .. 256x256);
# 2^18, 2^19: three passes (32x32x128, 32x32x256)
@pytest.mark.parametrize("log2n", [9, 10, 12, 13, 14, 15, 16, 17, 18, 19])
def test_spectrum(emu, log2n):
    N = 1 << log2n
    x = synth.make_series(N, 4242 + log2n, [synth.Signal(0.2, N / 8 + 0.3, 2.0, 0.5)])
    x[: N // 2] += 3.0
    plan = emu.Plan(N, 4.0, 2.0, 16, 256, quad_points=64)
    d_S, d_mu = plan.spectrum(x)
    S = d_S.np()[0]
    S_ref, mu = oracle.spectrum(x)
    assert float(d_mu.np()[0]) == pytest.approx(mu, rel=2e-6)
    assert np.max(np.abs(S[:, 0] + 1j * S[:, 1] - S_ref)) <= 3e-6 * np.max(np.abs(S_ref)) + 2e-5
    assert fdas.fdas_plan_status(plan.handle) == 0
    plan.close()


def test_spectrum_paths_agree_and_fall_back(emu):
    """The TMA-staged passes and the generic kernels give the same spectrum to rounding (each within 1e-6 rms of
    the oracle); a series that is only 8-byte aligned (tensor maps need 16) silently takes the generic kernels."""
    N = 1 << 15
    xs = np.stack([synth.make_series(N, 500 + b) * (1.0 + 0.5 * b) for b in range(2)])
    S = {}
    for generic in (0, 1):
        plan = emu.Plan(N, 4.0, 2.0, 16, 256, max_batch=2, quad_points=64)
        fdas.fdas_plan_set_option(plan.handle, fdas.FDAS_OPT_TUNE_SPEC_GENERIC, generic)
        d_S, d_mu = plan.spectrum(xs)
        S[generic] = d_S.np().copy()
        for b in range(2):
            S_ref, mu = oracle.spectrum(xs[b])
            z = S[generic][b][:, 0] + 1j * S[generic][b][:, 1]
            assert np.sqrt(np.mean(np.abs(z - S_ref) ** 2)) < 1e-6 and float(d_mu.np()[b]) == pytest.approx(mu, rel=2e-6)
        plan.close()
    assert np.max(np.abs(S[0] - S[1])) < 5e-6
    plan = emu.Plan(N, 4.0, 2.0, 16, 256, quad_points=64)
    buf = E.DevBuf(N + 2, np.float32)
    buf.np()[2:] = xs[0]

    class Shifted:
        def data_ptr(self):
            return buf.ptr + 8

    d_S = E.DevBuf((1, N // 2, 2), np.float32)
    fdas.fdas_spectrum(plan.handle, Shifted(), 1, d_S, None, plan.workspace)
    assert np.max(np.abs(d_S.np()[0] - S[1][0])) == 0.0                  # bit for bit the generic kernels' result
    plan.close()


def test_spectrum_selftest_and_fallback(emu):
    """fdas_build_templates compares the TMA-staged passes with the generic kernels on one seeded series: in the
    normal case the status word stays 0 and the TMA passes are used; if the comparison fails (test hook: option
    value 2) the plan reports FDAS_STATUS_TMA_FALLBACK and its spectra are the generic kernels', bit for bit."""
    N = 1 << 14
    x = synth.make_series(N, 321)
    ok = emu.Plan(N, 4.0, 2.0, 16, 256, quad_points=64)
    assert fdas.fdas_plan_status(ok.handle) == 0
    spec = lambda plan: (lambda d: d[0].np().copy())(plan.spectrum(x))     # (the buffers stay alive while they are copied)
    S_tma = spec(ok)
    fdas.fdas_plan_set_option(ok.handle, fdas.FDAS_OPT_TUNE_SPEC_GENERIC, 1)
    S_gen = spec(ok)
    ok.close()
    bad = emu.Plan(N, 4.0, 2.0, 16, 256, quad_points=64, options=[(fdas.FDAS_OPT_TUNE_SPEC_SELFTEST, 2)])
    assert fdas.fdas_plan_status(bad.handle) == fdas.FDAS_STATUS_TMA_FALLBACK
    S_bad = spec(bad)
    bad.close()
    assert np.array_equal(S_bad, S_gen) and not np.array_equal(S_tma, S_gen)
    skipped = emu.Plan(N, 4.0, 2.0, 16, 256, quad_points=64, options=[(fdas.FDAS_OPT_TUNE_SPEC_SELFTEST, 1)])
    assert fdas.fdas_plan_status(skipped.handle) == 0 and np.array_equal(spec(skipped), S_tma)
    skipped.close()


def test_all_zero_series(emu):
    """Degenerate input (G22): zero spectrum, zero plane, no candidates, nothing NaN."""
    N = 1 << 13
    plan = emu.Plan(N, 4.0, 2.0, 64, 2048, quad_points=256)
    d_S, d_mu = plan.spectrum(np.zeros(N, np.float32))
    assert float(d_mu.np()[0]) == 0.0 and not np.any(d_S.np())
    d_P, _, d_n = plan.correlate(d_S, True, 0.5, 16)
    assert not np.any(d_P.np()) and int(d_n.np()[0]) == 0
    c, n = plan.harmsum(d_P, 16, oracle.thresholds(16), 16)
    assert n == 0
    plan.close()


@pytest.mark.parametrize("N", [1 << 12, 1 << 13])
def test_spectrum_batched(emu, N):
    xs = np.stack([synth.make_series(N, 900 + b) * (1.0 + b) for b in range(3)])
    plan = emu.Plan(N, 4.0, 2.0, 16, 256, max_batch=3, quad_points=64)
    d_S, d_mu = plan.spectrum(xs)
    for b in range(3):
        S_ref, mu = oracle.spectrum(xs[b])
        S = d_S.np()[b]
        assert np.max(np.abs(S[:, 0] + 1j * S[:, 1] - S_ref)) < 2e-5
        assert float(d_mu.np()[b]) == pytest.approx(mu, rel=2e-6)
    plan.close()


# (N, z_max, m, L, interbin): the generic shared-memory kernel (L != 2048) and every template
# instance of the register-resident L = 2048 kernel, including a ragged last segment, m = L/2,
# one template (z_max = 0) and more than one template chunk (n_t > 29).
@pytest.mark.parametrize("N,zmax,m,L,ib", [
    (1 << 12, 6.0, 16, 256, 1), (1 << 13, 8.0, 128, 256, 0), (1 << 14, 4.0, 32, 4096, 1), (1 << 12, 0.0, 2, 1024, 0),
    (1 << 13, 8.0, 64, 2048, 1), (1 << 13, 8.0, 64, 2048, 0), (1 << 13, 60.0, 256, 2048, 0), (1 << 12, 2.0, 1024, 2048, 1), (1 << 13, 4.0, 256, 2048, 1),
])
def test_correlate_all_modes(emu, N, zmax, m, L, ib):
    cfg = synth.small_config(N, zmax, 2.0, m, L, interbin=ib, index=20 + ib)
    x = cfg.series()
    plan = emu.Plan(N, zmax, 2.0, m, L, interbin=ib, quad_points=max(2048, 32 * m))
    d_S, _ = plan.spectrum(x)
    d_P, d_c, d_n = plan.correlate(d_S, True, 9.0, 1 << 14)           # plane + candidates
    S, _ = oracle.spectrum(x)
    T = oracle.templates(zmax, 2.0, m, ib)
    assert np.max(np.abs(fdas.fdas_get_templates(plan.handle) - T)) <= 1e-6
    P_ref = oracle.correlate_direct(S, T, interbin=ib)                 # Eq. (1), the definition
    power_ok(d_P.np()[0], P_ref)
    n = int(d_n.np()[0])
    cand_ok(d_c.np()[0, :n], oracle.candidates(P_ref, 9.0), lambda h: 9.0)
    _, d_c2, d_n2 = plan.correlate(d_S, False, 9.0, 1 << 14)          # fused: plane not stored
    assert cset(d_c2.np()[0, :int(d_n2.np()[0])]) == cset(d_c.np()[0, :n])
    d_P3, _, _ = plan.correlate(d_S, True)                            # plane only
    assert np.array_equal(d_P3.np(), d_P.np())
    _, _, d_n4 = plan.correlate(d_S, False, 9.0, 3)                   # overflow: true count, 3 records
    assert int(d_n4.np()[0]) == n
    c5, n5 = plan.candidates(d_P, 9.0, 1 << 14)                       # fdas_candidates on the stored plane
    assert n5 == n and cset(c5) == cset(d_c.np()[0, :n])
    plan.close()


@pytest.mark.parametrize("N", [1 << 9, 1 << 12])
@pytest.mark.parametrize("max_harm", [1, 2, 4, 8, 16])
def test_harmsum(emu, N, max_harm):
    plan = emu.Plan(N, 8.0, 2.0, 16, 256, quad_points=64)
    n_z, n_cols = plan.info.n_z, plan.info.n_cols
    P = np.random.default_rng(77).exponential(1.0, size=(n_z, n_cols)).astype(np.float32)
    P[4, n_cols // 4] = 40.0; P[6, n_cols // 2 + 1] = 35.0; P[1, 7] = 50.0
    thr = oracle.thresholds(max_harm, 1e-3)
    c, n = plan.harmsum(E.to_dev(P), max_harm, thr, 1 << 16)
    c_ref = oracle.harmsum(P.astype(np.float64), max_harm, thr, bin0=1)
    assert len(c_ref) >= 3 and n == len(c)
    thr32 = thr.astype(np.float32)
    cand_ok(c, c_ref, lambda h: float(thr32[int(h).bit_length() - 1]))
    plan.close()


def test_pulse_train_is_found_by_the_harmonic_sum(emu):
    """A multi-harmonic workload for row a7: eight harmonics of a fundamental at
    bin 250, z0 = 1, each near the single-harmonic threshold (A^2 N/4 = 12.4), in N(0,1) noise.  The CUDA path
    (spectrum -> correlate -> harmonic sum) must give the oracle's candidates, and the most significant
    one must be the 8-harmonic sum labelled by the TOP harmonic: (8 r0, 8 z0)."""
    N, r0, z0, nh = 1 << 14, 250, 1, 8
    x = synth.make_series(N, 4711, synth.pulse_train(0.055, r0, z0, nh, phi=0.4))
    plan = emu.Plan(N, 8.0, 1.0, 64, 2048, quad_points=2048)
    d_S, _ = plan.spectrum(x)
    d_P, _, _ = plan.correlate(d_S, True)
    thr = oracle.thresholds(16, 1e-5)
    c, n = plan.harmsum(d_P, 16, thr, 1 << 14)
    S, _ = oracle.spectrum(x)
    P_ref = oracle.correlate_direct(S, oracle.templates(8.0, 1.0, 64))
    c_ref = oracle.harmsum(P_ref, 16, thr, bin0=1)
    thr32 = thr.astype(np.float32)
    cand_ok(c, c_ref, lambda h: float(thr32[int(h).bit_length() - 1]))
    sig = lambda r: oracle.gamma_q(int(r["nharm"]), float(r["power"]))  # false-alarm probability: smaller = stronger
    best = min(c, key=sig)
    assert (int(best["nharm"]), int(best["col"]), int(best["zi"])) == (8, r0 * nh - 1, 8 + z0 * nh)


@pytest.mark.parametrize("beta", [0.0, 0.004, -0.3, 0.49])
def test_resample_is_bit_exact(emu, beta):
    N = 1 << 13
    x = synth.make_series(N, 31)
    plan = emu.Plan(N, 0.0, 2.0, 2, 2048, quad_points=64)
    assert np.array_equal(plan.resample(x, beta), oracle.resample(x, beta))
    plan.close()


def test_time_domain_trial_end_to_end(emu):
    """PAPER.md:17 through the CUDA path: resample at beta = z/(2 r0), spectrum, |S|^2 by the z_max = 0 plan
    (one delta template), candidates -- the accelerated sinusoid comes back as a tone at r0."""
    N, r0, z = 1 << 14, 1500, 12.0
    x = synth.make_series(N, 32, [synth.Signal(0.2, r0, z, 0.3)])
    plan = emu.Plan(N, 0.0, 2.0, 2, 2048, quad_points=64)
    y = plan.resample(x, z / (2.0 * r0))
    assert np.array_equal(y, oracle.resample(x, z / (2.0 * r0)))
    d_S, _ = plan.spectrum(y)
    d_P, d_c, d_n = plan.correlate(d_S, True, 40.0, 64)
    S_ref, _ = oracle.spectrum(y)
    power_ok(d_P.np()[0, 0], np.abs(S_ref) ** 2)                      # the delta template: plane row = |S|^2
    c = d_c.np()[0, :int(d_n.np()[0])]
    assert len(c) >= 1 and int(c[np.argmax(c["power"])]["col"]) == r0 - 1
    d_S0, _ = plan.spectrum(x)                                        # without the resampling the tone is smeared
    d_P0, _, _ = plan.correlate(d_S0, True)
    assert d_P0.np().max() < 0.5 * d_P.np().max()
    plan.close()


def test_correlate_variants_agree(emu):
    """The tuning keys (FDAS_OPT_TUNE_*) change instruction selection and launch geometry only: the packed f32x2
    butterflies give the scalar ones' plane bit for bit, the number of template chunks per segment does not
    matter, and the harmonic sum does not depend on its sector count, warps per CTA or tile width."""
    cfg = synth.small_config(1 << 13, 12.0, 2.0, 256, 2048, n_sig=2, index=7, amp=0.2)
    plan = emu.Plan(cfg.n_samples, cfg.z_max, cfg.dz, cfg.width, cfg.seg_len, quad_points=2048)
    d_S, _ = plan.spectrum(cfg.series())
    planes = {}
    for name, opts in (("packed", {}), ("scalar", {fdas.FDAS_OPT_TUNE_SCALAR: 1}), ("one_chunk", {fdas.FDAS_OPT_TUNE_T_CHUNKS: 1}),
                       ("five_chunks", {fdas.FDAS_OPT_TUNE_T_CHUNKS: 5}), ("staged", {fdas.FDAS_OPT_TUNE_STAGE_TEMPLATES: 1}),
                       ("staged_one_chunk", {fdas.FDAS_OPT_TUNE_STAGE_TEMPLATES: 1, fdas.FDAS_OPT_TUNE_T_CHUNKS: 1})):
        for k, v in opts.items():
            fdas.fdas_plan_set_option(plan.handle, k, v)
        try:
            d_P = plan.correlate(d_S, True)[0]                        # keep the buffer alive while it is copied
            planes[name] = d_P.np().copy()
        finally:
            for k in opts:
                fdas.fdas_plan_set_option(plan.handle, k, 0)
    for other in ("scalar", "one_chunk", "five_chunks", "staged", "staged_one_chunk"):
        assert np.array_equal(planes["packed"], planes[other]), other
    thr = oracle.thresholds(16, 1e-3)
    lists = []
    for opts in ({fdas.FDAS_OPT_TUNE_HS_SECTORS: 1}, {}, {fdas.FDAS_OPT_TUNE_HS_SECTORS: 7},
                 {fdas.FDAS_OPT_TUNE_HS_ROWS: 8}, {fdas.FDAS_OPT_TUNE_HS_VARIANT: 1}):
        for k, v in opts.items():
            fdas.fdas_plan_set_option(plan.handle, k, v)
        try:
            c, n = plan.harmsum(E.to_dev(planes["packed"][0]), 16, thr, 1 << 16)
        finally:
            for k in opts:
                fdas.fdas_plan_set_option(plan.handle, k, 0)
        lists.append(sorted((int(r["nharm"]), int(r["zi"]), int(r["col"]), float(r["power"])) for r in c))
    assert all(l == lists[0] for l in lists) and len(lists[0]) > 0
    plan.close()


@pytest.mark.parametrize("N,zmax,m,ib,nb", [(1 << 14, 8.0, 64, 1, 1), (1 << 14, 30.0, 256, 0, 2), (1 << 13, 2.0, 1024, 0, 1)])
def test_staged_templates_kernel(emu, N, zmax, m, ib, nb):
    """k_correlate_2048_staged (four segments per CTA share every template spectrum through a bulk-copy ring,
    FDAS_OPT_TUNE_STAGE_TEMPLATES): plane bit for bit the default kernel's, candidates identical; 5 segments (a
    last CTA with idle groups), interbinning, a batch, one and several template chunks, a ragged last segment."""
    cfg = synth.small_config(N, zmax, 2.0, m, 2048, interbin=ib, n_dm=nb, n_sig=2, index=51, amp=0.2)
    xs = np.stack([cfg.series(d) for d in range(nb)])
    plan = emu.Plan(N, zmax, 2.0, m, 2048, interbin=ib, max_batch=nb, quad_points=512)
    d_S, _ = plan.spectrum(xs)
    out = {}
    for staged in (0, 1):
        fdas.fdas_plan_set_option(plan.handle, fdas.FDAS_OPT_TUNE_STAGE_TEMPLATES, staged)
        d_P, d_c, d_n = plan.correlate(d_S, True, 12.0, 1 << 12)
        out[staged] = (d_P.np().copy(), [cset(d_c.np()[b, :int(d_n.np()[b])]) for b in range(nb)])
        _, d_c, d_n = plan.correlate(d_S, False, 12.0, 1 << 12)           # fused mode: plane not stored
        assert [cset(d_c.np()[b, :int(d_n.np()[b])]) for b in range(nb)] == out[staged][1]
    assert np.array_equal(out[0][0], out[1][0]) and out[0][1] == out[1][1] and sum(len(c) for c in out[0][1]) > 0
    assert fdas.fdas_plan_status(plan.handle) == 0
    plan.close()


def test_plane_offset_by_four_bytes(emu):
    """include/fdas.h promises that fdas_candidates and fdas_harmsum accept a plane that is only 4-byte aligned
    (k_candidates once took its 16-byte loads from the row offset alone)."""
    N = 1 << 12
    plan = emu.Plan(N, 4.0, 2.0, 16, 256, quad_points=64)
    n_z, n_cols = plan.info.n_z, plan.info.n_cols
    rng = np.random.default_rng(5)
    P = rng.exponential(1.0, size=(n_z, n_cols)).astype(np.float32)
    buf = E.DevBuf(n_z * n_cols + 1, np.float32)
    buf.np()[1:] = P.ravel()

    class Shifted:
        def data_ptr(self):
            return buf.ptr + 4

    c, n = plan.candidates(Shifted(), 6.0, 1 << 14)
    assert n == int((P > 6.0).sum()) and cset(c) == cset(oracle.candidates(P.astype(np.float64), 6.0))
    thr = oracle.thresholds(16, 1e-3)
    c, n = plan.harmsum(Shifted(), 16, thr, 1 << 16)
    thr32 = thr.astype(np.float32)
    cand_ok(c, oracle.harmsum(P.astype(np.float64), 16, thr, bin0=1), lambda h: float(thr32[int(h).bit_length() - 1]))
    plan.close()


def test_b200_geometry(monkeypatch):
    """The persistent harmonic-sum grid and the batched fused-threshold grid at the REAL device geometry
    (148 SMs x the occupancy ptxas gives: 2 CTAs of 128 threads for k_harmsum<5,2,2>), not the 3 x 2 pretend
    device of the other tests: the item arithmetic (sector -> item ranges, items per CTA <= 1 for most CTAs)."""
    monkeypatch.setenv("EMU_SMS", "148")
    monkeypatch.setenv("EMU_CTAS_PER_SM", "2")
    for align in ("end", "start"):
        monkeypatch.setenv("EMU_ALIGN", align)
        N = 1 << 16
        plan = E.Plan(N, 16.0, 2.0, 16, 256, quad_points=64)
        rng = np.random.default_rng(11)
        P = rng.exponential(1.0, size=(plan.info.n_z, plan.info.n_cols)).astype(np.float32)
        P[3, 20000] = 60.0
        thr = oracle.thresholds(16, 1e-4)
        c, n = plan.harmsum(E.to_dev(P), 16, thr, 1 << 16)
        thr32 = thr.astype(np.float32)
        cand_ok(c, oracle.harmsum(P.astype(np.float64), 16, thr, bin0=1), lambda h: float(thr32[int(h).bit_length() - 1]))
        plan.close()
        small = synth.small_config(1 << 13, 4.0, 2.0, 64, 2048, n_dm=64, n_sig=1, index=35, amp=0.3)   # config-3 shape: 64 DMs
        xs = np.stack([small.series(d) for d in range(64)])
        plan = E.Plan(1 << 13, 4.0, 2.0, 64, 2048, max_batch=64, quad_points=512)
        d_S, _ = plan.spectrum(xs)
        _, d_c, d_n = plan.correlate(d_S, False, 12.0, 1 << 10)
        T = oracle.templates(4.0, 2.0, 64)
        for d in (0, 17, 63):
            S, _ = oracle.spectrum(xs[d])
            cand_ok(d_c.np()[d, :int(d_n.np()[d])], oracle.candidates(oracle.correlate_direct(S, T), 12.0), lambda h: 12.0)
        plan.close()


def test_fused_batch(emu):
    small = synth.small_config(1 << 13, 8.0, 2.0, 64, 2048, n_dm=5, n_sig=1, index=33, amp=0.3)
    xs = np.stack([small.series(d) for d in range(5)])
    plan = emu.Plan(1 << 13, 8.0, 2.0, 64, 2048, max_batch=5, quad_points=2048)
    d_S, _ = plan.spectrum(xs)
    _, d_c, d_n = plan.correlate(d_S, False, 12.0, 1 << 10)
    T = oracle.templates(8.0, 2.0, 64)
    for d in range(5):
        S, _ = oracle.spectrum(xs[d])
        c_ref = oracle.candidates(oracle.correlate_direct(S, T), 12.0)
        cand_ok(d_c.np()[d, :int(d_n.np()[d])], c_ref, lambda h: 12.0)
    plan.close()


def test_search_host(emu):
    N = 1 << 13
    cfg = synth.small_config(N, 8.0, 2.0, 64, 2048, n_sig=2, index=41, amp=0.3)
    x = cfg.series()
    plan = emu.Plan(N, 8.0, 2.0, 64, 2048, quad_points=2048)
    thr = fdas.thresholds(8, 1e-3)
    h_c, h_n = fdas.fdas_search_host(plan.handle, x.reshape(1, -1), 8, thr, 1 << 14)
    d_S, _ = plan.spectrum(x)
    d_P, _, _ = plan.correlate(d_S, True)
    c, n = plan.harmsum(d_P, 8, thr, 1 << 14)
    assert int(h_n[0]) == n and n > 0 and cset(h_c[0, :n]) == cset(c)
    xs = np.stack([x, x[::-1].copy(), x])                             # batch larger than MAX_BATCH = 1
    h_c, h_n = fdas.fdas_search_host(plan.handle, xs, 0, np.array([12.0]), 1 << 10)
    c1, n1 = plan.candidates(d_P, 12.0, 1 << 10)
    assert h_n[0] == h_n[2] == n1 and cset(h_c[0, :n1]) == cset(h_c[2, :n1]) == cset(c1)
    h_c, h_n = fdas.fdas_search_host(plan.handle, xs, 4, fdas.thresholds(4, 1e-3), 1 << 14)
    assert h_n[0] == h_n[2] and cset(h_c[0, :h_n[0]]) == cset(h_c[2, :h_n[2]])
    plan.close()


def test_the_emulator_catches_out_of_bounds_and_misaligned_accesses():
    """The harness itself: a plane buffer that is too short, or a misaligned one, must stop the run (guard page:
    exit code 99 with the kernel named; alignment sanitizer: abort) -- otherwise the tests above prove nothing."""
    import subprocess
    prog = r'''
import sys, numpy as np
sys.path.insert(0, %r)
from emu import harness as E
plan = E.Plan(1 << 12, 4.0, 2.0, 16, 256, quad_points=64)
n = plan.info.n_z * plan.info.n_cols
mode = sys.argv[1]
if mode == "short":
    buf = E.DevBuf(n - 64, np.float32); buf.np()[...] = 1.0
    class P:                                            # the kernel reads n cells from a buffer of n - 64
        def data_ptr(self): return buf.ptr
    plan.candidates(P(), 0.5, 16)
else:
    d_S, _ = plan.spectrum(np.zeros(1 << 12, np.float32))
    buf = E.DevBuf(n + 4, np.float32)
    class P:
        def data_ptr(self): return buf.ptr + 4          # 4-byte offset: the boundary must refuse it
    try:
        E.fdas.fdas_correlate(plan.handle, d_S, 1, P(), 0.0, None, None, 0)
    except E.fdas.FdasError as e:
        sys.exit(0 if e.code == E.fdas.FDAS_E_INVALID else 3)
    sys.exit(4)
''' % os.path.dirname(os.path.abspath(__file__))
    short = subprocess.run([sys.executable, "-c", prog, "short"], capture_output=True, text=True, timeout=300)
    assert short.returncode == 99 and "illegal access" in short.stderr and "k_candidates" in short.stderr, short.stderr[-500:]
    mis = subprocess.run([sys.executable, "-c", prog, "misaligned"], capture_output=True, text=True, timeout=300)
    assert mis.returncode == 0, mis.stderr[-500:]


def test_the_emulator_models_the_asynchronous_copies():
    """The emulator's model of mbarriers and TMA copies (tests/emu/emu_tma.h), tried on small kernels that use them
    correctly and incorrectly (tests/emu/selftest_tma.cpp): a read before the wait sees poison, a byte count that
    does not match is a reported deadlock, a store that is not waited for, a misaligned box buffer and a source
    buffer reused too early are all caught.  Without this the TMA-staged kernels' emulator runs would prove little."""
    import subprocess
    prog = r'''
import ctypes, sys
sys.path.insert(0, %r)
from emu import build
L = ctypes.CDLL(build.build())
sys.exit(10 + L.emu_selftest_tma(int(sys.argv[1])))
''' % os.path.dirname(os.path.abspath(__file__))
    env = dict(os.environ, EMU_ORDER="fwd", EMU_THREADS="1")
    def run(mode):
        return subprocess.run([sys.executable, "-c", prog, str(mode)], capture_output=True, text=True, timeout=300, env=env)
    assert run(0).returncode == 10                                      # correct use: output right
    assert run(1).returncode == 11                                      # early read saw NaN poison
    r = run(2)
    assert r.returncode not in (10, 11) and "mbarrier wait can never be satisfied" in r.stderr, r.stderr[-300:]
    r = run(3)
    assert r.returncode not in (10, 11) and "not committed and waited for" in r.stderr, r.stderr[-300:]
    r = run(4)
    assert r.returncode not in (10, 11) and "not aligned" in r.stderr, r.stderr[-300:]
    assert run(5).returncode == 11                                      # buffer reused too early: output corrupted


def test_search_host_stream_ordering(tmp_path):
    """fdas_search_host overlaps the copy of series c+1 with the kernels of series c on three streams; the emulator
    runs everything synchronously, so the ORDER the library asks for is checked instead: every stream and event
    call is logged (EMU_STREAM_TRACE), the happens-before graph is rebuilt from stream order, record -> wait pairs
    and host synchronisations, and every buffer hazard of the pipeline must be ordered by it:
    the copy into a series buffer after the spectrum kernels that last read it, those kernels after the copy, the
    counts and candidate copies after the harmonic sum that wrote them, and nothing outstanding at return."""
    import subprocess
    trace = str(tmp_path / "trace.txt")
    prog = r'''
import os, sys, numpy as np
sys.path.insert(0, %r); sys.path.insert(0, %r)
from paper_1511_07343_b200 import synth
from emu import harness as E
N = 1 << 13
x = synth.small_config(N, 8.0, 2.0, 64, 2048, n_sig=2, index=41, amp=0.3).series()
plan = E.Plan(N, 8.0, 2.0, 64, 2048, quad_points=512)
open(os.environ["EMU_STREAM_TRACE"], "w").close()                    # drop the plan's own operations
h_c, h_n = E.fdas.fdas_search_host(plan.handle, np.stack([x] * 6), 4, E.fdas.thresholds(4, 1e-3), 1 << 12)
assert len(set(h_n.tolist())) == 1 and h_n[0] > 0
''' % (ROOT_DIR, os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, EMU_STREAM_TRACE=trace)
    r = subprocess.run([sys.executable, "-c", prog], capture_output=True, text=True, timeout=600, env=env)
    assert r.returncode == 0, r.stderr[-800:]
    ops = [l.split() for l in open(trace) if l.strip()]
    n = len(ops)
    anc = [0] * n                                    # bitset of the operations that happen before operation i
    last_on_stream, last_record, host_before = {}, {}, 0
    for i, o in enumerate(ops):
        kind, stream = o[0], o[1]
        before = host_before                          # whatever the host has synchronised with
        if kind in ("memcpy", "memset", "launch", "record", "wait"):
            j = last_on_stream.get(stream)
            if j is not None:
                before |= anc[j] | (1 << j)
            last_on_stream[stream] = i
        if kind == "wait" and o[2] in last_record:
            j = last_record[o[2]]
            before |= anc[j] | (1 << j)
        if kind == "record":
            last_record[o[2]] = i
        anc[i] = before
        if kind == "eventsync" and o[2] in last_record:
            j = last_record[o[2]]
            host_before |= anc[j] | (1 << j)
        if kind == "streamsync" and stream in last_on_stream:
            j = last_on_stream[stream]
            host_before |= anc[j] | (1 << j)
    hb = lambda a, b: bool(anc[b] >> a & 1)
    h2d = [i for i, o in enumerate(ops) if o[0] == "memcpy" and int(o[4]) == (1 << 13) * 4]
    spec_first = [i for i, o in enumerate(ops) if o[0] == "launch" and o[2] == "k_spec_cols"]
    spec_last = [i for i, o in enumerate(ops) if o[0] == "launch" and o[2] == "k_spec_rows"]
    harm = [i for i, o in enumerate(ops) if o[0] == "launch" and o[2] == "k_harmsum"]
    counts = [i for i, o in enumerate(ops) if o[0] == "memcpy" and int(o[4]) == 4]
    cands = [i for i, o in enumerate(ops) if o[0] == "memcpy" and o[1] not in (ops[spec_first[0]][1], ops[h2d[0]][1])]
    assert len(h2d) == len(spec_first) == len(spec_last) == len(harm) == len(counts) == len(cands) == 6
    assert len({ops[i][2] for i in h2d}) == 2                              # two series buffers, alternating
    for c in range(6):
        assert ops[h2d[c]][2] == ops[h2d[c % 2]][2]
        assert hb(h2d[c], spec_first[c]), "spectrum %d may start before its series has arrived" % c
        if c >= 2:
            assert hb(spec_last[c - 2], h2d[c]), "series %d may overwrite a buffer the spectrum of %d still reads" % (c, c - 2)
        if c + 1 < 6:
            assert not hb(harm[c], h2d[c + 1]), "the copy of series %d is serialised behind the kernels of %d: no overlap" % (c + 1, c)
        assert hb(harm[c], counts[c]) and hb(counts[c], cands[c]), "candidates of %d copied before they are complete" % c
    assert all(anc[n - 1] >> i & 1 or i == n - 1 for i in range(n - 1)) or ops[-1][0] == "streamsync"
    final = host_before
    assert all(final >> i & 1 for i in h2d + harm + counts + cands), "work outstanding when fdas_search_host returns"
