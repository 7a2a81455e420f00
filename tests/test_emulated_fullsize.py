"""BASELINE.json configs[2] + configs[4] at FULL size (2^23 samples, 85 templates, 16-harmonic sum) through the
emulator, at the B200's geometry (148 SMs x 3 resident CTAs), in the launch configuration bench.py times:
the TMA-staged three-pass spectrum, the fused segment kernel (default and staged variant), the persistent
harmonic sum.  About two minutes on 8 cores; it is the only full-size evidence there is while no GPU answers
(DESIGN.md section 9).  Test infrastructure only (tests/emu/README.md)."""
import os
import sys

import numpy as np
import pytest

import oracle
from paper_1511_07343_b200 import synth

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))


def test_config2_and_config4_at_full_size(monkeypatch):
    monkeypatch.setenv("EMU_SMS", "148")
    monkeypatch.setenv("EMU_CTAS_PER_SM", "3")
    from emu import harness as E
    fdas = E.fdas
    cfg = synth.config(2)
    x = cfg.series()
    plan = E.Plan(cfg.n_samples, cfg.z_max, cfg.dz, cfg.width, cfg.seg_len)
    d_S, d_mu = plan.spectrum(x)
    S_ref, mu = oracle.spectrum(x)
    S = d_S.np()[0]
    S = S[:, 0] + 1j * S[:, 1]
    assert np.sqrt(np.mean(np.abs(S - S_ref) ** 2)) < 5e-7 and abs(float(d_mu.np()[0]) / mu - 1) < 2e-6
    d_P, _, _ = plan.correlate(d_S, True)
    P = d_P.np()[0].copy()
    T = oracle.templates(cfg.z_max, cfg.dz, cfg.width)
    P_ref = oracle.correlate_fft(S_ref, T, cfg.seg_len)
    pmax = float(P_ref.max())
    for zi in range(P.shape[0]):                                      # north_star tolerance, row by row (memory)
        assert not (np.abs(P[zi] - P_ref[zi]) > 1e-4 * pmax + 1e-5 * P_ref[zi]).any(), zi
    del P_ref
    fdas.fdas_plan_set_option(plan.handle, fdas.FDAS_OPT_TUNE_STAGE_TEMPLATES, 1)
    d_P2, _, _ = plan.correlate(d_S, True)
    assert np.array_equal(d_P2.np()[0], P)                            # staged variant: bit for bit
    del d_P2
    fdas.fdas_plan_set_option(plan.handle, fdas.FDAS_OPT_TUNE_STAGE_TEMPLATES, 0)
    thr = oracle.thresholds(16)
    c, n = plan.harmsum(d_P, 16, thr, 1 << 22)
    c_ref = oracle.harmsum(P.astype(np.float64), 16, thr, bin0=1)     # the kernel alone: the same fp32 plane
    key = lambda r: (int(r["nharm"]), int(r["zi"]), int(r["col"]))
    g, r = {key(q) for q in c}, {key(q) for q in c_ref}
    assert n == len(g) and len(r) > 100000
    pw = {key(q): float(q["power"]) for q in c_ref}
    thr32 = thr.astype(np.float32)
    for k in g ^ r:                                                   # only entries within 1e-4 of their threshold may differ
        t = float(thr32[k[0].bit_length() - 1])
        assert k in pw and abs(pw[k] - t) <= 1e-4 * t, k
    assert fdas.fdas_plan_status(plan.handle) == 0
    plan.close()


@pytest.mark.skipif(not os.environ.get("FDAS_EMU_ALL"), reason="a minute of oracle time: run with FDAS_EMU_ALL=1 (profiles/r2_emulator_fullsize.md)")
def test_config1_interbinned_at_full_size(monkeypatch):
    """BASELINE.json configs[1]: 2^20 samples, 101 z x 2 template sets (202 templates, 7 chunks), column interleave."""
    monkeypatch.setenv("EMU_SMS", "148")
    monkeypatch.setenv("EMU_CTAS_PER_SM", "3")
    from emu import harness as E
    cfg = synth.config(1)
    x = cfg.series()
    plan = E.Plan(cfg.n_samples, cfg.z_max, cfg.dz, cfg.width, cfg.seg_len, interbin=1)
    d_S, _ = plan.spectrum(x)
    d_P, d_c, d_n = plan.correlate(d_S, True, 30.0, 1 << 20)
    S, _ = oracle.spectrum(x)
    P_ref = oracle.correlate_fft(S, oracle.templates(cfg.z_max, cfg.dz, cfg.width, 1), cfg.seg_len, interbin=1)
    P = d_P.np()[0]
    assert P.shape == (101, 1 << 20)
    assert not (np.abs(P - P_ref) > 1e-4 * P_ref.max() + 1e-5 * P_ref).any()
    c_ref = oracle.candidates(P_ref, 30.0)
    got = {(int(r["zi"]), int(r["col"])) for r in d_c.np()[0, :int(d_n.np()[0])]}
    assert got == {(int(r["zi"]), int(r["col"])) for r in c_ref} and len(got) > 100
    plan.close()


def test_maximum_series_length(monkeypatch):
    """2^25 samples (the largest the plan accepts): three passes of 256 x 256 x 256, 2^24 columns per row --
    index arithmetic at its limits (k h, plane offsets, twiddle exponents), 3 templates."""
    monkeypatch.setenv("EMU_SMS", "148")
    monkeypatch.setenv("EMU_CTAS_PER_SM", "3")
    from emu import harness as E
    N = 1 << 25
    x = synth.make_series(N, 77, [synth.Signal(0.02, 9.0e6 + 0.25, 1.5, 0.3), synth.Signal(0.02, 1.6e7 - 3.5, -2.0, 1.0)])
    plan = E.Plan(N, 2.0, 2.0, 256, 2048)
    d_S, _ = plan.spectrum(x)
    d_P, d_c, d_n = plan.correlate(d_S, True, 30.0, 1 << 16)
    thr = oracle.thresholds(16)
    c, n = plan.harmsum(d_P, 16, thr, 1 << 20)
    S, _ = oracle.spectrum(x)
    P_ref = oracle.correlate_fft(S, oracle.templates(2.0, 2.0, 256), 2048)
    P = d_P.np()[0]
    assert not (np.abs(P - P_ref) > 1e-4 * P_ref.max() + 1e-5 * P_ref).any()
    assert int(d_n.np()[0]) == len(oracle.candidates(P_ref, 30.0)) > 10
    c_ref = oracle.harmsum(P.astype(np.float64), 16, thr, bin0=1)
    key = lambda r: (int(r["nharm"]), int(r["zi"]), int(r["col"]))
    assert {key(q) for q in c} == {key(q) for q in c_ref} and n == len(c_ref) > 100
    plan.close()
