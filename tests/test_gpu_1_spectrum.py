"""GPU parity, row a1: real-to-complex FFT + normalisation (k_spec_pass1, k_spec_pass2) (see tests/gpu_common.py for the tolerances and the order of the session)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1511_07343_b200 import synth
from gpu_common import assert_cand_parity, assert_power_parity, cand_set, make_plan, run_gpu_plane  # noqa: F401

pytestmark = pytest.mark.gpu


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
    assert plan.status() & fdas.FDAS_STATUS_COPY_TIMEOUT == 0   # no asynchronous copy timed out


def test_spectrum_paths_agree(fdas):
    """The TMA-staged multi-pass transform (default from 2^13 samples) against the generic two-pass kernels
    (tuning key): same spectrum to rounding, both within 1e-6 rms of the oracle, two and three passes."""
    for log2n in (14, 18):
        N = 1 << log2n
        xs = np.stack([synth.make_series(N, 500 + b) * (1.0 + 0.5 * b) for b in range(2)])
        S = {}
        for generic in (0, 1):
            plan = fdas.Plan(N, 4.0, 2.0, 16, 256, max_batch=2)
            fdas.fdas_plan_set_option(plan.handle, fdas.FDAS_OPT_TUNE_SPEC_GENERIC, generic)
            d_S, d_mu = plan.spectrum(torch.from_numpy(xs).cuda())
            S[generic] = d_S.cpu().numpy()
            assert plan.status() & fdas.FDAS_STATUS_COPY_TIMEOUT == 0
            for b in range(2):
                S_ref, mu = oracle.spectrum(xs[b])
                z = S[generic][b][:, 0] + 1j * S[generic][b][:, 1]
                assert np.sqrt(np.mean(np.abs(z - S_ref) ** 2)) < 1e-6
                assert float(d_mu[b]) == pytest.approx(mu, rel=2e-6)
        assert np.max(np.abs(S[0] - S[1])) < 5e-6


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
