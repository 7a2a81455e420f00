"""GPU parity, the asynchronous-copy (TMA) paths STRICTLY: the modules before this one accept a plan whose init-stage
self-test fell back to the generic spectrum kernels (they check results, and that no copy wait timed out); this one
requires the TMA-staged passes to be the ones in use, and runs the opt-in staged segment kernel.  It sits after the
small modules and before the full-size ones (see tests/gpu_common.py)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1511_07343_b200 import synth
from gpu_common import make_plan  # noqa: F401

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("log2n", [13, 16, 18, 23])
def test_tma_spectrum_is_in_use_and_right(fdas, log2n):
    N = 1 << log2n
    x = synth.make_series(N, 4300 + log2n, [synth.Signal(0.1, N / 8 + 0.3, 2.0, 0.5)])
    plan = fdas.Plan(N, 4.0, 2.0, 16, 256)
    assert plan.status() == 0, "the TMA-staged spectrum passes failed their init-stage self-test (fallback in use)"
    d_S, d_mu = plan.spectrum(torch.from_numpy(x).cuda().view(1, -1))
    assert plan.status() == 0
    S = d_S.cpu().numpy()[0]
    S_ref, mu = oracle.spectrum(x)
    assert np.sqrt(np.mean(np.abs(S[:, 0] + 1j * S[:, 1] - S_ref) ** 2)) < 1e-6
    assert float(d_mu[0]) == pytest.approx(mu, rel=2e-6)


def test_staged_segment_kernel(fdas):
    """FDAS_OPT_TUNE_STAGE_TEMPLATES: four segments per CTA share each template spectrum through a bulk-copy ring;
    plane and candidates bit for bit the default kernel's (5 segments: an idle group; a batch of 2; fused mode)."""
    cfg = synth.small_config(1 << 14, 30.0, 2.0, 256, 2048, n_dm=2, n_sig=2, index=51, amp=0.2)
    xs = np.stack([cfg.series(d) for d in range(2)])
    plan = make_plan(fdas, cfg, max_batch=2)
    d_S, _ = plan.spectrum(torch.from_numpy(xs).cuda())
    out = {}
    for staged in (0, 1):
        fdas.fdas_plan_set_option(plan.handle, fdas.FDAS_OPT_TUNE_STAGE_TEMPLATES, staged)
        d_P = plan.empty_plane(2)
        cands = plan.empty_cands(1 << 12, n_batch=2)
        plan.correlate(d_S, d_P, threshold=12.0, cands=cands, capacity=1 << 12)
        fused = plan.empty_cands(1 << 12, n_batch=2)
        plan.correlate(d_S, None, threshold=12.0, cands=fused, capacity=1 << 12)
        sets = []
        for b in range(2):
            a = {(int(r["zi"]), int(r["col"])) for r in fdas.cands_to_numpy(cands[0], cands[1], b)}
            assert a == {(int(r["zi"]), int(r["col"])) for r in fdas.cands_to_numpy(fused[0], fused[1], b)}
            sets.append(a)
        out[staged] = (d_P.cpu().numpy(), sets)
    assert np.array_equal(out[0][0], out[1][0]) and out[0][1] == out[1][1] and sum(len(s) for s in out[0][1]) > 0
    assert plan.status() == 0
