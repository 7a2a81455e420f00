"""GPU parity, rows a2-a6, a6': fused overlap-save segment kernels at small sizes (see tests/gpu_common.py for the tolerances and the order of the session)."""
import numpy as np
import pytest
import torch

import oracle
from paper_1511_07343_b200 import synth
from gpu_common import assert_cand_parity, assert_power_parity, cand_set, make_plan, run_gpu_plane  # noqa: F401

pytestmark = pytest.mark.gpu


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
