"""Helpers of the `-m gpu` parity tests: the CUDA path (through the C ABI) against the fp64 oracle, element by
element on the same seeded inputs.  Tolerances are BASELINE.json north_star's:
  power:  |P_gpu - P_ref| <= 1e-4*max(P_ref) + 1e-5*P_ref      (max over the plane of that series; for harmonic
                                                                  sums, max over that stage: SURVEY G20)
  candidate (col, zi, nharm) sets identical except entries within 1e-4 relative of the threshold.

Order of the GPU session: the modules are named so that `pytest -m gpu -x` runs every kernel
family at config-0 size first (test_gpu_0_* ... test_gpu_4_*), then the strict checks of the asynchronous-copy
paths (test_gpu_5_async_copies.py), and the full-size cases (2^20 ... 2^25 samples) last
(test_gpu_9_fullsize.py); the first failure stops the run.
"""
import numpy as np
import torch


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


def assert_cand_parity(c_gpu, c_ref, thr_of_nharm):
    """Sets equal except entries whose (reference) power is within 1e-4 relative of the threshold; powers of the
    common entries within the plane tolerance, with max(P_ref) taken per harmonic stage."""
    g, r = cand_set(c_gpu), cand_set(c_ref)
    assert len(c_gpu) == len(g), "duplicate candidates"
    pw_ref = {(int(x["nharm"]), int(x["zi"]), int(x["col"])): float(x["power"]) for x in c_ref}
    pw_gpu = {(int(x["nharm"]), int(x["zi"]), int(x["col"])): float(x["power"]) for x in c_gpu}
    for key in g ^ r:
        p = pw_ref.get(key, pw_gpu.get(key))
        T = thr_of_nharm(key[0])
        assert abs(p - T) <= 1e-4 * T, "candidate mismatch %s power %g thr %g" % (key, p, T)
    pmax = {}
    for key, p in pw_ref.items():
        pmax[key[0]] = max(pmax.get(key[0], 0.0), p)
    for key in g & r:
        assert abs(pw_gpu[key] - pw_ref[key]) <= 1e-4 * pmax[key[0]] + 1e-5 * pw_ref[key], key


def make_plan(fdas, cfg, max_batch=1):
    return fdas.Plan(cfg.n_samples, cfg.z_max, cfg.dz, cfg.width, cfg.seg_len, interbin=cfg.interbin,
                     max_batch=max_batch)


def run_gpu_plane(fdas, plan, x, thr=None, cap=1 << 16):
    d_x = torch.from_numpy(np.ascontiguousarray(x)).cuda().view(1, -1)
    d_S, _ = plan.spectrum(d_x)
    d_P = plan.empty_plane(1)
    cands = plan.empty_cands(cap) if thr is not None else None
    plan.correlate(d_S, d_P, threshold=thr or 0.0, cands=cands, capacity=cap if thr is not None else 0)
    torch.cuda.synchronize()
    c = fdas.cands_to_numpy(*cands) if thr is not None else None
    return d_P[0], c
