"""N > 1 path on the CPU: two gloo ranks shard a batch of DM trials (dm mod world), each searches its
shard with the kernels running in the host emulator (tests/emu), rank 0 gathers the candidate lists;
the result must equal a single-process search of all trials and the oracle's candidates."""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_1511_07343_b200 import shard, synth

HERE = os.path.dirname(os.path.abspath(__file__))
N, ZMAX, M, L, N_DM, THR = 1 << 13, 8.0, 64, 2048, 5, 12.0


def _series():
    cfg = synth.small_config(N, ZMAX, 2.0, M, L, n_dm=N_DM, n_sig=1, index=33, amp=0.3)
    return np.stack([cfg.series(d) for d in range(N_DM)])


def _search(xs, dms):
    sys.path.insert(0, HERE)
    from emu import harness as E
    plan = E.Plan(N, ZMAX, 2.0, M, L, max_batch=max(1, len(dms)), quad_points=2048)
    out = {}
    if dms:
        h_c, h_n = E.fdas.fdas_search_host(plan.handle, xs[dms], 0, np.array([THR]), 1 << 10)
        out = {dm: h_c[i, :h_n[i]].copy() for i, dm in enumerate(dms)}
    plan.close()
    return out


def _rank_main(rank, world, port, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), EMU_THREADS="2")
    dist.init_process_group("gloo", rank=rank, world_size=world)
    local = _search(_series(), shard.dm_shard(N_DM, rank, world))
    merged = shard.gather_candidates(local, N_DM)
    if rank == 0:
        q.put({dm: [(int(r["zi"]), int(r["col"])) for r in c] for dm, c in merged.items()})
    else:
        assert merged is None
    dist.barrier()
    dist.destroy_process_group()


def test_dm_shard_partition():
    for world in (1, 2, 3, 8):
        parts = [shard.dm_shard(64, r, world) for r in range(world)]
        assert sorted(sum(parts, [])) == list(range(64))
        assert max(map(len, parts)) - min(map(len, parts)) <= 1
    with pytest.raises(ValueError):
        shard.dm_shard(4, 2, 2)


def test_two_rank_search_equals_single_process():
    import oracle
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_rank_main, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=300)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    xs = _series()
    single = _search(xs, list(range(N_DM)))
    T = oracle.templates(ZMAX, 2.0, M)
    n_total = 0
    for dm in range(N_DM):
        one = sorted((int(r["zi"]), int(r["col"])) for r in single[dm])
        assert sorted(got[dm]) == one
        S, _ = oracle.spectrum(xs[dm])
        ref = oracle.candidates(oracle.correlate_direct(S, T), THR)
        assert set(one) == {(int(r["zi"]), int(r["col"])) for r in ref}
        n_total += len(one)
    assert n_total > 0
