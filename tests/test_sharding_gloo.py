"""N > 1 host logic on CPU: two gloo ranks shard an ensemble by samples (paper_1012_0385_b200.shard), each runs its
block with the global sample index as RNG key, the records are gathered - and equal the single-process ensemble
row for row (no collective on the data path).  The per-rank engine here is the CPU oracle (tests may
use it); on the GPU box bench.py drives the CUDA path with the same first_sample arithmetic."""
import os
import socket

import numpy as np
import pytest

from paper_1012_0385_b200 import shard


def test_shard_samples_partitions_exactly():
    for total in (0, 1, 5, 16, 1024, 1000):
        for world in (1, 2, 3, 8):
            blocks = [shard.shard_samples(total, world, r) for r in range(world)]
            assert blocks[0][0] == 0
            assert sum(c for _, c in blocks) == total
            for (f0, c0), (f1, _) in zip(blocks, blocks[1:]):
                assert f1 == f0 + c0
            assert max(c for _, c in blocks) - min(c for _, c in blocks) <= 1
    assert shard.weak_first_sample(1024, 3) == 3072
    with pytest.raises(ValueError):
        shard.shard_samples(4, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, total, L, n_mcs, times, q):
    import torch.distributed as dist
    from oracle import kpzref as R
    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        first, count = shard.shard_samples(total, world, rank)
        sim = R.KpzRef(L, count, 0.75, 0.25, seed=11, first_sample=first)
        sim.set_record_times(times)
        sim.run(n_mcs)
        rec = sim.roughness()
        local = {"sum_h": rec["sum_h"], "sum_h2": rec["sum_h2"], "t": np.asarray(rec["t"]),
                 "lattice": sim.lattice().T.copy()}         # samples on the last axis
        full = shard.gather_records(local)
        dist.barrier()
        if rank == 0:
            q.put({k: np.asarray(v) for k, v in full.items()})
    finally:
        dist.destroy_process_group()


def test_two_gloo_ranks_reproduce_the_single_process_ensemble():
    import torch.multiprocessing as mp
    from oracle import build as oracle_build
    from oracle import kpzref as R
    oracle_build.build()
    total, L, n_mcs, times = 5, 128, 30, [1, 7, 30]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, total, L, n_mcs, times, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    ref = R.KpzRef(L, total, 0.75, 0.25, seed=11)
    ref.set_record_times(times)
    ref.run(n_mcs)
    rr = ref.roughness()
    assert list(got["t"]) == times
    assert np.array_equal(got["sum_h"], rr["sum_h"]) and np.array_equal(got["sum_h2"], rr["sum_h2"])
    assert np.array_equal(got["lattice"].T, ref.lattice())
    # the blocks really differ (distinct global sample indices), so the agreement is not trivial
    assert len({tuple(row) for row in ref.lattice()}) == total
