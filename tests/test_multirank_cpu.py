"""The N>1 path of bench.py on CPU: world_size 2 over gloo (rendezvous on 127.0.0.1).

The path shards over SEEDS (field replicated, no data-path collective); the
only cross-rank traffic is bench.Reducer (barrier, MAX of the timed region, SUM of the work
counters).  Each rank draws its own shard (bench.shard_seed), traces it with the CPU oracle as a
stand-in for the per-rank work, and the whole-job value must equal the hand-computed aggregate.
"""
import os
import socket
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank),
                      WORLD_SIZE=str(world), OMP_NUM_THREADS="2")
    import torch.distributed as dist
    import bench
    import oracle
    import workloads as wl
    dist.init_process_group("gloo", rank=rank, world_size=world)
    red = bench.Reducer(world, "cpu")
    fld = wl.turb_field_cpu(24, 16, 1.0, 4.0)
    seeds = wl.seeds_uniform(bench.shard_seed(rank), 512, [23.0] * 3)
    g = oracle.grid(fld.data, fld.dims, fld.origin, fld.spacing)
    r = oracle.streamlines(g, seeds, oracle.params(integrator=0, h=0.25, max_steps=200, vmin=1e-6,
                                                   capacity=8, stride=32), "f32")
    attempts = int(r.totals[0])
    ms = 10.0 * (rank + 1)                      # rank 1 is the slow one
    red.barrier()
    value, total_ms, job_attempts = bench.job_value(attempts, 3, ms, red)
    q.put((rank, attempts, value, total_ms, job_attempts, seeds[:2].tolist()))
    dist.destroy_process_group()


def test_world2_seed_sharding_and_reduction():
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, a0, v0, t0, j0, s0), (r1, a1, v1, t1, j1, s1) = out
    assert s0 != s1, "ranks must trace different seeds"
    assert a0 > 0 and a1 > 0
    assert t0 == t1 == 20.0, "timed region = MAX over ranks"
    assert j0 == j1 == float(a0 + a1), "work = SUM over ranks"
    assert v0 == v1 == pytest.approx((a0 + a1) * 3 / 20e-3)


def test_rank0_shard_is_baseline_seed():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.shard_seed(0) == 42
    assert len({bench.shard_seed(r) for r in range(8)}) == 8
