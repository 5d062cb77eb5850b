"""Host-side logic of bench.py's N > 1 path (replicas only: no data-path collective),
on CPU with the gloo backend, world size 2: per-rank seeding gives disjoint batches, the whole-job time is the
max over ranks, the whole-job value aggregates all ranks."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def _worker(rank, world, port, q):
    import bench
    import workloads as wl
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 10.0 + 5.0 * rank                        # rank 1 is the slow one
        ms = bench.max_over_ranks(ms_local, dist, torch.device("cpu"))
        cfg = wl.get_config("cfg2_small")
        h = bench.host_inputs(cfg, seed=bench.shard_seed(rank, 0))
        q.put((rank, ms, float(h["K"].sum()), bench.whole_job_value(world, 100, ms)))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_replicas_time_is_max_over_ranks_and_batches_differ():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ms0, k0, v0), (r1, ms1, k1, v1) = res
    assert ms0 == ms1 == 15.0                               # max over ranks, identical on every rank
    assert k0 != k1                                         # different seeds -> different users per rank
    assert np.isclose(v0, 2 * 100 / 15e-3) and v0 == v1     # whole-job SIDs/s counts both ranks


def test_single_rank_passthrough_and_seed_layout():
    import bench
    assert bench.max_over_ranks(3.5) == 3.5
    assert bench.shard_seed(0, 0) == 0 and bench.shard_seed(2, 3) == 2003
    assert len({bench.shard_seed(r, s) for r in range(8) for s in range(16)}) == 128
