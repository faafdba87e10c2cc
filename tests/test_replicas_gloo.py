"""Multi-GPU is "replicas only": no data-path collective.  The rank plumbing of bench.py
(rank-specific seeds, MAX over ranks of the device time, aggregate value) is covered here on CPU with gloo, world 2."""
import os
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp  # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    import bench
    from paper_2302_02474_b200 import inputs
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        ms_local = 10.0 + 5.0 * rank                         # rank 1 is the slow replica
        ms = bench.max_over_ranks(dist, ms_local, "cpu")
        cfg = inputs.C1
        in_seed, ph_seed = bench.replica_seeds(cfg, rank)
        st = inputs.make_state(cfg, seed=in_seed)
        out.put((rank, ms, bench.aggregate_value(cfg.n, 4, world, ms), in_seed, ph_seed, float(st.x.sum())))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_replicas_max_time_and_independent_inputs():
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(out.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ms0, v0, s0, k0, x0), (r1, ms1, v1, s1, k1, x1) = res
    assert ms0 == ms1 == 15.0                                # both ranks see the slowest replica's time
    assert v0 == v1 == pytest.approx(2 * 2000 * 4 / 15e-3)   # whole-job aggregate, weak scaling
    assert s0 != s1 and k0 != k1 and x0 != x1                # independent replicas: different inputs and noise keys


def test_single_process_path_needs_no_collective():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(None, 3.5, "cpu") == 3.5
    assert bench.aggregate_value(100, 10, 1, 2.0) == pytest.approx(100 * 10 / 2e-3)
