"""The path shards by walker with no data-path collective.  These world_size-2 gloo tests
cover the host logic bench.py runs for N > 1 (every function of sharding.py): rank -> ensemble assignment, max-over-ranks
timing, whole-job aggregation on rank 0."""
import os
import socket
import sys

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.distributed as dist          # noqa: E402
import torch.multiprocessing as mp        # noqa: E402

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    from paper_2311_17174_b200 import sharding, workloads as W
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = W.scaled(W.CONFIGS[1], K=6, N=1 << 10)
    # weak scaling: every rank owns a full ensemble, drawn from its own seed
    rcfg = sharding.rank_config(cfg, rank)
    P = W.draw_params(rcfg)
    # timing: the slowest rank defines the step time
    t = sharding.max_over_ranks(10.0 + rank, world)
    total = sharding.whole_job_value(cfg.K * cfg.N, 3, t, world)
    firsts = [None] * world
    dist.all_gather_object(firsts, float(P[0, 0]))
    if rank == 0:
        out.put(dict(t=t, total=total, firsts=firsts, seed0=rcfg.seed))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_shard_time_and_aggregate():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res["t"] == 11.0                                   # max over ranks
    assert res["total"] == pytest.approx(2 * 6 * 1024 * 3 / 11.0e-3)
    assert res["firsts"][0] != res["firsts"][1]               # distinct ensembles per rank
    assert res["seed0"] == 1                                  # rank 0 keeps the config's seed
