"""world_size-2 gloo test of the multi-GPU host logic used by bench.py (replicas, max-over-ranks timing)."""
import os
import socket

import pytest


def _worker(rank, world, port, out):
    import torch.distributed as dist
    from paper_1804_03310_b200 import dist as D
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    t = D.max_over_ranks(1.0 + rank)            # rank 1 is the slow one
    out[rank] = (t, D.rank_seed(1000, rank), D.whole_job_rate(2048 * 4, world, t))
    dist.barrier()
    dist.destroy_process_group()


def test_replicas_max_time_and_seeds():
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Manager().dict()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    assert out[0][0] == out[1][0] == 2.0                     # every rank sees the max
    assert out[0][1] != out[1][1]                            # independent field streams
    assert out[0][2] == pytest.approx(2 * 2048 * 4 / 2.0)    # whole-job aggregate over both replicas


def test_single_process_is_identity():
    from paper_1804_03310_b200 import dist as D
    assert D.max_over_ranks(3.5) == 3.5
