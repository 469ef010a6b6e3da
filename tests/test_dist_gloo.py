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


def _comb_worker(rank, world, port, out):
    """Routing of the sharded comb (dist.comb_splits) under gloo: the counts of the two sides agree and the exchanged
    records arrive in slot order.  Records are stood in for by the parents' global indices (no kernels on CPU)."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from oracle import afqmc_oracle as orc
    from paper_1804_03310_b200 import dist as D
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nw = 37
    ok = True
    for seed, u in ((1, 0.0), (2, 0.41), (3, 0.97)):
        rng = np.random.default_rng(seed)
        w_local = rng.random((world, nw)) ** 4
        w_local[1, :20] = 0.0                               # rank 1 is mostly dead: it must be refilled from rank 0
        gathered = [torch.zeros(nw, dtype=torch.float64) for _ in range(world)]
        dist.all_gather(gathered, torch.tensor(w_local[rank]))
        w_all = torch.cat(gathered).numpy()
        parent_all = torch.tensor(orc.o_comb(w_all, u))
        slot_lo, count, send_counts, recv_counts = D.comb_splits(parent_all, nw, world, rank)
        sendbuf = parent_all[slot_lo:slot_lo + count].tolist()   # "records" = the parents' global ids, slot order
        assert all(rank * nw <= p < (rank + 1) * nw for p in sendbuf)
        everyone = [None] * world
        dist.all_gather_object(everyone, (send_counts, sendbuf))
        recv = []
        for s in range(world):
            sc, sb = everyone[s]
            off = sum(sc[:rank])
            ok &= sc[rank] == recv_counts[s]
            recv += sb[off:off + sc[rank]]
        ok &= recv == parent_all[rank * nw:(rank + 1) * nw].tolist()
        ok &= sum(send_counts) == count and sum(recv_counts) == nw
    out[rank] = bool(ok)
    dist.barrier()
    dist.destroy_process_group()


def test_sharded_comb_routing_gloo():
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Manager().dict()
    procs = [ctx.Process(target=_comb_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(180)
        assert p.exitcode == 0
    assert out[0] and out[1]
