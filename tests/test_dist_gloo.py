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


class _StubCtx:
    """Stands in for AfqmcContext on CPU: every ABI call run_sharded makes is recorded, and the ones whose output steers the
    control flow (energies, weights, sums, the comb) are filled with simple deterministic numbers.  Walker 'records' are one
    float64 per walker (its global id of origin), so the routing through all_to_all_single can be checked exactly."""

    def __init__(self, nw, rank, world):
        import types
        self.params = types.SimpleNamespace(n_walkers=nw)
        self.rank, self.world, self.nw = rank, world, nw
        self.calls, self.steps_done, self.stream = [], 0, None
        self.afqmc_comb_record_bytes = 8

    def afqmc_run(self, phi, weight, ovlp, theta, fb, x, n, ee, oe, pc, u, eloc, wm, parents, flags):
        import torch
        assert pc == 0 and u is None and x.shape[0] == n            # segments never comb inside afqmc_run
        self.calls.append(("run", self.steps_done, n))
        for j in range(n // ee if ee else 0):
            step = self.steps_done + (j + 1) * ee
            eloc[j] = torch.full((self.nw,), complex(-1.0 - 0.01 * step, 0.5), dtype=torch.complex128)
            wm[j] = weight                                           # weights at the measurement
        self.steps_done += n

    def afqmc_mixed_sums(self, w, e, out3):
        out3[0] = w.sum(); out3[1] = (w * e.real).sum(); out3[2] = (w * e.imag).sum()

    def afqmc_mixed_energy(self, sums, m, emix):
        for k in range(m):
            emix[k] = complex(float(sums[k, 1] / sums[k, 0]), float(sums[k, 2] / sums[k, 0]))

    def afqmc_comb_map(self, w_all, u, cum, parent_all, w_new):
        import numpy as np
        import torch
        from oracle import afqmc_oracle as orc
        self.calls.append(("comb", float(u), float(w_all.sum())))
        parent_all.copy_(torch.tensor(orc.o_comb(w_all.numpy(), u), dtype=torch.int32))
        w_new[0] = float(np.cumsum(w_all.numpy())[-1]) / w_all.numel()

    def afqmc_comb_pack(self, phi, ovlp, theta, fb, parent_all, slot_lo, count, first_local, sendbuf):
        import torch
        ids = parent_all[slot_lo:slot_lo + count].to(torch.int64) - first_local
        sendbuf.view(torch.float64)[:count] = phi[ids]

    def afqmc_comb_unpack(self, recvbuf, phi, weight, ovlp, theta, fb, w_new):
        phi.copy_(recvbuf.view(torch_f64())[:self.nw])
        weight.fill_(float(w_new[0]))


def torch_f64():
    import torch
    return torch.float64


def _run_sharded_worker(rank, world, port, out):
    """dist.run_sharded's control flow under gloo with a stubbed context: segment boundaries (afqmc_run is called per
    pc_every steps, never with its own comb), us[k] indexing, all-reduce of sums[:m], E_mix identical on both ranks, and
    walkers really crossing ranks in the comb."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from oracle import afqmc_oracle as orc
    from paper_1804_03310_b200 import dist as D
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    nw, ns, ee, oe, pe = 16, 50, 10, 2, 20
    ctx = _StubCtx(nw, rank, world)
    phi = torch.arange(rank * nw, (rank + 1) * nw, dtype=torch.float64)            # "walker" = its global id of origin
    wts = [np.random.default_rng(5 + r).random(nw) ** 3 * (4.0 if r == 0 else 0.25) for r in range(world)]
    weight = torch.tensor(wts[rank])
    z = torch.zeros(nw, dtype=torch.float64)
    x = torch.zeros(ns, nw, 3)
    us = [0.37, 0.81]
    D.COMB_STATS.clear()
    en = D.run_sharded(ctx, phi, weight, z, z, z, x, ns, ee, oe, pe, us=us)
    # expected, from the same stub rules: segments of 20, 20, 10 steps; combs after steps 20 and 40 with us[0], us[1]
    ok = [c for c in ctx.calls if c[0] == "run"] == [("run", 0, 20), ("run", 20, 20), ("run", 40, 10)]
    combs = [c for c in ctx.calls if c[0] == "comb"]
    ok &= [c[1] for c in combs] == us
    w_all = np.concatenate(wts)
    ids = np.arange(world * nw, dtype=np.float64)
    exp_e = []
    for k in range(2):
        for j in (1, 2):
            step = 20 * k + 10 * j
            exp_e.append(complex(-1.0 - 0.01 * step, 0.5))              # every walker has the same E_L: E_mix = that value
        par = orc.o_comb(w_all, us[k])
        ids = ids[par]
        w_all = np.full(world * nw, np.cumsum(w_all)[-1] / (world * nw))
    exp_e.append(complex(-1.5, 0.5))
    ok &= len(en) == 5 and all(abs(a - b) < 1e-12 for a, b in zip(en, exp_e))
    ok &= np.array_equal(phi.numpy(), ids[rank * nw:(rank + 1) * nw])    # the right walkers, in slot order, across ranks
    ok &= np.allclose(weight.numpy(), w_all[rank * nw:(rank + 1) * nw])
    moved = sum(c["walkers_sent_to_peers"] for c in D.COMB_STATS)
    out[rank] = (bool(ok), int(moved), [complex(e) for e in en])
    dist.barrier()
    dist.destroy_process_group()


def test_run_sharded_control_flow_gloo():
    import torch.multiprocessing as mp
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    out = ctx.Manager().dict()
    procs = [ctx.Process(target=_run_sharded_worker, args=(r, 2, port, out)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(180)
        assert p.exitcode == 0
    assert out[0][0] and out[1][0]
    assert out[0][2] == out[1][2]                      # the all-reduced estimator is the same on both ranks
    assert out[0][1] > 0                               # rank 0 (heavy weights) really sent walkers to rank 1
