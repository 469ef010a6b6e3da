"""Multi-GPU plumbing.  The walker step has no exchange step ("subsets which are independently
propagated"), so for bench.py N GPUs run N independent replicas of the batch and the only cross-rank traffic is the
max-over-ranks of the measured time.  The one real exchange step of the method is the comb population control over a
population sharded across ranks: `population_control_sharded` runs it with an all-gather of
the weights and one all-to-all of walker records; the map, the packing and the unpacking are CUDA kernels behind the
C ABI (afqmc_comb_map / _pack / _unpack), this module only routes buffers.  Works on any torch.distributed backend
(nccl on GPUs; the routing logic is covered with gloo in tests)."""
from __future__ import annotations


COMB_STATS = []   # one dict per sharded comb on this rank (walkers / bytes sent to other ranks); bench.py --sharded reads it


def rank_seed(base: int, rank: int) -> int:
    """Distinct, reproducible field seed per replica."""
    return int(base) + 7919 * int(rank)


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of a scalar (identity when torch.distributed is not initialised)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank: int, world: int, seconds_max: float) -> float:
    """Aggregate throughput of `world` replicas that each processed `units_per_rank` units."""
    return world * units_per_rank / seconds_max


def comb_splits(parent_all, n_local: int, world: int, rank: int):
    """Routing of the sharded comb from the global parent map (index bookkeeping only, no method arithmetic).

    parent_all: integer tensor [world * n_local], monotone non-decreasing, parent_all[g] = global index of the walker
    that global slot g receives.  Returns (slot_lo, count, send_counts, recv_counts): the global slots whose parent
    lives on `rank` are the contiguous range [slot_lo, slot_lo + count); send_counts[d] of them belong to rank d (in
    slot order, so the send buffer is already grouped by destination); recv_counts[s] of this rank's own slots have
    their parent on rank s (in slot order, so the receive buffer arrives in slot order)."""
    import torch
    p = parent_all.to(torch.int64)
    owner = torch.div(p, n_local, rounding_mode="floor")
    dest = torch.arange(p.numel(), device=p.device, dtype=torch.int64) // n_local
    mine = owner == rank
    count = int(mine.sum().item())
    slot_lo = int(torch.nonzero(mine)[0].item()) if count else 0
    send_counts = torch.bincount(dest[mine], minlength=world).tolist()
    recv_counts = torch.bincount(owner[rank * n_local:(rank + 1) * n_local], minlength=world).tolist()
    return slot_lo, count, send_counts, recv_counts


def population_control_sharded(ctx, phi, weight, ovlp, theta, fb, u: float, group=None):
    """Comb population control (R22) over a population sharded across the ranks of
    `group`: every rank holds ctx.params.n_walkers walkers and calls this with the SAME u.  In place.  Returns the
    global parent map (device int32 [world * N_w]).  One all-gather of N_w doubles and one all-to-all of walker
    records; with a single rank (or torch.distributed not initialised) it needs no collective at all."""
    import torch
    import torch.distributed as dist
    if weight.is_cuda and torch.cuda.current_stream(weight.device) != ctx.stream:
        # the library enqueues on ctx.stream; torch ops and collectives on torch's current stream: make them the same
        with torch.cuda.stream(ctx.stream):
            return population_control_sharded(ctx, phi, weight, ovlp, theta, fb, u, group=group)
    on = dist.is_available() and dist.is_initialized()
    world = dist.get_world_size(group) if on else 1
    rank = dist.get_rank(group) if on else 0
    nw = int(ctx.params.n_walkers)
    dev = weight.device
    if world > 1:
        w_all = torch.empty(world * nw, dtype=torch.float64, device=dev)
        dist.all_gather_into_tensor(w_all, weight.contiguous(), group=group)
    else:
        w_all = weight
    cum = torch.empty(world * nw, dtype=torch.float64, device=dev)
    parent_all = torch.empty(world * nw, dtype=torch.int32, device=dev)
    w_new = torch.empty(2, dtype=torch.float64, device=dev)
    ctx.afqmc_comb_map(w_all, u, cum, parent_all, w_new)
    slot_lo, count, send_counts, recv_counts = comb_splits(parent_all, nw, world, rank)
    rec = ctx.afqmc_comb_record_bytes
    sendbuf = torch.empty(max(count, 1) * rec, dtype=torch.uint8, device=dev)
    ctx.afqmc_comb_pack(phi, ovlp, theta, fb, parent_all, slot_lo, count, rank * nw, sendbuf)
    if world > 1:
        recvbuf = torch.empty(nw * rec, dtype=torch.uint8, device=dev)
        dist.all_to_all_single(recvbuf, sendbuf[:count * rec], [c * rec for c in recv_counts],
                               [c * rec for c in send_counts], group=group)
    else:
        recvbuf = sendbuf
    ctx.afqmc_comb_unpack(recvbuf, phi, weight, ovlp, theta, fb, w_new)
    to_peers = sum(c for d, c in enumerate(send_counts) if d != rank)
    COMB_STATS.append(dict(walkers_sent_to_peers=int(to_peers), bytes_sent_to_peers=int(to_peers) * int(rec)))
    return parent_all


def run_sharded(ctx, phi, weight, ovlp, theta, fb, x, n_steps, energy_every=20, ortho_every=2, pc_every=20, us=(),
                flags=None, group=None):
    """The paper's schedule (afqmc_run) for a population sharded across the ranks of `group`: every rank
    steps its own N_w walkers with its own fields x [n_steps][N_w][n_chol]; the comb runs over the WHOLE population
    (population_control_sharded, same us on every rank) and every measurement all-reduces the three estimator sums of
    afqmc_mixed_sums.  pc_every must be a multiple of energy_every and of ortho_every (the paper's 20 / 2 / 20), or 0.
    Returns the list of global mixed-estimator energies (complex) of the measurements, identical on every rank."""
    import torch
    import torch.distributed as dist
    if weight.is_cuda and torch.cuda.current_stream(weight.device) != ctx.stream:
        with torch.cuda.stream(ctx.stream):      # one stream for the library's kernels, torch's ops and the collectives
            return run_sharded(ctx, phi, weight, ovlp, theta, fb, x, n_steps, energy_every, ortho_every, pc_every, us,
                               flags, group)
    on = dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1
    nw = int(ctx.params.n_walkers)
    seg = pc_every if pc_every else n_steps
    assert seg > 0 and (not energy_every or seg % energy_every == 0) and (not ortho_every or seg % ortho_every == 0)
    n_meas_seg = seg // energy_every if energy_every else 0
    eloc = torch.zeros(max(n_meas_seg, 1), nw, dtype=torch.complex128, device=weight.device)
    wm = torch.zeros(max(n_meas_seg, 1), nw, dtype=torch.float64, device=weight.device)
    sums = torch.zeros(max(n_meas_seg, 1), 3, dtype=torch.float64, device=weight.device)
    emix = torch.zeros(max(n_meas_seg, 1), dtype=torch.complex128, device=weight.device)
    energies, done, k = [], 0, 0
    while done < n_steps:
        n = min(seg, n_steps - done)
        ctx.afqmc_run(phi, weight, ovlp, theta, fb, x[done:done + n], n, energy_every, ortho_every, 0, None, eloc, wm,
                      None, flags)
        m = n // energy_every if energy_every else 0
        for j in range(m):
            ctx.afqmc_mixed_sums(wm[j], eloc[j], sums[j])
        if m:
            if on:
                dist.all_reduce(sums[:m], group=group)
            ctx.afqmc_mixed_energy(sums, m, emix)      # the estimator's division runs in the library too
            energies.extend(complex(v) for v in emix[:m].tolist())
        done += n
        if pc_every and n == seg:
            population_control_sharded(ctx, phi, weight, ovlp, theta, fb, us[k], group=group)
            k += 1
    return energies
