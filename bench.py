#!/usr/bin/env python
"""bench.py -- walker-steps/s of the ph-AFQMC walker step (propagate + energy every step, both spins).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--cfg 5] [--impl ours|reference]

One "step" = one pass of the whole hot path (shift -> assemble -> Taylor -> overlap/weights -> force
bias -> local energy) over all N_w walkers of the workload.  The workload is BASELINE.json's config 5
(M=200, 13+12 electrons, N_chol=1000, 2048 complex64 walkers) unless --cfg says otherwise; inputs are
seeded synthetic tensors of that shape (workloads/gen.py).
Prints ONE JSON line on rank 0 (contract in the task statement; keys `roofline`, `cpu_baseline`, `e2e`,
`clocks`, `gpu_launches` included).  N > 1: launched under torchrun, every rank runs an independent
replica of the batch ("weak"), time = max over ranks (NCCL all-reduce of the device time).
--impl reference times the FP64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "walker-steps/sec (propagate+energy)"
UNIT = "walker-steps/s"


def workload_name(wl):
    return (f"cfg{wl.cfg} M={wl.M} N=({wl.n_alpha},{wl.n_beta}) N_chol={wl.n_chol} N_w={wl.n_walkers} "
            f"{wl.precision} K={wl.K} n_det={wl.n_det}")


def flops_per_walker_step(wl):
    """Algorithmic (useful, real) flops per stage per walker-step."""
    M, na, nb, ng, K = wl.M, wl.n_alpha, wl.n_beta, wl.n_chol, wl.K
    nt = na + nb
    return dict(assemble=4.0 * ng * M * M,                       # real x complex: 2 planes x 2 flop
                force_bias=4.0 * ng * M * nt,
                taylor=8.0 * M * M * nt * K + 2 * 4.0 * M * M * nt,
                energy=2.0 * ((M * na) ** 2 + (M * nb) ** 2),   # v^T Y v with Y symmetric: upper triangle only
                green=4.0 * M * (na * na + nb * nb) + 8.0 * M * (na * na + nb * nb))


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16_burst=d["bf16_tflops"], bf16_sust=d["bf16_tflops_sustained"],
                    sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
    return dict(hbm=6650.0, bf16_burst=1590.0, bf16_sust=1400.0, sm_max_mhz=1965.0, source="fallback")


def measure_peaks(device):
    """Self-written microbenchmarks (csrc/peaks.cuh, afqmc_peak_probe): the TF32 / FP32 / FP64 / L2 denominators the fractions are
    quoted against.  ~50 ms in total."""
    import torch
    import paper_1804_03310_b200 as afq
    scr = torch.zeros(96 << 20, dtype=torch.uint8, device=device)

    def best(kind, n, iters, rep=3):
        r = [afq.afqmc_peak_probe(kind, n, iters, scr) for _ in range(rep)]
        return min(r, key=lambda t: t[0])
    out = {}
    for key, kind in (("tf32_ss_n256", 0), ("tf32_ts_n256", 1), ("tf32_pair_n256", 2)):
        ms, fl, clk = best(kind, 256, 8000)
        out[key] = dict(tflops=fl / ms / 1e9, clk_per_mma=clk)
    ms, fl, clk = best(0, 128, 8000)
    out["tf32_ss_n128"] = dict(tflops=fl / ms / 1e9, clk_per_mma=clk)
    ms, fl, clk = best(0, 64, 8000)
    out["tf32_ss_n64"] = dict(tflops=fl / ms / 1e9, clk_per_mma=clk)
    ms, fl, _ = best(3, 0, 100000)
    out["ffma_tflops"] = fl / ms / 1e9
    ms, fl, _ = best(4, 0, 100000)
    out["dfma_tflops"] = fl / ms / 1e9
    ms, by, _ = best(5, 48, 3000)
    out["l2_to_smem_tma_gbs"] = by / ms / 1e6
    out["note"] = ("back-to-back tcgen05.mma.kind::tf32 M=128 (pair: M=256) K=8 from shared memory (ss), with the a-operand in TMEM (ts), "
                   "on CTA pairs; FFMA / DFMA 8 chains per thread; TMA stream of a 48 MiB (L2-resident) buffer into shared memory")
    return out


class ClockSampler(threading.Thread):
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        super().__init__(daemon=True)
        self.index, self.rows, self._halt = index, [], threading.Event()

    def _nvml_loop(self):
        import pynvml as nv
        nv.nvmlInit()
        h = nv.nvmlDeviceGetHandleByIndex(self.index)
        mx = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
        bits = {"hw_slowdown": 0x8, "sw_power_cap": 0x4, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40}
        get_reasons = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
        while not self._halt.is_set():
            sm = nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)
            r = int(get_reasons(h))
            pw = nv.nvmlDeviceGetPowerUsage(h) / 1000.0
            row = [str(sm), str(mx), str(pw)] + [("Active" if r & bits[n] else "Not Active")
                                                 for n in ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")]
            self.rows.append(row)
            self._halt.wait(0.002)

    def run(self):
        try:
            self._nvml_loop()        # NVML in-process: ~1 ms per sample, so even a 50 ms timed region is covered
            return
        except Exception:
            pass
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                      "-i", str(self.index)], capture_output=True, text=True, timeout=5).stdout
                self.rows.append([c.strip() for c in out.strip().split(",")])
            except Exception:
                pass
            self._halt.wait(0.1)

    def stop(self):
        self._halt.set()
        self.join(timeout=6)
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        pw = []
        for r in self.rows:
            try:
                pw.append(float(r[2]))
            except Exception:
                pass
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=mx or None, reasons=sorted(reasons),
                    samples=len(sm), power_w_max=max(pw) if pw else None)


def time_oracle(wl, target_s=12.0, one_thread_s=0.0):
    """The FP64 numpy oracle as it stands, on the host cores: walker-steps/s on a bounded sample."""
    from oracle import afqmc_oracle as orc
    cores = len(os.sched_getaffinity(0))
    ini = orc.o_init(wl.h, wl.L, wl.dt, wl.psi_a, wl.psi_b)
    trial = orc.MultiDetTrial(wl.C_act, wl.det_coeff, wl.det_exc, wl.n_alpha, wl.n_beta) if wl.n_det > 1 else None
    nw = min(wl.n_walkers, 8)
    done, t_total, nsteps = 0, 0.0, 0
    def start(n):
        phi = wl.walkers(n)
        if trial is not None:
            # The workload's initial walkers ARE the reference determinant: their overlap with every excited determinant is
            # exactly zero and the oracle's SMW path (one small inverse per walker and determinant) raises on the exactly
            # singular matrix.  Timing is value independent: start from seeded walkers a little away from the reference.
            g = np.random.default_rng(7)
            phi = phi + 0.05 * (g.standard_normal(phi.shape) + 1j * g.standard_normal(phi.shape))
        return orc.o_seed_state(ini, phi, wl.n_alpha, trial=trial)

    while True:
        ost = start(nw)
        x = wl.fields(1, nw)[0]
        t0 = time.perf_counter()
        orc.o_step(ini, ost, x, wl.n_alpha, K=wl.K, E0=wl.E0, trial=trial)
        dt = time.perf_counter() - t0
        t_total += dt; done += nw; nsteps += 1
        if t_total >= target_s or nsteps >= 64:
            break
        if dt < 1.0 and nw < wl.n_walkers:
            nw = min(wl.n_walkers, nw * 4)
    out = dict(value=done / t_total, unit=UNIT, cores=cores, kind="oracle",
               sample=f"{nsteps} oracle step(s) over {done} walker-steps of {workload_name(wl)} "
                      f"({t_total:.1f} s CPU wall, numpy/BLAS threads = all {cores} cores, init excluded"
                      + ("; walkers = reference determinant + 0.05 complex normal noise, seed 7" if trial is not None else "") + ")")
    if one_thread_s > 0:
        # the paper's comparator is ONE CPU core in double precision: same oracle, BLAS limited to 1 thread
        try:
            from threadpoolctl import threadpool_limits
            n1 = min(wl.n_walkers, 4)
            ost = start(n1)
            x = wl.fields(1, n1)[0]
            d1, t1 = 0, 0.0
            with threadpool_limits(limits=1):
                while t1 < one_thread_s:
                    t0 = time.perf_counter()
                    orc.o_step(ini, ost, x, wl.n_alpha, K=wl.K, E0=wl.E0, trial=trial)
                    t1 += time.perf_counter() - t0
                    d1 += n1
            out["value_1thread"] = d1 / t1
            out["sample_1thread"] = f"{d1} walker-steps in {t1:.1f} s with BLAS limited to 1 thread (threadpoolctl)"
        except Exception as e:          # the baseline is a reported figure only
            out["value_1thread"] = None
            out["sample_1thread"] = f"unavailable: {e}"
    return out


def run_reference(args):
    from workloads import make_workload
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    wl = make_workload(args.cfg, args.variant)
    budget = max(4.0, min(120.0, 8.0 * (args.steps + args.warmup)))
    t0 = time.perf_counter()
    base = time_oracle(wl, target_s=budget)
    line = dict(metric=METRIC, value=base["value"], unit=UNIT, n_gpus=args.gpus, steps=args.steps, warmup=args.warmup,
                ms_per_step=1e3 * wl.n_walkers / base["value"], higher_is_better=True, scaling="weak",
                vs_baseline=None, dtype="f64", data="synthetic", impl="reference",
                config=dict(workload=workload_name(wl), variant=args.variant),
                cpu_baseline=base,
                e2e=dict(value=base["value"], unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                wall_s=time.perf_counter() - t0)
    print(json.dumps(line))


def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1804_03310_b200.state import WalkerState
    from workloads import make_workload

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))

    wl = make_workload(args.cfg, args.variant)
    nw, K, W = wl.n_walkers, args.steps, max(args.warmup, 3)
    import paper_1804_03310_b200 as afq
    p = afq.make_params(wl.M, wl.n_alpha, wl.n_beta, wl.n_chol, nw, wl.precision, wl.dt, taylor_order=wl.K,
                        E0=wl.E0, n_det=wl.n_det, n_act=wl.n_act, gemm_path=args.gemm_path)
    kw = {}
    if wl.n_det > 1:
        kw = dict(C_act=wl.C_act, det_coeff=wl.det_coeff, det_exc=wl.det_exc)
    ctx = afq.AfqmcContext(p, wl.h, wl.L, wl.psi_a, wl.psi_b, device=f"cuda:{local}", **kw)
    dev = ctx.device
    # fields: every rank its own seed (replicas are independent); a fresh draw per step, resident in HBM
    from paper_1804_03310_b200 import dist as D
    rng = np.random.default_rng(D.rank_seed(1000, rank))
    nfield = min(K, 8)
    x = torch.tensor(rng.standard_normal((nfield, nw, wl.n_chol)), dtype=ctx.rdtype, device=dev)
    phi0 = torch.tensor(wl.walkers(nw), dtype=ctx.cdtype, device=dev)
    st = WalkerState(ctx, wl.walkers(nw))
    eloc = torch.zeros(1, nw, dtype=torch.complex128, device=dev)

    def reseed():
        # walkers restart from the trial (the literal configs kill every walker in ~8 steps)
        st.phi.copy_(phi0); st.weight.fill_(1.0); st.flags.zero_()
        st.seed()

    def one_step(i):
        ctx.afqmc_step(st.phi, st.weight, st.ovlp, st.theta, st.fb, x[i % nfield], 1, eloc, st.flags)

    reseed()
    for i in range(W):
        one_step(i)
    torch.cuda.synchronize()
    reseed()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    ctx.afqmc_profile_enable(True)
    l0 = ctx.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for i in range(K):
        if i and i % 6 == 0:
            reseed()           # inside the timed region: counted (2 extra small kernels + copies)
        one_step(i)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    launches = ctx.launch_count - l0
    prof = ctx.afqmc_profile_read()
    ctx.afqmc_profile_enable(False)
    clocks = sampler.stop() if sampler else None
    if world > 1:
        dist.barrier()
    ms_max = D.max_over_ranks(ms, dev)

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----
    Ke = K          # every step uploads its fields and downloads its energies; the walkers go in and out once per call
    phi_h = torch.tensor(wl.walkers(nw), dtype=ctx.cdtype).pin_memory()
    w_h = torch.ones(nw, dtype=torch.float64).pin_memory()
    S_h = torch.zeros(nw, dtype=torch.complex128).pin_memory()
    x_h = torch.tensor(rng.standard_normal((Ke, nw, wl.n_chol)), dtype=ctx.rdtype).pin_memory()
    e_h = torch.zeros(Ke, nw, dtype=torch.complex128).pin_memory()
    f_h = torch.zeros(nw, dtype=torch.int32).pin_memory()
    phi_keep = phi_h.clone()
    ctx.afqmc_step_host(phi_h, w_h, S_h, x_h, 1, e_h, f_h)      # warm
    phi_h.copy_(phi_keep); w_h.fill_(1.0)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t0 = time.perf_counter()
    up, down = ctx.afqmc_step_host(phi_h, w_h, S_h, x_h, Ke, e_h, f_h)   # synchronises internally
    t_e2e = time.perf_counter() - t0
    t_e2e = D.max_over_ranks(t_e2e, dev)

    # ---- the paper's production schedule: hybrid weights, E_L every 20 steps,
    # orthonormalisation every 2, comb population control every 20 -- one afqmc_run call of 20 steps, reported beside
    # the headline (which measures E_L on every step, BASELINE.json's metric)
    sched = None
    if not args.no_schedule:
        ns, ee, oe, pe = 20, 20, 2, 20
        xs20 = x[torch.arange(ns, device=dev) % nfield].contiguous()
        el20 = torch.zeros(1, nw, dtype=torch.complex128, device=dev)
        par20 = torch.zeros(1, nw, dtype=torch.int32, device=dev)
        reseed()
        ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xs20, ns, ee, oe, pe, [0.5], el20, None, par20, st.flags)
        reseed()
        ctx.afqmc_profile_enable(True)
        l1 = ctx.launch_count
        torch.cuda.synchronize()
        e0.record()
        ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xs20, ns, ee, oe, pe, [0.5], el20, None, par20, st.flags)
        e1.record()
        torch.cuda.synchronize()
        ms20 = e0.elapsed_time(e1)
        prof20 = ctx.afqmc_profile_read()
        ctx.afqmc_profile_enable(False)
        # the literal configs kill the whole population within ~8 steps, so the comb inside the run moves
        # nothing; its cost is measured on the same state with seeded log-normal weights (sigma 0.5) instead
        wr = torch.tensor(np.exp(0.5 * np.random.default_rng(7).standard_normal(nw)), dtype=torch.float64, device=dev)
        st.weight.copy_(wr)
        ctx.afqmc_profile_enable(True)
        ctx.afqmc_population_control(st.phi, st.weight, st.ovlp, st.theta, st.fb, 0.5, par20[0])
        torch.cuda.synchronize()
        prof_pc = ctx.afqmc_profile_read()
        ctx.afqmc_profile_enable(False)
        moved = int((par20[0] != torch.arange(nw, device=dev, dtype=torch.int32)).sum().item())
        cb_ = 8 if wl.precision == "c64" else 16
        ob = nw * (2 * wl.M * wl.n_t * cb_ + 32)                       # read + write the walker, read + write S
        o_ms = prof20["ortho"][0] / max(prof20["ortho"][1], 1)
        p_ms = prof_pc["popctl"][0] / max(prof_pc["popctl"][1], 1)
        pb = moved * 4 * ((2 * wl.M * wl.n_t + wl.n_chol) * cb_ + 16) + nw * 28
        hbm = peaks()["hbm"]
        sched = dict(value=world * nw * ns / (ms20 * 1e-3), unit=UNIT, ms_per_step=ms20 / ns, steps=ns, energy_every=ee,
                     ortho_every=oe, pc_every=pe, gpu_launches=ctx.launch_count - l1,
                     ortho=dict(ms_per_launch=o_ms, bytes=ob, achieved_gbs=ob / (o_ms * 1e-3) / 1e9 if o_ms else None,
                                frac_hbm=ob / (o_ms * 1e-3) / 1e9 / hbm if o_ms else None),
                     popctl=dict(ms_per_launch=p_ms, ms_inside_run=prof20["popctl"][0], walkers_moved=moved, bytes=pb,
                                 weights="seeded log-normal, sigma 0.5",
                                 achieved_gbs=pb / (p_ms * 1e-3) / 1e9 if p_ms else None),
                     note="one afqmc_run call: propagate-only steps (no energy contraction) except the measured one")

    # ---- launch-latency-bound configs (M < 96: cfgs 1-4): the same K steps as ONE CUDA graph replay ----
    graph = None
    if wl.M < 96 and not args.no_graph:
        xg = x[torch.arange(K, device=dev) % nfield].contiguous()
        elg = torch.zeros(K, nw, dtype=torch.complex128, device=dev)
        reseed()
        side = torch.cuda.Stream(device=dev)
        side.wait_stream(torch.cuda.current_stream(dev))
        g = torch.cuda.CUDAGraph()
        with torch.cuda.stream(side):
            ctx.use_stream(side)
            ctx.afqmc_step(st.phi, st.weight, st.ovlp, st.theta, st.fb, xg, K, elg, st.flags)   # warm on the capture stream
            side.synchronize()
            reseed()
            lg = ctx.launch_count
            with torch.cuda.graph(g, stream=side):
                ctx.afqmc_step(st.phi, st.weight, st.ovlp, st.theta, st.fb, xg, K, elg, st.flags)
            lg = ctx.launch_count - lg
            g.replay(); side.synchronize()
            reseed(); side.synchronize()
            eg0, eg1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            eg0.record(side)
            g.replay()
            eg1.record(side)
            side.synchronize()
            ms_g = eg0.elapsed_time(eg1)
            # empty-launch floor: the library's smallest kernel (k_mixed_ratio, one thread of work), launched back to back
            o3 = torch.ones(3, dtype=torch.float64, device=dev)
            o1 = torch.zeros(1, dtype=torch.complex128, device=dev)
            for _ in range(20):
                ctx.afqmc_mixed_energy(o3, 1, o1)
            side.synchronize()
            eg0.record(side)
            for _ in range(200):
                ctx.afqmc_mixed_energy(o3, 1, o1)
            eg1.record(side)
            side.synchronize()
            floor_us = eg0.elapsed_time(eg1) * 1e3 / 200
        ctx.use_stream(torch.cuda.current_stream(dev))
        ms_g = D.max_over_ranks(ms_g, dev)
        graph = dict(value=world * nw * K / (ms_g * 1e-3), unit=UNIT, us_per_step=ms_g * 1e3 / K, kernels_in_graph=lg,
                     eager_us_per_step=ms_max * 1e3 / K, launch_floor_us_per_kernel=floor_us,
                     floor_us_per_step=floor_us * lg / K,
                     note="one afqmc_step(n_steps) call captured into a CUDA graph and replayed; the floor is the measured "
                          "back-to-back launch rate of a one-CTA kernel times the kernels per step")

    mp = measure_peaks(dev)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    pk = peaks()
    fl = flops_per_walker_step(wl)
    headline_ms = ms_max
    if graph is not None:          # latency-bound configs: the graph replay is the library's fast path and the headline
        headline_ms = graph["us_per_step"] * K * 1e-3
    value = D.whole_job_rate(nw * K, world, headline_ms * 1e-3)
    M_, ng_, nt_ = wl.M, wl.n_chol, wl.n_t
    tensor_path = ctx.gemm_path >= 2
    tay_tc = tensor_path and 96 <= M_ <= 256 and nt_ <= 32
    if tensor_path:
        fl["assemble"] = 4.0 * ng_ * M_ * (M_ + 1) / 2       # the tcgen05 assembly GEMM exploits A = A^T: upper triangle only
    if wl.n_det > 1:
        # H10: TT = C_act^T X Theta_0 for all X (one GEMM), W / WT per operator, E x E work per determinant
        nact, nd = wl.n_act, wl.n_det
        fl["energy"] = (4.0 * (ng_ + 1) * nact * M_ * nt_ + sum(16.0 * (nact - n) * n * n for n in (wl.n_alpha, wl.n_beta)) * (ng_ + 1)
                        + 120.0 * nd * (ng_ + 1))
    tf32_peak = max(mp["tf32_ss_n256"]["tflops"], mp["tf32_pair_n256"]["tflops"])
    tensor_note = (f"TF32 dense MEASURED by back-to-back tcgen05.mma.kind::tf32 N=256 on every SM (afqmc_peak_probe): {tf32_peak:.0f} TFLOP/s "
                   f"(nominal-ratio estimate 0.5 x BF16 {pk['bf16_burst']:.0f} = {0.5 * pk['bf16_burst']:.0f}); achieved counts ALGORITHMIC flops and "
                   "3xTF32 issues 3x of them, so frac <= 1/3 by construction")
    fp32_note = f"FP32 FMA MEASURED (8 chains per thread, afqmc_peak_probe): {mp['ffma_tflops']:.1f} TFLOP/s (nominal 148 x 128 x 2 x {pk['sm_max_mhz']:.0f} MHz = {148 * 128 * 2 * pk['sm_max_mhz'] * 1e-6:.1f})"
    fp64_note = f"FP64 FMA MEASURED (afqmc_peak_probe): {mp['dfma_tflops']:.1f} TFLOP/s"
    alu_peak, alu_note = (mp["dfma_tflops"], fp64_note) if wl.precision == "c128" else (mp["ffma_tflops"], fp32_note)
    kind = dict(assemble="tensor" if tensor_path else "alu", force_bias="tensor" if tensor_path else "alu",
                taylor="tensor" if tay_tc else "alu", energy="alu" if wl.n_det > 1 else ("tensor" if tensor_path else "alu"), green="hbm")
    names = dict(assemble="H6 assembly GEMM A_w = sum_g z_g L_g (" + ("tc::k_gemm_tf32_pair_ps<EpiAssembleSym>" if tensor_path else "k_gemm_nt") + ")",
                 taylor="H7 Taylor propagator (" + ("tt::k_taylor_tc" if tay_tc else "k_taylor, FP32/FP64 SIMT") + ")",
                 energy=("H10 multi-determinant energy (TT GEMM + k_md_energy_b, FP32 SIMT)" if wl.n_det > 1 else
                         "H9 energy GEMM (both spins, one persistent launch) + fused dot (" + ("tc::k_gemm_tf32_pair_ps<EpiEnergy>" if tensor_path else "k_gemm_nt") + ")"),
                 force_bias="H4 force-bias GEMMs", green="H1-H3/H8 overlap, LU, Theta, weights (k_green)")
    dtype = "tf32x3" if tensor_path else ("f32" if wl.precision == "c64" else "f64")
    traffic_ncu = load_traffic(args.cfg, ctx.gemm_path)

    def roof(stage):
        ms, n = prof[stage]
        if not n or ms <= 0 or stage not in fl:
            return None
        ach = fl[stage] * nw * n / (ms * 1e-3) / 1e12
        if kind[stage] == "tensor":
            peak, note = tf32_peak, tensor_note
        else:
            peak, note = alu_peak, alu_note
        r = dict(bound=kind[stage] if kind[stage] != "hbm" else "hbm", kernel=names[stage], achieved=ach, peak=peak, unit="TFLOP/s",
                 frac=ach / peak, traffic=traffic_ncu.get(stage), peak_source=note, launches_timed=n, ms_per_launch=ms / n)
        if kind[stage] == "tensor":
            r["issued_frac"] = 3.0 * ach / peak
        if stage == "green":      # HBM-bound stage: bytes, not flops
            cb = 8 if wl.precision == "c64" else 16
            byts = nw * wl.M * wl.n_t * cb * (2 + (2 if tensor_path else 1))
            r.update(bound="hbm", achieved=byts * n / (ms * 1e-3) / 1e9, peak=pk["hbm"], unit="GB/s",
                     peak_source=f"{pk['source']} HBM copy bandwidth")
            r["frac"] = r["achieved"] / r["peak"]
            r.pop("issued_frac", None)
        if wl.M < 96:
            r["note"] = ("launch/latency-bound config (SURVEY 8(d)): no roofline fraction is meaningful here; see `latency` for us/step "
                         "against the launch floor")
        return r

    timed = {k: v[0] / v[1] for k, v in prof.items() if v[1] and k in names}
    dominant = max(timed, key=timed.get) if timed else "assemble"
    stage_ms = {k: (v[0] / v[1] if v[1] else None) for k, v in prof.items()}
    stage_tflops = {k: (fl[k] * nw / (stage_ms[k] * 1e-3) / 1e12 if stage_ms.get(k) else None) for k in fl}
    base = None
    if not args.no_cpu_baseline:
        base = time_oracle(wl, target_s=args.cpu_seconds, one_thread_s=min(6.0, args.cpu_seconds / 2))
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=W, ms_per_step=headline_ms / K,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype=dtype, data="synthetic",
                config=dict(workload=workload_name(wl), variant=args.variant, global_walkers=world * nw,
                            parallelism=f"replicas x{world}" if world > 1 else "single GPU",
                            l2="per-step working set (A_w buffer %.0f MB + operands) exceeds the 126 MB L2; no flush"
                               % (nw * wl.M * wl.M * 2 * (4 if wl.precision == "c64" else 8) / 1e6),
                            gemm_path={1: "simt", 2: "tcgen05-3xtf32", 3: "tcgen05-3xtf32-ctapair"}[ctx.gemm_path],
                            launch="CUDA graph replay of afqmc_step(n_steps)" if graph is not None else "eager afqmc_step"),
                clocks=clocks, gpu_launches=launches,
                e2e=dict(value=world * nw * Ke / t_e2e, unit=UNIT, h2d_bytes_per_step=up / Ke, d2h_bytes_per_step=down / Ke,
                         steps=Ke, note="afqmc_step_host: pinned host buffers, H2D of walkers+fields and D2H of "
                                        "walkers/weights/overlaps/energies inside the timed region"),
                roofline=roof(dominant), roofline_h6=roof("assemble"), latency=graph, eager_ms_per_step=ms_max / K,
                stages_ms=stage_ms, stages_tflops=stage_tflops, measured_peaks=mp, schedule=sched, cpu_baseline=base)
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def load_traffic(cfg, gemm_path):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch from the tracked ncu summary profiles/r2_traffic.csv
    (columns: stage,cfg,gemm_path,dram_bytes,kernel,capture).  Null when no capture matches the running kernel."""
    import csv
    out = {}
    p = os.path.join(ROOT, "profiles", "r2_traffic.csv")
    if os.path.exists(p):
        for row in csv.DictReader(open(p)):
            if int(row["cfg"]) == cfg and int(row["gemm_path"]) == gemm_path:
                out[row["stage"]] = float(row["dram_bytes"])
    return out


def run_ndet_scan(args):
    """cfg 4 (multi-determinant trial) at N_det = 10 / 100 / 1000: ms per walker step and the ratio to N_det = 10, beside the paper's
    "10 -> 1200 determinants multiplies the propagation time by 3.9" (Fig. 1 :74; other hardware, other workload,
    energy every 20 steps there, every step here: context, not a target)."""
    import torch
    from paper_1804_03310_b200.state import WalkerState, make_context
    from workloads import make_workload, random_walkers
    rows = []
    for nd in (10, 100, 1000):
        wl = make_workload(4, args.variant, overrides=dict(n_det=nd))
        nw, K = wl.n_walkers, args.steps
        ctx = make_context(wl, nw, gemm_path=args.gemm_path)
        dev = ctx.device
        x = torch.tensor(np.random.default_rng(1000).standard_normal((4, nw, wl.n_chol)), dtype=ctx.rdtype, device=dev)
        phi0 = random_walkers(wl, nw, seed=21, spread=0.05)
        st = WalkerState(ctx, phi0)
        p0 = st.phi.clone()
        eloc = torch.zeros(1, nw, dtype=torch.complex128, device=dev)

        def reseed():
            st.phi.copy_(p0); st.weight.fill_(1.0); st.flags.zero_(); st.seed()
        out = {}
        for mode, ee in (("energy_every_step", 1), ("energy_every_20", 20)):
            reseed()
            xs = x[torch.arange(20, device=dev) % 4].contiguous()
            e20 = torch.zeros(20, nw, dtype=torch.complex128, device=dev)
            ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xs, 20, ee, 2, 0, None, e20, None, None, st.flags)   # warm
            reseed()
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xs, 20, ee, 2, 0, None, e20, None, None, st.flags)
            e1.record()
            torch.cuda.synchronize()
            out[mode] = e0.elapsed_time(e1) / 20
        rows.append(dict(n_det=nd, ms_per_step=out["energy_every_step"], ms_per_step_paper_schedule=out["energy_every_20"]))
        ctx.close()
    r0 = rows[0]
    for r in rows:
        r["ratio_to_10"] = r["ms_per_step"] / r0["ms_per_step"]
        r["ratio_to_10_paper_schedule"] = r["ms_per_step_paper_schedule"] / r0["ms_per_step_paper_schedule"]
    print(json.dumps(dict(metric="ms per walker step vs N_det (cfg 4 shapes, 512 walkers)", rows=rows,
                          paper="x3.9 for 10 -> 1200 determinants (Mn QZ, 20 walkers, GTX 1080, energy every 20 steps; PAPER.md:68, :74)",
                          note="20 steps per afqmc_run call, orthonormalisation every 2; energy_every_20 is the paper's schedule")))


def run_sharded(args):
    """NEXT-4: the paper's schedule over a population SHARDED across the ranks --
    every rank steps its own N_w walkers, every measurement all-reduces three estimator sums, every pc_every steps the comb runs over
    the whole population (all-gather of the weights + one all-to-all of walker records).  One dist.run_sharded call of 40 steps
    (E/20, QR/2, comb/20).  "weak": the global population is N_w x ranks."""
    import torch
    import torch.distributed as dist
    from paper_1804_03310_b200 import dist as D
    from paper_1804_03310_b200.state import WalkerState, make_context
    from workloads import make_workload
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("NCCL_DEBUG", "INFO")          # the communicator line (nranks) stays visible in the log
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    # the literal / mf inputs kill the whole population within ~8 steps: the 40-step schedule runs on the tame
    # variant of the same shapes, so that the estimator is finite and the comb has live weights to route (timing is value independent)
    variant = {"mf": "tame_mf", "raw": "tame"}.get(args.variant, args.variant)
    wl = make_workload(args.cfg, variant)
    nw = wl.n_walkers
    ctx = make_context(wl, nw, gemm_path=args.gemm_path, device=f"cuda:{local}")
    dev = ctx.device
    ns, ee, oe, pe = 40, 20, 2, 20
    rng = np.random.default_rng(D.rank_seed(1000, rank))
    x = torch.tensor(rng.standard_normal((8, nw, wl.n_chol)), dtype=ctx.rdtype, device=dev)
    xs = x[torch.arange(ns, device=dev) % 8].contiguous()
    st = WalkerState(ctx, wl.walkers(nw))
    phi0 = st.phi.clone()
    # seeded log-normal start weights (sigma 0.5, every rank its own mean) so that the comb really moves walkers across ranks
    w0 = torch.tensor(np.exp(0.5 * rng.standard_normal(nw) + 0.3 * (rank - (world - 1) / 2)), dtype=torch.float64, device=dev)

    def reseed():
        st.phi.copy_(phi0); st.weight.copy_(w0); st.flags.zero_(); st.seed()
    reseed()
    D.run_sharded(ctx, st.phi, st.weight, st.ovlp, st.theta, st.fb, xs, ns, ee, oe, pe, us=[0.37, 0.81], flags=st.flags)   # warm
    reseed()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    l0 = ctx.launch_count
    D.COMB_STATS.clear()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    energies = D.run_sharded(ctx, st.phi, st.weight, st.ovlp, st.theta, st.fb, xs, ns, ee, oe, pe, us=[0.37, 0.81], flags=st.flags)
    e1.record()
    torch.cuda.synchronize()
    ms = D.max_over_ranks(e0.elapsed_time(e1), dev)
    if world > 1:
        dist.barrier()
    if rank == 0:
        sent = [c["bytes_sent_to_peers"] for c in D.COMB_STATS]
        line = dict(metric=METRIC, value=world * nw * ns / (ms * 1e-3), unit=UNIT, n_gpus=world, steps=ns, warmup=ns,
                    ms_per_step=ms / ns, higher_is_better=True, scaling="weak", vs_baseline=None,
                    dtype="tf32x3" if ctx.gemm_path >= 2 else ("f32" if wl.precision == "c64" else "f64"), data="synthetic",
                    config=dict(workload=workload_name(wl), variant=variant, global_walkers=world * nw,
                                parallelism=f"walkers sharded x{world}, global comb", schedule=dict(energy_every=ee, ortho_every=oe, pc_every=pe)),
                    gpu_launches=ctx.launch_count - l0,
                    sharded=dict(combs=len(D.COMB_STATS), record_bytes=ctx.afqmc_comb_record_bytes,
                                 rank0_walkers_sent_to_peers=[c["walkers_sent_to_peers"] for c in D.COMB_STATS],
                                 rank0_bytes_sent_to_peers=sent, allgather_bytes=world * nw * 8, allreduce_bytes_per_measurement=24,
                                 e_mix=[[e.real, e.imag] for e in energies]),
                    note="energy every 20 steps (the paper's schedule), not every step: compare with `schedule`, not with the headline")
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=12)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--cfg", type=int, default=5)
    ap.add_argument("--variant", default="mf")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--gemm-path", type=int, default=0)
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-schedule", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="M < 96: time eager launches only (no CUDA graph replay)")
    ap.add_argument("--sharded", action="store_true", help="NEXT-4: the paper's schedule over a population sharded across the ranks")
    ap.add_argument("--ndet-scan", action="store_true", help="cfg 4 at N_det = 10 / 100 / 1000 (PAPER.md Fig. 1)")
    ap.add_argument("--peaks", action="store_true", help="print the measured peak microbenchmarks only")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.peaks:
        import torch
        print(json.dumps(dict(measured_peaks=measure_peaks(torch.device("cuda:0")), driver_peaks=peaks())))
    elif args.ndet_scan:
        run_ndet_scan(args)
    elif args.sharded:
        run_sharded(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
