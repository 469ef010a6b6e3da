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
    while True:
        ost = orc.o_seed_state(ini, wl.walkers(nw), wl.n_alpha, trial=trial)
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
                      f"({t_total:.1f} s CPU wall, numpy/BLAS threads = all {cores} cores, init excluded)")
    if one_thread_s > 0:
        # the paper's comparator is ONE CPU core in double precision: same oracle, BLAS limited to 1 thread
        try:
            from threadpoolctl import threadpool_limits
            n1 = min(wl.n_walkers, 4)
            ost = orc.o_seed_state(ini, wl.walkers(n1), wl.n_alpha, trial=trial)
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

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    pk = peaks()
    fl = flops_per_walker_step(wl)
    value = D.whole_job_rate(nw * K, world, ms_max * 1e-3)
    # roofline of the dominant kernel = the stage with the largest device time (CUDA events on the launching
    # stream, afqmc_profile_*); the H6 assembly GEMM is always reported beside it as `roofline_h6`
    M_, ng_ = wl.M, wl.n_chol
    if ctx.gemm_path >= 2:
        # the tcgen05 assembly GEMM exploits A = A^T: its algorithmic work is the upper triangle only
        fl["assemble"] = 4.0 * ng_ * M_ * (M_ + 1) / 2
        peak, peak_note = 0.5 * pk["bf16_burst"], (
            f"TF32 dense = {pk['source']} burst BF16 {pk['bf16_burst']} TF/s x nominal TF32/BF16 ratio 0.5 (each kernel runs "
            f"0.2-1.6 ms inside a ~3.4 ms step, no power-cap reason active; sustained figure would be {0.5 * pk['bf16_sust']:.0f}); "
            "achieved counts ALGORITHMIC flops and 3xTF32 issues 3x of them, so frac <= 1/3 by construction")
        bound, dtype = "tensor", "tf32x3"
    else:
        fp32_peak = 148 * 128 * 2 * pk["sm_max_mhz"] * 1e6 / 1e12
        bound, peak, peak_note = "alu", fp32_peak, "FP32 FMA: 148 SMs x 128 lanes x 2 flop x clocks.max.sm (DESIGN.md)"
        dtype = "f32" if wl.precision == "c64" else "f64"
        if wl.precision == "c128":
            peak, peak_note = fp32_peak / 2, "FP64 FMA: 148 SMs x 64 lanes x 2 flop x clocks.max.sm (DESIGN.md)"
    names = dict(assemble="H6 assembly GEMM A_w = sum_g z_g L_g (tc::k_gemm_tf32_pair<EpiAssembleSym> / k_gemm_tf32 / k_gemm_nt)",
                 taylor="H7 Taylor propagator (tt::k_taylor_tc / k_taylor)",
                 energy="H9 energy GEMMs + fused dot (or H10 multi-det energy)", force_bias="H4 force-bias GEMMs",
                 green="H1-H3/H8 overlap, LU, Theta, weights (k_green)")
    traffic_ncu = {"assemble": 2.227e9, "taylor": 2.131e9} if (ctx.gemm_path >= 2 and args.cfg == 5) else {}

    def roof(stage):
        ms, n = prof[stage]
        if not n or ms <= 0 or stage not in fl:
            return None
        ach = fl[stage] * nw * n / (ms * 1e-3) / 1e12
        r = dict(bound=bound, kernel=names[stage], achieved=ach, peak=peak, unit="TFLOP/s", frac=ach / peak,
                 traffic=traffic_ncu.get(stage), peak_source=peak_note, launches_timed=n, ms_per_launch=ms / n)
        if ctx.gemm_path >= 2:
            r["issued_frac"] = 3.0 * ach / peak
        if stage == "green":      # HBM-bound stage: bytes, not flops
            cb = 8 if wl.precision == "c64" else 16
            byts = nw * wl.M * wl.n_t * cb * (2 + (2 if ctx.gemm_path >= 2 else 1))
            r.update(bound="hbm", achieved=byts * n / (ms * 1e-3) / 1e9, peak=pk["hbm"], unit="GB/s",
                     peak_source=f"{pk['source']} HBM copy bandwidth")
            r["frac"] = r["achieved"] / r["peak"]
            r.pop("issued_frac", None)
        return r

    timed = {k: v[0] / v[1] for k, v in prof.items() if v[1] and k in names}
    dominant = max(timed, key=timed.get) if timed else "assemble"
    stage_ms = {k: (v[0] / v[1] if v[1] else None) for k, v in prof.items()}
    stage_tflops = {k: (fl[k] * nw / (stage_ms[k] * 1e-3) / 1e12 if stage_ms.get(k) else None) for k in fl}
    base = None
    if not args.no_cpu_baseline:
        base = time_oracle(wl, target_s=args.cpu_seconds, one_thread_s=min(6.0, args.cpu_seconds / 2))
    line = dict(metric=METRIC, value=value, unit=UNIT, n_gpus=world, steps=K, warmup=W, ms_per_step=ms_max / K,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype=dtype, data="synthetic",
                config=dict(workload=workload_name(wl), variant=args.variant, global_walkers=world * nw,
                            parallelism=f"replicas x{world}" if world > 1 else "single GPU",
                            l2="per-step working set (A_w buffer %.0f MB + operands) exceeds the 126 MB L2; no flush"
                               % (nw * wl.M * wl.M * 2 * (4 if wl.precision == "c64" else 8) / 1e6),
                            gemm_path={1: "simt", 2: "tcgen05-3xtf32", 3: "tcgen05-3xtf32-ctapair"}[ctx.gemm_path]),
                clocks=clocks, gpu_launches=launches,
                e2e=dict(value=world * nw * Ke / t_e2e, unit=UNIT, h2d_bytes_per_step=up / Ke, d2h_bytes_per_step=down / Ke,
                         steps=Ke, note="afqmc_step_host: pinned host buffers, H2D of walkers+fields and D2H of "
                                        "walkers/weights/overlaps/energies inside the timed region"),
                roofline=roof(dominant), roofline_h6=roof("assemble"),
                stages_ms=stage_ms, stages_tflops=stage_tflops, schedule=sched, cpu_baseline=base)
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
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
