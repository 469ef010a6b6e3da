"""GPU parity, round 2 additions (VERDICT r1 "Next round" 1b-1f and the advisor's Taylor edge cases):

  * weight_mode 1 (local-energy weights) through afqmc_propagate and afqmc_step against o_step(mode=1);
  * protocol B (free-running, alive walkers) on cfg 5; full-size sampled-walker checks for cfg 3 (1024 walkers) and
    cfg 4 (512 walkers, 100 determinants);
  * free-running WITH orthonormalisation through afqmc_run(energy_every=1, ortho_every=2): flat 2e-4 on the `tame`
    variants; on the literal / mean-field-subtracted configs graded against the measured error of a plain numpy
    complex64 pipeline on the same walkers (tests/fp32_pipeline.py; tests/test_fp32_floor.py shows why a flat 2e-4 is out
    of reach of any FP32 implementation there);
  * the tensor-pipe Taylor kernel at sizes where its tiles are ragged (M = 97 ... 255, odd N_t), paths 2 and 3.
Raw worst errors go to gpurun_out/parity_raw.jsonl (H.record) and from there to profiles/parity_r2.md."""
import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from workloads import make_workload, random_walkers

from . import fp32_pipeline as F
from . import gpu_harness as H

pytestmark = pytest.mark.gpu

SMALL = {1: 64, 2: 96, 3: 40, 4: 12, 5: 6}


# ---- weight_mode 1 ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("cfg,variant", [(1, "raw"), (2, "raw"), (3, "mf"), (5, "mf")])
def test_weight_mode1_propagate(cfg, variant):
    """One afqmc_propagate with local-energy weights from random non-orthonormal walkers; E_0 != 0 so that the projector
    shift is exercised; eloc_pre comes from afqmc_local_energy.  w' = w exp(-dt (Re E_L(pre) - E_0)) max(0, cos dtheta)."""
    import torch
    wl = make_workload(cfg, variant)
    nw = SMALL[cfg]
    tol = H.tol_for(wl)
    ini, _ = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=5, spread=0.1)
    ost = orc.o_seed_state(ini, phi, wl.n_alpha, w=np.linspace(0.5, 2.0, nw))
    E0 = float(np.median(ost.eloc.real)) + 3.0
    x = wl.fields(1, nw)[0]
    new, rec = orc.o_step(ini, ost, x, wl.n_alpha, K=wl.K, E0=E0, mode=1)
    ctx = H.make_ctx(wl, nw, weight_mode=1, E0=E0)
    st = H.DeviceState(ctx, phi, weight=ost.w)
    st.seed()
    epre = torch.zeros(nw, dtype=torch.complex128, device=ctx.device)
    ctx.afqmc_local_energy(st.phi, st.theta, epre)
    xd = torch.tensor(x, dtype=ctx.rdtype, device=ctx.device)
    ctx.afqmc_propagate(st.phi, xd, st.fb, st.ovlp, st.weight, st.theta, epre, st.flags)
    out = st.host()
    fac = ost.w * np.exp(-wl.dt * (ost.eloc.real - E0))            # un-projected magnitude (R11's weight metric)
    alive_o, alive_g = rec["w"] > 0, out["w"] > 0
    flip = alive_o != alive_g
    assert np.all(np.abs(rec["cosd"][flip]) < tol), "dead/alive flip away from cos = 0"
    errs = dict(phi=H.rel_fro(out["phi"], rec["phi"]), S=H.rel_abs(out["S"], rec["S"]),
                w=float(np.max(np.abs(out["w"] - rec["w"])[~flip] / fac[~flip])),
                Epre=H.rel_abs(epre.cpu().numpy(), ost.eloc))
    killed = (out["flags"] & 4) != 0
    assert np.array_equal(killed[~flip], ~alive_o[~flip])
    print(f"cfg{cfg}/{variant} weight_mode 1 propagate: {errs}, killed {int(killed.sum())}/{nw}")
    H.record("weight_mode1_propagate", cfg=cfg, variant=variant, **errs)
    for k, v in errs.items():
        assert v < tol, (k, v)
    # the two modes really differ on this input (the test would not notice a mode mix-up otherwise)
    _, rec0 = orc.o_step(ini, ost, x, wl.n_alpha, K=wl.K, E0=E0, mode=0)
    assert np.max(np.abs(rec0["w"] - rec["w"])[alive_o] / fac[alive_o]) > 100 * tol


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_weight_mode1_step(cfg):
    """afqmc_step(n_steps = 3) with weight_mode 1 on the `tame` variant: the first step uses E_L of the walkers on entry
    (computed inside the call), every later one the E_L the previous step measured."""
    wl = make_workload(cfg, "tame")
    nw, steps = SMALL[cfg], 3
    tol = H.tol_for(wl)
    ini, _ = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=9, spread=0.05)
    ost = orc.o_seed_state(ini, phi, wl.n_alpha)
    E0 = float(np.median(ost.eloc.real))
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw, weight_mode=1, E0=E0)
    st = H.DeviceState(ctx, phi)
    st.seed()
    eloc = st.step(xs)
    worst = {}
    for n in range(steps):
        ost, rec = orc.o_step(ini, ost, xs[n], wl.n_alpha, K=wl.K, E0=E0, mode=1)
        worst["E"] = max(worst.get("E", 0.0), H.rel_abs(eloc[n], rec["eloc"]))
    out = st.host()
    assert np.all(ost.w > 0)
    worst.update(phi=H.rel_fro(out["phi"], ost.phi), S=H.rel_abs(out["S"], ost.S), w=H.rel_abs(out["w"], ost.w),
                 f=H.rel_fro(out["f"], ost.f_a + ost.f_b))
    print(f"cfg{cfg}/tame weight_mode 1, afqmc_step x{steps}: {worst}")
    H.record("weight_mode1_step", cfg=cfg, **worst)
    for k, v in worst.items():
        assert v < tol, (k, v)
    # and the weights are NOT the hybrid ones
    h = orc.o_seed_state(ini, phi, wl.n_alpha)
    for n in range(steps):
        h, _ = orc.o_step(ini, h, xs[n], wl.n_alpha, K=wl.K, E0=E0, mode=0)
    assert H.rel_abs(out["w"], h.w) > 10 * H.rel_abs(out["w"], ost.w)


# ---- protocol B on cfg 5, full-size sampled walkers for cfg 3 and cfg 4 ------------------------------------------
def test_protocol_B_cfg5():
    """cfg 5 / mf, free-running 10 steps in one afqmc_step call, graded on the walkers alive in the oracle with the
    per-step tolerance accumulated over the steps taken and scaled by the largest kappa met (as protocol B elsewhere)."""
    wl = make_workload(5, "mf")
    nw, steps = SMALL[5], 10
    ini, _ = H.oracle_init(wl)
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, wl.walkers(nw))
    st.seed()
    eloc = st.step(xs)
    ost = orc.o_seed_state(ini, wl.walkers(nw), wl.n_alpha)
    kappa = np.ones(nw)
    worstE, rawE, n_alive = 0.0, 0.0, []
    for n in range(steps):
        ost, rec = orc.o_step(ini, ost, xs[n], wl.n_alpha, K=wl.K, E0=wl.E0)
        with np.errstate(all="ignore"):
            kn = H.cond_number(wl, rec["phi"])
        kappa = np.maximum(kappa, np.where(np.isfinite(kn), kn, np.inf))
        alive = (rec["w"] > 0) & np.isfinite(kappa)
        n_alive.append(int(alive.sum()))
        if np.any(alive):
            e = H.energy_err_w(eloc[n], rec["eloc"], rec["f"])
            worstE = max(worstE, H.worst_ratio(e, (n + 1) * H.walker_tol(wl, kappa), alive))
            rawE = max(rawE, float(np.max(e[alive])))
    out = st.host()
    alive = (ost.w > 0) & np.isfinite(kappa)
    ratio, raw = dict(E=worstE), dict(E=rawE)
    if np.any(alive):
        tw = steps * H.walker_tol(wl, kappa)
        for k, e in (("phi", H.rel_fro_w(out["phi"], ost.phi)), ("S", H.rel_abs_w(out["S"], ost.S)),
                     ("w", H.rel_abs_w(out["w"], ost.w))):
            ratio[k], raw[k] = H.worst_ratio(e, tw, alive), float(np.max(e[alive]))
    print(f"cfg5/mf protocol B alive per step {n_alive}: err/tol {ratio} raw {raw} kappa max {kappa[np.isfinite(kappa)].max():.0f}")
    H.record("protocol_B_cfg5", alive_last=n_alive[-1], **{f"raw_{k}": v for k, v in raw.items()})
    assert n_alive[0] > 0
    for k, v in ratio.items():
        assert v < 1.0, (k, v)


def test_full_size_cfg3_sampled_walkers():
    """cfg 3 at its full 1024 walkers (the launch configuration `bench.py --cfg 3` times), two free-running steps, sampled
    walkers recomputed one by one by the oracle; flat tolerance."""
    wl = make_workload(3, "mf")
    nw, steps = wl.n_walkers, 2
    tol = H.tol_for(wl)
    ini, _ = H.oracle_init(wl)
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, wl.walkers(nw))
    st.seed()
    eloc = st.step(xs)
    out = st.host()
    idx = np.array([0, 1, 127, 128, 255, 256, 511, 640, 777, 1022, 1023])
    ost = orc.o_seed_state(ini, wl.walkers(nw)[idx], wl.n_alpha)
    for n in range(steps):
        ost, rec = orc.o_step(ini, ost, xs[n][idx], wl.n_alpha, K=wl.K, E0=wl.E0)
    errs = dict(phi=H.rel_fro(out["phi"][idx], ost.phi), S=H.rel_abs(out["S"][idx], ost.S),
                w=H.rel_abs(out["w"][idx], ost.w), f=H.rel_fro(out["f"][idx], ost.f_a + ost.f_b),
                E=H.rel_abs(eloc[-1][idx], rec["eloc"]))
    print(f"cfg3 full size (path {ctx.gemm_path}), sampled walkers: {errs}")
    H.record("full_size_cfg3", **errs)
    assert np.all(np.isfinite(out["phi"].view(np.float64)))
    for k, v in errs.items():
        assert v < tol, (k, v)


def test_full_size_cfg4_sampled_walkers():
    """cfg 4 at its full size (512 walkers, 100 determinants: the configuration in which k_md_energy_b and the TT GEMM
    are timed): stage quantities on random walkers and one full step, on sampled walkers against the oracle's definition
    path (every determinant recomputed directly)."""
    import torch
    wl = make_workload(4, "mf")
    nw = wl.n_walkers
    tol = H.tol_for(wl)
    ini, trial = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=11, spread=0.2)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, phi)
    st.seed()
    eloc0 = torch.zeros(nw, dtype=torch.complex128, device=ctx.device)
    ctx.afqmc_local_energy(st.phi, st.theta, eloc0)
    g0 = st.host()
    idx = np.array([0, 1, 127, 128, 255, 256, 300, 510, 511])
    S, f, E = orc.o_multidet_definition(ini, trial, phi[idx], wl.n_alpha)
    errs = dict(S=H.rel_abs(g0["S"][idx], S), f=H.rel_fro(g0["f"][idx], f), E=H.rel_abs(eloc0.cpu().numpy()[idx], E))
    x = wl.fields(1, nw)
    eloc = st.step(x)
    out = st.host()
    ost = orc.o_seed_state(ini, phi[idx], wl.n_alpha, trial=trial)
    new, rec = orc.o_step(ini, ost, x[0][idx], wl.n_alpha, K=wl.K, E0=wl.E0, trial=trial)
    kappa = np.maximum(H.cond_number(wl, phi[idx]), H.cond_number(wl, rec["phi"]))
    tw = H.walker_tol(wl, kappa)
    den_w = np.where(rec["absI"] > 0, rec["absI"], 1.0)
    step_e = dict(phi=H.rel_fro_w(out["phi"][idx], rec["phi"]), S1=H.rel_abs_w(out["S"][idx], rec["S"]),
                  f1=H.rel_fro_w(out["f"][idx], rec["f"]), E1=H.energy_err_w(eloc[0][idx], rec["eloc"], rec["f"]),
                  w=np.abs(out["w"][idx] - rec["w"]) / den_w)
    print(f"cfg4 full size (512 walkers, 100 dets), stage {errs}; one step raw {({k: float(v.max()) for k, v in step_e.items()})} "
          f"kappa max {kappa.max():.0f}")
    H.record("full_size_cfg4", **errs, **{k: float(v.max()) for k, v in step_e.items()})
    for k, v in errs.items():
        assert v < tol, (k, v)
    amp_w = np.maximum(1.0, wl.dt * np.sum(np.abs(rec["f_used"]) ** 2, axis=-1))
    for k, v in step_e.items():
        assert np.all(v < (tw * amp_w if k == "w" else tw)), (k, float(v.max()))


# ---- free-running with orthonormalisation through afqmc_run ------------------------------------------------------
def _run_ortho(wl, nw, steps, idx=None):
    """afqmc_run(energy_every = 1, ortho_every = 2) on the device; the oracle and the plain complex64 pipeline follow the
    same schedule.  Returns per-step error arrays (GPU vs oracle, complex64 pipeline vs oracle) over the selected walkers."""
    import torch
    ini, _ = H.oracle_init(wl)
    i32 = F.init32(wl, ini)
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, wl.walkers(nw))
    st.seed()
    xd = torch.tensor(np.ascontiguousarray(xs), dtype=ctx.rdtype, device=ctx.device)
    eloc = torch.zeros(steps, nw, dtype=torch.complex128, device=ctx.device)
    wm = torch.zeros(steps, nw, dtype=torch.float64, device=ctx.device)
    ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, steps, 1, 2, 0, None, eloc, wm, None, st.flags)
    out = st.host()
    eloc, wm = eloc.cpu().numpy(), wm.cpu().numpy()
    sel = np.arange(nw) if idx is None else idx
    ost = orc.o_seed_state(ini, wl.walkers(nw)[sel], wl.n_alpha)
    s32 = F.seed32(i32, wl.walkers(nw)[sel], wl.n_alpha)
    per_step = []
    kappa = np.ones(sel.shape[0])
    for n in range(1, steps + 1):
        w_prev = ost.w
        ost, rec = orc.o_step(ini, ost, xs[n - 1][sel], wl.n_alpha, K=wl.K, E0=wl.E0)
        s32 = F.step32(i32, s32, xs[n - 1][sel], wl.n_alpha, K=wl.K, E0=wl.E0)
        alive = (ost.w > 0) & np.isfinite(ost.eloc) & np.isfinite(ost.S)
        # R11: weight errors are measured against the UN-PROJECTED magnitude w e^{dt E0} |I| (cos dtheta -> 0 makes the plain
        # relative error unbounded for a walker about to be killed)
        den = w_prev * np.exp(wl.dt * wl.E0) * rec["absI"]
        den = np.where(den > 0, den, 1.0)
        with np.errstate(all="ignore"):
            kn = H.cond_number(wl, ost.phi)
        kappa = np.maximum(kappa, np.where(np.isfinite(kn), kn, np.inf))
        per_step.append(dict(alive=alive & np.isfinite(kappa), kappa=kappa.copy(),
                             amp_w=np.maximum(1.0, wl.dt * np.sum(np.abs(rec["f_used"]) ** 2, axis=-1)),
                             E_gpu=H.energy_err_w(eloc[n - 1][sel], ost.eloc, rec["f"]), E_32=H.energy_err_w(s32.eloc, ost.eloc, rec["f"]),
                             w_gpu=np.abs(wm[n - 1][sel] - ost.w) / den, w_32=np.abs(s32.w - ost.w) / den))
        if n % 2 == 0:
            q, s = orc.o_orthonormalize(ost.phi, ost.S, wl.n_alpha)
            ost = orc.OracleState(q, ost.w, s, ost.theta, ost.f_a, ost.f_b, ost.eloc)
            s32 = F.ortho32(s32, wl.n_alpha)
    final = dict(alive=(ost.w > 0) & np.isfinite(ost.S) & np.isfinite(kappa), kappa=kappa,
                 phi_gpu=H.rel_fro_w(out["phi"][sel], ost.phi), phi_32=H.rel_fro_w(s32.phi.astype(np.complex128), ost.phi),
                 S_gpu=H.rel_abs_w(out["S"][sel], ost.S), S_32=H.rel_abs_w(s32.S, ost.S),
                 f_gpu=H.rel_fro_w(out["f"][sel], ost.f_a + ost.f_b, H.fb_floor(ini)),
                 f_32=H.rel_fro_w((s32.fa + s32.fb).astype(np.complex128), ost.f_a + ost.f_b, H.fb_floor(ini)))
    return per_step, final, out


@pytest.mark.parametrize("cfg,variant", [(2, "tame"), (2, "tame_mf"), (3, "tame"), (3, "tame_mf"), (5, "tame"), (5, "tame_mf")])
def test_free_run_ortho_flat_tolerance(cfg, variant):
    """10 free-running steps (cfg 2: 20) through afqmc_run with E_L every step and orthonormalisation every 2,
    `tame` variants (||A||_2 ~ 0.2, the regime of molecule-like Cholesky vectors): every walker, flat 2e-4, no kappa scaling,
    no step accumulation."""
    wl = make_workload(cfg, variant)
    nw, steps = SMALL[cfg], (20 if cfg == 2 else 10)
    tol = H.tol_for(wl)
    per_step, final, out = _run_ortho(wl, nw, steps)
    assert all(np.all(p["alive"]) for p in per_step)
    worst = dict(E=max(float(p["E_gpu"].max()) for p in per_step), w=max(float(p["w_gpu"].max()) for p in per_step),
                 phi=float(final["phi_gpu"].max()), S=float(final["S_gpu"].max()), f=float(final["f_gpu"].max()))
    ref32 = dict(E=max(float(p["E_32"].max()) for p in per_step), w=max(float(p["w_32"].max()) for p in per_step),
                 phi=float(final["phi_32"].max()), S=float(final["S_32"].max()), f=float(final["f_32"].max()))
    q = out["phi"][:, :, :wl.n_alpha]
    qhq = float(np.abs(np.einsum("wia,wib->wab", q.conj(), q) - np.eye(wl.n_alpha)).max())
    print(f"cfg{cfg}/{variant} afqmc_run E/1 QR/2, {steps} free-running steps: GPU {worst}; plain complex64 numpy {ref32}; |Q^H Q - 1| {qhq:.1e}")
    H.record("free_run_ortho_flat", cfg=cfg, variant=variant, steps=steps, **worst, **{f"numpy_c64_{k}": v for k, v in ref32.items()})
    assert qhq < 1e-5
    for k, v in worst.items():
        assert v < tol, (k, v)


@pytest.mark.parametrize("cfg,variant", [(2, "raw"), (2, "mf"), (3, "raw"), (3, "mf"), (5, "raw"), (5, "mf")])
def test_free_run_ortho_vs_fp32_floor(cfg, variant):
    """The same schedule on the literal / mean-field-subtracted configs (violent: ||A||_2 ~ 1.8, walkers die within ~8 steps,
    errors of ANY FP32 pipeline are amplified chaotically once kappa grows -- tests/test_fp32_floor.py).  Graded over the walkers
    alive in the oracle, per step, two ways:
      * the TYPICAL walker (median, steps with >= 4 alive) against the measured floor, no kappa model: median error <=
        max(2e-4, 16 x median error of the plain numpy complex64 pipeline on the same walkers).  Why 16: at step 1 (kappa ~ 2,
        nothing amplified yet) the 3xTF32 tensor-pipe GEMMs leave S at 4e-6 where plain FP32 leaves 4e-7 (the tensor pipe
        accumulates with truncation; gemm_path 1 reproduces the numpy figures digit for digit);
      * the WORST walker against protocol B's budget (per-step tolerance scaled by the largest kappa met, times the steps taken):
        the maximum over a chaotic ensemble is a single-sample quantity, two FP32 pipelines differ by an order of magnitude on it."""
    wl = make_workload(cfg, variant)
    nw, steps = SMALL[cfg], 10
    tol = H.tol_for(wl)
    per_step, final, out = _run_ortho(wl, nw, steps)
    med_ratio, worst_ratio, raw, raw32, n_alive = 0.0, 0.0, {}, {}, []
    for n, p in enumerate(per_step):
        a = p["alive"]
        n_alive.append(int(a.sum()))
        if not np.any(a):
            continue
        tw = (n + 1) * H.walker_tol(wl, p["kappa"])
        for k in ("E", "w"):
            g, r = p[f"{k}_gpu"][a], p[f"{k}_32"][a]
            raw[k], raw32[k] = max(raw.get(k, 0.0), float(g.max())), max(raw32.get(k, 0.0), float(r.max()))
            # log w' contains c = x.xbar - xbar.xbar/2 of size dt ||f||^2 (protocol A): the weight budget carries that factor,
            # accumulated like the rest
            amp = np.maximum.accumulate(np.stack([q["amp_w"] for q in per_step[:n + 1]]), axis=0)[-1][a] if k == "w" else 1.0
            worst_ratio = max(worst_ratio, float(np.max(g / (tw[a] * amp))))
            if a.sum() >= 4:
                med_ratio = max(med_ratio, float(np.median(g)) / max(tol, 16 * float(np.median(r))))
    a = final["alive"]
    if np.any(a):
        tw = steps * H.walker_tol(wl, final["kappa"])
        for k in ("phi", "S", "f"):
            g, r = final[f"{k}_gpu"][a], final[f"{k}_32"][a]
            raw[k], raw32[k] = float(g.max()), float(r.max())
            worst_ratio = max(worst_ratio, float(np.max(g / tw[a])))
    print(f"cfg{cfg}/{variant} afqmc_run E/1 QR/2, 10 free-running steps, alive per step {n_alive}: GPU raw max {raw}; "
          f"plain complex64 numpy max {raw32}; median err / max(2e-4, 16 x numpy median) = {med_ratio:.3f}; worst err / protocol-B budget = {worst_ratio:.3f}")
    H.record("free_run_ortho_vs_floor", cfg=cfg, variant=variant, alive=n_alive, median_ratio=med_ratio, worst_ratio=worst_ratio,
             **{f"gpu_{k}": v for k, v in raw.items()}, **{f"numpy_c64_{k}": v for k, v in raw32.items()})
    assert n_alive[0] > 0
    assert med_ratio < 1.0 and worst_ratio < 1.0
    assert np.all(np.isfinite(out["phi"].view(np.float64)[np.isfinite(out["w"]) & (out["w"] > 0)]))


# ---- tensor-pipe Taylor kernel: ragged tiles (advisor, round 1) --------------------------------------------------
@pytest.mark.parametrize("path", [2, 3])
@pytest.mark.parametrize("M,na,nb,ng,nw", [(97, 3, 2, 37, 5), (101, 5, 4, 33, 3), (128, 7, 6, 64, 4), (130, 4, 3, 41, 6),
                                           (255, 9, 8, 50, 3), (256, 16, 16, 40, 2), (96, 1, 0, 33, 7), (200, 13, 12, 70, 149)])
def test_taylor_tc_ragged_sizes(M, na, nb, ng, nw, path):
    """96 <= M <= 256 runs tt::k_taylor_tc: M = 97 / 101 (one tile, rows_last rounded up past M, MP > M), 128 (exactly one
    tile), 130 (two tiles, the second almost empty: its TMA box reaches into the next walker's rows), 255 / 256 (two full
    tiles; 256 with N_t = 32 is the largest shape), M % 4 != 0 (non-staged assembly epilogue + k_symmetrize writing the lo
    plane), n_beta = 0, and more walkers than SMs (persistent loop, walker boundary).  Two full steps against o_step."""
    wl = make_workload(5, "tame", overrides=dict(M=M, n_alpha=na, n_beta=nb, n_chol=ng, n_walkers=nw, sigma_L=0.3 * (200.0 / M) ** 0.5 * (1000.0 / ng) ** 0.5 * 0.1))
    tol = H.tol_for(wl)
    ini, _ = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=3, spread=0.1)
    ost = orc.o_seed_state(ini, phi, wl.n_alpha)
    ctx = H.make_ctx(wl, nw, gemm_path=path)
    assert ctx.gemm_path == path
    st = H.DeviceState(ctx, phi)
    st.seed()
    xs = wl.fields(2, nw)
    eloc = st.step(xs)
    for n in range(2):
        ost, rec = orc.o_step(ini, ost, xs[n], wl.n_alpha, K=wl.K)
    out = st.host()
    errs = dict(phi=H.rel_fro(out["phi"], ost.phi), S=H.rel_abs(out["S"], ost.S), E=H.rel_abs(eloc[-1], rec["eloc"]),
                f=H.rel_fro(out["f"], ost.f_a + ost.f_b, H.fb_floor(ini)), w=H.rel_abs(out["w"], ost.w))
    print(f"taylor_tc M={M} N=({na},{nb}) Ng={ng} Nw={nw} path {path}: {errs}")
    H.record("taylor_tc_ragged", M=M, na=na, nb=nb, path=path, **errs)
    assert np.all(ost.w > 0)
    for k, v in errs.items():
        assert v < tol, (k, v)


def test_large_M_accepted_on_tensor_path_only():
    """check_params no longer applies the one-CTA SIMT Taylor kernel's size limit where the tensor-pipe kernel runs
    (advisor, round 1): M = 256, N_t = 32 complex64 is accepted on gemm_path 0/2/3 and rejected on the SIMT path."""
    import paper_1804_03310_b200 as afq
    for gp, ok in ((0, True), (2, True), (3, True), (1, False)):
        p = afq.make_params(256, 16, 16, 40, 2, "c64", 0.005, gemm_path=gp)
        if ok:
            afq.afqmc_query_bytes(p)
        else:
            with pytest.raises(afq.AfqmcError) as ei:
                afq.afqmc_query_bytes(p)
            assert ei.value.status == afq.AFQMC_EUNSUPPORTED


def test_multidet_large_expansion():
    """N_det = 1000 (the paper's expansions reach 1266 determinants, Fig. 1 :68): S, mixed f and mixed E_L on
    random walkers against the oracle's definition path.  Runs the general multi-determinant energy kernel (8 determinants
    per thread) with Z read from its FP64 copy -- a second copy does not fit one CTA's shared memory at this size."""
    import torch
    wl = make_workload(4, "raw", overrides=dict(n_det=1000))
    nw = 4
    tol = H.tol_for(wl)
    ini, trial = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=11, spread=0.2)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, phi)
    st.seed()
    eloc = torch.zeros(nw, dtype=torch.complex128, device=ctx.device)
    ctx.afqmc_local_energy(st.phi, st.theta, eloc)
    out = st.host()
    S, f, E = orc.o_multidet_definition(ini, trial, phi, wl.n_alpha)
    errs = dict(S=H.rel_abs(out["S"], S), f=H.rel_fro(out["f"], f), E=H.rel_abs(eloc.cpu().numpy(), E))
    print(f"cfg4 shapes, 1000 determinants: {errs}")
    H.record("multidet_1000", **errs)
    for k, v in errs.items():
        assert v < tol, (k, v)


def _high_rank_trial(wl, n_det, seed=5):
    """Determinants with excitation rank 0..4 per spin (in-place column replacement, distinct holes / particles per spin)."""
    rng = np.random.default_rng(seed)
    exc = -np.ones((n_det, 2, 4, 2), dtype=np.int32)
    seen = {()}
    i = 1
    while i < n_det:
        key = []
        for s, n in enumerate((wl.n_alpha, wl.n_beta)):
            rk = int(rng.integers(0, 5)) if i > 4 else (i if s == 0 else 4 - (i - 1))      # dets 1-4 force ranks (1,4) (2,3) (3,2) (4,1)
            rk = min(rk, n, wl.n_act - n)
            holes = rng.permutation(n)[:rk]
            parts = n + rng.permutation(wl.n_act - n)[:rk]
            key += [(s, int(h), int(p)) for h, p in zip(holes, parts)]
        if not key or tuple(sorted(key)) in seen:
            continue
        seen.add(tuple(sorted(key)))
        cnt = [0, 0]
        for s, h, p in key:
            exc[i, s, cnt[s]] = (h, p)
            cnt[s] += 1
        i += 1
    c = rng.standard_normal(n_det)
    c[0] = 3.0
    return c / np.linalg.norm(c), exc


@pytest.mark.parametrize("path", [0, 1])
def test_multidet_excitation_rank_up_to_4(path):
    """excitation rank > 2.  Eq. (4) holds for any rank E_i; the GPU inverts the E x E matrices
    Q[P_i, H_i] by a small pivoted elimination for E = 3, 4 (closed forms for E <= 2).  S, mixed G, mixed f, mixed E_L and one full
    step against the oracle's definition path (every determinant recomputed directly)."""
    import torch
    wl = make_workload(4, "raw", overrides=dict(M=26, n_alpha=6, n_beta=5, n_chol=22, n_act=12, n_det=2, n_walkers=8))
    wl.n_det = 24
    wl.det_coeff, wl.det_exc = _high_rank_trial(wl, wl.n_det)
    ranks = {(int((wl.det_exc[i, 0, :, 0] >= 0).sum()), int((wl.det_exc[i, 1, :, 0] >= 0).sum())) for i in range(wl.n_det)}
    assert {(1, 4), (2, 3), (3, 2), (4, 1)} <= ranks
    nw = 8
    tol = H.tol_for(wl)
    ini, trial = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=11, spread=0.25)
    ctx = H.make_ctx(wl, nw, gemm_path=path)
    st = H.DeviceState(ctx, phi)
    G = torch.zeros(nw, 2, wl.M, wl.M, dtype=ctx.cdtype, device=ctx.device)
    ctx.afqmc_overlap_green(st.phi, st.ovlp, st.theta, G, st.flags)
    ctx.afqmc_force_bias(st.phi, st.theta, st.fb)
    eloc = torch.zeros(nw, dtype=torch.complex128, device=ctx.device)
    ctx.afqmc_local_energy(st.phi, st.theta, eloc)
    out = st.host()
    S, f, E, Gref = orc.o_multidet_definition(ini, trial, phi, wl.n_alpha, want_G=True)
    errs = dict(S=H.rel_abs(out["S"], S), G=H.rel_fro(G.cpu().numpy().astype(np.complex128), Gref),
                f=H.rel_fro(out["f"], f), E=H.rel_abs(eloc.cpu().numpy(), E))
    x = wl.fields(1, nw)
    e1 = st.step(x)
    o1 = st.host()
    ost = orc.o_seed_state(ini, phi, wl.n_alpha, trial=trial)
    new, rec = orc.o_step(ini, ost, x[0], wl.n_alpha, K=wl.K, E0=wl.E0, trial=trial)
    kappa = np.maximum(H.cond_number(wl, phi), H.cond_number(wl, rec["phi"]))
    tw = H.walker_tol(wl, kappa)
    step = dict(phi=H.rel_fro_w(o1["phi"], rec["phi"]), S1=H.rel_abs_w(o1["S"], rec["S"]),
                E1=H.energy_err_w(e1[0], rec["eloc"], rec["f"]))
    print(f"rank <= 4 trial ({wl.n_det} determinants, gemm_path {ctx.gemm_path}): stage {errs}; step {({k: float(v.max()) for k, v in step.items()})}")
    H.record("multidet_rank4", path=path, **errs, **{k: float(v.max()) for k, v in step.items()})
    assert np.all(out["flags"] == 0)
    for k, v in errs.items():
        assert v < tol, (k, v)
    for k, v in step.items():
        assert np.all(v < tw), (k, float(v.max()))
