"""GPU parity: the CUDA path (through the C-ABI binding) against the FP64 oracle, same seeded inputs.

Protocols:
  stage  : each entry point alone on random complex non-orthonormal walkers
  A      : per-step re-synchronised, all walkers, 10 steps
  B      : free-running from the common initial state, graded on walkers alive in the oracle
  C      : free-running on the `tame` variant (sigma_L / 10), all walkers
Tolerances: 1e-5 (FP64 path) / 2e-4 (FP32 path) per north_star.
"""
import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from workloads import make_workload, random_walkers

from . import gpu_harness as H

pytestmark = pytest.mark.gpu

# (cfg, variant, n_walkers used in the element-by-element comparison, steps)
SMALL = {1: 64, 2: 96, 3: 40, 4: 12, 5: 6}


def _wl(cfg, variant="raw"):
    return make_workload(cfg, variant)


@pytest.mark.parametrize("cfg", [1, 2, 3, 5])
def test_stage_overlap_green_forcebias_energy(cfg):
    import torch
    wl = _wl(cfg)
    nw = SMALL[cfg]
    tol = H.tol_for(wl)
    ini, _ = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=11)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, phi)
    G = torch.zeros(nw, 2, wl.M, wl.M, dtype=ctx.cdtype, device=ctx.device)
    ctx.afqmc_overlap_green(st.phi, st.ovlp, st.theta, G, st.flags)
    ctx.afqmc_force_bias(st.phi, st.theta, st.fb)
    eloc = torch.zeros(nw, dtype=torch.complex128, device=ctx.device)
    ctx.afqmc_local_energy(st.phi, st.theta, eloc)
    out = st.host()
    S, theta, Gref = orc.o_green(wl.psi_a, wl.psi_b, phi, want_G=True)
    fa, fb = orc.o_force_bias(ini["R"], theta, wl.n_alpha)
    E = orc.o_local_energy(ini, theta, fa, fb, wl.n_alpha)
    errs = dict(S=H.rel_abs(out["S"], S), theta=H.rel_fro(out["theta"], theta),
                G=H.rel_fro(G.cpu().numpy().astype(np.complex128), Gref), f=H.rel_fro(out["f"], fa + fb),
                E=H.rel_abs(eloc.cpu().numpy(), E))
    print(f"cfg{cfg} stage errors: {errs}")
    H.record("stage", cfg=cfg, **errs)
    assert np.all(out["flags"] == 0)
    for k, v in errs.items():
        assert v < tol, (k, v)


@pytest.mark.parametrize("path", [0, 1])
def test_stage_multidet_overlap_forcebias_energy(path):
    """cfg 4 (100 determinants): S, mixed G, mixed f, mixed E_L against the oracle's DEFINITION path (every
    determinant recomputed directly) -- the GPU uses SMW rank-E closed forms (Eq.(4)).  path 0: tcgen05 GEMMs and the
    batched-gamma energy kernel; path 1: SIMT GEMMs and the one-operator-at-a-time energy kernel."""
    import torch
    wl = _wl(4)
    nw = SMALL[4]
    tol = H.tol_for(wl)
    ini, trial = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=11, spread=0.2)
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
    print(f"cfg4 multi-det stage errors (gemm_path {ctx.gemm_path}): {errs}")
    for k, v in errs.items():
        assert v < tol, (k, v)


@pytest.mark.parametrize("cfg", [1, 2, 3, 5])
def test_stage_propagate(cfg):
    import torch
    wl = _wl(cfg)
    nw = SMALL[cfg]
    tol = H.tol_for(wl)
    ini, _ = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=5, spread=0.1)
    ost = orc.o_seed_state(ini, phi, wl.n_alpha)
    x = wl.fields(1, nw)[0]
    new, rec = orc.o_step(ini, ost, x, wl.n_alpha, K=wl.K, E0=wl.E0)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, phi)
    st.seed()
    xd = torch.tensor(x, dtype=ctx.rdtype, device=ctx.device)
    ctx.afqmc_propagate(st.phi, xd, st.fb, st.ovlp, st.weight, st.theta, None, st.flags)
    out = st.host()
    errs = dict(phi=H.rel_fro(out["phi"], rec["phi"]), S=H.rel_abs(out["S"], rec["S"]),
                theta=H.rel_fro(out["theta"], rec["theta"]),
                w=H.weight_err(out["w"], rec, ost.w, wl.dt, wl.E0))
    print(f"cfg{cfg} propagate errors: {errs}")
    for k, v in errs.items():
        assert v < tol, (k, v)


def _protocol_A(wl, nw, steps, gemm_path=0):
    """Per-step re-synchronised: the GPU starts every step from the oracle's recorded state.  Every walker
    is graded; its tolerance is H.walker_tol (stated tolerance, scaled by cond(A)/100 beyond 100 on FP32)."""
    tol = H.tol_for(wl)
    ini, trial = H.oracle_init(wl)
    ost = orc.o_seed_state(ini, H.start_walkers(wl, nw), wl.n_alpha, trial=trial)
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw, gemm_path=gemm_path)
    ratio, raw, kmax = {}, {}, 1.0
    floor = H.fb_floor(ini)
    for n in range(steps):
        new, rec = orc.o_step(ini, ost, xs[n], wl.n_alpha, K=wl.K, E0=wl.E0, trial=trial)
        st = H.DeviceState(ctx, ost.phi, weight=ost.w)
        st.seed()
        g0 = st.host()
        eloc = st.step(xs[n:n + 1])[0]
        out = st.host()
        ok = np.isfinite(rec["S"]) & np.isfinite(rec["eloc"])
        kappa = np.maximum(H.cond_number(wl, ost.phi), H.cond_number(wl, rec["phi"]))
        ok &= np.isfinite(kappa)
        tw = H.walker_tol(wl, np.where(np.isfinite(kappa), kappa, 1.0))
        kmax = max(kmax, float(np.max(kappa[ok])))
        den_w = ost.w * np.exp(wl.dt * wl.E0) * rec["absI"]
        den_w = np.where(den_w > 0, den_w, 1.0)
        errs = dict(S0=H.rel_abs_w(g0["S"], ost.S), f_used=H.rel_fro_w(g0["f"], rec["f_used"], floor),
                    phi=H.rel_fro_w(out["phi"], rec["phi"]), S=H.rel_abs_w(out["S"], rec["S"]),
                    f=H.rel_fro_w(out["f"], rec["f"], floor), E=H.energy_err_w(eloc, rec["eloc"], rec["f"]),
                    w=np.abs(out["w"] - rec["w"]) / den_w)
        # a dead/alive flip is accepted iff |cos dtheta|_ora < tolerance of that walker
        flip = ((out["w"] == 0) != (rec["w"] == 0)) & ok
        assert np.all(np.abs(rec["cosd"][flip]) < tw[flip]), "dead/alive flip away from cos=0"
        ok_w = ok & ~flip
        # log w' contains c = x.xbar - xbar.xbar/2 of size dt ||f||^2: a relative error eps in f moves log w' by
        # eps * dt ||f||^2, so the weight tolerance carries that factor (raw configs: ||f||^2 ~ 1e3..1e4)
        amp_w = np.maximum(1.0, wl.dt * np.sum(np.abs(rec["f_used"]) ** 2, axis=-1))
        for k, v in errs.items():
            m = ok_w if k == "w" else ok
            ratio[k] = max(ratio.get(k, 0.0), H.worst_ratio(v, tw * amp_w if k == "w" else tw, m))
            raw[k] = max(raw.get(k, 0.0), float(np.max(v[m])) if np.any(m) else 0.0)
        ost = new
    print(f"cfg{wl.cfg}/{wl.variant} protocol A over {steps} steps, {nw} walkers (max cond {kmax:.0f}): "
          f"worst err/tol {({k: round(v, 3) for k, v in ratio.items()})} raw {({k: float('%.2g' % v) for k, v in raw.items()})}")
    for k, v in ratio.items():
        assert v < 1.0, (k, v, raw[k])
    return raw


@pytest.mark.parametrize("cfg,variant", [(1, "raw"), (1, "mf"), (2, "raw"), (2, "mf"), (3, "raw"), (3, "mf"), (4, "raw"), (4, "mf"),
                                         (5, "raw"), (5, "mf")])
def test_protocol_A_resync(cfg, variant):
    """north_star: "per step, over 10 steps" -- 10 steps on every config."""
    wl = _wl(cfg, variant)
    raw = _protocol_A(wl, SMALL[cfg], 10)
    H.record("protocol_A", cfg=cfg, variant=variant, steps=10, **raw)


def _free_run(wl, nw, steps):
    ini, trial = H.oracle_init(wl)
    ost = orc.o_seed_state(ini, H.start_walkers(wl, nw), wl.n_alpha, trial=trial)
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, H.start_walkers(wl, nw))
    st.seed()
    eloc = st.step(xs)           # one afqmc_step call over all steps
    recs = []
    for n in range(steps):
        w_prev = ost.w
        ost, rec = orc.o_step(ini, ost, xs[n], wl.n_alpha, K=wl.K, E0=wl.E0, trial=trial)
        rec["w_prev"] = w_prev
        recs.append(rec)
    return st.host(), eloc, recs, ost


@pytest.mark.parametrize("cfg,variant", [(1, "raw"), (2, "raw"), (3, "mf"), (4, "mf")])
def test_protocol_B_free_running_alive(cfg, variant):
    """Free-running from the common initial state, one afqmc_step call over all steps; graded on the walkers
    alive in the oracle (energies at every step, state at the last step).  Per-walker tolerance from the
    largest condition number met along the trajectory (errors accumulate)."""
    wl = _wl(cfg, variant)
    nw, steps = SMALL[cfg], (10 if cfg != 4 else 5)
    out, eloc, recs, ost = _free_run(wl, nw, steps)
    kappa = np.ones(nw)
    worstE, rawE, n_alive = 0.0, 0.0, []
    for n in range(steps):
        with np.errstate(all="ignore"):
            kn = H.cond_number(wl, recs[n]["phi"])
        kappa = np.maximum(kappa, np.where(np.isfinite(kn), kn, np.inf))
        alive = (recs[n]["w"] > 0) & np.isfinite(kappa)
        n_alive.append(int(alive.sum()))
        if np.any(alive):
            e = H.energy_err_w(eloc[n], recs[n]["eloc"], recs[n]["f"])
            worstE = max(worstE, H.worst_ratio(e, (n + 1) * H.walker_tol(wl, kappa), alive))
            rawE = max(rawE, float(np.max(e[alive])))
    alive = (ost.w > 0) & np.isfinite(kappa)
    ratio = dict(E=worstE)
    if np.any(alive):
        tw = steps * H.walker_tol(wl, kappa)      # per-step tolerance accumulated over the steps taken
        ratio.update(phi=H.worst_ratio(H.rel_fro_w(out["phi"], ost.phi), tw, alive),
                     S=H.worst_ratio(H.rel_abs_w(out["S"], ost.S), tw, alive),
                     w=H.worst_ratio(H.rel_abs_w(out["w"], ost.w), tw, alive))
    print(f"cfg{cfg}/{variant} protocol B alive per step {n_alive}: err/tol {ratio} raw E {rawE:.2g}")
    assert n_alive[0] > 0
    for k, v in ratio.items():
        assert v < 1.0, (k, v)


@pytest.mark.parametrize("cfg", [1, 2, 3])
def test_protocol_C_tame(cfg):
    wl = _wl(cfg, "tame")
    nw = SMALL[cfg]
    steps = 10 if cfg != 2 else 50
    tol = H.tol_for(wl)
    out, eloc, recs, ost = _free_run(wl, nw, steps)
    assert np.all(ost.w > 0)
    errs = dict(phi=H.rel_fro(out["phi"], ost.phi), S=H.rel_abs(out["S"], ost.S), w=H.rel_abs(out["w"], ost.w),
                f=H.rel_fro(out["f"], ost.f_a + ost.f_b), E=H.rel_abs(eloc[-1], recs[-1]["eloc"]))
    print(f"cfg{cfg}/tame protocol C after {steps} steps: {errs}")
    H.record("protocol_C_tame", cfg=cfg, steps=steps, **errs)
    for k, v in errs.items():
        assert v < tol, (k, v)


def test_step_host_matches_device_step():
    wl = _wl(2, "tame")
    nw, steps = 64, 3
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, wl.walkers(nw))
    st.seed()
    xs = wl.fields(steps, nw)
    eloc_d = st.step(xs)
    d = st.host()
    phi_h = wl.walkers(nw).astype(np.complex64)
    w_h = np.ones(nw)
    S_h = np.zeros(nw, dtype=np.complex128)
    e_h = np.zeros((steps, nw), dtype=np.complex128)
    f_h = np.zeros(nw, dtype=np.int32)
    up, down = ctx.afqmc_step_host(phi_h, w_h, S_h, xs.astype(np.float32), steps, e_h, f_h)
    assert up == phi_h.nbytes + w_h.nbytes + xs.astype(np.float32).nbytes
    assert down == phi_h.nbytes + w_h.nbytes + S_h.nbytes + e_h.nbytes + f_h.nbytes
    np.testing.assert_array_equal(phi_h.astype(np.complex128), d["phi"])
    np.testing.assert_array_equal(w_h, d["w"])
    np.testing.assert_array_equal(S_h, d["S"])
    np.testing.assert_allclose(e_h, eloc_d, rtol=1e-12)
    assert ctx.launch_count > 0


def test_edge_cases():
    import torch
    import paper_1804_03310_b200 as afq
    # ragged / odd sizes, n_beta = 0, a single walker, and the empty batch
    for (M, na, nb, ng, nw, prec) in [(7, 3, 2, 5, 3, "c128"), (9, 2, 0, 33, 1, "c64"), (13, 4, 3, 17, 5, "c64"),
                                      (6, 2, 2, 4, 0, "c64")]:
        wl = make_workload(1, "raw", overrides=dict(M=M, n_alpha=na, n_beta=nb, n_chol=ng, n_walkers=max(nw, 1),
                                                    precision=prec))
        ini, _ = H.oracle_init(wl)
        ctx = H.make_ctx(wl, nw)
        if nw == 0:
            empty = torch.zeros(1, M, na + nb, dtype=ctx.cdtype, device=ctx.device)   # never touched: N_w = 0
            z = torch.zeros(1, dtype=torch.complex128, device=ctx.device)
            ctx.afqmc_overlap_green(empty, z, empty, None, None)
            assert ctx.launch_count == 0
            continue
        phi = random_walkers(wl, nw, seed=3, spread=0.1)
        ost = orc.o_seed_state(ini, phi, wl.n_alpha)
        st = H.DeviceState(ctx, phi)
        st.seed()
        xs = wl.fields(2, nw)
        eloc = st.step(xs)
        for n in range(2):
            ost, rec = orc.o_step(ini, ost, xs[n], wl.n_alpha, K=wl.K)
        out = st.host()
        tol = H.tol_for(wl)
        assert H.rel_fro(out["phi"], ost.phi) < tol
        assert H.rel_abs(out["S"], ost.S) < tol
        assert H.rel_abs(eloc[-1], rec["eloc"]) < tol


def test_singular_walker_sets_flag():
    wl = _wl(1)
    ctx = H.make_ctx(wl, 4)
    phi = wl.walkers(4).copy()
    phi[2, :, 1] = phi[2, :, 0]          # two equal alpha columns -> singular overlap matrix
    st = H.DeviceState(ctx, phi)
    st.seed()
    out = st.host()
    assert out["flags"][2] & 1
    assert np.all(out["flags"][[0, 1, 3]] == 0)


# ---- tcgen05 3xTF32 contraction path (gemm_path = 2: one CTA per tile, 3: CTA pairs): same oracle, same tolerances
@pytest.mark.parametrize("path", [2, 3])
@pytest.mark.parametrize("cfg", [2, 3, 5])
def test_tcgen05_stage_forcebias_energy_propagate(cfg, path):
    import torch
    wl = _wl(cfg)
    nw = {2: 200, 3: 136, 5: 6}[cfg]      # ragged against the 256-column tile (2 nw = 400 / 272 / 12)
    tol = H.tol_for(wl)
    ini, _ = H.oracle_init(wl)
    phi = random_walkers(wl, nw, seed=5, spread=0.1)
    ctx = H.make_ctx(wl, nw, gemm_path=path)
    assert ctx.gemm_path == path
    st = H.DeviceState(ctx, phi)
    st.seed()
    eloc = torch.zeros(nw, dtype=torch.complex128, device=ctx.device)
    ctx.afqmc_local_energy(st.phi, st.theta, eloc)
    g0 = st.host()
    ost = orc.o_seed_state(ini, phi, wl.n_alpha)
    x = wl.fields(1, nw)[0]
    new, rec = orc.o_step(ini, ost, x, wl.n_alpha, K=wl.K, E0=wl.E0)
    xd = torch.tensor(x, dtype=ctx.rdtype, device=ctx.device)
    ctx.afqmc_propagate(st.phi, xd, st.fb, st.ovlp, st.weight, st.theta, None, st.flags)
    out = st.host()
    errs = dict(f=H.rel_fro(g0["f"], ost.f_a + ost.f_b), E=H.rel_abs(eloc.cpu().numpy(), ost.eloc),
                phi=H.rel_fro(out["phi"], rec["phi"]), S=H.rel_abs(out["S"], rec["S"]),
                w=H.weight_err(out["w"], rec, ost.w, wl.dt, wl.E0))
    print(f"cfg{cfg} tcgen05 3xTF32 (gemm_path {path}) stage errors: {errs}")
    for k, v in errs.items():
        assert v < tol, (k, v)


@pytest.mark.parametrize("path", [2, 3])
@pytest.mark.parametrize("cfg,variant", [(3, "mf"), (5, "mf")])
def test_protocol_A_resync_tcgen05(cfg, variant, path):
    wl = _wl(cfg, variant)
    raw = _protocol_A(wl, SMALL[cfg], 10, gemm_path=path)
    H.record("protocol_A_tcgen05", cfg=cfg, variant=variant, path=path, steps=10, **raw)


def test_full_size_sampled_walkers():
    """bench.py's launch configuration (cfg 5, all 2048 walkers, default contraction path): two free-running steps,
    compared on sampled walkers the oracle recomputes one by one (walkers are independent)."""
    wl = _wl(5, "mf")
    nw, steps = wl.n_walkers, 2
    tol = H.tol_for(wl)
    ini, _ = H.oracle_init(wl)
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, wl.walkers(nw))
    st.seed()
    eloc = st.step(xs)
    out = st.host()
    idx = np.array([0, 1, 255, 256, 1023, 1531, 2046, 2047])
    ost = orc.o_seed_state(ini, wl.walkers(nw)[idx], wl.n_alpha)
    for n in range(steps):
        ost, rec = orc.o_step(ini, ost, xs[n][idx], wl.n_alpha, K=wl.K, E0=wl.E0)
    errs = dict(phi=H.rel_fro(out["phi"][idx], ost.phi), S=H.rel_abs(out["S"][idx], ost.S),
                w=H.rel_abs(out["w"][idx], ost.w), f=H.rel_fro(out["f"][idx], ost.f_a + ost.f_b),
                E=H.rel_abs(eloc[-1][idx], rec["eloc"]))
    print(f"cfg5 full size (path {ctx.gemm_path}), sampled walkers: {errs}")
    H.record("full_size_cfg5", **errs)
    assert np.all(np.isfinite(out["phi"].view(np.float64)))
    for k, v in errs.items():
        assert v < tol, (k, v)
