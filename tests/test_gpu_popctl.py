"""GPU parity of the steps either side of the walker step: orthonormalisation,
comb population control and the paper's schedule, through the C ABI against the FP64 oracle.

Orthonormalisation: R has a real positive diagonal on both sides (R21), so Q is unique and compared per walker in
the Frobenius norm.  Comb: the parent map is an integer decision taken in FP64 on the same weights on both sides:
bit-exact; the moved walkers are compared bit for bit with a gather of the inputs."""
import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from workloads import make_workload, random_walkers

from . import gpu_harness as H

pytestmark = pytest.mark.gpu

SMALL = {1: 64, 2: 96, 3: 40, 4: 12, 5: 6}


def _rounded(wl, phi):
    """What the device sees: the walker rounded to its storage precision."""
    return phi.astype(np.complex64).astype(np.complex128) if wl.precision == "c64" else phi


@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_stage_orthonormalize(cfg):
    import torch
    wl = make_workload(cfg)
    nw = SMALL[cfg]
    tol = H.tol_for(wl)
    phi = _rounded(wl, random_walkers(wl, nw, seed=13, spread=0.5))
    rng = np.random.default_rng(4)
    S = rng.standard_normal(nw) + 1j * rng.standard_normal(nw)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, phi, ovlp=S)
    ctx.afqmc_orthonormalize(st.phi, st.ovlp, st.flags)
    out = st.host()
    Q, S2 = orc.o_orthonormalize(phi, S, wl.n_alpha)
    errs = dict(Q=H.rel_fro(out["phi"], Q), S=H.rel_abs(out["S"], S2))
    qa = out["phi"][:, :, :wl.n_alpha]
    errs["QhQ"] = float(np.abs(np.einsum("wia,wib->wab", qa.conj(), qa) - np.eye(wl.n_alpha)).max())
    print(f"cfg{cfg} orthonormalize: {errs}")
    assert np.all(out["flags"] == 0)
    for k, v in errs.items():
        assert v < tol, (k, v)
    # Theta / overlap consistency through the library itself: S' == <Psi_T|Q> when S was <Psi_T|Phi>
    if wl.n_det == 1:
        st2 = H.DeviceState(ctx, phi)
        ctx.afqmc_overlap_green(st2.phi, st2.ovlp, st2.theta, None, st2.flags)
        th0 = st2.theta.clone()
        ctx.afqmc_orthonormalize(st2.phi, st2.ovlp, st2.flags)
        s_after = st2.ovlp.clone()
        ctx.afqmc_overlap_green(st2.phi, st2.ovlp, st2.theta, None, st2.flags)
        torch.cuda.synchronize()
        assert H.rel_abs(s_after.cpu().numpy(), st2.ovlp.cpu().numpy()) < tol
        assert H.rel_fro(st2.theta.cpu().numpy().astype(complex), th0.cpu().numpy().astype(complex)) < tol


def test_orthonormalize_edge_cases():
    """odd sizes, n_beta = 0, a single walker, an ill-conditioned walker (cond ~ 1e4: MGS in FP64 keeps the FP32
    result at rounding level), and a walker with two equal columns (flagged, left untouched)."""
    for over in (dict(M=7, n_alpha=3, n_beta=0, n_chol=5), dict(M=33, n_alpha=5, n_beta=4, n_chol=9),
                 dict(M=9, n_alpha=9, n_beta=1, n_chol=3)):
        wl = make_workload(2, overrides=over)
        for nw in (1, 5):
            phi = _rounded(wl, random_walkers(wl, nw, seed=2, spread=0.6))
            S = np.full(nw, 2.0 - 1.0j)
            ctx = H.make_ctx(wl, nw)
            st = H.DeviceState(ctx, phi, ovlp=S)
            ctx.afqmc_orthonormalize(st.phi, st.ovlp, None)
            out = st.host()
            Q, S2 = orc.o_orthonormalize(phi, S, wl.n_alpha)
            assert H.rel_fro(out["phi"], Q) < 2e-4 and H.rel_abs(out["S"], S2) < 2e-4, over
    wl = make_workload(3)
    phi = random_walkers(wl, 4, seed=8, spread=0.5)
    phi[1][:, 3] = phi[1][:, 2] + 1e-4 * phi[1][:, 3]           # nearly dependent columns
    phi = _rounded(wl, phi)
    phi[2][:, wl.n_alpha + 1] = phi[2][:, wl.n_alpha]            # exactly dependent (beta block)
    S = np.ones(4, dtype=complex)
    ctx = H.make_ctx(wl, 4)
    st = H.DeviceState(ctx, phi, ovlp=S)
    ctx.afqmc_orthonormalize(st.phi, st.ovlp, st.flags)
    out = st.host()
    ok = np.array([0, 1, 3])
    Q, S2 = orc.o_orthonormalize(phi[ok], S[ok], wl.n_alpha)
    assert H.rel_fro(out["phi"][ok], Q) < 2e-4 and H.rel_abs(out["S"][ok], S2) < 2e-4
    assert out["flags"][2] & 1 and np.all(out["flags"][ok] == 0)
    assert np.array_equal(out["phi"][2], phi[2]) and out["S"][2] == 1.0


def _random_state(wl, ctx, nw, seed):
    rng = np.random.default_rng(seed)
    phi = _rounded(wl, random_walkers(wl, nw, seed=seed))
    st = H.DeviceState(ctx, phi)
    st.seed()
    w = rng.random(nw) ** 2
    w[rng.random(nw) < 0.15] = 0.0
    w[0] = max(w[0], 0.5)
    return st, w


@pytest.mark.parametrize("cfg,nw", [(1, 1), (1, 7), (2, 1024), (2, 3001), (4, 33)])
def test_population_control_bit_exact(cfg, nw):
    import torch
    wl = make_workload(cfg)
    ctx = H.make_ctx(wl, nw)
    st, w = _random_state(wl, ctx, nw, seed=cfg + nw)
    st.weight.copy_(torch.tensor(w, dtype=torch.float64))
    before = st.host()
    parent = torch.full((nw,), -1, dtype=torch.int32, device=ctx.device)
    for u in (0.0, 0.37, 0.999999):
        st.phi.copy_(torch.tensor(before["phi"], dtype=ctx.cdtype)); st.theta.copy_(torch.tensor(before["theta"], dtype=ctx.cdtype))
        st.fb.copy_(torch.tensor(before["f"], dtype=ctx.cdtype)); st.ovlp.copy_(torch.tensor(before["S"]))
        st.weight.copy_(torch.tensor(w, dtype=torch.float64))
        ctx.afqmc_population_control(st.phi, st.weight, st.ovlp, st.theta, st.fb, u, parent)
        out = st.host()
        par = orc.o_comb(w, u)
        assert np.array_equal(parent.cpu().numpy(), par), (cfg, nw, u)
        assert np.array_equal(out["w"], np.full(nw, np.cumsum(w)[-1] / nw))
        for k in ("phi", "theta", "f", "S"):
            assert np.array_equal(out[k], before[k][par]), k
    # a dead population: nothing moves, weights kept
    st.weight.zero_()
    ref = st.host()
    ctx.afqmc_population_control(st.phi, st.weight, st.ovlp, st.theta, st.fb, 0.5, parent)
    out = st.host()
    assert np.array_equal(parent.cpu().numpy(), np.arange(nw)) and np.all(out["w"] == 0)
    assert np.array_equal(out["phi"], ref["phi"])
    with pytest.raises(Exception):
        ctx.afqmc_population_control(st.phi, st.weight, st.ovlp, st.theta, st.fb, 1.0, parent)


def _run_both(wl, nw, steps, ee, oe, pe, us, idx=None):
    """afqmc_run on the device, the same schedule on the oracle.  The comb decision is an integer taken from the
    weights: it is checked bit-exactly against o_comb on the DEVICE's weights at that point, compared with the
    oracle's own map, and the oracle then follows the device's map so that the states stay comparable."""
    import torch
    ini, trial = H.oracle_init(wl)
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, H.start_walkers(wl, nw))
    st.seed()
    xd = torch.tensor(np.ascontiguousarray(xs), dtype=ctx.rdtype, device=ctx.device)
    n_meas, n_pc = (steps // ee if ee else 0), (steps // pe if pe else 0)
    eloc = torch.zeros(max(n_meas, 1), nw, dtype=torch.complex128, device=ctx.device)
    wm = torch.zeros(max(n_meas, 1), nw, dtype=torch.float64, device=ctx.device)
    par = torch.zeros(max(n_pc, 1), nw, dtype=torch.int32, device=ctx.device)
    ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, steps, ee, oe, pe, us, eloc, wm, par, st.flags)
    out = st.host()
    eloc, wm, par = eloc.cpu().numpy(), wm.cpu().numpy(), par.cpu().numpy()
    sel = np.arange(nw) if idx is None else idx
    assert idx is None or not pe, "sampling walkers and combing the population do not go together"
    ost = orc.o_seed_state(ini, H.start_walkers(wl, nw)[sel], wl.n_alpha, trial=trial)
    meas, flips = [], 0
    for n in range(1, steps + 1):
        ost, _ = orc.o_step(ini, ost, xs[n - 1][sel], wl.n_alpha, K=wl.K, E0=wl.E0, trial=trial)
        if ee and n % ee == 0:
            meas.append((ost.w.copy(), ost.eloc.copy()))
        if oe and n % oe == 0:
            phi, S = orc.o_orthonormalize(ost.phi, ost.S, wl.n_alpha)
            ost = orc.OracleState(phi, ost.w, S, ost.theta, ost.f_a, ost.f_b, ost.eloc)
        if pe and n % pe == 0:
            k = n // pe - 1
            if ee and n % ee == 0:      # device weights at this point are known: the decision must be bit-exact
                assert np.array_equal(par[k], orc.o_comb(wm[n // ee - 1], us[k]))
            po = orc.o_comb(ost.w, us[k])
            bad = np.nonzero(po != par[k])[0]
            cum = np.cumsum(ost.w)
            for i in bad:               # a differing parent must come from a tooth within rounding of a boundary
                t = (i + us[k]) * cum[-1] / nw
                assert abs(int(po[i]) - int(par[k][i])) == 1 and np.min(np.abs(cum - t)) < 1e-3 * cum[-1] / nw
            flips += bad.size
            g = par[k]
            ost = orc.OracleState(ost.phi[g], np.full(nw, np.cumsum(ost.w)[-1] / nw), ost.S[g], ost.theta[g],
                                  ost.f_a[g], ost.f_b[g], ost.eloc[g])
    return ctx, out, eloc, wm, par, ost, meas, flips


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_run_schedule_tame(cfg):
    """energy every 4, orthonormalise every 2, comb every 4 steps over 8 steps (the paper's 20 / 2 / 20 scaled down) on
    the `tame` variant, all walkers, free running."""
    wl = make_workload(cfg, "tame")
    nw = SMALL[cfg]
    tol = H.tol_for(wl)
    us = [0.3, 0.85]
    ctx, out, eloc, wm, par, ost, meas, flips = _run_both(wl, nw, 8, 4, 2, 4, us)
    errs = dict(phi=H.rel_fro(out["phi"], ost.phi), S=H.rel_abs(out["S"], ost.S), w=H.rel_abs(out["w"], ost.w),
                f=H.rel_fro(out["f"], ost.f_a + ost.f_b), theta=H.rel_fro(out["theta"], ost.theta))
    for k, (w_o, e_o) in enumerate(meas):
        errs[f"E{k}"] = H.rel_abs(eloc[k], e_o)
        errs[f"w{k}"] = H.rel_abs(wm[k], w_o)
    print(f"cfg{cfg}/tame schedule 8 steps (E/4, QR/2, comb/4): {errs}; comb flips {flips}")
    assert np.all(ost.w > 0) and flips <= 1
    for k, v in errs.items():
        assert v < tol, (k, v)


def test_run_equals_step_when_schedule_is_trivial():
    """energy_every = 1, no QR, no comb: afqmc_run leaves the state afqmc_step leaves, bit for bit; a propagate-only run (energy_every = 0)
    leaves the same walkers, weights and force bias."""
    import torch
    wl = make_workload(2, "tame")
    nw, steps = 64, 3
    xs = wl.fields(steps, nw)
    ctx = H.make_ctx(wl, nw)
    res = []
    for mode in ("step", "run", "noE"):
        st = H.DeviceState(ctx, wl.walkers(nw))
        st.seed()
        xd = torch.tensor(np.ascontiguousarray(xs), dtype=ctx.rdtype, device=ctx.device)
        eloc = torch.zeros(steps, nw, dtype=torch.complex128, device=ctx.device)
        if mode == "step":
            ctx.afqmc_step(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, steps, eloc, st.flags)
        else:
            ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, steps, 1 if mode == "run" else 0, 0, 0, None,
                          eloc, None, None, st.flags)
        res.append((st.host(), eloc.cpu().numpy()))
    for k in ("phi", "w", "S", "f", "theta"):
        assert np.array_equal(res[0][0][k], res[1][0][k]) and np.array_equal(res[0][0][k], res[2][0][k]), k
    # E_L is accumulated with FP64 atomics (order not fixed): equal to rounding, not bit for bit
    assert H.rel_abs(res[1][1], res[0][1]) < 1e-12 and np.all(res[2][1] == 0)


def test_full_size_schedule_sampled_walkers():
    """bench.py --schedule's launch configuration (cfg 5, 2048 walkers): 4 steps, energy at step 4, QR every 2 steps,
    no comb (walkers stay independent, so the oracle recomputes the sampled ones one by one); then one comb at full
    size, bit-exact against the oracle's map on the device's weights."""
    import torch
    wl = make_workload(5, "mf")
    nw = wl.n_walkers
    tol = H.tol_for(wl)
    idx = np.array([0, 1, 255, 1024, 1531, 2047])
    ctx, out, eloc, wm, par, ost, meas, _ = _run_both(wl, nw, 4, 4, 2, 0, None, idx=idx)
    errs = dict(phi=H.rel_fro(out["phi"][idx], ost.phi), S=H.rel_abs(out["S"][idx], ost.S),
                w=H.rel_abs(out["w"][idx], ost.w), f=H.rel_fro(out["f"][idx], ost.f_a + ost.f_b),
                E=H.rel_abs(eloc[0][idx], meas[0][1]))
    q = out["phi"][:, :, :wl.n_alpha]
    errs["QhQ"] = float(np.abs(np.einsum("wia,wib->wab", q.conj(), q) - np.eye(wl.n_alpha)).max())
    print(f"cfg5 full-size schedule, sampled walkers: {errs}")
    for k, v in errs.items():
        assert v < 4 * tol, (k, v)       # 4 free-running steps
    st = H.DeviceState(ctx, out["phi"], weight=out["w"], ovlp=out["S"])
    st.theta.copy_(torch.tensor(out["theta"], dtype=ctx.cdtype)); st.fb.copy_(torch.tensor(out["f"], dtype=ctx.cdtype))
    parent = torch.zeros(nw, dtype=torch.int32, device=ctx.device)
    ctx.afqmc_population_control(st.phi, st.weight, st.ovlp, st.theta, st.fb, 0.4321, parent)
    o2 = st.host()
    p = orc.o_comb(out["w"], 0.4321)
    assert np.array_equal(parent.cpu().numpy(), p)
    assert np.array_equal(o2["phi"], out["phi"][p]) and np.array_equal(o2["S"], out["S"][p])
    assert np.array_equal(o2["w"], np.full(nw, np.cumsum(out["w"])[-1] / nw))


def test_run_argument_errors_and_ragged_schedule():
    """EINVAL before any launch: weight_mode 1, u outside [0, 1), missing u / eloc; an empty batch and n_steps = 0 are
    no-ops; a step count that is not a multiple of the intervals measures / combs floor(n / every) times."""
    import torch
    import paper_1804_03310_b200 as afq
    wl = make_workload(1, "tame")
    nw = 8
    xs = wl.fields(5, nw)
    ctx = H.make_ctx(wl, nw)
    st = H.DeviceState(ctx, wl.walkers(nw))
    st.seed()
    xd = torch.tensor(np.ascontiguousarray(xs), dtype=ctx.rdtype, device=ctx.device)
    eloc = torch.full((2, nw), -7.0, dtype=torch.complex128, device=ctx.device)
    par = torch.full((1, nw), -1, dtype=torch.int32, device=ctx.device)
    l0 = ctx.launch_count
    for kw in (dict(u=[1.0]), dict(u=[-0.1]), dict(u=None)):
        with pytest.raises(afq.AfqmcError) as ei:
            ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, 5, 2, 2, 3, kw["u"], eloc, None, par, st.flags)
        assert ei.value.status == afq.AFQMC_EINVAL
    with pytest.raises(afq.AfqmcError):
        ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, 5, 2, 0, 0, None, None, None, None, st.flags)
    with pytest.raises(afq.AfqmcError):
        ctx.afqmc_orthonormalize(None, st.ovlp, None)
    assert ctx.launch_count == l0
    ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, 0, 1, 1, 1, [0.5], eloc, None, par, st.flags)
    assert ctx.launch_count == l0
    ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, 5, 2, 2, 3, [0.5], eloc, None, par, st.flags)
    torch.cuda.synchronize()
    assert torch.all(eloc.real != -7.0) and torch.all(par >= 0)          # 2 measurements, 1 comb
    ctx1 = H.make_ctx(wl, nw, weight_mode=1)
    with pytest.raises(afq.AfqmcError):
        ctx1.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, 2, 1, 0, 0, None, eloc, None, None, st.flags)
    ctx0 = H.make_ctx(wl, 0)
    e = torch.zeros(0, dtype=ctx0.cdtype, device=ctx0.device)
    ctx0.afqmc_orthonormalize(e, e, None)
    ctx0.afqmc_population_control(e, e, e, e, e, 0.5, None)
    assert ctx0.launch_count == 0


@pytest.mark.parametrize("world", [1, 2, 3])
def test_sharded_comb_emulated_ranks(world):
    """The comb over a population sharded across `world` ranks (afqmc_comb_map / _pack / _unpack + dist.comb_splits),
    with the ranks played one after the other on this GPU and the all-to-all replaced by slicing the send buffers the
    way torch.distributed.all_to_all_single would (no kernel waits on another rank).  Bit-exact against
    afqmc_population_control on the whole population in one context, and against the oracle's map."""
    import torch
    from paper_1804_03310_b200 import dist as D
    wl = make_workload(2)
    nl = 50
    nt = world * nl
    ctx_all = H.make_ctx(wl, nt)
    full, w = _random_state(wl, ctx_all, nt, seed=31 + world)
    w[nl // 2:nl] = 0.0                                   # a dead stretch: its slots are refilled from other ranks
    full.weight.copy_(torch.tensor(w, dtype=torch.float64))
    before = full.host()
    u = 0.613
    ranks = []
    for r in range(world):
        c = H.make_ctx(wl, nl)
        sl = slice(r * nl, (r + 1) * nl)
        st = H.DeviceState(c, before["phi"][sl], weight=w[sl], ovlp=before["S"][sl])
        st.theta.copy_(torch.tensor(before["theta"][sl], dtype=c.cdtype)); st.fb.copy_(torch.tensor(before["f"][sl], dtype=c.cdtype))
        ranks.append((c, st))
    w_all = torch.cat([st.weight for _, st in ranks])      # the all-gather
    sends, plans = [], []
    for r, (c, st) in enumerate(ranks):
        cum = torch.empty(nt, dtype=torch.float64, device=c.device)
        parent_all = torch.empty(nt, dtype=torch.int32, device=c.device)
        w_new = torch.empty(2, dtype=torch.float64, device=c.device)
        c.afqmc_comb_map(w_all, u, cum, parent_all, w_new)
        slot_lo, count, sc, rc = D.comb_splits(parent_all, nl, world, r)
        rec = c.afqmc_comb_record_bytes
        sb = torch.zeros(max(count, 1) * rec, dtype=torch.uint8, device=c.device)
        c.afqmc_comb_pack(st.phi, st.ovlp, st.theta, st.fb, parent_all, slot_lo, count, r * nl, sb)
        sends.append(sb); plans.append((parent_all, w_new, sc, rc, rec))
    par_o = orc.o_comb(w, u)
    for r, (c, st) in enumerate(ranks):
        parent_all, w_new, sc, rc, rec = plans[r]
        assert np.array_equal(parent_all.cpu().numpy(), par_o)
        parts = []
        for s in range(world):                              # what all_to_all_single delivers to rank r
            off = sum(plans[s][2][:r]) * rec
            assert plans[s][2][r] == rc[s]
            parts.append(sends[s][off:off + plans[s][2][r] * rec])
        rb = torch.cat(parts)
        assert rb.numel() == nl * rec
        c.afqmc_comb_unpack(rb, st.phi, st.weight, st.ovlp, st.theta, st.fb, w_new)
    ctx_all.afqmc_population_control(full.phi, full.weight, full.ovlp, full.theta, full.fb, u, None)
    ref = full.host()
    for r, (c, st) in enumerate(ranks):
        got = st.host()
        sl = slice(r * nl, (r + 1) * nl)
        for k in ("phi", "theta", "f", "S", "w"):
            assert np.array_equal(got[k], ref[k][sl]), (world, r, k)
    assert np.array_equal(ref["phi"], before["phi"][par_o])
    if world == 1:      # the public helper, single rank: no collective
        c, st = ranks[0]
        st2 = H.DeviceState(c, before["phi"], weight=w, ovlp=before["S"])
        st2.theta.copy_(torch.tensor(before["theta"], dtype=c.cdtype)); st2.fb.copy_(torch.tensor(before["f"], dtype=c.cdtype))
        pm = D.population_control_sharded(c, st2.phi, st2.weight, st2.ovlp, st2.theta, st2.fb, u)
        g2 = st2.host()
        assert np.array_equal(pm.cpu().numpy(), par_o)
        for k in ("phi", "theta", "f", "S", "w"):
            assert np.array_equal(g2[k], ref[k]), k


def test_mixed_sums_and_sharded_run_single_rank():
    """afqmc_mixed_sums against the oracle's mixed estimator; dist.run_sharded with one rank (no collective) leaves
    exactly the state afqmc_run leaves with the same schedule, and its energies are the oracle's mixed estimator of the
    device's own measurements."""
    import torch
    from paper_1804_03310_b200 import dist as D
    wl = make_workload(2, "tame")
    nw, steps = 1031, 8
    ctx = H.make_ctx(wl, nw)
    rng = np.random.default_rng(3)
    w = rng.random(nw); w[::7] = 0.0
    e = rng.standard_normal(nw) + 1j * rng.standard_normal(nw)
    e[::7] = np.nan                                        # dead walkers may carry garbage energies
    out3 = torch.zeros(3, dtype=torch.float64, device=ctx.device)
    ctx.afqmc_mixed_sums(torch.tensor(w, device=ctx.device), torch.tensor(e, device=ctx.device), out3)
    o = out3.cpu().numpy()
    alive = w > 0
    assert abs(o[0] - w.sum()) < 1e-12 * w.sum()
    assert abs(o[1] / o[0] - orc.o_mixed_energy(w[alive], e[alive])) < 1e-12
    assert abs(o[2] - np.sum(w[alive] * e[alive].imag)) < 1e-11
    xs = wl.fields(steps, nw)
    xd = torch.tensor(np.ascontiguousarray(xs), dtype=ctx.rdtype, device=ctx.device)
    us = [0.3, 0.85]
    a = H.DeviceState(ctx, wl.walkers(nw)); a.seed()
    eloc = torch.zeros(2, nw, dtype=torch.complex128, device=ctx.device)
    wm = torch.zeros(2, nw, dtype=torch.float64, device=ctx.device)
    ctx.afqmc_run(a.phi, a.weight, a.ovlp, a.theta, a.fb, xd, steps, 4, 2, 4, us, eloc, wm, None, a.flags)
    b = H.DeviceState(ctx, wl.walkers(nw)); b.seed()
    en = D.run_sharded(ctx, b.phi, b.weight, b.ovlp, b.theta, b.fb, xd, steps, 4, 2, 4, us, flags=b.flags)
    ha, hb = a.host(), b.host()
    for k in ("phi", "w", "S", "theta", "f"):
        assert np.array_equal(ha[k], hb[k]), k
    assert len(en) == 2
    for j in range(2):
        ref = orc.o_mixed_energy(wm[j].cpu().numpy(), eloc[j].cpu().numpy())
        assert abs(en[j].real - ref) < 1e-10 * abs(ref)


@pytest.mark.parametrize("precision", ["c128", "c64"])
def test_long_run_on_gpu_vs_fci(precision):
    """The whole CUDA path end to end against brute-force FCI (the north_star's validation, here on the GPU): cfg 1
    shapes, `tame_mf` inputs, dt = 0.05, 640 walkers (complex128: FP64 SIMT path; complex64: the FP32 / 3xTF32 tcgen05
    path, the paper's single-precision claim PAPER.md:135), 700 steps in ONE afqmc_run call with E_L every step,
    orthonormalisation every 5 and comb every 10 steps (the recipe of the oracle's pin P10b).  The mixed estimator over the
    last 500 steps must agree with the lowest eigenvalue of the sector Hamiltonian within 3 sigma (reblocked) plus 2 % of
    the correlation energy (the phaseless bias allowance of P10b)."""
    import dataclasses
    import torch
    from tests.fockspace import sector_one_body_ops
    from tests.test_oracle_fci import _sector_hamiltonian
    wl = dataclasses.replace(make_workload(1, "tame_mf"), dt=0.05, precision=precision)
    fk, idx, E = sector_one_body_ops(wl.M, 2, 2)
    Hs = _sector_hamiltonian(wl, E) + wl.e_const * np.eye(idx.size)
    e_fci = np.linalg.eigvalsh(Hs)[0]
    nw, n_steps, n_eq = 640, 700, 200
    rng = np.random.default_rng(12345)
    xs = rng.standard_normal((n_steps, nw, wl.n_chol))
    us = rng.random(n_steps // 10)
    ini = orc.o_init(wl.h, wl.L, wl.dt, wl.psi_a, wl.psi_b)
    e_hf = orc.o_seed_state(ini, wl.walkers(1), 2).eloc[0].real
    ctx = H.make_ctx(wl, nw, E0=e_hf)
    st = H.DeviceState(ctx, wl.walkers(nw))
    st.seed()
    xd = torch.tensor(xs, dtype=ctx.rdtype, device=ctx.device)
    eloc = torch.zeros(n_steps, nw, dtype=torch.complex128, device=ctx.device)
    wm = torch.zeros(n_steps, nw, dtype=torch.float64, device=ctx.device)
    ctx.afqmc_run(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd, n_steps, 1, 5, 10, us, eloc, wm, None, st.flags)
    torch.cuda.synchronize()
    eloc, wm = eloc.cpu().numpy(), wm.cpu().numpy()
    assert np.all(np.isfinite(wm)) and np.all(wm.sum(axis=1) > 0)
    num = np.sum(wm * eloc.real, axis=1)[n_eq:]
    den = wm.sum(axis=1)[n_eq:]
    e_mix = num.sum() / den.sum() + wl.e_const
    nb = 20
    blocks = np.array([b.sum() for b in np.array_split(num, nb)]) / np.array(
        [b.sum() for b in np.array_split(den, nb)]) + wl.e_const
    sigma = blocks.std(ddof=1) / np.sqrt(nb)
    corr = abs(e_hf + wl.e_const - e_fci)
    print(f"GPU long run ({precision}, gemm_path {ctx.gemm_path}): E_mix {e_mix:.6f} +- {sigma:.6f}, E_FCI {e_fci:.6f}, E_HF {e_hf + wl.e_const:.6f}")
    assert e_fci < e_hf + wl.e_const
    assert abs(e_mix - e_fci) <= 3 * sigma + 0.02 * corr, (e_mix, e_fci, sigma)
    assert abs(e_mix - e_fci) < 0.2 * corr
