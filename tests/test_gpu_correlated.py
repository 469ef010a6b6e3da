"""Correlated sampling (SURVEY.md 8(f) NEXT-3; PAPER.md:181 "pairs of walkers sample the same auxiliary fields", :235): a
neutral species (N_alpha, N_beta) and its cation (N_alpha - 1, N_beta) on the same h, L are stepped by two contexts that read
the SAME device field buffer.  Each must equal its own oracle run, and the spread of the energy difference over repeats must
be well below the one obtained with independent fields (the variance reduction the paper uses for ionisation potentials)."""
import numpy as np
import pytest

from oracle import afqmc_oracle as orc
from workloads import make_workload

from . import gpu_harness as H

pytestmark = pytest.mark.gpu

OV = dict(M=12, n_alpha=4, n_beta=3, n_chol=30, n_walkers=64)


def _species():
    wn = make_workload(2, "tame", overrides=OV)
    wc = make_workload(2, "tame", overrides=dict(OV, n_alpha=OV["n_alpha"] - 1))
    assert np.array_equal(wn.L, wc.L) and np.array_equal(wn.h, wc.h)      # same Hamiltonian, one electron removed
    return wn, wc


def test_correlated_sampling_shared_field_buffer():
    import torch
    wn, wc = _species()
    nw, steps, reps = 48, 12, 10
    ctxs = [H.make_ctx(w, nw) for w in (wn, wc)]
    inis = [H.oracle_init(w)[0] for w in (wn, wc)]
    dev = ctxs[0].device

    def gpu_run(k, xd):
        wl, ctx = (wn, wc)[k], ctxs[k]
        st = H.DeviceState(ctx, wl.walkers(nw))
        st.seed()
        eloc = torch.zeros(steps, nw, dtype=torch.complex128, device=dev)
        wts = []
        for n in range(steps):          # one step per call so that the weights at every measurement are available
            ctx.afqmc_step(st.phi, st.weight, st.ovlp, st.theta, st.fb, xd[n], 1, eloc[n:n + 1], st.flags)
            wts.append(st.weight.clone())
        torch.cuda.synchronize()
        e, w = eloc.cpu().numpy(), torch.stack(wts).cpu().numpy()
        emix = np.array([np.real(np.sum(w[n] * e[n])) / np.sum(w[n]) for n in range(steps)])
        return st.host(), e, float(np.mean(emix[steps // 2:]))

    d_corr, d_unc = [], []
    for r in range(reps):
        x1 = np.random.default_rng(100 + r).standard_normal((steps, nw, wn.n_chol))
        x2 = np.random.default_rng(900 + r).standard_normal((steps, nw, wn.n_chol))
        xd1 = torch.tensor(x1, dtype=ctxs[0].rdtype, device=dev)       # ONE buffer, handed to both contexts
        xd2 = torch.tensor(x2, dtype=ctxs[0].rdtype, device=dev)
        outN, eN, EN = gpu_run(0, xd1)
        outC, eC, EC = gpu_run(1, xd1)
        _, _, EC2 = gpu_run(1, xd2)
        d_corr.append(EN - EC)
        d_unc.append(EN - EC2)
        if r == 0:      # each species against its own oracle run on the shared fields
            for k, (wl, out, e) in enumerate(((wn, outN, eN), (wc, outC, eC))):
                ost = orc.o_seed_state(inis[k], wl.walkers(nw), wl.n_alpha)
                worstE = 0.0
                for n in range(steps):
                    ost, rec = orc.o_step(inis[k], ost, x1[n], wl.n_alpha, K=wl.K, E0=wl.E0)
                    worstE = max(worstE, H.rel_abs(e[n], rec["eloc"]))
                errs = dict(phi=H.rel_fro(out["phi"], ost.phi), S=H.rel_abs(out["S"], ost.S), w=H.rel_abs(out["w"], ost.w), E=worstE)
                print(f"correlated sampling, species N=({wl.n_alpha},{wl.n_beta}): {errs}")
                H.record("correlated_sampling_parity", n_alpha=wl.n_alpha, **errs)
                assert np.all(ost.w > 0)
                for q, v in errs.items():
                    assert v < H.tol_for(wl), (q, v)
    ratio = float(np.var(d_corr) / np.var(d_unc))
    print(f"E(neutral) - E(cation) over {reps} repeats: shared fields {np.mean(d_corr):.5f} +- {np.std(d_corr):.5f}, "
          f"independent fields {np.mean(d_unc):.5f} +- {np.std(d_unc):.5f}; variance ratio {ratio:.3f}")
    H.record("correlated_sampling_variance", ratio=ratio, std_shared=float(np.std(d_corr)), std_independent=float(np.std(d_unc)))
    assert abs(np.mean(d_corr) - np.mean(d_unc)) < 4 * np.std(d_unc) / np.sqrt(reps) + 4 * np.std(d_corr) / np.sqrt(reps)   # same estimate
    assert ratio < 0.3          # the oracle alone gives 0.08 on these inputs (the point of the method)
