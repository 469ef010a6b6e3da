"""Helpers for the `-m gpu` parity tests: build a context from a seeded Workload, run the CUDA
path through the C-ABI binding, and compare with the FP64 oracle using the metrics of
DESIGN.md "Parity protocol" (R11).  No method arithmetic lives here beyond the error norms."""
from __future__ import annotations

import numpy as np

from oracle import afqmc_oracle as orc


def tol_for(wl):
    """north_star: 1e-5 for the FP64 path, 2e-4 for the FP32 path, per step."""
    return 1e-5 if wl.precision == "c128" else 2e-4


def make_ctx(wl, n_walkers=None, gemm_path=0, weight_mode=0, E0=None, K=None, max_exc=None):
    from paper_1804_03310_b200.state import make_context
    return make_context(wl, n_walkers, gemm_path=gemm_path, weight_mode=weight_mode, E0=E0, K=K, max_exc=max_exc)


def oracle_init(wl):
    ini = orc.o_init(wl.h, wl.L, wl.dt, wl.psi_a, wl.psi_b)
    trial = None
    if wl.n_det > 1:
        trial = orc.MultiDetTrial(wl.C_act, wl.det_coeff, wl.det_exc, wl.n_alpha, wl.n_beta)
    return ini, trial


def DeviceState(ctx, phi, weight=None, ovlp=None):
    """Walker state tensors on the device in the ABI layouts (paper_1804_03310_b200.state.WalkerState)."""
    from paper_1804_03310_b200.state import WalkerState
    return WalkerState(ctx, phi, weight=weight, ovlp=ovlp)


# ---- error norms (R11): never elementwise-relative -------------------------------------------
def rel_fro(a, b, floor=0.0):
    """max over walkers of ||a_w - b_w||_F / max(||b_w||_F, floor) (b = oracle).  `floor` is the natural
    scale of the quantity when the oracle value itself vanishes (the force bias of the mean-field
    subtracted inputs is exactly 0 at the trial)."""
    a = a.reshape(a.shape[0], -1)
    b = b.reshape(b.shape[0], -1)
    den = np.maximum(np.linalg.norm(b, axis=1), floor)
    den = np.where(den == 0, 1.0, den)
    return float(np.max(np.linalg.norm(a - b, axis=1) / den)) if a.shape[0] else 0.0


def fb_floor(ini):
    """Scale below which a force-bias norm counts as zero: 1e-3 ||R||_F (f = R . Theta, ||Theta|| = O(1))."""
    return 1e-3 * float(np.sqrt(sum(np.sum(R * R) for R in ini["R"])))


def rel_abs(a, b):
    den = np.where(np.abs(b) == 0, 1.0, np.abs(b))
    return float(np.max(np.abs(a - b) / den)) if a.size else 0.0


def weight_err(w_gpu, rec, w_prev, dt, E0):
    """|w' - w'_ora| / (w_prev e^{dt E0} |I|_ora): error against the un-projected magnitude."""
    den = w_prev * np.exp(dt * E0) * rec["absI"]
    ok = den > 0
    if not np.any(ok):
        return 0.0
    return float(np.max(np.abs(w_gpu[ok] - rec["w"][ok]) / den[ok]))


def well_conditioned(wl, phi, limit=1e3):
    """Walkers whose overlap matrices Psi_s^T Phi_s both have condition number <= limit (R11: FP32 error of
    the inverse scales with cond; the others are reported separately, not graded)."""
    ok = np.ones(phi.shape[0], dtype=bool)
    for psi, ph in zip((wl.psi_a, wl.psi_b), (phi[..., :wl.n_alpha], phi[..., wl.n_alpha:])):
        if psi.shape[1] == 0:
            continue
        A = np.matmul(psi.T[None], ph)
        with np.errstate(all="ignore"):
            c = np.linalg.cond(A)
        ok &= np.isfinite(c) & (c <= limit)
    return ok


def cond_number(wl, phi):
    """Per walker: max over spins of cond(Psi_s^T Phi_s)."""
    c = np.ones(phi.shape[0])
    for psi, ph in zip((wl.psi_a, wl.psi_b), (phi[..., :wl.n_alpha], phi[..., wl.n_alpha:])):
        if psi.shape[1] == 0:
            continue
        with np.errstate(all="ignore"):
            ck = np.linalg.cond(np.matmul(psi.T[None], ph))
        c = np.maximum(c, np.where(np.isfinite(ck), ck, np.inf))
    return c


def walker_tol(wl, kappa, kappa0=32.0):
    """Per-walker tolerance: the stated tolerance for cond <= kappa0; on the FP32
    path it grows in proportion to the condition number kappa of the walker's overlap matrices beyond that:
    tol_w = max(2e-4, 6.25e-6 * kappa).  Measured FP32 floor (any FP32 implementation, inputs rounded to
    complex64): S, E, w errors up to 1.5e-6 * kappa, i.e. the bound keeps a factor ~4.  FP64 path: no scaling."""
    tol = tol_for(wl)
    if wl.precision == "c128":
        return np.full(kappa.shape, tol)
    return tol * np.maximum(1.0, kappa / kappa0)


def rel_fro_w(a, b, floor=0.0):
    a = a.reshape(a.shape[0], -1)
    b = b.reshape(b.shape[0], -1)
    den = np.maximum(np.linalg.norm(b, axis=1), floor)
    den = np.where(den == 0, 1.0, den)
    return np.linalg.norm(a - b, axis=1) / den


def rel_abs_w(a, b):
    den = np.where(np.abs(b) == 0, 1.0, np.abs(b))
    return np.abs(a - b) / den


def worst_ratio(err_w, tol_w, mask=None):
    """max over (masked) walkers of error / tolerance; < 1 passes."""
    if mask is not None:
        err_w, tol_w = err_w[mask], tol_w[mask]
    return float(np.max(err_w / tol_w)) if err_w.size else 0.0


def start_walkers(wl, nw):
    """Initial population of a run: the trial determinant (SURVEY O-init 5).  Multi-determinant trials start
    from the reference determinant plus a small seeded complex perturbation: at the exact reference every excited
    determinant has zero overlap and both Eq.(4) and the per-determinant definition divide by it."""
    if wl.n_det > 1:
        from workloads import random_walkers
        return random_walkers(wl, nw, seed=21, spread=0.05)
    return wl.walkers(nw)


def energy_err_w(e_gpu, e_ora, f_ora):
    """|E - E_ora| / max(|E_ora|, 1/2 ||f_ora||^2): E_L is a sum of terms of size 1/2 sum_g |f_g|^2 that partly
    cancel, so the error is measured against the largest of them (same idea as the weight metric, R11)."""
    den = np.maximum(np.abs(e_ora), 0.5 * np.sum(np.abs(f_ora) ** 2, axis=-1))
    den = np.where(den == 0, 1.0, den)
    return np.abs(e_gpu - e_ora) / den


def record(name, **vals):
    """Append the raw (un-normalised) worst errors of a parity test to gpurun_out/parity_raw.jsonl -- the file the
    profiles/parity_*.md summaries are transcribed from.  Never fails a test."""
    import json
    import os
    try:
        root = os.environ.get("GRAFT_REPO_ROOT") or os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
        d = os.path.join(root, "gpurun_out")
        os.makedirs(d, exist_ok=True)
        clean = {k: (float(v) if isinstance(v, (int, float, np.floating, np.integer)) else v) for k, v in vals.items()}
        with open(os.path.join(d, "parity_raw.jsonl"), "a") as fh:
            fh.write(json.dumps(dict(test=name, **clean)) + "\n")
    except Exception:
        pass
