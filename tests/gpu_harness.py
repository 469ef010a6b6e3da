"""Helpers for the `-m gpu` parity tests: build a context from a seeded Workload, run the CUDA
path through the C-ABI binding, and compare with the FP64 oracle using the metrics of
DESIGN.md "Parity protocol" (R11).  No method arithmetic lives here beyond the error norms."""
from __future__ import annotations

import numpy as np

from oracle import afqmc_oracle as orc


def tol_for(wl):
    """north_star: 1e-5 for the FP64 path, 2e-4 for the FP32 path, per step."""
    return 1e-5 if wl.precision == "c128" else 2e-4


def make_ctx(wl, n_walkers=None, gemm_path=0, weight_mode=0, E0=None, K=None):
    import paper_1804_03310_b200 as afq
    nw = wl.n_walkers if n_walkers is None else n_walkers
    p = afq.make_params(wl.M, wl.n_alpha, wl.n_beta, wl.n_chol, nw, wl.precision, wl.dt,
                        taylor_order=wl.K if K is None else K, weight_mode=weight_mode,
                        E0=wl.E0 if E0 is None else E0, n_det=wl.n_det, n_act=wl.n_act, max_exc=2,
                        gemm_path=gemm_path)
    if wl.n_det > 1:
        return afq.AfqmcContext(p, wl.h, wl.L, wl.psi_a, wl.psi_b, C_act=wl.C_act, det_coeff=wl.det_coeff,
                                det_exc=wl.det_exc)
    return afq.AfqmcContext(p, wl.h, wl.L, wl.psi_a, wl.psi_b)


def oracle_init(wl):
    ini = orc.o_init(wl.h, wl.L, wl.dt, wl.psi_a, wl.psi_b)
    trial = None
    if wl.n_det > 1:
        trial = orc.MultiDetTrial(wl.C_act, wl.det_coeff, wl.det_exc, wl.n_alpha, wl.n_beta)
    return ini, trial


class DeviceState:
    """Walker state tensors on the device in the ABI layouts."""

    def __init__(self, ctx, phi, weight=None, ovlp=None):
        import torch
        dev = ctx.device
        nw = phi.shape[0]
        self.ctx = ctx
        self.phi = torch.tensor(np.ascontiguousarray(phi), dtype=ctx.cdtype, device=dev)
        self.theta = torch.zeros_like(self.phi)
        self.weight = torch.tensor(np.ones(nw) if weight is None else weight, dtype=torch.float64, device=dev)
        self.ovlp = torch.zeros(nw, dtype=torch.complex128, device=dev)
        if ovlp is not None:
            self.ovlp.copy_(torch.tensor(ovlp, dtype=torch.complex128))
        self.fb = torch.zeros(nw, ctx.params.n_chol, dtype=ctx.cdtype, device=dev)
        self.flags = torch.zeros(nw, dtype=torch.int32, device=dev)

    def seed(self):
        self.ctx.afqmc_overlap_green(self.phi, self.ovlp, self.theta, None, self.flags)
        self.ctx.afqmc_force_bias(self.phi, self.theta, self.fb)

    def step(self, x, n_steps=None):
        """x numpy [steps][nw][ng]; returns eloc [steps][nw] complex128 (numpy)."""
        import torch
        n_steps = x.shape[0] if n_steps is None else n_steps
        xd = torch.tensor(np.ascontiguousarray(x), dtype=self.ctx.rdtype, device=self.ctx.device)
        eloc = torch.zeros(n_steps, self.phi.shape[0], dtype=torch.complex128, device=self.ctx.device)
        self.ctx.afqmc_step(self.phi, self.weight, self.ovlp, self.theta, self.fb, xd, n_steps, eloc, self.flags)
        torch.cuda.synchronize()
        return eloc.cpu().numpy()

    def host(self):
        import torch
        torch.cuda.synchronize()
        return dict(phi=self.phi.cpu().numpy().astype(np.complex128), theta=self.theta.cpu().numpy().astype(np.complex128),
                    w=self.weight.cpu().numpy(), S=self.ovlp.cpu().numpy(), f=self.fb.cpu().numpy().astype(np.complex128),
                    flags=self.flags.cpu().numpy())


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
