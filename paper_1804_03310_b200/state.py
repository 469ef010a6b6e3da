"""Device-side walker state in the ABI layouts (include/afqmc.h) and a context factory for a seeded Workload.

Marshalling only: allocates the torch tensors the C ABI takes and forwards to the binding.  No method arithmetic
and nothing from the CPU reference side -- bench.py's GPU arm and the parity tests both build their state here."""
from __future__ import annotations

import numpy as np

from .binding import AfqmcContext, make_params


def make_context(wl, n_walkers=None, gemm_path=0, weight_mode=0, E0=None, K=None, max_exc=None, device="cuda:0", stream=None):
    """AfqmcContext for a workloads.Workload (single- or multi-determinant trial)."""
    nw = wl.n_walkers if n_walkers is None else n_walkers
    if max_exc is None:
        max_exc = int(wl.det_exc.shape[2]) if wl.n_det > 1 else 2
    p = make_params(wl.M, wl.n_alpha, wl.n_beta, wl.n_chol, nw, wl.precision, wl.dt,
                    taylor_order=wl.K if K is None else K, weight_mode=weight_mode,
                    E0=wl.E0 if E0 is None else E0, n_det=wl.n_det, n_act=wl.n_act, max_exc=max_exc,
                    gemm_path=gemm_path)
    if wl.n_det > 1:
        return AfqmcContext(p, wl.h, wl.L, wl.psi_a, wl.psi_b, C_act=wl.C_act, det_coeff=wl.det_coeff,
                            det_exc=wl.det_exc, device=device, stream=stream)
    return AfqmcContext(p, wl.h, wl.L, wl.psi_a, wl.psi_b, device=device, stream=stream)


class WalkerState:
    """Walker state tensors on the device: phi, theta, weight, ovlp, fb, flags (+ eloc of the current walkers)."""

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
