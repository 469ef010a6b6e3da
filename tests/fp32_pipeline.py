"""A plain numpy complex64 restatement of the walker step -- TEST INFRASTRUCTURE ONLY.

It exists to MEASURE what any single-precision implementation of the step can reach against the FP64 oracle
(the condition-number scaling of the FP32 tolerance), so that the tolerance of the GPU
parity tests rests on a committed measurement instead of a model.  Same formulas and order as oracle/afqmc_oracle.py
(readings R1-R3, R5, R6), every matrix in complex64 / float32; the per-walker scalars
(S, w, c) are FP64 as in the ABI (R17).  The N x N overlap matrix is formed in complex64 and inverted in complex128
(what the CUDA path does; a complex64 inverse would only be worse).  numpy only; shares no code with csrc/."""
from __future__ import annotations

import numpy as np

from oracle import afqmc_oracle as orc


def c64(a):
    return np.asarray(a).astype(np.complex64)


def init32(wl, ini):
    return dict(L=wl.L.astype(np.float32), Eh=ini["Eh"].astype(np.float32),
                psi=tuple(p.astype(np.float32) for p in ini["psi"]), R=tuple(r.astype(np.float32) for r in ini["R"]),
                hrot=tuple(h.astype(np.float32) for h in ini["hrot"]), Y=tuple(y.astype(np.float32) for y in ini["Y"]),
                dt=float(wl.dt))


def green32(i32, phi, na):
    S = np.ones(phi.shape[0], dtype=np.complex128)
    ths = []
    for psi, ph in zip(i32["psi"], (phi[..., :na], phi[..., na:])):
        if psi.shape[1] == 0:
            ths.append(ph)
            continue
        A = np.matmul(psi.T[None], ph).astype(np.complex64)
        A64 = A.astype(np.complex128)
        S = S * np.linalg.det(A64)
        ths.append(np.matmul(ph, c64(np.linalg.inv(A64))).astype(np.complex64))
    return S, np.concatenate(ths, axis=2)


def fb32(i32, theta, na):
    out = []
    for Rs, th in zip(i32["R"], (theta[..., :na], theta[..., na:])):
        out.append(c64(np.einsum("gak,wka->wg", Rs, th, optimize=True)))
    return out[0], out[1]


def energy32(i32, theta, fa, fb, na):
    E = np.einsum("wg,wg->w", fa.astype(np.complex128), fb.astype(np.complex128))
    for hr, Ys, th in zip(i32["hrot"], i32["Y"], (theta[..., :na], theta[..., na:])):
        E = E + np.einsum("ak,wka->w", hr, th).astype(np.complex128)
        v = th.reshape(th.shape[0], -1)
        u = np.matmul(v, Ys).astype(np.complex64)
        E = E + 0.5 * np.einsum("wi,wi->w", v.astype(np.complex128), u.astype(np.complex128))
    return E


class State32:
    def __init__(self, phi, w, S, theta, fa, fb, eloc):
        self.phi, self.w, self.S, self.theta, self.fa, self.fb, self.eloc = phi, w, S, theta, fa, fb, eloc


def seed32(i32, phi, na, w=None, S=None):
    phi = c64(phi)
    w = np.ones(phi.shape[0]) if w is None else np.asarray(w, dtype=np.float64)
    S0, th = green32(i32, phi, na)
    fa, fb = fb32(i32, th, na)
    return State32(phi, w, S0 if S is None else np.asarray(S, dtype=np.complex128), th, fa, fb, energy32(i32, th, fa, fb, na))


def step32(i32, st, x, na, K=6, E0=0.0):
    dt = i32["dt"]
    sdt = np.float32(np.sqrt(dt))
    f = (st.fa + st.fb).astype(np.complex64)
    x32 = np.asarray(x).astype(np.float32)
    xbar = (-1j * sdt * f).astype(np.complex64)
    xs = (x32 - xbar).astype(np.complex64)
    xb, xd = xbar.astype(np.complex128), x32.astype(np.float64)
    c = np.sum(xd * xb, axis=-1) - 0.5 * np.sum(xb * xb, axis=-1)
    A = (1j * sdt * np.tensordot(xs, i32["L"], axes=(1, 0))).astype(np.complex64)
    T = np.matmul(i32["Eh"][None], st.phi).astype(np.complex64)
    P = T.copy()
    for k in range(1, K + 1):
        T = (np.matmul(A, T) / np.float32(k)).astype(np.complex64)
        P = (P + T).astype(np.complex64)
    phi = np.matmul(i32["Eh"][None], P).astype(np.complex64)
    S, th = green32(i32, phi, na)
    fa, fb = fb32(i32, th, na)
    w, absI, cosd = orc.o_weight(st.S, S, c, st.w, dt, E0)        # FP64 scalars: the rule itself is the oracle's
    return State32(phi, w, S, th, fa, fb, energy32(i32, th, fa, fb, na))


def ortho32(st, na):
    """orthonormalise the complex64 walker (FP64 arithmetic, stored back in complex64), S <- S / det R."""
    q, s = orc.o_orthonormalize(st.phi.astype(np.complex128), st.S, na)
    return State32(c64(q), st.w, s, st.theta, st.fa, st.fb, st.eloc)
