"""FP64 CPU oracle for the phaseless AFQMC walker step -- TEST INFRASTRUCTURE ONLY.

Plain numpy, complex128 throughout, no blocking / fusion / reordering beyond what the
definitions state.  It shares no code with the CUDA path (paper_1804_03310_b200/) and
neither imports the other.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import it.

Everything is batched over a leading walker axis (numpy broadcasting of `@`), which is
the same arithmetic as a per-walker loop.

Citations are PAPER.md:<line>.  Where the paper is silent the
reading is the one listed in DESIGN.md "Readings" (R1..R18).

Pins (tests/test_oracle_*.py, all `-m "not gpu"`):
  o_init / h'            P1  operator identity in Fock space
  o_green, o_force_bias  P2  Fock-space overlaps / mixed expectation values
  o_local_energy         P3  Hartree-Fock closed form, Fock space, Y-form == Cholesky form
  o_propagate            P4  Thouless theorem in Fock space, Taylor vs scipy expm bound
  o_step weights         P5  force-bias sign: odd-in-x part of log I cancels
  o_weight               P15 hand-derived values of the phaseless rule, hybrid and local-energy form (both modes),
                             kill boundary at arg(rho) = +-pi/2, dead walkers stay dead, no overflow at |rho| = 1e200
  multi-det SMW          P6  Eq. (4) == direct recomputation
  Cholesky <-> V         P7  pivoted Cholesky reproduces V and the energies
  multi-det mixed        P8  Fock-space brute force;  P9 FCI trial => E_L == E_FCI
  whole method           P10 long run vs FCI on cfg 1
  o_orthonormalize       P12 Fock-space |Phi> = det(R_a) det(R_b) |Q>, Q^+Q = 1, R upper / positive diagonal,
                             Theta / f / E_L invariance, S' == overlap recomputed from Q
  o_comb / o_population_control  P13 brute-force tooth counting, copies in {floor, ceil}(N w_i / W),
                             mean copies over u == N w_i / W, total weight kept
  o_run                  P14 schedule == hand-unrolled o_step / ortho / comb sequence; mixed estimator unchanged
                             by orthonormalisation
No step-level worked numeric example is printed in the paper: parity is pinned only by
P1-P14 (DESIGN.md says so too).
"""
from __future__ import annotations

import numpy as np


# --------------------------------------------------------------------------------------
# O-init: PAPER.md:34-39 (Hamiltonian, H_2 = -1/2 sum v^2), :80 and Eq. (5) :78 (Y tensor)
# --------------------------------------------------------------------------------------
def o_init(h, L, dt, psi_a, psi_b):
    """Precompute the step's constants.

    h [M][M] real symmetric (T_ij of Eq. 1), L [N_g][M][M] real symmetric with
    V_ijkl = sum_g L_g[i,k] L_g[j,l], psi_s [M][N_s] real trial orbitals.

    Returns dict with
      hp   = h - 1/2 sum_g L_g L_g            (H = sum hp c+c + 1/2 sum_g Lhat_g^2, R3)
      Eh   = expm(-(dt/2) hp)                  via eigh (R3: exact, symmetric split)
      R_s  = psi_s^T L_g                       [N_g][N_s][M]
      hrot_s = psi_s^T h                       [N_s][M]
      Y_s[(k,a),(l,b)] = sum_g R_s[g,a,k] R_s[g,b,l] - R_s[g,a,l] R_s[g,b,k]   (Eq. 5 per spin, R8)
    """
    h = np.asarray(h, dtype=np.float64)
    L = np.asarray(L, dtype=np.float64)
    hp = h - 0.5 * np.matmul(L, L).sum(axis=0)
    ev, U = np.linalg.eigh(hp)
    Eh = (U * np.exp(-0.5 * dt * ev)) @ U.T
    out = dict(h=h, L=L, hp=hp, Eh=Eh, dt=float(dt), psi=(np.asarray(psi_a), np.asarray(psi_b)))
    R, hrot, Y = [], [], []
    for psi in out["psi"]:
        Rs = np.matmul(psi.T[None], L)                      # [g][a][k]
        R.append(Rs)
        hrot.append(psi.T @ h)                              # [a][k]
        ns, M = Rs.shape[1], Rs.shape[2]
        Rflat = Rs.transpose(0, 2, 1).reshape(Rs.shape[0], M * ns)   # [g][(k,a)]
        coul = Rflat.T @ Rflat                              # sum_g R[g,a,k] R[g,b,l]
        exch = np.tensordot(Rs, Rs, axes=(0, 0))            # [a][l][b][k]
        exch = exch.transpose(3, 0, 1, 2).reshape(M * ns, M * ns)    # [(k,a)][(l,b)]
        Y.append(coul - exch)
    out["R"], out["hrot"], out["Y"] = tuple(R), tuple(hrot), tuple(Y)
    return out


def split_spin(phi, n_alpha):
    """phi [...][M][N_t] -> (phi_alpha [...][M][N_a], phi_beta [...][M][N_b])."""
    return phi[..., :n_alpha], phi[..., n_alpha:]


# --------------------------------------------------------------------------------------
# O-green: PAPER.md:51, :61, :68  (A = [psi_T]^dagger [phi_k]; overlap; Green's function)
# --------------------------------------------------------------------------------------
def o_green(psi_a, psi_b, phi, want_G=False):
    """Overlap S = det(A_a) det(A_b), Theta_s = Phi_s A_s^{-1}, optional G_s = (Theta_s psi_s^T)^T.

    G_s[i,j] = <Psi_T| c+_i c_j |phi> / <Psi_T|phi>  (R15).  phi [N_w][M][N_t] complex.
    Returns S [N_w] complex128, theta [N_w][M][N_t], and G [N_w][2][M][M] if want_G.
    """
    phi = np.asarray(phi, dtype=np.complex128)
    na = psi_a.shape[1]
    S = np.ones(phi.shape[0], dtype=np.complex128)
    thetas, Gs = [], []
    for psi, ph in zip((psi_a, psi_b), split_spin(phi, na)):
        A = np.matmul(psi.T[None], ph)                      # [w][N_s][N_s]
        S = S * np.linalg.det(A)
        th = np.matmul(ph, np.linalg.inv(A))                # [w][M][N_s]
        thetas.append(th)
        if want_G:
            Gs.append(np.matmul(th, psi.T[None]).transpose(0, 2, 1))
    theta = np.concatenate(thetas, axis=2)
    if want_G:
        return S, theta, np.stack(Gs, axis=1)
    return S, theta


# --------------------------------------------------------------------------------------
# O-fb: PAPER.md:51 ("shifted by a force-bias"), north_star: f_g = Tr(L_g G)
# --------------------------------------------------------------------------------------
def o_force_bias(R, theta, n_alpha):
    """f^s_g = sum_{a,k} R_s[g,a,k] Theta_s[k,a] (= sum_ij L_g[i,j] G_s[i,j]).

    Returns (f_alpha, f_beta), each [N_w][N_g] complex; the API quantity is their sum (R2)."""
    out = []
    for Rs, th in zip(R, split_spin(theta, n_alpha)):
        out.append(np.einsum("gak,wka->wg", Rs, th, optimize=True))
    return out[0], out[1]


# --------------------------------------------------------------------------------------
# Local energy: PAPER.md:51 (E_L definition), :70-80 + Eq. (5) (Y form), R8 (spin structure)
# --------------------------------------------------------------------------------------
def o_local_energy(ini, theta, f_a, f_b, n_alpha):
    """E_L = sum_s Tr(hrot_s Theta_s) + 1/2 sum_s vec(Theta_s)^T Y_s vec(Theta_s) + sum_g f^a_g f^b_g."""
    E = np.einsum("wg,wg->w", f_a, f_b)
    for hr, Ys, th in zip(ini["hrot"], ini["Y"], split_spin(theta, n_alpha)):
        E = E + np.einsum("ak,wka->w", hr, th)
        v = th.reshape(th.shape[0], -1)                     # row-major (k,a) -> k*N_s + a
        E = E + 0.5 * np.einsum("wi,wi->w", v, v @ Ys)      # Y symmetric
    return E


def o_local_energy_chol(ini, theta, n_alpha):
    """Cholesky-form cross-check: E_2 = 1/2 sum_g f_g^2 - 1/2 sum_s sum_g Tr(T^s_g T^s_g), T = R Theta."""
    f_a, f_b = o_force_bias(ini["R"], theta, n_alpha)
    f = f_a + f_b
    E = 0.5 * np.einsum("wg,wg->w", f, f)
    for hr, Rs, th in zip(ini["hrot"], ini["R"], split_spin(theta, n_alpha)):
        E = E + np.einsum("ak,wka->w", hr, th)
        T = np.einsum("gak,wkb->wgab", Rs, th, optimize=True)
        E = E - 0.5 * np.einsum("wgab,wgba->w", T, T, optimize=True)
    return E


# --------------------------------------------------------------------------------------
# O-step pieces: PAPER.md:41-53 (Eq. 2, 3, Thouless, force bias, phaseless rule), :97 (hybrid)
# --------------------------------------------------------------------------------------
def o_shift(x, f, dt):
    """Step 1: xbar = -i sqrt(dt) f;  xs = x - xbar;  c = sum x xbar - 1/2 sum xbar^2 (no conj) (R2)."""
    xbar = -1j * np.sqrt(dt) * f
    xs = x - xbar
    c = np.sum(x * xbar, axis=-1) - 0.5 * np.sum(xbar * xbar, axis=-1)
    return xs, c


def o_assemble(L, xs, dt):
    """Step 2: A = i sqrt(dt) sum_g xs_g L_g  (Eq. 2's exponent with v_g = i L_g, R1)."""
    return 1j * np.sqrt(dt) * np.tensordot(xs, L, axes=(1, 0))      # [w][M][M]


def o_propagate(Eh, A, phi, K):
    """Step 3: Phi' = Eh [sum_{k=0..K} A^k / k!] Eh Phi (Taylor order K; R3, R9)."""
    T = np.matmul(Eh[None], phi)
    P = T.copy()
    for k in range(1, K + 1):
        T = np.matmul(A, T) / k
        P = P + T
    return np.matmul(Eh[None], P)


def o_weight(S_old, S_new, c, w, dt, E0, mode=0, E_pre=None):
    """Step 5: rho = S'/S, dtheta = arg rho, I = rho e^c.

    hybrid (mode 0): w' = w e^{dt E0} |I| max(0, cos dtheta);
    local-energy (mode 1): w' = w exp(-dt (Re E_L(pre) - E0)) max(0, cos dtheta).
    Returns w', |I|, cos dtheta."""
    rho = S_new / S_old
    dtheta = np.arctan2(rho.imag, rho.real)
    cosd = np.cos(dtheta)
    with np.errstate(over="ignore"):
        absI = np.exp(np.log(np.abs(rho)) + c.real)
    if mode == 0:
        fac = np.exp(dt * E0) * absI
    else:
        fac = np.exp(-dt * (E_pre.real - E0))
    # max{0, cos dtheta}: cos dtheta = Re(rho)/|rho|, so the walker is killed iff Re(rho) <= 0.  The
    # decision is taken on Re(rho) itself (reading R6b): cos(atan2(y, x)) in floating point is 6e-17 > 0 at x = 0 and
    # for tiny negative x, i.e. it misses exactly the boundary the rule is about.
    killed = (rho.real <= 0.0) | (w == 0.0)        # a dead walker stays dead (0 * anything = 0)
    with np.errstate(invalid="ignore", over="ignore"):
        w_new = np.where(killed, 0.0, w * fac * cosd)
    return w_new, absI, cosd


class OracleState:
    """Walker population state carried between steps: {Phi, w, S, Theta, f_a, f_b, E_L}."""

    def __init__(self, phi, w, S, theta, f_a, f_b, eloc):
        self.phi, self.w, self.S, self.theta = phi, w, S, theta
        self.f_a, self.f_b, self.eloc = f_a, f_b, eloc


def o_seed_state(ini, phi, n_alpha, w=None, trial=None):
    """State of a fresh population: O-green + O-fb + E_L on the given walkers (O-init item 5)."""
    phi = np.asarray(phi, dtype=np.complex128)
    w = np.ones(phi.shape[0]) if w is None else np.asarray(w, dtype=np.float64)
    if trial is not None:
        S, theta, f, eloc = o_multidet_smw(ini, trial, phi, n_alpha)[:4]
        return OracleState(phi, w, S, theta, f, np.zeros_like(f), eloc)
    S, theta = o_green(ini["psi"][0], ini["psi"][1], phi)
    f_a, f_b = o_force_bias(ini["R"], theta, n_alpha)
    eloc = o_local_energy(ini, theta, f_a, f_b, n_alpha)
    return OracleState(phi, w, S, theta, f_a, f_b, eloc)


def o_step(ini, st, x, n_alpha, K=6, E0=0.0, mode=0, trial=None):
    """One walker step for the whole population (order R10): shift -> assemble -> propagate ->
    new overlap/Theta -> weight -> force bias and E_L on the new walker.

    x [N_w][N_g] real fields.  Returns (new state, record dict for parity)."""
    dt = ini["dt"]
    f = st.f_a + st.f_b
    xs, c = o_shift(x, f, dt)
    A = o_assemble(ini["L"], xs, dt)
    phi_new = o_propagate(ini["Eh"], A, st.phi, K)
    if trial is not None:
        S_new, theta_new, f_new, eloc_new = o_multidet_smw(ini, trial, phi_new, n_alpha)[:4]
        fa_new, fb_new = f_new, np.zeros_like(f_new)
    else:
        S_new, theta_new = o_green(ini["psi"][0], ini["psi"][1], phi_new)
        fa_new, fb_new = o_force_bias(ini["R"], theta_new, n_alpha)
        eloc_new = o_local_energy(ini, theta_new, fa_new, fb_new, n_alpha)
    w_new, absI, cosd = o_weight(st.S, S_new, c, st.w, dt, E0, mode, st.eloc)
    rec = dict(f_used=f, xs=xs, c=c, phi=phi_new, S=S_new, w=w_new, absI=absI, cosd=cosd,
               eloc=eloc_new, theta=theta_new, f=fa_new + fb_new)
    return OracleState(phi_new, w_new, S_new, theta_new, fa_new, fb_new, eloc_new), rec


def o_mixed_energy(w, eloc):
    """Population mixed estimator E_mix = Re(sum w E_L) / sum w."""
    return float(np.real(np.sum(w * eloc)) / np.sum(w))


# --------------------------------------------------------------------------------------
# O-multidet: PAPER.md:61-68 (Eq. 4, |Psi_T> = sum_i c_i |psi_T,i>, orthonormal determinants)
# --------------------------------------------------------------------------------------
class MultiDetTrial:
    """C_act [M][n_act]; determinant i, spin s has columns occ[i][s] of C_act (in-place
    replacement of reference columns by particles, no re-sorting => no sign; R13)."""

    def __init__(self, C_act, coeff, exc, n_alpha, n_beta):
        self.C = np.asarray(C_act, dtype=np.float64)
        self.coeff = np.asarray(coeff, dtype=np.float64)
        self.exc = np.asarray(exc)
        self.n_sigma = (n_alpha, n_beta)
        self.n_det = self.coeff.shape[0]

    def occ(self, i, s):
        occ = list(range(self.n_sigma[s]))
        for hole, part in self.exc[i, s]:
            if hole >= 0:
                occ[int(hole)] = int(part)
        return occ

    def holes_particles(self, i, s):
        hp = [(int(a), int(p)) for a, p in self.exc[i, s] if a >= 0]
        return [a for a, _ in hp], [p for _, p in hp]


def o_multidet_definition(ini, trial, phi, n_alpha, want_G=False):
    """Definition path (the truth): every determinant recomputed directly.

    S = sum_i c_i* S_i;  G_s = sum_i c_i* S_i G_i^s / S;  f_g = sum_s sum_jk L_g[j,k] G_s[j,k];
    E_L = sum_i c_i* S_i E_L^(i) / S with E_L^(i) in Cholesky form for determinant i.
    Returns S, f, E_L (, G [N_w][2][M][M])."""
    phi = np.asarray(phi, dtype=np.complex128)
    nw, M = phi.shape[0], phi.shape[1]
    h, L = ini["h"], ini["L"]
    S = np.zeros(nw, dtype=np.complex128)
    Gacc = np.zeros((nw, 2, M, M), dtype=np.complex128)
    Eacc = np.zeros(nw, dtype=np.complex128)
    for i in range(trial.n_det):
        Si = np.ones(nw, dtype=np.complex128)
        Gi, fi, e1, exch = [], [], 0.0, 0.0
        for s, ph in enumerate(split_spin(phi, n_alpha)):
            psi = trial.C[:, trial.occ(i, s)]
            A = np.matmul(psi.T[None], ph)
            Si = Si * np.linalg.det(A)
            th = np.matmul(ph, np.linalg.inv(A))
            Gi.append(np.matmul(th, psi.T[None]).transpose(0, 2, 1))
            Rs = np.matmul(psi.T[None], L)                  # [g][a][k]
            T = np.einsum("gak,wkb->wgab", Rs, th, optimize=True)
            fi.append(np.einsum("wgaa->wg", T))
            e1 = e1 + np.einsum("ak,wka->w", psi.T @ h, th)
            exch = exch + np.einsum("wgab,wgba->w", T, T, optimize=True)
        ft = fi[0] + fi[1]
        Ei = e1 + 0.5 * np.einsum("wg,wg->w", ft, ft) - 0.5 * exch
        ci = np.conj(trial.coeff[i])
        S += ci * Si
        Eacc += ci * Si * Ei
        Gacc += (ci * Si)[:, None, None, None] * np.stack(Gi, axis=1)
    G = Gacc / S[:, None, None, None]
    f = np.einsum("gjk,wsjk->wg", L, G, optimize=True)
    E = Eacc / S
    if want_G:
        return S, f, E, G
    return S, f, E


def o_smw_det_inverse(A0_inv, detA0, U, Vt):
    """Eq. (4), for one matrix: returns det(A0 + U V^T) and its inverse."""
    E = U.shape[1]
    Kmat = np.eye(E) + Vt @ A0_inv @ U
    det = np.linalg.det(Kmat) * detA0
    inv = A0_inv - A0_inv @ U @ np.linalg.inv(Kmat) @ Vt @ A0_inv
    return det, inv


def o_multidet_smw(ini, trial, phi, n_alpha, want_G=False):
    """SMW path (second, independent function): reference determinant first, then Eq. (4)
    updates for all i != 0 with U_i = e_{H_i}, V_i^T = (C_{P_i}^T - C_{H_i}^T) Phi_s.

    Returns S, theta (of the reference determinant), f, E_L (, G)."""
    phi = np.asarray(phi, dtype=np.complex128)
    nw, M = phi.shape[0], phi.shape[1]
    h, L, C = ini["h"], ini["L"], trial.C
    S = np.zeros(nw, dtype=np.complex128)
    Gacc = np.zeros((nw, 2, M, M), dtype=np.complex128)
    Eacc = np.zeros(nw, dtype=np.complex128)
    ref = []
    for s, ph in enumerate(split_spin(phi, n_alpha)):
        ns = trial.n_sigma[s]
        A0 = np.matmul(C[:, :ns].T[None], ph)
        ref.append((ph, np.linalg.det(A0), np.linalg.inv(A0)))
    theta0 = np.concatenate([np.matmul(ph, Ai) for ph, _, Ai in ref], axis=2)
    for i in range(trial.n_det):
        Si = np.ones(nw, dtype=np.complex128)
        Gi, fi, e1, exch = [], [], 0.0, 0.0
        for s in range(2):
            ph, det0, inv0 = ref[s]
            ns = trial.n_sigma[s]
            holes, parts = trial.holes_particles(i, s)
            if holes:
                U = np.zeros((ns, len(holes)))
                U[holes, np.arange(len(holes))] = 1.0
                Vt = np.matmul((C[:, parts] - C[:, holes]).T[None], ph)   # [w][E][ns]
                Kmat = np.eye(len(holes))[None] + np.matmul(np.matmul(Vt, inv0), U[None])
                det = np.linalg.det(Kmat) * det0
                inv = inv0 - np.matmul(np.matmul(np.matmul(inv0, U[None]), np.linalg.inv(Kmat)),
                                       np.matmul(Vt, inv0))
            else:
                det, inv = det0, inv0
            psi = C[:, trial.occ(i, s)]
            Si = Si * det
            th = np.matmul(ph, inv)
            Gi.append(np.matmul(th, psi.T[None]).transpose(0, 2, 1))
            Rs = np.matmul(psi.T[None], L)
            T = np.einsum("gak,wkb->wgab", Rs, th, optimize=True)
            fi.append(np.einsum("wgaa->wg", T))
            e1 = e1 + np.einsum("ak,wka->w", psi.T @ h, th)
            exch = exch + np.einsum("wgab,wgba->w", T, T, optimize=True)
        ft = fi[0] + fi[1]
        Ei = e1 + 0.5 * np.einsum("wg,wg->w", ft, ft) - 0.5 * exch
        ci = np.conj(trial.coeff[i])
        S += ci * Si
        Eacc += ci * Si * Ei
        Gacc += (ci * Si)[:, None, None, None] * np.stack(Gi, axis=1)
    G = Gacc / S[:, None, None, None]
    f = np.einsum("gjk,wsjk->wg", L, G, optimize=True)
    E = Eacc / S
    if want_G:
        return S, theta0, f, E, G
    return S, theta0, f, E


# --------------------------------------------------------------------------------------
# NEXT-1 / NEXT-2: the two steps either side of the walker step and the paper's
# schedule.  PAPER.md:97 ("Walker orbitals are orthonormalized after every two propagation steps",
# local energy "measured every 0.1 Ha^-1", population control "at intervals of 0.1 Ha^-1"),
# PAPER.md:295 ("a simple combing method").  Also used by the FCI pin P10.
# --------------------------------------------------------------------------------------
def o_orthonormalize(phi, S, n_alpha):
    """Thin QR of each spin block, Phi_s = Q_s R_s; the walker becomes Q and S <- S / (det R_a det R_b),
    because |Phi> = det(R_a) det(R_b) |Q> (a determinant is multilinear and alternating in its columns).

    Reading R21: R has a real positive diagonal -- the one thin QR that is unique -- so LAPACK's
    Householder factors are re-phased column by column: Q <- Q D, R <- D^* R, D = diag(R_jj / |R_jj|).
    Returns (Q, S')."""
    out = []
    S = np.array(S, dtype=np.complex128, copy=True)
    for ph in split_spin(phi, n_alpha):
        if ph.shape[2] == 0:
            out.append(ph)
            continue
        Q, R = np.linalg.qr(ph)
        d = np.diagonal(R, axis1=1, axis2=2)
        D = d / np.abs(d)
        Q = Q * D[:, None, :]
        S = S / np.prod(np.abs(d), axis=1)
        out.append(Q)
    return np.concatenate(out, axis=2), S


def o_comb(w, u):
    """'Simple combing' population control: returns the parent index of each new walker.

    Reading R22: N_w teeth at t_i = (i + u) W / N_w, W = sum w, u in [0,1) drawn by the caller; tooth i
    selects the first walker p whose running sum c_p = w_0 + ... + w_p (accumulated in index order)
    exceeds t_i.  Every new walker then carries the weight W / N_w (the population keeps its total weight)."""
    n = w.shape[0]
    cum = np.cumsum(w)
    teeth = (np.arange(n) + u) * (cum[-1] / n)
    return np.searchsorted(cum, teeth, side="right").clip(0, n - 1)


def o_population_control(st, u):
    """Comb the population: every per-walker quantity of the state follows its parent; weights = W / N_w.
    Returns (new state, parent indices)."""
    par = o_comb(st.w, u)
    n = st.w.shape[0]
    w = np.full(n, np.cumsum(st.w)[-1] / n)            # W = the running sum's last element (R22)
    return OracleState(st.phi[par], w, st.S[par], st.theta[par], st.f_a[par], st.f_b[par], st.eloc[par]), par


def o_run(ini, st, xs, n_alpha, K=6, E0=0.0, energy_every=1, ortho_every=0, pc_every=0, us=(), trial=None):
    """The paper's schedule around o_step, hybrid weights (mode 0) only.  After step n
    (1-based): E_L is recorded if n % energy_every == 0; then the walkers are orthonormalised if
    n % ortho_every == 0; then combed if n % pc_every == 0 with offset us[n / pc_every - 1] (reading R23:
    measure, orthonormalise, comb, in that order; 0 switches a part off).  Theta, f and E_L do not change
    under orthonormalisation (Theta = Phi A^-1 is invariant under Phi -> Phi R^-1), so the order of the first
    two is immaterial.  Returns (state, [(n, w at measurement, E_L)], [parents per comb])."""
    meas, parents = [], []
    for n in range(1, xs.shape[0] + 1):
        st, _ = o_step(ini, st, xs[n - 1], n_alpha, K=K, E0=E0, mode=0, trial=trial)
        if energy_every and n % energy_every == 0:
            meas.append((n, st.w.copy(), st.eloc.copy()))
        if ortho_every and n % ortho_every == 0:
            phi, S = o_orthonormalize(st.phi, st.S, n_alpha)
            st = OracleState(phi, st.w, S, st.theta, st.f_a, st.f_b, st.eloc)
        if pc_every and n % pc_every == 0:
            st, par = o_population_control(st, us[n // pc_every - 1])
            parents.append(par)
    return st, meas, parents
