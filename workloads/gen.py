"""Seeded synthetic inputs for the ph-AFQMC walker step (BASELINE.json configs 1-5).

This module is shared by the CPU oracle's tests and by the CUDA path's tests/bench.
It only *constructs inputs* (Hamiltonian tensors, trial orbitals, determinant lists,
initial walkers, Gaussian field draws).  It holds none of the method's arithmetic:
no overlap, Green's function, force bias, propagator, weight or energy code lives here.

Recipe:
  * one numpy default_rng(0) stream: h first, then L_0 .. L_{N_gamma-1};
  * a "random real symmetric" matrix = upper triangle incl. diagonal filled row-major
    from the stream, then mirrored (every entry keeps the stated standard deviation);
  * h entries N(0,1)/sqrt(M); L entries N(0, sigma_L);
  * trial orbitals = lowest eigenvectors of F = h + sum_g L_g @ L_g, ascending, each
    eigenvector sign-fixed so its largest-magnitude component is positive;
  * fields: default_rng(1).standard_normal((steps, N_w, N_gamma)) in float64;
  * cfg 4 determinants from default_rng(2).
Variants: "raw" (literal), "mf" (mean-field-subtracted h and L: same Hamiltonian on the
(N_alpha, N_beta) sector up to the returned constant), "tame" (sigma_L / 10).

The paper's real inputs (PySCF integrals, CD/DF vectors, UHF/CASSCF trials)
are not available here; these tensors take their shapes and stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field
import numpy as np

# cfg -> parameters.  K = Taylor order, sigma_L per SURVEY R9 (cfg 5: 0.03).
CONFIGS = {
    1: dict(M=8, n_alpha=2, n_beta=2, n_chol=24, n_walkers=64, precision="c128",
            dt=0.01, steps=10, K=6, sigma_L=0.3, n_det=1, n_act=0),
    2: dict(M=20, n_alpha=5, n_beta=5, n_chol=100, n_walkers=1024, precision="c64",
            dt=0.005, steps=50, K=6, sigma_L=0.3, n_det=1, n_act=0),
    3: dict(M=60, n_alpha=15, n_beta=15, n_chol=300, n_walkers=1024, precision="c64",
            dt=0.005, steps=10, K=6, sigma_L=0.1, n_det=1, n_act=0),
    4: dict(M=60, n_alpha=10, n_beta=10, n_chol=300, n_walkers=512, precision="c64",
            dt=0.005, steps=10, K=6, sigma_L=0.1, n_det=100, n_act=20),
    5: dict(M=200, n_alpha=13, n_beta=12, n_chol=1000, n_walkers=2048, precision="c64",
            dt=0.005, steps=10, K=6, sigma_L=0.03, n_det=1, n_act=0),
}


@dataclass
class Workload:
    """Everything one run needs.  All arrays float64 / complex128 on the host."""
    cfg: int
    variant: str
    M: int
    n_alpha: int
    n_beta: int
    n_chol: int
    n_walkers: int
    precision: str          # "c64" or "c128": what the CUDA path computes in
    dt: float
    steps: int
    K: int
    E0: float
    h: np.ndarray           # [M][M]
    L: np.ndarray           # [n_chol][M][M]
    psi_a: np.ndarray       # [M][n_alpha]  (multi-det: reference determinant)
    psi_b: np.ndarray       # [M][n_beta]
    e_const: float = 0.0    # constant to add to energies ("mf" variant), else 0
    n_det: int = 1
    n_act: int = 0
    C_act: np.ndarray | None = None      # [M][n_act]
    det_coeff: np.ndarray | None = None  # [n_det] real, normalised
    det_exc: np.ndarray | None = None    # [n_det][2][max_exc][2] int32 (hole, particle) or -1
    extra: dict = field(default_factory=dict)

    @property
    def n_t(self) -> int:
        return self.n_alpha + self.n_beta

    def walkers(self, n_walkers: int | None = None) -> np.ndarray:
        """Initial walkers = trial (reference) determinant, [N_w][M][N_t] complex128."""
        nw = self.n_walkers if n_walkers is None else n_walkers
        phi0 = np.concatenate([self.psi_a, self.psi_b], axis=1).astype(np.complex128)
        return np.ascontiguousarray(np.broadcast_to(phi0, (nw,) + phi0.shape))

    def fields(self, steps: int | None = None, n_walkers: int | None = None) -> np.ndarray:
        """Gaussian auxiliary fields [steps][N_w][N_gamma], float64, seed 1 (R14).

        The full [steps][N_w][N_gamma] array of the config is always drawn and then
        sliced, so a sub-population sees the same numbers as in the full run."""
        st = self.steps if steps is None else steps
        nw = self.n_walkers if n_walkers is None else n_walkers
        rng = np.random.default_rng(1)
        full_st = max(st, self.steps)
        full_nw = max(nw, self.n_walkers)
        x = rng.standard_normal((full_st, full_nw, self.n_chol))
        return np.ascontiguousarray(x[:st, :nw])


def sym_normal(rng: np.random.Generator, M: int, sigma: float) -> np.ndarray:
    """Random real symmetric M x M: upper triangle (incl. diagonal) row-major, mirrored."""
    iu = np.triu_indices(M)
    vals = rng.standard_normal(iu[0].size) * sigma
    a = np.zeros((M, M))
    a[iu] = vals
    a = a + np.triu(a, 1).T
    return a


def sign_fix(C: np.ndarray) -> np.ndarray:
    """Flip each column so that its largest-magnitude component is positive."""
    C = C.copy()
    idx = np.argmax(np.abs(C), axis=0)
    s = np.sign(C[idx, np.arange(C.shape[1])])
    s[s == 0] = 1.0
    return C * s


def random_walkers(wl: Workload, n_walkers: int, seed: int = 7, spread: float = 0.3) -> np.ndarray:
    """Non-trivial complex, non-orthonormal walkers near the trial (for stage parity tests)."""
    rng = np.random.default_rng(seed)
    phi = wl.walkers(n_walkers).copy()
    noise = rng.standard_normal(phi.shape) + 1j * rng.standard_normal(phi.shape)
    return phi + spread * noise / np.sqrt(wl.M)


def _gen_determinants(n_det: int, n_sigma: tuple[int, int], n_act: int, seed: int = 2):
    """cfg 4 determinant list.  Returns (coeff[n_det], exc[n_det][2][2][2])."""
    rng = np.random.default_rng(seed)
    max_exc = 2
    exc = -np.ones((n_det, 2, max_exc, 2), dtype=np.int32)
    seen = {()}
    dets = [()]
    while len(dets) < n_det:
        rank = 1 if rng.random() < 0.5 else 2
        moves = []
        ok = True
        for _ in range(rank):
            s = int(rng.integers(0, 2))
            hole = int(rng.integers(0, n_sigma[s]))
            part = int(rng.integers(n_sigma[s], n_act))
            # a hole or particle may be used once per spin within one determinant
            if any(m[0] == s and (m[1] == hole or m[2] == part) for m in moves):
                ok = False
            moves.append((s, hole, part))
        if not ok:
            continue
        key = tuple(sorted(moves))
        if key in seen:
            continue
        seen.add(key)
        dets.append(key)
    for i, key in enumerate(dets):
        cnt = [0, 0]
        for (s, hole, part) in key:
            exc[i, s, cnt[s], 0] = hole
            exc[i, s, cnt[s], 1] = part
            cnt[s] += 1
    c = rng.standard_normal(n_det)
    c = c / np.linalg.norm(c)
    # reference-dominated trial: put the largest coefficient on the reference
    if abs(c[0]) < 0.1 * np.max(np.abs(c)):
        j = int(np.argmax(np.abs(c)))
        c[0], c[j] = c[j], c[0]
    return c, exc


def occupations(exc_i: np.ndarray, n_sigma: int) -> list[int]:
    """Column list of determinant i for one spin: (0..n_sigma-1) with holes replaced in place."""
    occ = list(range(n_sigma))
    for e in range(exc_i.shape[0]):
        hole, part = int(exc_i[e, 0]), int(exc_i[e, 1])
        if hole >= 0:
            occ[hole] = part
    return occ


def make_workload(cfg: int, variant: str = "raw", *, n_walkers: int | None = None,
                  overrides: dict | None = None) -> Workload:
    """Build config `cfg` (1..5) in variant raw | mf | tame | tame_mf.

    `overrides` may shrink a config for tests (e.g. {"M": 5, "n_chol": 7}); the recipe
    is unchanged."""
    p = dict(CONFIGS[cfg])
    if overrides:
        p.update(overrides)
    M, na, nb, ng = p["M"], p["n_alpha"], p["n_beta"], p["n_chol"]
    sigma_L = p["sigma_L"] * (0.1 if variant.startswith("tame") else 1.0)
    rng = np.random.default_rng(0)
    h = sym_normal(rng, M, 1.0 / np.sqrt(M))
    L = np.empty((ng, M, M))
    for g in range(ng):
        L[g] = sym_normal(rng, M, sigma_L)
    F = h + np.matmul(L, L).sum(axis=0)
    _, C = np.linalg.eigh(F)
    C = sign_fix(C)
    psi_a = np.ascontiguousarray(C[:, :na])
    psi_b = np.ascontiguousarray(C[:, :nb])
    e_const = 0.0
    E0 = 0.0
    if variant in ("mf", "tame_mf"):
        P = psi_a @ psi_a.T + psi_b @ psi_b.T
        lbar = np.einsum("gij,ji->g", L, P)
        n_e = na + nb
        Lp = L - (lbar / n_e)[:, None, None] * np.eye(M)[None]
        h = (h - 0.5 * np.matmul(L, L).sum(axis=0)
             + 0.5 * np.matmul(Lp, Lp).sum(axis=0)
             + np.einsum("g,gij->ij", lbar, Lp))
        L = Lp
        e_const = 0.5 * float(lbar @ lbar)
    elif variant not in ("raw", "tame"):
        raise ValueError(f"unknown variant {variant!r}")
    wl = Workload(cfg=cfg, variant=variant, M=M, n_alpha=na, n_beta=nb, n_chol=ng,
                  n_walkers=p["n_walkers"] if n_walkers is None else n_walkers,
                  precision=p["precision"], dt=p["dt"], steps=p["steps"], K=p["K"], E0=E0,
                  h=h, L=L, psi_a=psi_a, psi_b=psi_b, e_const=e_const,
                  n_det=p["n_det"], n_act=p["n_act"])
    if p["n_det"] > 1:
        n_act = p["n_act"]
        wl.C_act = np.ascontiguousarray(C[:, :n_act])
        wl.det_coeff, wl.det_exc = _gen_determinants(p["n_det"], (na, nb), n_act, seed=2)
    return wl
