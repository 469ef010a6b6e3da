"""Pins P12-P14 for the oracle's orthonormalisation, comb population control and schedule (no GPU).
PAPER.md:97 (orthonormalise every 2 steps, energy / population control every 0.1 Ha^-1), :295 (comb).
Each pin checks the oracle against something other than itself: Fock-space vectors, explicit loops,
algebraic invariants."""
import numpy as np
import pytest

from oracle import afqmc_oracle as O
from workloads import make_workload, random_walkers
from tests.fockspace import Fock

SMALL = dict(M=4, n_alpha=2, n_beta=1, n_chol=5, n_walkers=3)


@pytest.fixture(scope="module")
def small():
    wl = make_workload(1, overrides=SMALL)
    ini = O.o_init(wl.h, wl.L, wl.dt, wl.psi_a, wl.psi_b)
    return wl, ini, Fock(wl.M)


def test_P12_orthonormalize_fock(small):
    """|Phi> = det(R_a) det(R_b) |Q> as explicit Fock vectors, with det R = S / S' real positive (R21)."""
    wl, ini, fk = small
    phi = random_walkers(wl, 3, seed=5, spread=0.8)
    S, theta = O.o_green(wl.psi_a, wl.psi_b, phi)
    Q, S2 = O.o_orthonormalize(phi, S, wl.n_alpha)
    for w in range(3):
        ket = fk.determinant(phi[w][:, :wl.n_alpha], phi[w][:, wl.n_alpha:])
        ketq = fk.determinant(Q[w][:, :wl.n_alpha], Q[w][:, wl.n_alpha:])
        ratio = S[w] / S2[w]
        assert abs(ratio.imag) < 1e-13 * abs(ratio) and ratio.real > 0
        assert np.abs(ket - ratio * ketq).max() < 1e-12 * np.abs(ket).max()
        assert abs(np.vdot(ketq, ketq) - 1.0) < 1e-12          # orthonormal orbitals: normalised determinant


def test_P12_orthonormalize_factors_and_invariants():
    """Q^+Q = 1; R = Q^+ Phi upper triangular with a real positive diagonal and Q R = Phi; the overlap recomputed
    from Q equals S'; Theta, force bias and E_L do not change."""
    wl = make_workload(2, overrides=dict(n_walkers=6))
    ini = O.o_init(wl.h, wl.L, wl.dt, wl.psi_a, wl.psi_b)
    phi = random_walkers(wl, 6, seed=9, spread=0.7)
    S, theta = O.o_green(wl.psi_a, wl.psi_b, phi)
    f_a, f_b = O.o_force_bias(ini["R"], theta, wl.n_alpha)
    E = O.o_local_energy(ini, theta, f_a, f_b, wl.n_alpha)
    Q, S2 = O.o_orthonormalize(phi, S, wl.n_alpha)
    lo = 0
    for n in (wl.n_alpha, wl.n_beta):
        q, p = Q[:, :, lo:lo + n], phi[:, :, lo:lo + n]
        lo += n
        qhq = np.einsum("wia,wib->wab", q.conj(), q)
        assert np.abs(qhq - np.eye(n)).max() < 1e-13
        R = np.einsum("wia,wib->wab", q.conj(), p)
        assert np.abs(np.tril(R, -1)).max() < 1e-12
        d = np.diagonal(R, axis1=1, axis2=2)
        assert np.all(d.real > 0) and np.abs(d.imag).max() < 1e-13
        assert np.abs(q @ R - p).max() < 1e-12
    Sq, thq = O.o_green(wl.psi_a, wl.psi_b, Q)
    assert np.abs(Sq - S2).max() < 1e-12 * np.abs(S2).max()
    assert np.abs(thq - theta).max() < 1e-10 * np.abs(theta).max()
    fqa, fqb = O.o_force_bias(ini["R"], thq, wl.n_alpha)
    Eq = O.o_local_energy(ini, thq, fqa, fqb, wl.n_alpha)
    assert np.abs(fqa + fqb - f_a - f_b).max() < 1e-9 * np.abs(f_a + f_b).max()
    assert np.abs(Eq - E).max() < 1e-9 * np.abs(E).max()


def test_P12_orthonormalize_already_orthonormal_and_scaling():
    """Special cases with a closed form: an orthonormal walker is returned unchanged (R = 1); scaling one of its
    columns by a complex s leaves |s| in R and the phase s/|s| in the column (positive diagonal, R21), so
    S' = S_in / |s|."""
    rng = np.random.default_rng(3)
    M, na, nb = 7, 3, 2
    X = rng.standard_normal((2, M, na + nb)) + 1j * rng.standard_normal((2, M, na + nb))
    Q0 = np.concatenate([np.linalg.qr(X[:, :, :na])[0], np.linalg.qr(X[:, :, na:])[0]], axis=2)
    S0 = np.array([1.5 - 0.5j, -0.3 + 2j])
    Q1, S1 = O.o_orthonormalize(Q0, S0, na)
    assert np.abs(Q1 - Q0).max() < 1e-13 and np.abs(S1 - S0).max() < 1e-13
    s = 0.3 - 1.1j
    X2 = Q0.copy()
    X2[:, :, 1] *= s                      # |Phi'> = s |Phi>, so the overlap handed in is s S0
    Q2, S2 = O.o_orthonormalize(X2, s * S0, na)
    ph = s / abs(s)
    Q0p = Q0.copy()
    Q0p[:, :, 1] *= ph                    # positive diagonal: the phase stays in the column
    assert np.abs(Q2 - Q0p).max() < 1e-13
    assert np.abs(S2 - s * S0 / abs(s)).max() < 1e-13


def _comb_bruteforce(w, u):
    """Definition by explicit loops: tooth i at (i+u) W/N falls into the interval [c_{p-1}, c_p) of walker p."""
    n = len(w)
    W = 0.0
    for v in w:
        W += v
    out = []
    for i in range(n):
        t = (i + u) * (W / n)
        c, p = 0.0, 0
        for p in range(n):
            c += w[p]
            if c > t:
                break
        out.append(p)
    return np.array(out)


def test_P13_comb_bruteforce_and_counts():
    rng = np.random.default_rng(11)
    for n in (1, 2, 7, 64, 257):
        w = rng.random(n) ** 3
        w[rng.random(n) < 0.2] = 0.0                    # dead walkers
        if w.sum() == 0:
            w[0] = 1.0
        for u in (0.0, 0.25, 0.999999, rng.random()):
            par = O.o_comb(w, u)
            assert np.array_equal(par, _comb_bruteforce(w, u))
            assert np.all(np.diff(par) >= 0)
            cnt = np.bincount(par, minlength=n)
            ideal = n * w / w.sum()
            assert np.all(cnt >= np.floor(ideal - 1e-9)) and np.all(cnt <= np.ceil(ideal + 1e-9))
            assert np.all(cnt[w == 0.0] == 0)           # a dead walker is never copied


def test_P13_comb_unbiased_and_uniform_identity():
    """Mean number of copies over the offset u equals N w_i / W (the comb is unbiased); equal weights give the
    identity map; total weight is preserved by o_population_control."""
    rng = np.random.default_rng(5)
    n = 16
    w = rng.random(n)
    us = (np.arange(20000) + 0.5) / 20000
    cnt = np.zeros(n)
    for u in us:
        cnt += np.bincount(O.o_comb(w, u), minlength=n)
    assert np.abs(cnt / us.size - n * w / w.sum()).max() < 2e-3
    assert np.array_equal(O.o_comb(np.full(n, 0.37), 0.4), np.arange(n))
    st = O.OracleState(rng.random((n, 3, 2)) + 0j, w, rng.random(n) + 0j, rng.random((n, 3, 2)) + 0j,
                       rng.random((n, 4)) + 0j, rng.random((n, 4)) + 0j, rng.random(n) + 0j)
    st2, par = O.o_population_control(st, 0.3)
    assert abs(st2.w.sum() - w.sum()) < 1e-13 and np.ptp(st2.w) == 0.0
    for a, b in ((st2.phi, st.phi), (st2.S, st.S), (st2.theta, st.theta), (st2.f_a, st.f_a), (st2.eloc, st.eloc)):
        assert np.array_equal(a, b[par])


def test_P14_schedule_matches_unrolled_sequence():
    """o_run == the hand-unrolled sequence of o_step / o_orthonormalize / o_population_control, and
    orthonormalising more often changes neither the weights nor the energies (up to rounding)."""
    wl = make_workload(1, "tame_mf")
    nw, n = 12, 8
    ini = O.o_init(wl.h, wl.L, wl.dt, wl.psi_a, wl.psi_b)
    xs = wl.fields(n, nw)
    us = [0.3, 0.8]
    st0 = O.o_seed_state(ini, wl.walkers(nw), wl.n_alpha)
    st, meas, parents = O.o_run(ini, st0, xs, wl.n_alpha, K=wl.K, energy_every=4, ortho_every=2, pc_every=4, us=us)
    assert [m[0] for m in meas] == [4, 8] and len(parents) == 2
    s2 = O.o_seed_state(ini, wl.walkers(nw), wl.n_alpha)
    for k in range(n):
        s2, _ = O.o_step(ini, s2, xs[k], wl.n_alpha, K=wl.K)
        if k in (3, 7):
            assert np.array_equal(meas[k // 4][2], s2.eloc) and np.array_equal(meas[k // 4][1], s2.w)
        if k % 2 == 1:
            phi, S = O.o_orthonormalize(s2.phi, s2.S, wl.n_alpha)
            s2 = O.OracleState(phi, s2.w, S, s2.theta, s2.f_a, s2.f_b, s2.eloc)
        if k in (3, 7):
            par = O.o_comb(s2.w, us[k // 4])
            assert np.array_equal(par, parents[k // 4])
            s2 = O.OracleState(s2.phi[par], np.full(nw, np.cumsum(s2.w)[-1] / nw), s2.S[par], s2.theta[par], s2.f_a[par],
                               s2.f_b[par], s2.eloc[par])
    assert np.array_equal(st.phi, s2.phi) and np.array_equal(st.w, s2.w) and np.array_equal(st.S, s2.S)
    # no population control: orthonormalisation every step vs never -> same weights and energies
    a, ma, _ = O.o_run(ini, st0, xs, wl.n_alpha, K=wl.K, energy_every=1, ortho_every=1)
    b, mb, _ = O.o_run(ini, st0, xs, wl.n_alpha, K=wl.K, energy_every=1, ortho_every=0)
    assert np.abs(a.w - b.w).max() < 1e-9 * np.abs(b.w).max()
    assert np.abs(ma[-1][2] - mb[-1][2]).max() < 1e-8 * np.abs(mb[-1][2]).max()
    assert O.o_mixed_energy(*ma[-1][1:]) == pytest.approx(O.o_mixed_energy(*mb[-1][1:]), rel=1e-9)
