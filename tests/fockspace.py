"""Brute-force second quantisation on the full Fock space (test helper, not the oracle).

Spin orbital p = s*M + i (s = 0 alpha, 1 beta); a basis state is the bitmask of occupied
spin orbitals; c+_p |n> = (-1)^{#occupied below p} |n + p>.  Everything is built from this
single rule, so it shares nothing with oracle/ or the CUDA path.
"""
import numpy as np
import scipy.sparse as sp


class Fock:
    def __init__(self, M):
        self.M = M
        self.n_so = 2 * M
        self.dim = 1 << self.n_so
        states = np.arange(self.dim, dtype=np.int64)
        self._cre = []
        for p in range(self.n_so):
            free = (states >> p) & 1 == 0
            src = states[free]
            below = src & ((1 << p) - 1)
            par = np.zeros_like(below)
            b = below.copy()
            while np.any(b):
                par ^= b & 1
                b >>= 1
            sign = 1.0 - 2.0 * par
            self._cre.append(sp.csr_matrix((sign, (src | (1 << p), src)), shape=(self.dim, self.dim)))
        self._ann = [c.T.tocsr() for c in self._cre]
        self.popcount_a = np.array([bin(int(s) & ((1 << M) - 1)).count("1") for s in states])
        self.popcount_b = np.array([bin(int(s) >> M).count("1") for s in states])

    def cre(self, i, s):
        return self._cre[s * self.M + i]

    def ann(self, i, s):
        return self._ann[s * self.M + i]

    def sector(self, na, nb):
        return np.nonzero((self.popcount_a == na) & (self.popcount_b == nb))[0]

    def one_body(self, mat):
        """sum_ij mat[i,j] sum_s c+_is c_js (sparse)."""
        out = sp.csr_matrix((self.dim, self.dim), dtype=np.result_type(mat.dtype, np.float64))
        for s in range(2):
            for i in range(self.M):
                for j in range(self.M):
                    if mat[i, j] != 0:
                        out = out + mat[i, j] * (self.cre(i, s) @ self.ann(j, s))
        return out

    def hamiltonian_eq1(self, h, V):
        """Eq. (1) literally: sum h_ij c+_is c_js + 1/2 sum V_ijkl c+_is c+_jt c_lt c_ks."""
        M = self.M
        H = self.one_body(h).astype(np.float64)
        for s in range(2):
            for t in range(2):
                for i in range(M):
                    for k in range(M):
                        left = self.cre(i, s)
                        right = self.ann(k, s)
                        for j in range(M):
                            for l in range(M):
                                v = V[i, j, k, l]
                                if v != 0:
                                    H = H + 0.5 * v * (left @ self.cre(j, t) @ self.ann(l, t) @ right)
        return H

    def determinant(self, phi_a, phi_b):
        """|phi> = prod_a (sum_i Phi_a[i,a] c+_i,alpha) prod_b (...beta) |0>, dense vector."""
        vec = np.zeros(self.dim, dtype=np.complex128)
        vec[0] = 1.0
        cols = [(phi_b, 1, b) for b in reversed(range(phi_b.shape[1]))]
        cols += [(phi_a, 0, a) for a in reversed(range(phi_a.shape[1]))]
        for mat, s, a in cols:
            new = np.zeros_like(vec)
            for i in range(self.M):
                if mat[i, a] != 0:
                    new += mat[i, a] * (self.cre(i, s) @ vec)
            vec = new
        return vec


def sector_one_body_ops(M, na, nb):
    """Dense E_ij = sum_s c+_is c_js restricted to the (na, nb) sector: [M][M][d][d], plus Fock."""
    fk = Fock(M)
    idx = fk.sector(na, nb)
    E = np.zeros((M, M, idx.size, idx.size))
    for i in range(M):
        for j in range(M):
            op = fk.cre(i, 0) @ fk.ann(j, 0) + fk.cre(i, 1) @ fk.ann(j, 1)
            E[i, j] = op[idx][:, idx].toarray()
    return fk, idx, E
