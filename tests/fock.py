"""Explicit many-body (Fock-space) matrices by Jordan-Wigner, for pinning the oracle.

Independent of `oracle/`: builds a+_j as dense 2^n x 2^n matrices and determinant states
as products of creation operators on the vacuum.  Spin orbital index = sigma * M + p.
Only usable for n = 2M <= 10 or so.
"""
import numpy as np


def creation_ops(n):
    """List of n creation operators a+_j (dense, real)."""
    cd = np.array([[0.0, 0.0], [1.0, 0.0]])
    Z = np.diag([1.0, -1.0])
    I2 = np.eye(2)
    ops = []
    for j in range(n):
        m = np.array([[1.0]])
        for k in range(n):
            m = np.kron(m, Z if k < j else (cd if k == j else I2))
        ops.append(m)
    return ops


class Fock:
    def __init__(self, M):
        self.M = M
        self.n = 2 * M
        self.cd = creation_ops(self.n)
        self.c = [a.T.copy() for a in self.cd]
        self.vac = np.zeros(2 ** self.n)
        self.vac[0] = 1.0

    def one_body(self, h):
        """sum_sigma sum_pq h_pq a+_{p sigma} a_{q sigma} for an M x M matrix h."""
        M = self.M
        out = np.zeros((2 ** self.n, 2 ** self.n), dtype=np.result_type(h, np.float64))
        for s in range(2):
            for p in range(M):
                for q in range(M):
                    if h[p, q] != 0:
                        out = out + h[p, q] * (self.cd[s * M + p] @ self.c[s * M + q])
        return out

    def hamiltonian(self, h, L):
        """Eq. (2) with (ps|qr) = sum_g L^g_ps L^g_qr (Eq. 3), spin summed:
        H = sum h_pq a+_p a_q + 1/2 sum_{sigma,sigma'} (ps|qr) a+_{p s} a+_{q s'} a_{r s'} a_{s s}."""
        M = self.M
        eri = np.einsum("gps,gqr->psqr", L, L)
        H = self.one_body(h).astype(np.float64)
        for s1 in range(2):
            for s2 in range(2):
                for p in range(M):
                    for q in range(M):
                        ap_aq = self.cd[s1 * M + p] @ self.cd[s2 * M + q]
                        for r in range(M):
                            for s in range(M):
                                H = H + 0.5 * eri[p, s, q, r] * (ap_aq @ self.c[s2 * M + r] @ self.c[s1 * M + s])
        return H

    def hamiltonian_eri(self, h, eri):
        """Eq. (2) for a given (possibly complex) h and four-index tensor eri[p, s, q, r] = (ps|qr)."""
        M = self.M
        H = self.one_body(h).astype(np.complex128)
        for s1 in range(2):
            for s2 in range(2):
                for p in range(M):
                    for q in range(M):
                        ap_aq = self.cd[s1 * M + p] @ self.cd[s2 * M + q]
                        for r in range(M):
                            for s in range(M):
                                if eri[p, s, q, r] != 0:
                                    H = H + 0.5 * eri[p, s, q, r] * (ap_aq @ self.c[s2 * M + r] @ self.c[s1 * M + s])
        return H

    def det_state(self, phi_a, phi_b):
        """prod_i (sum_p phi_a[p,i] a+_{p,up}) prod_j (sum_p phi_b[p,j] a+_{p,dn}) |0>."""
        M = self.M
        v = self.vac.astype(np.complex128)
        cols = [(1, phi_b[:, j]) for j in range(phi_b.shape[1])][::-1] + \
               [(0, phi_a[:, i]) for i in range(phi_a.shape[1])][::-1]
        for s, col in cols:          # rightmost operator acts first
            op = sum(col[p] * self.cd[s * M + p] for p in range(M))
            v = op @ v
        return v
