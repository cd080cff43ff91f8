"""CPU oracle for the walker step and local energy with COMPLEX Cholesky vectors.

TEST INFRASTRUCTURE ONLY (same rules as oracle/afqmc_oracle.py: only tests/ may import it; it shares no
code with the CUDA library).  Pins: tests/test_oracle_complex_pins.py (PC1-PC5, CPU); the CUDA path
(`complex_chol = 1`, csrc/cplx.cu) is compared with this file in tests/test_gpu_complex.py.

Source: /root/reference/PAPER.md Sec. IV.B, PAPER.md:326-328 ("Support of complex Cholesky vectors ... the
number of auxiliary fields is hence twice as many as the number of Cholesky vectors.  The implementation
details are available in Ref. 50") on top of Sec. II, Eqs. (2)-(18).  Ref. 50 is not in the container; what
follows is derived from the paper's own equations:

  * Complex orbitals: (ps|qr) = sum_g L^g_ps (L^g_rq)^*  (the Cholesky factorisation of the positive
    supermatrix V_(ps),(rq); for real orbitals this is Eq. 3).
  * Hermitian parts  A_g = (L_g + L_g^+)/2,  B_g = (L_g - L_g^+)/(2i),  L_g = A_g + i B_g:
        sum_g L^g_ps (L^g_rq)^* = sum_g [A_ps A_qr + B_ps B_qr] + i sum_g [B_ps A_qr - A_ps B_qr].
    The first sum is symmetric under (ps) <-> (qr), the second antisymmetric; electron repulsion integrals
    have (ps|qr) = (qr|ps), so the second sum vanishes and
        (ps|qr) = sum_{g'=1..2n} K^{g'}_ps K^{g'}_qr,   K = (A_1..A_n, B_1..B_n)  Hermitian.
    Every formula of the real case was derived from (ps|qr) = sum L_ps L_qr and one-body
    operators L_hat = sum L_pq a+_p a_q alone, so it holds with the 2n Hermitian K in place of the n real
    symmetric L: 2n auxiliary fields, v_g' = i K_g', m_g' = tr(K_g' P) (real), h' = h - 1/2 sum K K,
    h_mod = h' + sum m K (Hermitian), E1 = expm(-dt/2 h_mod), A = -i sqrt(dt) sum xs K, Lrot = psi^T K,
    X = tr(Lrot Theta), E_C = 1/2 sum X^2, E_X = -1/2 sum tr(T T), T = Lrot Theta.
  * Readings: h1 complex Hermitian; a vector set whose antisymmetric sum does not vanish (not a set of ERIs) is
    rejected at construction.
  * Complex trial (PAPER.md:219 Code Snippet 6 gives the trial no dtype; magnetic fields,
    spin-orbit coupling and Bloch orbitals make the wavefunctions complex; SURVEY S12 "formulas keep psi^+"):
    <Psi_T| = prod_i (sum_p conj(psi_pi) a_p), so every psi^T of the real-trial formulas is psi^+:
        O = psi^+ phi,  Theta = phi O^-1,  G_pq = <a+_p a_q> = [Theta psi^+]_qp,  P = psi psi^+ (Hermitian),
        m_g' = tr(K_g' P) (still real: K and P Hermitian),  Lrot = psi^+ K,  hrot = psi^+ h.
    A real trial is the special case; nothing else changes (the propagator does not see the trial).

Plain NumPy complex128; library primitives as single steps (matmul, det, solve, eigh, qr).
"""
from __future__ import annotations

import numpy as np

__all__ = ["ComplexCholOracle", "hermitian_parts"]


def hermitian_parts(L):
    """K[0:n] = A_g, K[n:2n] = B_g for complex vectors L [n, M, M]."""
    L = np.asarray(L, dtype=np.complex128)
    Ld = L.conj().transpose(0, 2, 1)
    return np.concatenate([(L + Ld) / 2, (L - Ld) / 2j], axis=0)


class ComplexCholOracle:
    def __init__(self, h1, L, trial, n_alpha, n_beta, walker_kind, taylor_order=6, e_shift=None, check=True,
                 xbar_bound=0.0, ehyb_bound=0.0):
        self.xbar_bound, self.ehyb_bound = float(xbar_bound), float(ehyb_bound)      # as in afqmc_oracle.py (S8b)
        h1 = np.asarray(h1, dtype=np.complex128)
        trial = np.asarray(trial)
        trial = trial.astype(np.complex128 if np.iscomplexobj(trial) else np.float64)
        self.M = M = h1.shape[0]
        self.n_alpha, self.n_beta, self.walker_kind = int(n_alpha), int(n_beta), int(walker_kind)
        self.K_order = int(taylor_order) if taylor_order else 6
        if self.walker_kind == 0:
            self.blocks, self.spin_factor = [(0, self.n_alpha)], 2.0
        else:
            self.blocks, self.spin_factor = [(0, self.n_alpha), (self.n_alpha, self.n_alpha + self.n_beta)], 1.0
        self.psi = [trial[:, a:b].copy() for a, b in self.blocks]
        self.h1 = h1
        L = np.asarray(L, dtype=np.complex128)
        self.Kmat = K = hermitian_parts(L)               # [2n, M, M]
        self.n_fields = K.shape[0]
        if check:
            n = L.shape[0]
            anti = np.einsum("gps,gqr->psqr", K[n:], K[:n]) - np.einsum("gps,gqr->psqr", K[:n], K[n:])
            if np.abs(anti).max() > 1e-10 * max(1.0, np.abs(K).max() ** 2):
                raise ValueError("the vectors do not factorise a (ps|qr) = (qr|ps) symmetric tensor")
        P_tot = sum(p @ p.conj().T for p in self.psi) * self.spin_factor      # P = psi psi^+
        self.m = np.einsum("gpq,qp->g", K, P_tot).real                    # tr(K P), real for Hermitian K, P
        hprime = h1 - 0.5 * np.einsum("gpq,gqr->pr", K, K)
        self.h_mod = hprime + np.einsum("g,gpq->pq", self.m, K)
        self.E_const = -0.5 * float(self.m @ self.m)
        self.Lrot = [np.einsum("pi,gpq->giq", p.conj(), K) for p in self.psi]   # psi^+ K_g  [2n, Ns, M]
        self.hrot = [p.conj().T @ h1 for p in self.psi]
        if e_shift is None:
            w0 = np.concatenate(self.psi, axis=1).astype(np.complex128)[None]
            self.e_shift = float(self.local_energy(w0)[0, 0].real)
        else:
            self.e_shift = float(e_shift)

    def one_body_propagator(self, dt):
        lam, V = np.linalg.eigh(self.h_mod)
        return (V * np.exp(-0.5 * dt * lam)) @ V.conj().T

    def overlap(self, walkers):
        ov = np.ones(walkers.shape[0], dtype=np.complex128)
        for (a, b), p in zip(self.blocks, self.psi):
            for w in range(walkers.shape[0]):
                d = np.linalg.det(p.conj().T @ walkers[w, :, a:b])
                ov[w] *= d * d if self.walker_kind == 0 else d
        return ov

    def theta(self, walkers):
        th = np.empty_like(walkers)
        for (a, b), p in zip(self.blocks, self.psi):
            for w in range(walkers.shape[0]):
                phi = walkers[w, :, a:b]
                th[w, :, a:b] = np.linalg.solve((p.conj().T @ phi).T, phi.T).T
        return th

    def force_bias_X(self, th):
        X = np.zeros((th.shape[0], self.n_fields), dtype=np.complex128)
        for (a, b), lr in zip(self.blocks, self.Lrot):
            X += self.spin_factor * np.einsum("giq,wqi->wg", lr, th[:, :, a:b])
        return X

    def vhs(self, xs, dt):
        return (-1j * np.sqrt(dt)) * np.einsum("wg,gpq->wpq", xs, self.Kmat)

    def propagate(self, walkers, x, dt, xbar_override=None):
        """x: [nw, 2n] standard normal fields (first n for the A_g, last n for the B_g)."""
        walkers = np.asarray(walkers, dtype=np.complex128)
        sq = np.sqrt(dt)
        ov_old = self.overlap(walkers)
        X = self.force_bias_X(self.theta(walkers))
        xbar = 1j * sq * (X - self.m[None, :])
        if xbar_override is not None:
            xbar = np.broadcast_to(np.asarray(xbar_override, dtype=np.complex128), X.shape)
        elif self.xbar_bound > 0.0:
            mag = np.abs(xbar)
            with np.errstate(all="ignore"):
                xbar = xbar * np.where(mag > self.xbar_bound, self.xbar_bound / mag, 1.0)
        xs = x - xbar
        c_fb = np.sum(x * xbar, axis=1) - 0.5 * np.sum(xbar * xbar, axis=1)
        c_mf = 1j * sq * (xs @ self.m)
        A = self.vhs(xs, dt)
        E1 = self.one_body_propagator(dt)
        new = np.empty_like(walkers)
        for w in range(walkers.shape[0]):
            phi = E1 @ walkers[w]
            T, acc = phi, phi.copy()
            for n in range(1, self.K_order + 1):
                T = (A[w] @ T) / n
                acc = acc + T
            new[w] = E1 @ acc
        ov_new = self.overlap(new)
        S = (ov_new / ov_old) * np.exp(c_mf)
        I = S * np.exp(c_fb) * np.exp(-dt * (self.E_const - self.e_shift))
        return new, dict(xbar=xbar, xs=xs, c_fb=c_fb, c_mf=c_mf, ovlp_old=ov_old, ovlp_new=ov_new, S=S, I=I, X=X, A=A)

    def step(self, walkers, weights, x, dt):
        new, info = self.propagate(walkers, x, dt)
        S, I = info["S"], info["I"]
        w = np.asarray(weights, dtype=np.float64).copy()
        for k in range(w.shape[0]):
            if not (np.isfinite(S[k]) and np.isfinite(I[k]) and abs(S[k]) > 0.0):
                w[k] = 0.0
                continue
            absI = abs(I[k])
            if self.ehyb_bound > 0.0 and absI > 0.0:
                D = -np.log(absI) / dt
                if abs(D) > self.ehyb_bound:
                    absI = np.exp(-dt * np.copysign(self.ehyb_bound, D))
            w[k] = w[k] * absI * max(0.0, S[k].real / abs(S[k]))
        return new, w, info["ovlp_new"].copy()

    def local_energy(self, walkers):
        walkers = np.asarray(walkers, dtype=np.complex128)
        nw = walkers.shape[0]
        th = self.theta(walkers)
        e1 = np.zeros(nw, dtype=np.complex128)
        ex = np.zeros(nw, dtype=np.complex128)
        for (a, b), hr, lr in zip(self.blocks, self.hrot, self.Lrot):
            e1 += self.spin_factor * np.einsum("iq,wqi->w", hr, th[:, :, a:b])
            T = np.einsum("giq,wqj->wgij", lr, th[:, :, a:b])
            ex += -0.5 * self.spin_factor * np.einsum("wgij,wgji->w", T, T)
        X = self.force_bias_X(th)
        ec = 0.5 * np.sum(X * X, axis=1)
        out = np.empty((nw, 3), dtype=np.complex128)
        out[:, 0], out[:, 1], out[:, 2] = e1 + ec + ex, e1, ec + ex
        return out
