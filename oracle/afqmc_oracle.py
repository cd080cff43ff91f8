"""CPU oracle for one batched phaseless-AFQMC walker step and the local energy.

TEST INFRASTRUCTURE ONLY.  This file is the slow, plain statement of what the hot
path computes.  Only `tests/`, `__graft_entry__.smoke()` and the `cpu_baseline` /
`--impl reference` legs of `bench.py` may import it.  It shares no code with the CUDA
library under `paper_2406_16238_b200/` and imports nothing from it.

Everything is NumPy float64 / complex128.  Library primitives used as single steps:
`@` (matmul), `numpy.linalg.det`, `numpy.linalg.solve`, `numpy.linalg.eigh`,
`numpy.linalg.qr`.  There is no blocking, fusion or reordering beyond the order of the
steps below, except that the Cholesky tensor L may be handed in as a provider of
gamma-slabs so that a 55 GB tensor never has to sit in host memory; sums over gamma are
then accumulated slab by slab in increasing gamma.

Source: /root/reference/PAPER.md ("Improved Modularity and New Features in ipie",
arXiv 2406.16238), Sec. II, Eqs. (1)-(18).  The paper states the method
at the level of those equations; the working formulas are derived from them in
SURVEY.md §8(c) D1-D7 and restated in DESIGN.md "Readings".  Each function cites the
passage it follows.

Conventions (DESIGN.md R-list):
  * H = sum h_pq a+_p a_q + 1/2 sum (ps|qr) a+_p a+_q a_r a_s, (ps|qr) = sum_g L^g_ps L^g_qr
    (Eqs. 2-3).  L_g real symmetric M x M.
  * v_g = i L_g (Eq. 6);  B(x) = exp(-dt/2 v0) exp(-sqrt(dt) x.v) exp(-dt/2 v0)
    (Eq. 9).
  * Trial: real orthonormal columns [alpha | beta] (Code Snippet 6).
  * walker_kind 0 (RHF, restricted walkers): one stored block [M x Nocc] used for both
    spins; walker_kind 1 (UHF): two stored blocks [alpha | beta].

Pins (tests/test_oracle_pins.py): P1-P13 of SURVEY.md §8(c); every function below is
pinned by at least one of them.
"""
from __future__ import annotations

import numpy as np

__all__ = ["AFQMCOracle"]


def _as_slab_iter(L, slab=64):
    """Yield (g0, L[g0:g1]) in increasing gamma.

    `L` is either an ndarray [n_chol, M, M] or a zero-argument callable returning an
    iterator of (g0, ndarray[g, M, M]) pairs (used for the 55 GB configuration)."""
    if callable(L):
        for g0, blk in L():
            yield int(g0), np.asarray(blk, dtype=np.float64)
    else:
        n = L.shape[0]
        for g0 in range(0, n, slab):
            yield g0, np.asarray(L[g0:g0 + slab], dtype=np.float64)


class AFQMCOracle:
    """Plain statement of `afqmc_create / afqmc_step / afqmc_local_energy`.

    Parameters follow include/afqmc.h.  `L` is [n_chol, M, M] float64 (each L_g
    symmetric) or a slab provider (see `_as_slab_iter`)."""

    # ------------------------------------------------------------------ O0 create
    def __init__(self, h1, L, trial, n_alpha, n_beta, walker_kind,
                 taylor_order=6, ortho_every=0, e_shift=None, n_chol=None, xbar_bound=0.0, ehyb_bound=0.0):
        h1 = np.asarray(h1, dtype=np.float64)
        trial = np.asarray(trial, dtype=np.float64)
        self.M = M = h1.shape[0]
        self.n_alpha, self.n_beta = int(n_alpha), int(n_beta)
        self.walker_kind = int(walker_kind)
        self.K = int(taylor_order) if taylor_order else 6
        self.ortho_every = int(ortho_every)
        self.n_steps_done = 0
        self.L = L
        # optional bounds (reading S8b in DESIGN.md); 0 = off, the paper's own algorithm
        self.xbar_bound, self.ehyb_bound = float(xbar_bound), float(ehyb_bound)
        if self.walker_kind == 0:
            if n_alpha != n_beta:
                raise ValueError("RHF walkers need n_alpha == n_beta")
            # one stored block serving both spins (reading S11)
            self.blocks = [(0, self.n_alpha)]
            self.spin_factor = 2.0
        else:
            # [alpha | beta] columns, PAPER.md:219 (np.hstack([orbs_a, orbs_b]))
            self.blocks = [(0, self.n_alpha), (self.n_alpha, self.n_alpha + self.n_beta)]
            self.spin_factor = 1.0
        self.Nt = self.blocks[-1][1]
        if trial.shape != (M, self.Nt):
            raise ValueError("trial must be [M, Nt]")
        self.psi = [trial[:, a:b].copy() for a, b in self.blocks]
        for p in self.psi:                      # orthonormal columns, 1e-10
            if np.abs(p.T @ p - np.eye(p.shape[1])).max() > 1e-10:
                raise ValueError("trial columns are not orthonormal")
        self.h1 = h1

        # D3: P_tot = sum_sigma psi_sigma psi_sigma^T ; m_g = sum_pq L^g_pq P_tot_pq
        # (mean-field shift <v_g>_T = i m_g)
        P_tot = sum(p @ p.T for p in self.psi) * self.spin_factor
        self.P_tot = P_tot
        m_list, lrot = [], [[] for _ in self.psi]
        hprime = h1.copy()                       # D2 / Eq. (5): h' = h - 1/2 sum_g L_g L_g
        mL = np.zeros((M, M))                    # sum_g m_g L_g
        for g0, Ls in _as_slab_iter(L):
            ms = Ls.reshape(Ls.shape[0], -1) @ P_tot.ravel()
            m_list.append(ms)
            for g in range(Ls.shape[0]):
                hprime -= 0.5 * (Ls[g] @ Ls[g])
                mL += ms[g] * Ls[g]
            for s, p in enumerate(self.psi):     # S4 half rotation: Lrot^g_sigma = psi^T L_g
                lrot[s].append(p.T @ Ls)                 # [g, Ns, M]
        self.m = np.concatenate(m_list)
        self.n_chol = self.m.shape[0]
        if n_chol is not None and n_chol != self.n_chol:
            raise ValueError("n_chol mismatch")
        self.Lrot = [np.concatenate(x, axis=0) for x in lrot]   # [n_chol, Ns, M]
        self.hrot = [p.T @ h1 for p in self.psi]                # [Ns, M]
        self.h_mod = hprime + mL                                # D3
        self.E_const = -0.5 * float(self.m @ self.m)            # D3
        self._E1 = {}
        if e_shift is None:
            # E_shift = local energy of the trial itself (reading S7)
            w0 = np.concatenate(self.psi, axis=1).astype(np.complex128)[None]
            self.e_shift = float(self.local_energy(w0)[0, 0].real)
        else:
            self.e_shift = float(e_shift)

    # ------------------------------------------------------------------ O0 / S6
    def one_body_propagator(self, dt):
        """E1 = expm(-dt/2 h_mod) by symmetric eigendecomposition (Eq. 9, PAPER.md:82;
        reading S6)."""
        key = float(dt)
        if key not in self._E1:
            lam, V = np.linalg.eigh(self.h_mod)
            self._E1[key] = (V * np.exp(-0.5 * dt * lam)) @ V.T
        return self._E1[key]

    # ------------------------------------------------------------------ O1
    def overlap(self, walkers):
        """<Psi_T|phi_w> = prod_sigma det(psi_sigma^T phi_sigma) (Eq. 10/17 denominators,
        PAPER.md:89-92, 123; D6).  RHF restricted: det(O)^2."""
        nw = walkers.shape[0]
        ov = np.ones(nw, dtype=np.complex128)
        for (a, b), p in zip(self.blocks, self.psi):
            for w in range(nw):
                d = np.linalg.det(p.T @ walkers[w, :, a:b])
                ov[w] *= d * d if self.walker_kind == 0 else d
        return ov

    # ------------------------------------------------------------------ O2
    def theta(self, walkers):
        """Theta_sigma = phi_sigma (psi_sigma^T phi_sigma)^-1, [nw, M, Nt] (D6).  The
        mixed Green's function is G_sigma = (Theta_sigma psi_sigma^T)^T; only Theta is
        formed ("Green's function", "half rotation")."""
        th = np.empty_like(walkers)
        for (a, b), p in zip(self.blocks, self.psi):
            for w in range(walkers.shape[0]):
                phi = walkers[w, :, a:b]
                O = p.T @ phi
                try:
                    th[w, :, a:b] = np.linalg.solve(O.T, phi.T).T
                except np.linalg.LinAlgError:               # singular overlap: reading S10
                    th[w, :, a:b] = np.nan
        return th

    def greens_function(self, walkers):
        """Full G_sigma,pq = <a+_p a_q>_mixed = [Theta psi^T]_qp, list over stored blocks
        of [nw, M, M].  Only used by tests (pins P1, P3, P4)."""
        th = self.theta(walkers)
        out = []
        for (a, b), p in zip(self.blocks, self.psi):
            out.append(np.einsum("wqi,pi->wpq", th[:, :, a:b], p))
        return out

    # ------------------------------------------------------------------ O3
    def force_bias_X(self, th):
        """X_g = <Psi_T|L_g|phi>/<Psi_T|phi> = sum_sigma sum_iq Lrot^g_sigma,iq Theta_sigma,qi
        (D6; the quantity inside Eq. 14)."""
        nw = th.shape[0]
        X = np.zeros((nw, self.n_chol), dtype=np.complex128)
        for (a, b), lr in zip(self.blocks, self.Lrot):
            lf = lr.reshape(self.n_chol, -1)                       # [g, (i,q)]
            tf = th[:, :, a:b].transpose(0, 2, 1).reshape(nw, -1)  # [w, (i,q)] = Theta_qi
            X += self.spin_factor * ((tf.real @ lf.T) + 1j * (tf.imag @ lf.T))
        return X

    # ------------------------------------------------------------------ O5
    def vhs(self, xs, dt):
        """A_w = -i sqrt(dt) sum_g xs[w,g] L_g (Eq. 9 with v_g = i L_g, PAPER.md:69, 82;
        the "VHS step")."""
        nw, M = xs.shape[0], self.M
        acc = np.zeros((nw, M * M), dtype=np.complex128)
        for g0, Ls in _as_slab_iter(self.L):
            Lf = Ls.reshape(Ls.shape[0], M * M)
            c = xs[:, g0:g0 + Ls.shape[0]]
            acc += (c.real @ Lf) + 1j * (c.imag @ Lf)
        return (-1j * np.sqrt(dt)) * acc.reshape(nw, M, M)

    # ------------------------------------------------------------------ O1-O10
    def propagate(self, walkers, x, dt, xbar_override=None):
        """One application of B(x - xbar) to every walker, with all scalars.

        Returns (new_walkers, info) where info holds xbar, c_fb, c_mf, ovlp_old,
        ovlp_new, S (Eq. 17) and I (Eq. 16 times the constant of reading S7).
        Follows O1-O9 of SURVEY.md §8(c); Eqs. (9), (12), (14), (16), (17)."""
        walkers = np.asarray(walkers, dtype=np.complex128)
        x = np.asarray(x, dtype=np.float64)
        sq = np.sqrt(dt)
        ov_old = self.overlap(walkers)                       # O1
        th = self.theta(walkers)                             # O2
        X = self.force_bias_X(th)                            # O3
        # reading S1 (sign): xbar = +i sqrt(dt) (X - m) = +sqrt(dt) <v - <v>_T>_mixed
        xbar = 1j * sq * (X - self.m[None, :])
        if xbar_override is not None:
            xbar = np.broadcast_to(np.asarray(xbar_override, dtype=np.complex128), X.shape)
        elif self.xbar_bound > 0.0:
            # S8b: cap the modulus of every component, keep its phase.  Eqs. (12), (16) hold for ANY xbar, and
            # xs, c_fb, c_mf below are formed from the xbar actually used.
            mag = np.abs(xbar)
            with np.errstate(all="ignore"):
                xbar = xbar * np.where(mag > self.xbar_bound, self.xbar_bound / mag, 1.0)
        xs = x - xbar                                        # O4, Eq. (12)
        # Eq. (16) exponent; bilinear sums, no conjugation (reading S14)
        c_fb = np.sum(x * xbar, axis=1) - 0.5 * np.sum(xbar * xbar, axis=1)
        # scalar factor of the shifted HS field (D4): exp(+i sqrt(dt) xs.m)
        c_mf = 1j * sq * (xs @ self.m)
        A = self.vhs(xs, dt)                                 # O5
        E1 = self.one_body_propagator(dt)
        new = np.empty_like(walkers)
        for w in range(walkers.shape[0]):                    # O6-O8, Eq. (9)/(12)
            phi = E1 @ walkers[w]
            T = phi
            acc = phi.copy()
            for n in range(1, self.K + 1):                   # reading S5: Taylor order K
                T = (A[w] @ T) / n
                acc = acc + T
            new[w] = E1 @ acc
        ov_new = self.overlap(new)                           # O9
        with np.errstate(all="ignore"):
            S = (ov_new / ov_old) * np.exp(c_mf)             # Eq. (17)
            I = S * np.exp(c_fb) * np.exp(-dt * (self.E_const - self.e_shift))  # Eq. (16), S7
        info = dict(xbar=xbar, xs=xs, c_fb=c_fb, c_mf=c_mf, ovlp_old=ov_old,
                    ovlp_new=ov_new, S=S, I=I, X=X, A=A)
        return new, info

    def step(self, walkers, weights, x, dt):
        """`afqmc_step`: walkers <- B(x - xbar) walkers (Eq. 12), w <- I_ph w (Eqs. 13,
        15), then re-orthonormalise every `ortho_every`-th call (O10).

        Returns (walkers, weights, overlaps of the returned walkers)."""
        new, info = self.propagate(walkers, x, dt)
        S, I = info["S"], info["I"]
        w = np.asarray(weights, dtype=np.float64).copy()
        ov = info["ovlp_new"].copy()
        for k in range(w.shape[0]):
            ok = (np.isfinite(S[k]) and np.isfinite(I[k]) and abs(S[k]) > 0.0
                  and info["ovlp_old"][k] != 0 and np.isfinite(ov[k]))
            if not ok:
                w[k] = 0.0                                   # reading S10
                continue
            cos_theta = S[k].real / abs(S[k])                # Eq. (18) without a branch cut
            absI = abs(I[k])
            if self.ehyb_bound > 0.0 and absI > 0.0:
                # S8b: D = -log|I| / dt is the real part of the hybrid energy relative to E_shift; clip it
                D = -np.log(absI) / dt
                if abs(D) > self.ehyb_bound:
                    absI = np.exp(-dt * np.copysign(self.ehyb_bound, D))
            w[k] = w[k] * absI * max(0.0, cos_theta)         # Eqs. (13), (15)
        self.n_steps_done += 1
        if self.ortho_every > 0 and self.n_steps_done % self.ortho_every == 0:
            new, detR = self.reorthonormalise(new)
            ov = ov / detR
        return new, w, ov

    # ------------------------------------------------------------------ O10
    def reorthonormalise(self, walkers):
        """Per stored block phi_sigma = Q R with R_ii real > 0; phi_sigma <- Q
        ("stabilization"; reading S9).  Returns (walkers, detR) with
        detR[w] = prod_sigma det R_sigma (squared for restricted walkers)."""
        out = np.empty_like(walkers)
        detR = np.ones(walkers.shape[0], dtype=np.complex128)
        for a, b in self.blocks:
            for w in range(walkers.shape[0]):
                Q, R = np.linalg.qr(walkers[w, :, a:b])
                d = np.diagonal(R)
                ph = d / np.abs(d)
                out[w, :, a:b] = Q * ph[None, :]             # R <- diag(conj ph) R
                dr = np.prod(np.abs(d))
                detR[w] *= dr * dr if self.walker_kind == 0 else dr
        return out, detR

    # ------------------------------------------------------------------ O11
    def local_energy(self, walkers):
        """E_loc = <Psi_T|H|phi>/<Psi_T|phi> (Eq. 11) by Wick's theorem (D7):
        E1b = sum_sigma sum_iq hrot_iq Theta_qi;  E_C = 1/2 sum_g X_g^2;
        E_X = -1/2 sum_g sum_sigma tr(T^g_sigma T^g_sigma), T^g_sigma = Lrot^g_sigma Theta_sigma.
        Returns complex [nw, 3] = (E, E1b, E_C + E_X) as in `energy[:, 0..2]` of Code
        Snippet 9."""
        walkers = np.asarray(walkers, dtype=np.complex128)
        nw = walkers.shape[0]
        th = self.theta(walkers)
        e1 = np.zeros(nw, dtype=np.complex128)
        ex = np.zeros(nw, dtype=np.complex128)
        for (a, b), hr, lr in zip(self.blocks, self.hrot, self.Lrot):
            e1 += self.spin_factor * np.einsum("iq,wqi->w", hr, th[:, :, a:b])
            for w in range(nw):
                tw = th[w, :, a:b]
                T = (lr @ tw.real) + 1j * (lr @ tw.imag)     # [n_chol, Ns, Ns]
                ex[w] += -0.5 * self.spin_factor * np.einsum("gij,gji->", T, T)
        X = self.force_bias_X(th)
        ec = 0.5 * np.sum(X * X, axis=1)
        out = np.empty((nw, 3), dtype=np.complex128)
        out[:, 0] = e1 + ec + ex
        out[:, 1] = e1
        out[:, 2] = ec + ex
        return out
