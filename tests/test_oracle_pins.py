"""Pins P1-P16 (P14-P16 added in DESIGN.md §4): the oracle against what the paper and the mathematics fix.

None of these retype the oracle's formulas: they use explicit many-body matrices
(tests/fock.py), brute-force four-index sums, closed forms, scipy's matrix exponential,
Gauss-Hermite quadrature, and invariances.  CPU only.
"""
import numpy as np
import pytest
import scipy.linalg as sla

from oracle.afqmc_oracle import AFQMCOracle
from tests.fock import Fock


def small_problem(M, na, nb, ng, kind, seed, lscale=0.3, noise=0.2, nw=3):
    r = np.random.default_rng(seed)
    h = r.standard_normal((M, M)); h = 0.5 * (h + h.T)
    L = r.standard_normal((ng, M, M)) * lscale
    L = 0.5 * (L + L.transpose(0, 2, 1))
    if kind == 0:
        trial = np.linalg.qr(r.standard_normal((M, na)))[0]
        Nt = na
    else:
        trial = np.concatenate([np.linalg.qr(r.standard_normal((M, na)))[0],
                                np.linalg.qr(r.standard_normal((M, nb)))[0]], axis=1)
        Nt = na + nb
    walkers = trial[None] + noise * (r.standard_normal((nw, M, Nt)) + 1j * r.standard_normal((nw, M, Nt)))
    return h, L, trial, walkers.astype(np.complex128)


def spin_blocks(o, mat):
    """(alpha, beta) column blocks of a [M, Nt] array under the oracle's walker kind."""
    if o.walker_kind == 0:
        return mat[:, :o.n_alpha], mat[:, :o.n_alpha]
    return mat[:, :o.n_alpha], mat[:, o.n_alpha:o.n_alpha + o.n_beta]


# --------------------------------------------------------------------------- P1
@pytest.mark.parametrize("kind", [0, 1])
def test_P1_walker_equals_trial(kind):
    h, L, trial, _ = small_problem(8, 3, 2 if kind else 3, 5, kind, 1)
    o = AFQMCOracle(h, L, trial, 3, 2 if kind else 3, kind)
    w = trial[None].astype(np.complex128)
    assert abs(o.overlap(w)[0] - 1) < 1e-13
    for G, p in zip(o.greens_function(w), o.psi):
        assert np.abs(G[0] - (p @ p.T).T).max() < 1e-13          # G = P^T
    X = o.force_bias_X(o.theta(w))
    assert np.abs(X[0] - o.m).max() < 1e-12                       # X = m  =>  xbar = 0
    _, info = o.propagate(w, np.zeros((1, 5)), 0.01)
    assert np.abs(info["xbar"]).max() < 1e-12


# --------------------------------------------------------------------------- P2
@pytest.mark.parametrize("kind", [0, 1])
def test_P2_hartree_fock_closed_form(kind):
    na, nb = (3, 3) if kind == 0 else (3, 2)
    h, L, trial, _ = small_problem(9, na, nb, 7, kind, 2)
    o = AFQMCOracle(h, L, trial, na, nb, kind)
    pa = trial[:, :na]
    pb = pa if kind == 0 else trial[:, na:]
    Pa, Pb = pa @ pa.T, pb @ pb.T
    e1 = np.trace(h @ Pa) + np.trace(h @ Pb)
    ec = 0.5 * sum((np.trace(Lg @ Pa) + np.trace(Lg @ Pb)) ** 2 for Lg in L)
    ex = -0.5 * sum(np.trace(Lg @ Pa @ Lg @ Pa) + np.trace(Lg @ Pb @ Lg @ Pb) for Lg in L)
    E = o.local_energy(trial[None].astype(np.complex128))[0]
    assert abs(E[0] - (e1 + ec + ex)) < 1e-12 * abs(e1 + ec + ex) + 1e-12
    assert abs(E[1] - e1) < 1e-12
    assert abs(E[2] - (ec + ex)) < 1e-12
    assert abs(o.e_shift - (e1 + ec + ex)) < 1e-11                # auto shift = trial energy


# --------------------------------------------------------------------------- P3
@pytest.mark.parametrize("kind", [0, 1])
def test_P3_bruteforce_four_index(kind):
    na, nb = (3, 3) if kind == 0 else (4, 2)
    h, L, trial, walkers = small_problem(10, na, nb, 6, kind, 3)
    o = AFQMCOracle(h, L, trial, na, nb, kind)
    eri = np.einsum("gps,gqr->psqr", L, L)                        # (ps|qr), Eq. (3)
    Gs = o.greens_function(walkers)
    if kind == 0:
        Gs = [Gs[0], Gs[0]]
    E = o.local_energy(walkers)
    for w in range(walkers.shape[0]):
        Ga, Gb = Gs[0][w], Gs[1][w]
        Gt = Ga + Gb
        e1 = np.sum(h * Gt)
        # <a+_p a+_q a_r a_s> = G_ps G_qr - delta_spin G_pr G_qs  (Wick)
        e2 = 0.5 * (np.einsum("psqr,ps,qr->", eri, Gt, Gt)
                    - np.einsum("psqr,pr,qs->", eri, Ga, Ga)
                    - np.einsum("psqr,pr,qs->", eri, Gb, Gb))
        assert abs(E[w, 1] - e1) < 1e-12 * max(1, abs(e1))
        assert abs(E[w, 2] - e2) < 1e-11 * max(1, abs(e2))
        assert abs(E[w, 0] - (e1 + e2)) < 1e-11 * max(1, abs(e1 + e2))


# --------------------------------------------------------------------------- P4
@pytest.mark.parametrize("kind,na,nb", [(1, 2, 1), (0, 2, 2)])
def test_P4_fock_space(kind, na, nb):
    M, ng = 4, 3
    h, L, trial, walkers = small_problem(M, na, nb, ng, kind, 4)
    o = AFQMCOracle(h, L, trial, na, nb, kind)
    F = Fock(M)
    H = F.hamiltonian(h, L)
    ta, tb = spin_blocks(o, trial)
    bra = F.det_state(ta.astype(complex), tb.astype(complex)).conj()
    ov = o.overlap(walkers)
    E = o.local_energy(walkers)
    X = o.force_bias_X(o.theta(walkers))
    Gs = o.greens_function(walkers)
    for w in range(walkers.shape[0]):
        wa, wb = spin_blocks(o, walkers[w])
        ket = F.det_state(wa, wb)
        ov_mb = bra @ ket
        assert abs(ov[w] - ov_mb) < 1e-12
        assert abs(E[w, 0] - (bra @ H @ ket) / ov_mb) < 1e-11
        for g in range(ng):
            assert abs(X[w, g] - (bra @ F.one_body(L[g]) @ ket) / ov_mb) < 1e-12
        for p in range(M):
            for q in range(M):                                   # alpha Green's function
                g_mb = (bra @ F.cd[p] @ F.c[q] @ ket) / ov_mb
                assert abs(Gs[0][w][p, q] - g_mb) < 1e-12
    # Thouless: e^{A_hat}|phi> = |e^{A} phi> for a complex symmetric one-body A
    A = -1j * 0.1 * np.einsum("g,gpq->pq", np.array([0.3, -1.1, 0.7]), L)
    wa, wb = spin_blocks(o, walkers[0])
    lhs = sla.expm(F.one_body(A)) @ F.det_state(wa, wb)
    rhs = F.det_state(sla.expm(A) @ wa, sla.expm(A) @ wb)
    assert np.abs(lhs - rhs).max() < 1e-12


# --------------------------------------------------------------------------- P5
@pytest.mark.parametrize("seed", [5, 6])
def test_P5_mean_field_shift_identity(seed):
    """H = H1[h_mod] + E_const + 1/2 sum_g (L_g - m_g)^2 for the oracle's h_mod, E_const, m,
    whatever trial (hence whatever m) it was built from (Eqs. 4-6)."""
    M, ng = 3, 3
    h, L, trial, _ = small_problem(M, 2, 1, ng, 1, seed)
    o = AFQMCOracle(h, L, trial, 2, 1, 1)
    F = Fock(M)
    H = F.hamiltonian(h, L)
    I = np.eye(2 ** F.n)
    rhs = F.one_body(o.h_mod) + o.E_const * I
    for g in range(ng):
        d = F.one_body(L[g]) - o.m[g] * I
        rhs = rhs + 0.5 * d @ d
    assert np.abs(H - rhs).max() < 1e-12
    assert np.abs(o.m).max() > 1e-2


# --------------------------------------------------------------------------- P6
def _quadrature_error(dt, mode, kind=1):
    M, ng, na, nb = 3, 2, 2, 1
    if kind == 0:
        nb = na
    h, L, trial, walkers = small_problem(M, na, nb, ng, kind, 7, lscale=0.5, noise=0.15, nw=1)
    o = AFQMCOracle(h, L, trial, na, nb, kind, taylor_order=24)
    F = Fock(M)
    H = F.hamiltonian(h, L)
    wa, wb = spin_blocks(o, walkers[0])
    exact = sla.expm(-dt * H) @ F.det_state(wa, wb)
    nodes, wts = np.polynomial.hermite_e.hermegauss(28)
    wts = wts / wts.sum()
    xs = np.array([[a, b] for a in nodes for b in nodes])
    ws = np.array([u * v for u in wts for v in wts])
    batch = np.repeat(walkers, xs.shape[0], axis=0)
    override = {"fb": None, "zero": np.zeros(ng), "arb": np.array([0.11 - 0.07j, -0.05 + 0.13j])}[mode]
    new, info = o.propagate(batch, xs, dt, xbar_override=override)
    # exp(c_fb + c_mf - dt E_const) = I * ovlp_old/ovlp_new * exp(-dt E_shift)
    scal = info["I"] * info["ovlp_old"] / info["ovlp_new"] * np.exp(-dt * o.e_shift)
    acc = np.zeros_like(exact)
    for k in range(xs.shape[0]):
        a, b = spin_blocks(o, new[k])
        acc = acc + ws[k] * scal[k] * F.det_state(a, b)
    return np.linalg.norm(acc - exact) / np.linalg.norm(exact)


@pytest.mark.parametrize("kind", [0, 1])
def test_P6_hubbard_stratonovich_quadrature(kind):
    """int dx p(x) e^{x.xbar - xbar.xbar/2} B(x - xbar)|phi> = e^{-dt H}|phi> + O(dt^2)
    (Eqs. 8, 9, 12, 16) for the force bias, for xbar = 0 and for an arbitrary complex xbar."""
    e1 = {m: _quadrature_error(0.02, m, kind) for m in ("fb", "zero", "arb")}
    e2 = {m: _quadrature_error(0.01, m, kind) for m in ("fb", "zero", "arb")}
    for m in e1:
        assert e1[m] < 5e-3
        assert 3.3 < e1[m] / e2[m] < 4.7, (m, e1[m], e2[m])
    # independent of xbar to quadrature accuracy
    assert abs(e1["fb"] - e1["zero"]) < 1e-6 and abs(e1["arb"] - e1["zero"]) < 1e-6


# --------------------------------------------------------------------------- P7
@pytest.mark.parametrize("kind", [0, 1])
def test_P7_reorthonormalisation(kind):
    na, nb = (3, 3) if kind == 0 else (3, 2)
    h, L, trial, walkers = small_problem(8, na, nb, 5, kind, 8, noise=0.4)
    o = AFQMCOracle(h, L, trial, na, nb, kind)
    q, detR = o.reorthonormalise(walkers)
    for a, b in o.blocks:
        for w in range(walkers.shape[0]):
            Q = q[w, :, a:b]
            assert np.abs(Q.conj().T @ Q - np.eye(b - a)).max() < 1e-13
            R = Q.conj().T @ walkers[w, :, a:b]
            assert np.abs(np.tril(R, -1)).max() < 1e-13          # upper triangular
            assert np.all(np.diagonal(R).real > 0) and np.abs(np.diagonal(R).imag).max() < 1e-13
    assert np.abs(o.local_energy(q) - o.local_energy(walkers)).max() < 1e-11
    assert np.abs(o.force_bias_X(o.theta(q)) - o.force_bias_X(o.theta(walkers))).max() < 1e-11
    assert np.abs(o.overlap(walkers) / detR - o.overlap(q)).max() < 1e-12
    # and through step(): ortho_every=1 returns orthonormal walkers and the matching overlap
    o1 = AFQMCOracle(h, L, trial, na, nb, kind, ortho_every=1)
    x = np.random.default_rng(0).standard_normal((walkers.shape[0], 5))
    nwk, wts, ov = o1.step(walkers, np.ones(walkers.shape[0]), x, 0.01)
    assert np.abs(o1.overlap(nwk) - ov).max() < 1e-12
    o0 = AFQMCOracle(h, L, trial, na, nb, kind, ortho_every=0)
    nwk0, wts0, ov0 = o0.step(walkers, np.ones(walkers.shape[0]), x, 0.01)
    assert np.abs(wts - wts0).max() < 1e-14                       # weights untouched by QR
    assert np.abs(o0.local_energy(nwk0) - o0.local_energy(nwk)).max() < 1e-10


# --------------------------------------------------------------------------- P8
def _std_log_I(dt, flip):
    h, L, trial, walkers = small_problem(6, 2, 2, 8, 0, 9, lscale=0.4, noise=0.25, nw=1)
    o = AFQMCOracle(h, L, trial, 2, 2, 0, taylor_order=12)
    r = np.random.default_rng(11)
    x = r.standard_normal((300, 8))
    batch = np.repeat(walkers, 300, axis=0)
    override = None
    if flip:
        _, info0 = o.propagate(walkers, x[:1], dt)
        override = -info0["xbar"][0]
    _, info = o.propagate(batch, x, dt, xbar_override=override)
    return np.std(np.log(info["I"]))


def test_P8_force_bias_sign():
    """With xbar = +i sqrt(dt)(X - m) the O(sqrt dt) fluctuation of log I cancels:
    std(log I) ~ dt; with Eq. (14)'s printed sign it stays ~ sqrt(dt) (reading S1)."""
    r_good = _std_log_I(0.02, False) / _std_log_I(0.005, False)
    r_bad = _std_log_I(0.02, True) / _std_log_I(0.005, True)
    assert r_good > 3.0, r_good
    assert r_bad < 2.6, r_bad
    assert _std_log_I(0.005, False) < 0.5 * _std_log_I(0.005, True)


# --------------------------------------------------------------------------- P9
def test_P9_rhf_equals_uhf_on_duplicated_blocks():
    h, L, trial, walkers = small_problem(8, 3, 3, 6, 0, 10)
    o_r = AFQMCOracle(h, L, trial, 3, 3, 0)
    o_u = AFQMCOracle(h, L, np.concatenate([trial, trial], axis=1), 3, 3, 1)
    wu = np.concatenate([walkers, walkers], axis=2)
    assert np.abs(o_r.local_energy(walkers) - o_u.local_energy(wu)).max() < 1e-12
    assert abs(o_r.e_shift - o_u.e_shift) < 1e-12
    x = np.random.default_rng(1).standard_normal((3, 6))
    a, wa, ova = o_r.step(walkers, np.ones(3), x, 0.01)
    b, wb, ovb = o_u.step(wu, np.ones(3), x, 0.01)
    assert np.abs(a - b[:, :, :3]).max() < 1e-13 and np.abs(a - b[:, :, 3:]).max() < 1e-13
    assert np.abs(wa - wb).max() < 1e-13 and np.abs(ova - ovb).max() < 1e-12


# --------------------------------------------------------------------------- P10
def test_P10_taylor_vs_expm():
    h, L, trial, walkers = small_problem(8, 3, 3, 6, 0, 12, lscale=0.15)
    dt = 0.01
    x = np.random.default_rng(2).standard_normal((3, 6))
    for K, tol_fn in ((6, lambda a: a ** 7 / 5040 * np.exp(a)), (24, lambda a: 1e-13)):
        o = AFQMCOracle(h, L, trial, 3, 3, 0, taylor_order=K)
        new, info = o.propagate(walkers, x, dt)
        E1 = sla.expm(-0.5 * dt * o.h_mod)
        for w in range(3):
            A = info["A"][w]
            nA = np.linalg.norm(A, 2)
            assert nA <= 0.3
            mid = E1 @ walkers[w]
            exact = E1 @ (sla.expm(A) @ mid)
            err = np.linalg.norm(new[w] - exact, 2)
            scale = np.linalg.norm(mid, 2) * np.linalg.norm(E1, 2)
            assert err <= 1.05 * tol_fn(nA) * scale + 1e-14
            if K == 6:
                assert err > 1e-3 * tol_fn(nA) * scale             # the bound is not vacuous
            # A is complex symmetric (its value is pinned by P6's quadrature and P16's many-body propagator,
            # not by retyping the formula here)
            assert np.abs(A - A.T).max() < 1e-15


# --------------------------------------------------------------------------- P11
def test_P11_one_body_limit():
    M, na = 7, 3
    h, _, trial, walkers = small_problem(M, na, na, 4, 0, 13)
    L0 = np.zeros((4, M, M))
    dt = 0.05
    o = AFQMCOracle(h, L0, trial, na, na, 0, ortho_every=1)
    x = np.random.default_rng(3).standard_normal((3, 4))
    new, info = o.propagate(walkers, x, dt)
    assert np.abs(info["X"]).max() == 0 and np.abs(info["xbar"]).max() == 0 and np.abs(info["A"]).max() == 0
    ref = np.einsum("pq,wqi->wpi", sla.expm(-dt * h), walkers)
    assert np.abs(new - ref).max() < 1e-12
    r = o.overlap(ref) / o.overlap(walkers)
    _, wts, _ = o.step(walkers, np.ones(3), x, dt)
    expect = np.abs(r) * np.exp(dt * o.e_shift) * np.maximum(0, np.cos(np.angle(r)))
    assert np.abs(wts - expect).max() < 1e-12
    # long projection converges to the sum of the lowest na eigenvalues (x2 for RHF)
    wk, w = walkers, np.ones(3)
    for _ in range(1500):
        wk, w, _ = o.step(wk, w, x, dt)
    e0 = 2 * np.sort(np.linalg.eigvalsh(h))[:na].sum()
    assert np.abs(o.local_energy(wk)[:, 0] - e0).max() < 1e-8


# --------------------------------------------------------------------------- P12
def test_P12_conjugation_symmetry():
    h, L, trial, walkers = small_problem(8, 3, 2, 6, 1, 14)
    o = AFQMCOracle(h, L, trial, 3, 2, 1)
    x = np.random.default_rng(4).standard_normal((3, 6))
    a, wa, ova = o.step(walkers, np.ones(3), x, 0.01)
    b, wb, ovb = o.step(walkers.conj(), np.ones(3), -x, 0.01)
    assert np.abs(a.conj() - b).max() < 1e-13
    assert np.abs(wa - wb).max() < 1e-13 and np.abs(ova.conj() - ovb).max() < 1e-13
    assert np.abs(o.local_energy(walkers).conj() - o.local_energy(walkers.conj())).max() < 1e-12


# --------------------------------------------------------------------------- P13
def test_P13_weights_real_nonnegative_and_phaseless_cut():
    h, L, trial, walkers = small_problem(8, 3, 3, 6, 0, 15, lscale=0.8, noise=0.6, nw=40)
    o = AFQMCOracle(h, L, trial, 3, 3, 0)
    r = np.random.default_rng(5)
    wk, w = walkers, np.ones(40)
    killed = 0
    for s in range(6):
        x = r.standard_normal((40, 6))
        _, info = o.propagate(wk, x, 0.05)
        wk, w, _ = o.step(wk, w, x, 0.05)
        assert w.dtype == np.float64 and np.all(w >= 0) and np.all(np.isfinite(w))
        neg = info["S"].real <= 0
        assert np.all(w[neg] == 0)                                # max[0, cos theta], Eq. (15)
        killed += int(neg.sum())
    assert killed > 0                                             # the cut was exercised
    E = o.local_energy(wk)
    assert np.isfinite(np.sum(w * E[:, 0]) / np.sum(w))
    # a zero-overlap walker gets weight 0, not an error (reading S10)
    bad = walkers[:1].copy(); bad[:] = 0
    _, wb, _ = o.step(bad, np.ones(1), r.standard_normal((1, 6)), 0.05)
    assert wb[0] == 0.0


# --------------------------------------------------------------------------- P14 comb
from oracle.block_oracle import comb, estimators, run_block  # noqa: E402


def _random_weights(r, nw, dead=0):
    w = r.uniform(0.05, 3.0, nw) ** 2
    if dead:
        w[r.choice(nw, dead, replace=False)] = 0.0
    return w


@pytest.mark.parametrize("nw,dead", [(7, 0), (64, 5), (640, 40)])
def test_P14_comb_counts_closed_form(nw, dead):
    """Copies of walker i = number of integers k with c_{i-1} <= (k + xi) s < c_i, which has the
    closed form ceil(c_i/s - xi) - ceil(c_{i-1}/s - xi): an independent count (no search)."""
    r = np.random.default_rng(nw)
    w = _random_weights(r, nw, dead)
    c = np.concatenate([[0.0], np.cumsum(w)])
    s = c[-1] / nw
    for xi in (0.0, 0.123456789, 0.5, 0.999):
        m, wn = comb(w, xi)
        counts = np.bincount(m, minlength=nw)
        closed = np.ceil(c[1:] / s - xi) - np.ceil(c[:-1] / s - xi)
        closed[-1] += nw - closed.sum()          # the end point c_Nw/s = Nw is exact only up to rounding
        assert np.array_equal(counts, closed.astype(int))
        assert np.all(np.diff(m) >= 0)                              # a comb never reorders
        assert np.all(counts[w == 0.0] == 0)                        # dead walkers are never copied
        ideal = nw * w / c[-1]                                      # copies within one of the ideal
        assert np.all(counts >= np.floor(ideal - 1e-9)) and np.all(counts <= np.ceil(ideal + 1e-9))
        assert np.all(wn == wn[0]) and abs(wn.sum() - w.sum()) < 1e-13 * w.sum()   # total weight kept


def test_P14_comb_is_unbiased():
    """Averaged over xi (uniform grid), the number of copies of walker i is Nw w_i / W, i.e.
    sum_k w'_k f(phi'_k) has the expectation sum_i w_i f(phi_i) (Eq. 10)."""
    r = np.random.default_rng(5)
    nw, J = 24, 2000
    w = _random_weights(r, nw, 3)
    mean = np.zeros(nw)
    for j in range(J):
        m, _ = comb(w, (j + 0.5) / J)
        mean += np.bincount(m, minlength=nw)
    mean /= J
    assert np.abs(mean - nw * w / w.sum()).max() < 2.0 / J * nw


def test_P14_comb_special_cases():
    nw = 16
    for xi, v in ((0.0, 0.75), (0.3, 0.7), (0.99, 0.7)):             # equal weights: nothing moves
        m, wn = comb(np.full(nw, v), xi)                             # (xi = 0 puts the teeth ON the
        assert np.array_equal(m, np.arange(nw)) and np.allclose(wn, v, rtol=1e-15)   # boundaries: exact sums)
    w = np.zeros(nw); w[11] = 2.5                                    # one survivor takes every slot
    m, wn = comb(w, 0.4)
    assert np.all(m == 11) and np.allclose(wn, 2.5 / nw)
    for bad in (np.zeros(nw), np.full(nw, np.nan), np.full(nw, np.inf)):   # nothing to resample
        m, wn = comb(bad, 0.2)
        assert np.array_equal(m, np.arange(nw)) and np.array_equal(wn, bad, equal_nan=True)
    with pytest.raises(ValueError):
        comb(np.ones(4), 1.0)


# --------------------------------------------------------------------------- P15 estimator, block
def test_P15_estimator_and_block_loop():
    h, L, trial, walkers = small_problem(8, 3, 3, 6, 0, 21, lscale=0.15, noise=0.05, nw=6)
    o = AFQMCOracle(h, L, trial, 3, 3, 0, ortho_every=2)
    # (a) walkers = trial with arbitrary weights: ENumer/EDenom is the closed-form HF energy (P2),
    # EDenom the total weight, and the one- and two-body parts add up
    P = trial @ trial.T
    e1 = 2 * np.trace(h @ P)
    e2 = sum(2 * np.trace(Lg @ P) ** 2 - np.trace(Lg @ P @ Lg @ P) for Lg in L)
    wts = np.array([0.3, 1.7, 0.0, 2.2])
    Wt = np.repeat(trial[None].astype(np.complex128), 4, axis=0)
    est = estimators(wts, o.local_energy(Wt))
    assert abs(est[1] - 4.2) < 1e-14
    assert abs(est[0] / est[1] - (e1 + e2)) < 1e-12 * abs(e1 + e2)
    assert abs(est[2] / est[1] - e1) < 1e-12 * abs(e1) and abs(est[3] / est[1] - e2) < 1e-12 * abs(e2)
    assert np.allclose(estimators(3.0 * wts, o.local_energy(Wt)), 3.0 * est, rtol=1e-14)
    # (b) the block loop is the plain composition step -> comb -> ... -> local energy
    r = np.random.default_rng(3)
    x = r.standard_normal((4, 6, 6))
    xi = [0.37, 0.81]
    W, w, ov, E, est, maps = run_block(o, walkers, np.ones(6), x, xi, 0.01, 2)
    o2 = AFQMCOracle(h, L, trial, 3, 3, 0, ortho_every=2)
    W2, w2 = walkers, np.ones(6)
    for s in range(4):
        W2, w2, ov2 = o2.step(W2, w2, x[s], 0.01)
        if s in (1, 3):
            m, w2 = comb(w2, xi[s // 2])
            W2, ov2 = W2[m], ov2[m]
    assert np.array_equal(W, W2) and np.array_equal(w, w2) and np.array_equal(ov, ov2)
    assert len(maps) == 2 and np.array_equal(E, o2.local_energy(W2))
    assert np.allclose(ov, o.overlap(W), rtol=1e-10)                 # carried overlaps follow the walkers
    # (c) population control does not change the total weight, and the estimate it leaves is a
    # weighted mean of the local energies it was given
    assert abs(w.sum() - est[1]) < 1e-13 * est[1]
    assert E[:, 0].real.min() - 1e-12 <= est[0] / est[1] <= E[:, 0].real.max() + 1e-12
    # (d) pop_every = 0: no comb at all
    o3 = AFQMCOracle(h, L, trial, 3, 3, 0, ortho_every=2)
    _, w3, _, _, _, maps3 = run_block(o3, walkers, np.ones(6), x, [], 0.01, 0)
    assert maps3 == [] and not np.allclose(w3, w3[0])


# --------------------------------------------------------------------------- P16 weight rule, L != 0
def _many_body_step(o, h, L, trial, walkers, x, w0, dt, xbar_bound=0.0, ehyb_bound=0.0):
    """Weights and new overlaps of one step from explicit many-body matrices only (see P16's docstring); the optional
    bounds are applied as DESIGN.md reading S8b states them."""
    M, ng = h.shape[0], L.shape[0]
    F = Fock(M)
    dim = 2 ** F.n
    Id = np.eye(dim)
    H = F.hamiltonian(h, L)
    ta, tb = spin_blocks(o, trial)
    psiT = F.det_state(ta.astype(complex), tb.astype(complex))
    bra = psiT.conj()
    assert abs(bra @ psiT - 1.0) < 1e-12
    Lop = [F.one_body(L[g]) for g in range(ng)]
    m = np.array([(bra @ Lop[g] @ psiT).real for g in range(ng)])
    E_c = -0.5 * float(m @ m)
    e_shift = float((bra @ H @ psiT).real)
    V0 = H - E_c * Id
    for g in range(ng):
        d = Lop[g] - m[g] * Id
        V0 = V0 - 0.5 * d @ d
    half = sla.expm(-0.5 * dt * V0)
    expect_w, expect_ov, phases, xbars, absI = [], [], [], [], []
    for k in range(walkers.shape[0]):
        wa, wb = spin_blocks(o, walkers[k])
        ket = F.det_state(wa, wb)
        ov = bra @ ket
        X = np.array([(bra @ Lop[g] @ ket) / ov for g in range(ng)])
        xbar = 1j * np.sqrt(dt) * (X - m)
        if xbar_bound > 0:
            xbar = np.array([z * min(1.0, xbar_bound / abs(z)) if abs(z) > 0 else z for z in xbar])
        xs = x[k] - xbar
        two = sla.expm(-1j * np.sqrt(dt) * sum(xs[g] * (Lop[g] - m[g] * Id) for g in range(ng)))
        Bket = np.exp(-dt * E_c) * (half @ (two @ (half @ ket)))
        ratio = (bra @ Bket) / ov
        S = ratio * np.exp(dt * E_c)
        I = ratio * np.exp(np.sum(x[k] * xbar) - 0.5 * np.sum(xbar * xbar)) * np.exp(dt * e_shift)
        mod = abs(I)
        if ehyb_bound > 0:
            D = -np.log(mod) / dt
            mod = np.exp(-dt * min(max(D, -ehyb_bound), ehyb_bound))
        expect_w.append(w0[k] * mod * max(0.0, S.real / abs(S)))
        expect_ov.append(bra @ Bket * np.exp(dt * E_c) / np.exp(1j * np.sqrt(dt) * (xs @ m)))
        phases.append(np.angle(S))
        xbars.append(xbar)
        absI.append(abs(I))
    return dict(w=np.array(expect_w), ov=np.array(expect_ov), phases=np.array(phases), xbar=np.array(xbars),
                absI=np.array(absI), e_shift=e_shift, E_c=E_c)


@pytest.mark.parametrize("kind,na,nb,seed", [(1, 2, 1, 21), (0, 2, 2, 22)])
def test_P16_weight_rule_many_body(kind, na, nb, seed):
    """Eqs. (13), (15)-(18) with L != 0, from explicit many-body matrices only.

    In the 256-dimensional Fock space the one-sample propagator is built WITHOUT any of the oracle's one-body
    formulas: with m_g = <Psi_T|L_g|Psi_T>, E_c = -1/2 sum m_g^2 and V0 = H - E_c - 1/2 sum_g (L_g - m_g)^2
    (the operator the Trotter split of Eq. 7 calls v0 after the mean-field shift),
        B(x - xbar) = e^{-dt E_c} e^{-dt/2 V0} e^{-i sqrt(dt) sum_g (x - xbar)_g (L_g - m_g)} e^{-dt/2 V0},
    xbar_g = i sqrt(dt) (<L_g>_mixed - m_g).  Then S = <Psi_T|B|phi>/<Psi_T|phi> e^{+dt E_c} (Eq. 17; real
    positive factors do not enter theta), I = <Psi_T|B|phi>/<Psi_T|phi> e^{x.xbar - xbar.xbar/2} e^{dt E_shift}
    (Eq. 16 with the energy shift of reading S7) and w' = w |I| max(0, Re S/|S|) (Eqs. 13, 15, 18).  The oracle's
    `step` (Taylor order 24, i.e. the exact exponential to 1e-15) must give the same weights and overlaps."""
    M, ng, dt = 4, 3, 0.04
    h, L, trial, walkers = small_problem(M, na, nb, ng, kind, seed, lscale=0.45, noise=0.35, nw=6)
    o = AFQMCOracle(h, L, trial, na, nb, kind, taylor_order=24)
    x = np.random.default_rng(seed).standard_normal((walkers.shape[0], ng))
    w0 = np.linspace(0.5, 2.0, walkers.shape[0])
    mb = _many_body_step(o, h, L, trial, walkers, x, w0, dt)
    expect_w, expect_ov, phases, e_shift, E_c = mb["w"], mb["ov"], mb["phases"], mb["e_shift"], mb["E_c"]
    new, w, ov_new = o.step(walkers, w0, x, dt)
    assert abs(o.e_shift - e_shift) < 1e-12 and abs(o.E_const - E_c) < 1e-12
    assert np.max(np.abs(w - expect_w)) < 1e-10 * max(expect_w)
    # the propagated determinant itself: <Psi_T|phi'> = <Psi_T|B|phi> without the scalars B carries
    assert np.max(np.abs(ov_new - expect_ov) / np.abs(expect_ov)) < 1e-10
    assert np.max(np.abs(phases)) > 1e-2          # theta is not trivially zero: the cos factor is exercised
    assert np.all(expect_w > 0)


# --------------------------------------------------------------------------- P17 (optional bounds, reading S8b)
def test_P17_bounds():
    """SURVEY 8f NEXT-1 / DESIGN.md S8b: (a) bounds that never trigger leave every bit unchanged; (b) a force-bias
    bound that does trigger caps |xbar_g| at the bound, keeps the phases and the untouched components, and the step
    still equals the many-body step with THAT xbar (Eqs. 12, 16 hold for any xbar: the estimator stays exact);
    (c) a hybrid-energy bound that triggers replaces |I| by exp(-/+ dt b) and leaves max(0, cos theta) alone."""
    M, ng, dt, kind, na, nb = 4, 3, 0.04, 1, 2, 1
    h, L, trial, walkers = small_problem(M, na, nb, ng, kind, 31, lscale=0.45, noise=0.35, nw=6)
    x = np.random.default_rng(31).standard_normal((walkers.shape[0], ng))
    w0 = np.linspace(0.5, 2.0, walkers.shape[0])
    plain = AFQMCOracle(h, L, trial, na, nb, kind, taylor_order=24)
    W0, wt0, ov0 = plain.step(walkers, w0, x, dt)
    _, info0 = plain.propagate(walkers, x, dt)
    # (a)
    loose = AFQMCOracle(h, L, trial, na, nb, kind, taylor_order=24, xbar_bound=1e6, ehyb_bound=1e6)
    W1, wt1, ov1 = loose.step(walkers, w0, x, dt)
    assert np.array_equal(W0, W1) and np.array_equal(wt0, wt1) and np.array_equal(ov0, ov1)
    # (b)
    mags = np.abs(info0["xbar"])
    b = float(np.median(mags))                      # about half of the components get capped
    capped = AFQMCOracle(h, L, trial, na, nb, kind, taylor_order=24, xbar_bound=b)
    _, info = capped.propagate(walkers, x, dt)
    hit = mags > b
    assert hit.any() and (~hit).any()
    assert np.all(np.abs(info["xbar"]) <= b * (1 + 1e-15))
    assert np.array_equal(info["xbar"][~hit], info0["xbar"][~hit])
    assert np.abs(info["xbar"][hit] / np.abs(info["xbar"][hit]) - info0["xbar"][hit] / mags[hit]).max() < 1e-15
    mb = _many_body_step(capped, h, L, trial, walkers, x, w0, dt, xbar_bound=b)
    W2, wt2, ov2 = capped.step(walkers, w0, x, dt)
    assert np.abs(mb["xbar"] - info["xbar"]).max() < 1e-12
    assert np.max(np.abs(wt2 - mb["w"])) < 1e-10 * mb["w"].max()
    assert np.max(np.abs(ov2 - mb["ov"]) / np.abs(mb["ov"])) < 1e-10
    assert np.abs(wt2 - wt0).max() > 1e-6           # the bound did change the sample
    # (c)
    D = -np.log(np.abs(info0["I"])) / dt
    B = float(np.median(np.abs(D)))
    eb = AFQMCOracle(h, L, trial, na, nb, kind, taylor_order=24, ehyb_bound=B)
    W3, wt3, ov3 = eb.step(walkers, w0, x, dt)
    assert np.array_equal(W3, W0) and np.array_equal(ov3, ov0)      # the bound touches the weights only
    cos = np.maximum(0.0, info0["S"].real / np.abs(info0["S"]))
    trig = np.abs(D) > B
    assert trig.any() and (~trig).any()
    expect = np.where(trig, w0 * np.exp(-dt * np.sign(D) * B) * cos, wt0)
    assert np.max(np.abs(wt3 - expect)) < 1e-14 * expect.max()
    mb3 = _many_body_step(eb, h, L, trial, walkers, x, w0, dt, ehyb_bound=B)
    assert np.max(np.abs(wt3 - mb3["w"])) < 1e-10 * mb3["w"].max()
    # (d) reading S10 before S8b: a walker whose importance function is not finite is dead (weight exactly 0); the
    # bound clips finite values only and never turns inf into exp(dt b).  E_shift = 1e6: exp(-dt (E_const - E_shift))
    # overflows, every |I| is inf.
    dead = AFQMCOracle(h, L, trial, na, nb, kind, taylor_order=24, e_shift=1.0e6, ehyb_bound=B)
    _, info_d = dead.propagate(walkers, x, dt)
    assert not np.isfinite(info_d["I"]).any()
    _, wt4, _ = dead.step(walkers, w0, x, dt)
    assert np.array_equal(wt4, np.zeros_like(w0))


# --------------------------------------------------------------------------- P18 (the slab-provider branch)
@pytest.mark.parametrize("kind", [0, 1])
def test_P18_slab_provider_is_the_array_path(kind):
    """At c4 / c5 the oracle never sees the Cholesky tensor as one array: `_as_slab_iter` takes a callable that
    yields (g0, slab) pairs, and __init__ (m, h', h_mod, Lrot) and `vhs` accumulate slab by slab.  Pin that branch:
    UNEVEN slabs (5, 1, 7 vectors - a dropped or doubled slab, a wrong g0 offset into the fields, or a slab mistaken
    for the whole tensor all fail here) against (i) the array path and (ii) the closed forms that pin the array path
    itself - the Hartree-Fock energy of P2 and the definition A = -i sqrt(dt) sum_g x_g L_g of Eq. (9)."""
    na, nb = (3, 3) if kind == 0 else (3, 2)
    M, ng, dt = 9, 13, 0.01
    h, L, trial, walkers = small_problem(M, na, nb, ng, kind, 18)
    cuts = [0, 5, 6, 13]
    calls = []

    def provider():
        calls.append(1)
        for a, b in zip(cuts[:-1], cuts[1:]):
            yield a, L[a:b].copy()

    o_arr = AFQMCOracle(h, L, trial, na, nb, kind, ortho_every=2)
    o_slab = AFQMCOracle(h, provider, trial, na, nb, kind, ortho_every=2)
    assert o_slab.n_chol == ng
    for name in ("m", "h_mod", "E_const", "e_shift"):
        a, b = np.asarray(getattr(o_slab, name)), np.asarray(getattr(o_arr, name))
        assert np.max(np.abs(a - b)) <= 1e-14 * max(1.0, np.max(np.abs(b))), name
    for a, b in zip(o_slab.Lrot, o_arr.Lrot):
        assert a.shape == b.shape and np.max(np.abs(a - b)) <= 1e-14 * np.max(np.abs(b))
    # (ii) P2's closed form through the provider
    pa = trial[:, :na]
    pb = pa if kind == 0 else trial[:, na:]
    Pa, Pb = pa @ pa.T, pb @ pb.T
    e1 = np.trace(h @ Pa) + np.trace(h @ Pb)
    ec = 0.5 * sum((np.trace(Lg @ Pa) + np.trace(Lg @ Pb)) ** 2 for Lg in L)
    ex = -0.5 * sum(np.trace(Lg @ Pa @ Lg @ Pa) + np.trace(Lg @ Pb @ Lg @ Pb) for Lg in L)
    E = o_slab.local_energy(trial[None].astype(np.complex128))[0]
    assert abs(E[0] - (e1 + ec + ex)) < 1e-12 * abs(e1 + ec + ex)
    assert abs(o_slab.e_shift - (e1 + ec + ex)) < 1e-11
    # V_HS through the provider: the definition, with complex shifted fields, and the array path
    r = np.random.default_rng(180)
    xs = r.standard_normal((walkers.shape[0], ng)) + 1j * r.standard_normal((walkers.shape[0], ng))
    n0 = len(calls)
    A = o_slab.vhs(xs, dt)
    assert len(calls) == n0 + 1                                   # the tensor is streamed once per build
    A_def = -1j * np.sqrt(dt) * np.einsum("wg,gpq->wpq", xs, L)
    assert np.max(np.abs(A - A_def)) <= 1e-14 * np.max(np.abs(A_def))
    assert np.max(np.abs(A - o_arr.vhs(xs, dt))) <= 1e-14 * np.max(np.abs(A_def))
    # two full steps (the second re-orthonormalises) and the local energy
    x = r.standard_normal((2, walkers.shape[0], ng))
    Wa, wa = walkers.copy(), np.ones(walkers.shape[0])
    Wb, wb = walkers.copy(), np.ones(walkers.shape[0])
    for s in range(2):
        Wa, wa, ova = o_arr.step(Wa, wa, x[s], dt)
        Wb, wb, ovb = o_slab.step(Wb, wb, x[s], dt)
    assert np.max(np.abs(Wa - Wb)) <= 1e-13 * np.max(np.abs(Wa))
    assert np.max(np.abs(wa - wb)) <= 1e-13 * np.max(np.abs(wa))
    assert np.max(np.abs(ova - ovb)) <= 1e-13 * np.max(np.abs(ova))
    Ea, Eb = o_arr.local_energy(Wa), o_slab.local_energy(Wb)
    assert np.max(np.abs(Ea - Eb)) <= 1e-12 * np.max(np.abs(Ea))
