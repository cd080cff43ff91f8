"""Pins of oracle/complex_chol_oracle.py (complex Cholesky vectors): the
derivation in its header against explicit many-body matrices, a brute-force four-index tensor, quadrature and
the already pinned real oracle.  CPU only.  None of these retype the oracle's formulas."""
import numpy as np
import pytest
import scipy.linalg as sla

from oracle.afqmc_oracle import AFQMCOracle
from oracle.complex_chol_oracle import ComplexCholOracle, hermitian_parts
from tests.fock import Fock


def complex_problem(M, na, nb, nc, kind, seed, lscale=0.3, noise=0.2, nw=3, complex_trial=False):
    """Complex Hermitian h, vectors {C_k, C_k^+} (closed under +, so the tensor is (ps|qr) = (qr|ps) symmetric),
    real (or complex, orthonormal) trial, complex walkers."""
    r = np.random.default_rng(seed)
    h = r.standard_normal((M, M)) + 1j * r.standard_normal((M, M))
    h = 0.5 * (h + h.conj().T)
    C = (r.standard_normal((nc, M, M)) + 1j * r.standard_normal((nc, M, M))) * lscale
    L = np.concatenate([C, C.conj().transpose(0, 2, 1)], axis=0)
    blocks = [np.linalg.qr(r.standard_normal((M, na)))[0]]
    if kind == 1:
        blocks.append(np.linalg.qr(r.standard_normal((M, nb)))[0])
    if complex_trial:
        blocks = [np.linalg.qr(b + 1j * r.standard_normal(b.shape))[0] for b in blocks]
    trial = np.concatenate(blocks, axis=1)
    Nt = trial.shape[1]
    walkers = trial[None] + noise * (r.standard_normal((nw, M, Nt)) + 1j * r.standard_normal((nw, M, Nt)))
    return h, L, trial, walkers.astype(np.complex128)


def eri_of(L):
    """(ps|qr) = sum_g L_ps conj(L_rq), the definition (not the oracle's Hermitian-parts form)."""
    return np.einsum("gps,grq->psqr", L, L.conj())


def spin_blocks(o, mat):
    if o.walker_kind == 0:
        return mat[:, :o.n_alpha], mat[:, :o.n_alpha]
    return mat[:, :o.n_alpha], mat[:, o.n_alpha:o.n_alpha + o.n_beta]


def test_PC1_hermitian_parts_factorise_the_symmetric_tensor():
    _, L, _, _ = complex_problem(4, 2, 1, 3, 1, 0)
    K = hermitian_parts(L)
    assert K.shape[0] == 2 * L.shape[0]                       # twice as many fields as vectors
    assert np.abs(K - K.conj().transpose(0, 2, 1)).max() < 1e-15
    eri = eri_of(L)
    assert np.abs(eri - eri.transpose(2, 3, 0, 1)).max() < 1e-13          # (ps|qr) = (qr|ps)
    assert np.abs(eri - np.einsum("gps,gqr->psqr", K, K)).max() < 1e-13
    # a set that is not closed under + is not such a tensor, and is rejected
    half = L[:3]
    e2 = eri_of(half)
    assert np.abs(e2 - e2.transpose(2, 3, 0, 1)).max() > 1e-3
    with pytest.raises(ValueError):
        ComplexCholOracle(np.eye(4), half, np.eye(4)[:, :2], 2, 2, 0)


@pytest.mark.parametrize("kind", [0, 1])
def test_PC2_reduces_to_the_real_oracle(kind):
    """Real symmetric vectors: A_g = L_g, B_g = 0; the extra fields multiply zero matrices."""
    r = np.random.default_rng(3)
    M, na, nb, ng, nw = 6, 2, 2 if kind == 0 else 1, 4, 3
    h = r.standard_normal((M, M)); h = 0.5 * (h + h.T)
    L = r.standard_normal((ng, M, M)) * 0.3; L = 0.5 * (L + L.transpose(0, 2, 1))
    blocks = [np.linalg.qr(r.standard_normal((M, na)))[0]]
    if kind == 1:
        blocks.append(np.linalg.qr(r.standard_normal((M, nb)))[0])
    trial = np.concatenate(blocks, axis=1)
    W = trial[None] + 0.2 * (r.standard_normal((nw, M, trial.shape[1])) + 1j * r.standard_normal((nw, M, trial.shape[1])))
    o = AFQMCOracle(h, L, trial, na, nb, kind)
    c = ComplexCholOracle(h, L, trial, na, nb, kind)
    x = r.standard_normal((nw, ng))
    x2 = np.concatenate([x, r.standard_normal((nw, ng))], axis=1)
    Wo, wo, ovo = o.step(W, np.ones(nw), x, 0.01)
    Wc, wc, ovc = c.step(W, np.ones(nw), x2, 0.01)
    assert np.abs(Wo - Wc).max() < 1e-13 and np.abs(wo - wc).max() < 1e-13 and np.abs(ovo - ovc).max() < 1e-12
    assert np.abs(o.local_energy(W) - c.local_energy(W)).max() < 1e-12
    assert abs(o.E_const - c.E_const) < 1e-13 and abs(o.e_shift - c.e_shift) < 1e-12


@pytest.mark.parametrize("kind,na,nb", [(1, 2, 1), (0, 2, 2)])
def test_PC3_fock_space(kind, na, nb):
    """Overlap, <K_g'>, the local energy and Thouless' theorem against explicit many-body matrices built from
    the DEFINITION of the tensor, sum_g L_ps conj(L_rq)."""
    M, nc = 4, 2
    h, L, trial, walkers = complex_problem(M, na, nb, nc, kind, 4)
    o = ComplexCholOracle(h, L, trial, na, nb, kind)
    F = Fock(M)
    H = F.hamiltonian_eri(h, eri_of(L))
    assert np.abs(H - H.conj().T).max() < 1e-12
    ta, tb = spin_blocks(o, trial)
    bra = F.det_state(ta.astype(complex), tb.astype(complex)).conj()
    ov, E = o.overlap(walkers), o.local_energy(walkers)
    X = o.force_bias_X(o.theta(walkers))
    for w in range(walkers.shape[0]):
        wa, wb = spin_blocks(o, walkers[w])
        ket = F.det_state(wa, wb)
        ov_mb = bra @ ket
        assert abs(ov[w] - ov_mb) < 1e-12
        assert abs(E[w, 0] - (bra @ H @ ket) / ov_mb) < 1e-11
        for g in range(o.n_fields):
            assert abs(X[w, g] - (bra @ F.one_body(o.Kmat[g]) @ ket) / ov_mb) < 1e-12
    A = o.vhs(np.array([[0.3, -1.1, 0.7, 0.2, -0.4, 0.9, 0.1, -0.6]]), 0.01)[0]
    wa, wb = spin_blocks(o, walkers[0])
    lhs = sla.expm(F.one_body(A)) @ F.det_state(wa, wb)
    rhs = F.det_state(sla.expm(A) @ wa, sla.expm(A) @ wb)
    assert np.abs(lhs - rhs).max() < 1e-12


def test_PC4_mean_field_shift_identity():
    """H = H1[h_mod] + E_const + 1/2 sum_g' (K_g' - m_g')^2 as many-body matrices (Eqs. 4-6 with 2n fields)."""
    M, nc = 3, 2
    h, L, trial, _ = complex_problem(M, 2, 1, nc, 1, 5)
    o = ComplexCholOracle(h, L, trial, 2, 1, 1)
    F = Fock(M)
    H = F.hamiltonian_eri(h, eri_of(L))
    I = np.eye(2 ** F.n)
    rhs = F.one_body(o.h_mod) + o.E_const * I
    for g in range(o.n_fields):
        d = F.one_body(o.Kmat[g]) - o.m[g] * I
        rhs = rhs + 0.5 * d @ d
    assert np.abs(H - rhs).max() < 1e-12
    assert np.abs(o.m).max() > 1e-2 and np.abs(o.h_mod - o.h_mod.conj().T).max() < 1e-13


def _quadrature_error(dt, mode):
    """One complex vector C and its adjoint: 4 Hermitian matrices, of which A(C^+) = A(C), B(C^+) = -B(C); the
    quadrature runs over the 4 fields with 12 nodes each."""
    M, na, nb = 3, 2, 1
    h, L, trial, walkers = complex_problem(M, na, nb, 1, 1, 7, lscale=0.45, noise=0.15, nw=1)
    o = ComplexCholOracle(h, L, trial, na, nb, 1, taylor_order=24)
    F = Fock(M)
    H = F.hamiltonian_eri(h, eri_of(L))
    wa, wb = spin_blocks(o, walkers[0])
    exact = sla.expm(-dt * H) @ F.det_state(wa, wb)
    nodes, wts = np.polynomial.hermite_e.hermegauss(12)
    wts = wts / wts.sum()
    grid = np.array(np.meshgrid(nodes, nodes, nodes, nodes, indexing="ij")).reshape(4, -1).T
    ws = np.prod(np.array(np.meshgrid(wts, wts, wts, wts, indexing="ij")).reshape(4, -1), axis=0)
    batch = np.repeat(walkers, grid.shape[0], axis=0)
    override = {"fb": None, "zero": np.zeros(4), "arb": np.array([0.11 - 0.07j, -0.05 + 0.13j, 0.02j, -0.04])}[mode]
    new, info = o.propagate(batch, grid, dt, xbar_override=override)
    scal = info["I"] * info["ovlp_old"] / info["ovlp_new"] * np.exp(-dt * o.e_shift)
    acc = np.zeros_like(exact)
    for k in range(grid.shape[0]):
        a, b = spin_blocks(o, new[k])
        acc = acc + ws[k] * scal[k] * F.det_state(a, b)
    return np.linalg.norm(acc - exact) / np.linalg.norm(exact)


def test_PC5_hubbard_stratonovich_quadrature():
    """int dx p(x) e^{x.xbar - xbar.xbar/2} B(x - xbar)|phi> = e^{-dt H}|phi> + O(dt^2) with the 2n fields, for the
    force bias, xbar = 0 and an arbitrary complex xbar: signs and scalars of the whole propagation."""
    e1 = {m: _quadrature_error(0.02, m) for m in ("fb", "zero", "arb")}
    e2 = {m: _quadrature_error(0.01, m) for m in ("zero",)}
    for m in e1:
        assert e1[m] < 5e-3
    assert 3.3 < e1["zero"] / e2["zero"] < 4.7, (e1, e2)
    assert abs(e1["fb"] - e1["zero"]) < 1e-5 and abs(e1["arb"] - e1["zero"]) < 1e-5


# ----------------------------------------------------------------------------------------------------------------
# Complex trial (SURVEY S12 "formulas keep psi^+"): the oracle's psi^+ against many-body matrices.
# <Psi_T| is the adjoint of the determinant state built from the trial's columns; none of the pins below uses a
# one-body formula of the oracle.

@pytest.mark.parametrize("kind,na,nb", [(1, 2, 1), (0, 2, 2)])
def test_PC6_complex_trial_fock_space(kind, na, nb):
    """Overlap, mixed <K_g'>, local energy, mean fields m_g' = <Psi_T|K_g'|Psi_T> and the trial energy."""
    M, nc = 4, 2
    h, L, trial, walkers = complex_problem(M, na, nb, nc, kind, 11, complex_trial=True)
    assert np.abs(trial.imag).max() > 0.1
    o = ComplexCholOracle(h, L, trial, na, nb, kind)
    F = Fock(M)
    H = F.hamiltonian_eri(h, eri_of(L))
    ta, tb = spin_blocks(o, trial)
    psiT = F.det_state(ta, tb)
    bra = psiT.conj()
    assert abs(bra @ psiT - 1.0) < 1e-12
    ov, E = o.overlap(walkers), o.local_energy(walkers)
    X = o.force_bias_X(o.theta(walkers))
    for w in range(walkers.shape[0]):
        wa, wb = spin_blocks(o, walkers[w])
        ket = F.det_state(wa, wb)
        ov_mb = bra @ ket
        assert abs(ov[w] - ov_mb) < 1e-12 * max(1.0, abs(ov_mb))
        assert abs(E[w, 0] - (bra @ H @ ket) / ov_mb) < 1e-11
        for g in range(o.n_fields):
            assert abs(X[w, g] - (bra @ F.one_body(o.Kmat[g]) @ ket) / ov_mb) < 1e-12
    for g in range(o.n_fields):
        mg = bra @ F.one_body(o.Kmat[g]) @ psiT
        assert abs(mg.imag) < 1e-13 and abs(o.m[g] - mg.real) < 1e-13
    assert abs(o.e_shift - (bra @ H @ psiT).real) < 1e-12
    assert abs(o.E_const + 0.5 * float(o.m @ o.m)) < 1e-14


def test_PC7_complex_trial_reductions():
    """(a) A complex trial with zero imaginary part is the real-trial oracle (to rounding).  (b) A unitary rotation
    U of the occupied columns is the same state up to the phase det(U): overlaps pick up conj(det U) per block,
    Theta-derived quantities (X, energies), the propagated walkers and the weights do not change."""
    M, na, nb, nc, kind = 6, 3, 2, 2, 1
    h, L, trial, walkers = complex_problem(M, na, nb, nc, kind, 13)
    a = ComplexCholOracle(h, L, trial, na, nb, kind)
    b = ComplexCholOracle(h, L, trial.astype(np.complex128), na, nb, kind)
    r = np.random.default_rng(5)
    x = r.standard_normal((walkers.shape[0], a.n_fields))
    Wa, wa, ova = a.step(walkers, np.ones(3), x, 0.01)
    Wb, wb, ovb = b.step(walkers, np.ones(3), x, 0.01)
    assert np.abs(Wa - Wb).max() < 1e-13 and np.abs(wa - wb).max() < 1e-13 and np.abs(ova - ovb).max() < 1e-13
    # (b)
    _, _, ctrial, _ = complex_problem(M, na, nb, nc, kind, 13, complex_trial=True)
    Ua = np.linalg.qr(r.standard_normal((na, na)) + 1j * r.standard_normal((na, na)))[0]
    Ub = np.linalg.qr(r.standard_normal((nb, nb)) + 1j * r.standard_normal((nb, nb)))[0]
    rot = np.concatenate([ctrial[:, :na] @ Ua, ctrial[:, na:] @ Ub], axis=1)
    c = ComplexCholOracle(h, L, ctrial, na, nb, kind)
    d = ComplexCholOracle(h, L, rot, na, nb, kind)
    ph = np.conj(np.linalg.det(Ua) * np.linalg.det(Ub))
    assert np.abs(d.overlap(walkers) - ph * c.overlap(walkers)).max() < 1e-12
    assert np.abs(d.m - c.m).max() < 1e-13 and abs(d.e_shift - c.e_shift) < 1e-12
    assert np.abs(d.local_energy(walkers) - c.local_energy(walkers)).max() < 1e-11
    Wc, wc, ovc = c.step(walkers, np.ones(3), x, 0.01)
    Wd, wd, ovd = d.step(walkers, np.ones(3), x, 0.01)
    assert np.abs(Wc - Wd).max() < 1e-12 and np.abs(wc - wd).max() < 1e-12 and np.abs(ovd - ph * ovc).max() < 1e-12


def test_PC8_complex_trial_hf_closed_form():
    """walker = trial: overlap 1, X = m, and the energy is the Hartree-Fock closed form written with the
    DEFINITION of the tensor and the density matrix G_pq = <a+_p a_q> = conj(P)_pq, P = psi psi^+ (Eq. 11 by Wick):
    E = sum h_pq G_pq + 1/2 sum (ps|qr) [G^tot_ps G^tot_qr - sum_sigma G_pr G_qs]."""
    M, na, nb, nc, kind = 5, 2, 1, 2, 1
    h, L, trial, _ = complex_problem(M, na, nb, nc, kind, 17, complex_trial=True)
    o = ComplexCholOracle(h, L, trial, na, nb, kind)
    W = trial[None].astype(np.complex128)
    assert abs(o.overlap(W)[0] - 1.0) < 1e-13
    assert np.abs(o.force_bias_X(o.theta(W))[0] - o.m).max() < 1e-13
    eri = eri_of(L)
    Gs = [(trial[:, :na] @ trial[:, :na].conj().T).T, (trial[:, na:] @ trial[:, na:].conj().T).T]
    Gt = Gs[0] + Gs[1]
    E = np.einsum("pq,pq->", h, Gt) + 0.5 * np.einsum("psqr,ps,qr->", eri, Gt, Gt)
    for G in Gs:
        E = E - 0.5 * np.einsum("psqr,pr,qs->", eri, G, G)
    assert abs(E.imag) < 1e-12
    assert abs(o.local_energy(W)[0, 0] - E) < 1e-12 * max(1.0, abs(E))


def test_PC9_complex_trial_weight_rule_many_body():
    """Eqs. (13), (15)-(18) with a complex trial from many-body matrices only (as P16 of the real oracle):
    B(x - xbar) = e^{-dt E_c} e^{-dt/2 V0} e^{-i sqrt(dt) sum (x - xbar)_g (K_g - m_g)} e^{-dt/2 V0},
    S = <Psi_T|B|phi>/<Psi_T|phi> e^{dt E_c}, I = ratio e^{x.xbar - xbar.xbar/2} e^{dt E_shift}."""
    M, na, nb, nc, kind, dt = 3, 2, 1, 1, 1, 0.04
    h, L, trial, walkers = complex_problem(M, na, nb, nc, kind, 19, lscale=0.45, noise=0.3, nw=5, complex_trial=True)
    o = ComplexCholOracle(h, L, trial, na, nb, kind, taylor_order=24)
    F = Fock(M)
    Id = np.eye(2 ** F.n)
    H = F.hamiltonian_eri(h, eri_of(L))
    ta, tb = spin_blocks(o, trial)
    psiT = F.det_state(ta, tb)
    bra = psiT.conj()
    Kop = [F.one_body(k) for k in hermitian_parts(L)]
    ng = len(Kop)
    m = np.array([(bra @ Kop[g] @ psiT).real for g in range(ng)])
    E_c = -0.5 * float(m @ m)
    e_shift = float((bra @ H @ psiT).real)
    V0 = H - E_c * Id
    for g in range(ng):
        dd = Kop[g] - m[g] * Id
        V0 = V0 - 0.5 * dd @ dd
    half = sla.expm(-0.5 * dt * V0)
    x = np.random.default_rng(23).standard_normal((walkers.shape[0], ng))
    w0 = np.linspace(0.5, 2.0, walkers.shape[0])
    ew, eov, phases = [], [], []
    for k in range(walkers.shape[0]):
        wa, wb = spin_blocks(o, walkers[k])
        ket = F.det_state(wa, wb)
        ov = bra @ ket
        X = np.array([(bra @ Kop[g] @ ket) / ov for g in range(ng)])
        xbar = 1j * np.sqrt(dt) * (X - m)
        xs = x[k] - xbar
        two = sla.expm(-1j * np.sqrt(dt) * sum(xs[g] * (Kop[g] - m[g] * Id) for g in range(ng)))
        Bket = np.exp(-dt * E_c) * (half @ (two @ (half @ ket)))
        ratio = (bra @ Bket) / ov
        S = ratio * np.exp(dt * E_c)
        I = ratio * np.exp(np.sum(x[k] * xbar) - 0.5 * np.sum(xbar * xbar)) * np.exp(dt * e_shift)
        ew.append(w0[k] * abs(I) * max(0.0, S.real / abs(S)))
        eov.append(bra @ Bket * np.exp(dt * E_c) / np.exp(1j * np.sqrt(dt) * (xs @ m)))
        phases.append(np.angle(S))
    _, w, ov_new = o.step(walkers, w0, x, dt)
    assert np.max(np.abs(w - np.array(ew))) < 1e-10 * max(ew)
    assert np.max(np.abs(ov_new - np.array(eov)) / np.abs(eov)) < 1e-10
    assert np.max(np.abs(phases)) > 1e-2
