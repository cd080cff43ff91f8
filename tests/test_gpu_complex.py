"""GPU parity for complex Cholesky vectors: `complex_chol = 1` against
oracle/complex_chol_oracle.py (pinned by tests/test_oracle_complex_pins.py), same tolerances as the real path."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2406_16238_b200 import inputs
from tests.gpu_util import planar_to_complex, rel_fro, rel_max

pytestmark = pytest.mark.gpu

TOL_STEP = 1e-10
TOL_RUN = 1e-8


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _pair(M, na, nb, npairs, kind, nw, seed=0, complex_trial=False, kernel_path=0, xbar_bound=0.0, ehyb_bound=0.0):
    torch = _torch()
    from oracle.complex_chol_oracle import ComplexCholOracle
    from paper_2406_16238_b200 import afqmc
    h, L, trial, walkers = inputs.make_complex_problem(M, na, nb, npairs, kind, seed, nw, complex_trial=complex_trial)
    assert np.iscomplexobj(trial) == complex_trial
    o = ComplexCholOracle(h, L, trial, na, nb, kind, xbar_bound=xbar_bound, ehyb_bound=ehyb_bound)
    Ld = torch.from_numpy(L).cuda()
    g = afqmc.AFQMC(h, Ld, trial, M=M, n_alpha=na, n_beta=nb, n_chol=L.shape[0], max_walkers=nw, walker_kind=kind,
                    complex_chol=True, complex_trial=complex_trial, kernel_path=kernel_path,
                    xbar_bound=xbar_bound, ehyb_bound=ehyb_bound)
    Ld.fill_(float("nan"))                 # the caller's tensor is not referenced after afqmc_create
    torch.cuda.synchronize()
    return o, g, walkers


def _step(g, W, wt, x, dt):
    torch = _torch()
    Wd = torch.from_numpy(np.ascontiguousarray(W)).cuda()
    wd = torch.from_numpy(np.ascontiguousarray(wt)).cuda()
    xd = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    ov = torch.empty(W.shape[0], dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    g.step(Wd, wd, xd, dt)
    g.get_overlaps(ov)
    g.sync()
    return Wd.cpu().numpy(), wd.cpu().numpy(), ov.cpu().numpy()


def _energy(g, W):
    torch = _torch()
    Wd = torch.from_numpy(np.ascontiguousarray(W)).cuda()
    E = torch.empty((W.shape[0], 3), dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    g.local_energy(Wd, E)
    g.sync()
    return E.cpu().numpy()


# the last case is UHF past half filling: Nt = n_alpha + n_beta = 19 > M = 16 (Nt x M setup products must not go
# through M x M scratch)
CASES = [(24, 5, 5, 12, 0, 8), (40, 9, 6, 10, 1, 5), (37, 7, 7, 9, 0, 3), (64, 16, 14, 20, 1, 6), (16, 10, 9, 6, 1, 4)]


@pytest.mark.parametrize("ctrial", [False, True])
@pytest.mark.parametrize("M,na,nb,npairs,kind,nw", CASES)
def test_setup_and_stages(M, na, nb, npairs, kind, nw, ctrial):
    o, g, walkers = _pair(M, na, nb, npairs, kind, nw, complex_trial=ctrial)
    c = g.constants()
    assert abs(c["E_const"] - o.E_const) <= 1e-12 * abs(o.E_const)
    assert abs(c["e_trial"] - o.e_shift) <= 1e-11 * abs(o.e_shift)
    x = inputs.make_complex_fields(0, 0, nw, o.n_fields)
    w0 = np.linspace(0.5, 1.5, nw)
    new_o, info = o.propagate(walkers, x, 0.005)
    Wg, wg, ovg = _step(g, walkers, w0, x, 0.005)
    X = planar_to_complex(g.debug_read(0), (nw, o.n_fields))
    assert rel_fro(X, info["X"]) < 1e-12
    A = planar_to_complex(g.debug_read(1), (nw, M, M))
    assert rel_fro(A, info["A"]) < 1e-11
    assert rel_fro(Wg, new_o) < TOL_STEP
    _, w_o, ov_o = o.step(walkers, w0, x, 0.005)
    assert rel_max(ovg, ov_o) < TOL_STEP
    assert rel_max(wg, w_o, scale=np.maximum(np.abs(w_o), 1e-3)) < TOL_STEP
    g.close()


@pytest.mark.parametrize("ctrial", [False, True])
@pytest.mark.parametrize("M,na,nb,npairs,kind,nw", CASES)
def test_local_energy(M, na, nb, npairs, kind, nw, ctrial):
    o, g, walkers = _pair(M, na, nb, npairs, kind, nw, complex_trial=ctrial)
    Eo = o.local_energy(walkers)
    Eg = _energy(g, walkers)
    X = o.force_bias_X(o.theta(walkers))
    ec = 0.5 * np.sum(X * X, axis=1)
    sc = np.abs(Eo[:, 1]) + np.abs(ec) + np.abs(Eo[:, 2] - ec)
    for k in range(3):
        assert rel_max(Eg[:, k], Eo[:, k], scale=sc) < 1e-11
    assert np.abs(Eo[:, 0].imag).max() > 1e-6          # genuinely complex energies: the cross term matters
    g.close()


@pytest.mark.parametrize("ctrial,kpath", [(False, 0), (True, 0), (True, 1), (True, 2)])
def test_free_running(ctrial, kpath):
    """10 free-running steps + energy; with a complex trial (oracle pins PC6-PC9) also on the
    cp.async kernels (kernel_path 1) and the one-kernel overlap route (kernel_path 2)."""
    o, g, walkers = _pair(40, 9, 6, 10, 1, 8, complex_trial=ctrial, kernel_path=kpath)
    Wo, wo = walkers, np.ones(8)
    Wg, wg = walkers.copy(), np.ones(8)
    for s in range(10):
        x = inputs.make_complex_fields(0, s, 8, o.n_fields)
        Wg, wg, ovg = _step(g, Wg, wg, x, 0.005)
        Wo, wo, ovo = o.step(Wo, wo, x, 0.005)
    assert rel_fro(Wg, Wo) < TOL_RUN
    assert rel_max(wg, wo, scale=np.maximum(np.abs(wo), 1e-3)) < TOL_RUN
    assert rel_max(ovg, ovo) < TOL_RUN
    Eo, Eg = o.local_energy(Wo), _energy(g, Wg)
    assert rel_max(Eg[:, 0], Eo[:, 0], scale=np.abs(Eo[:, 1]) + np.abs(Eo[:, 2])) < TOL_RUN
    assert wo.min() > 0.05
    g.close()


def test_bounds_complex():
    """Optional bounds (S8b, pin P17) in the complex mode with a complex trial; both set so that they
    trigger on part of the components / walkers."""
    o0, g0, walkers = _pair(40, 9, 6, 10, 1, 8, complex_trial=True)
    x = inputs.make_complex_fields(0, 0, 8, o0.n_fields)
    _, info = o0.propagate(walkers, x, 0.005)
    g0.close()
    b = float(np.median(np.abs(info["xbar"])))
    B = float(np.median(np.abs(np.log(np.abs(info["I"])) / 0.005)))
    o, g, walkers = _pair(40, 9, 6, 10, 1, 8, complex_trial=True, xbar_bound=b, ehyb_bound=B)
    Wo, wo, ovo = o.step(walkers, np.ones(8), x, 0.005)
    Wg, wg, ovg = _step(g, walkers, np.ones(8), x, 0.005)
    assert rel_fro(Wg, Wo) < TOL_STEP and rel_max(ovg, ovo) < TOL_STEP
    assert rel_max(wg, wo, scale=np.maximum(np.abs(wo), 1e-3)) < TOL_STEP
    W1, w1, _ = o0.step(walkers, np.ones(8), x, 0.005)
    assert rel_fro(Wo, W1) > 1e-6 and np.abs(wo - w1).max() > 1e-6          # the bounds did something
    g.close()


def test_vectors_that_are_no_repulsion_integrals_are_rejected():
    """Half of a {C, C^+} set: sum_g L_ps conj(L_rq) is not (ps|qr) = (qr|ps) symmetric; the oracle refuses it
    (PC1) and so does the library."""
    torch = _torch()
    from paper_2406_16238_b200 import afqmc
    h, L, trial, _ = inputs.make_complex_problem(24, 5, 5, 4, 0, 0, 2)
    Ld = torch.from_numpy(np.ascontiguousarray(L[:4])).cuda()
    with pytest.raises(afqmc.AfqmcError) as e:
        afqmc.AFQMC(h, Ld, trial, M=24, n_alpha=5, n_beta=5, n_chol=4, max_walkers=2, walker_kind=0, complex_chol=True)
    assert e.value.code == -1 and "symmetric tensor" in str(e.value)


def test_unsupported_combinations():
    torch = _torch()
    from paper_2406_16238_b200 import afqmc
    h, L, trial, _ = inputs.make_complex_problem(24, 5, 5, 4, 0, 0, 2)
    Ld = torch.from_numpy(L).cuda()
    kw = dict(M=24, n_alpha=5, n_beta=5, n_chol=L.shape[0], max_walkers=2, walker_kind=0, complex_chol=True)
    for extra in (dict(pack_chol=True), dict(mixed_precision=True), dict(group_size=2, group_rank=0)):
        with pytest.raises(afqmc.AfqmcError) as e:
            afqmc.AFQMC(h, Ld, trial, **kw, **extra)
        assert e.value.code == -6


def test_block_with_population_control():
    """afqmc_run_block in the complex mode: 10 steps, the comb every 5, energy and estimator sums, against the
    plain composition of the complex oracle's step, the (pinned) comb and the estimator sums; then the CUDA-graph
    replay of the same block gives the same bits."""
    torch = _torch()
    from oracle.block_oracle import run_block
    nw, n_steps, pop_every = 12, 10, 5
    o, g, walkers = _pair(40, 9, 6, 10, 1, nw)
    x = np.stack([inputs.make_complex_fields(0, s, nw, o.n_fields) for s in range(n_steps)])
    xi = inputs.make_pop_uniforms(0, n_steps // pop_every)
    Wo, wo, ovo, Eo, est_o, maps = run_block(o, walkers, np.ones(nw), x, xi, 0.005, pop_every)
    xd, xid = torch.from_numpy(x).cuda(), torch.from_numpy(xi).cuda()
    E = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")
    est = torch.empty(4, dtype=torch.float64, device="cuda")
    outs = []
    for rep in range(4):                   # eager, capture, two replays
        W = torch.from_numpy(walkers).cuda() if rep == 0 else W.copy_(torch.from_numpy(walkers))
        w = torch.ones(nw, dtype=torch.float64, device="cuda") if rep == 0 else w.fill_(1.0)
        torch.cuda.synchronize()
        g.run_block(W, w, xd, xid, 0.005, pop_every, E, est)
        g.sync()
        outs.append((W.cpu().numpy().copy(), w.cpu().numpy().copy(), E.cpu().numpy().copy(), est.cpu().numpy().copy()))
    Wg, wg, Eg, estg = outs[0]
    assert rel_fro(Wg, Wo) < TOL_RUN
    assert rel_max(wg, wo) < TOL_RUN
    sc = np.abs(Eo[:, 1]) + np.abs(Eo[:, 2])
    assert rel_max(Eg[:, 0], Eo[:, 0], scale=sc) < TOL_RUN
    assert abs(estg[0] / estg[1] - est_o[0] / est_o[1]) < TOL_RUN * np.mean(sc)
    for other in outs[1:]:
        for a, b in zip(outs[0], other):
            assert np.array_equal(a, b)
    assert g.set_block_graph(-1) >= 2
    g.close()


def test_create_destroy_releases_device_memory():
    """Handles of every flavour (double, pack_chol, mixed precision, complex, group member) give their device memory
    back: free memory after 5 create/destroy rounds equals free memory after the first one."""
    torch = _torch()
    from paper_2406_16238_b200 import afqmc
    cfg, h1, L, trial, _ = inputs.make_problem_host("c1", nw=4)
    Ld = torch.from_numpy(L).cuda()
    hc, Lc, tc, _ = inputs.make_complex_problem(24, 5, 5, 6, 0, 0, 4)
    Lcd = torch.from_numpy(Lc).cuda()
    kw = dict(M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta, max_walkers=4, walker_kind=0)

    def round_trip():
        for extra in (dict(), dict(pack_chol=True), dict(mixed_precision=True), dict(group_size=2, group_rank=1)):
            afqmc.AFQMC(h1, Ld, trial, n_chol=cfg.n_chol, **kw, **extra).close()
        afqmc.AFQMC(hc, Lcd, tc, n_chol=Lc.shape[0], complex_chol=True, **kw).close()
        torch.cuda.synchronize()
        return torch.cuda.mem_get_info()[0]

    first = round_trip()
    for _ in range(4):
        last = round_trip()
    assert last == first
