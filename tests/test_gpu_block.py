"""GPU parity for what sits between the steps of a block: population control
by the comb (index work: bit-exact), the estimator sums, and afqmc_run_block against the oracle's
block loop.  Through the C ABI via the ctypes binding."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2406_16238_b200 import inputs
from tests.gpu_util import Pair, energy_scale, rel_fro, rel_max

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _weight_cases(nw):
    r = np.random.default_rng(nw)
    w = r.uniform(0.05, 3.0, nw) ** 2
    out = [("random", w.copy())]
    wz = w.copy(); wz[r.choice(nw, max(1, nw // 8), replace=False)] = 0.0
    out.append(("with dead walkers", wz))
    out.append(("equal", np.full(nw, 0.7)))
    ws = np.zeros(nw); ws[nw // 2] = 2.5
    out.append(("one survivor", ws))
    wt = wz.copy(); wt[-3:] = 0.0
    out.append(("dead tail", wt))
    out.append(("all dead", np.zeros(nw)))
    wn = w.copy(); wn[0] = np.nan
    out.append(("nan", wn))
    out.append(("wide range", np.exp(r.uniform(-30, 3, nw))))
    return out


@pytest.mark.parametrize("nw", [1, 2, 16, 77, 640])
def test_comb_is_bit_exact(nw):
    """Map (int32) equal to the oracle's, new weights bit-equal, walkers and the stored overlaps
    permuted exactly, for every degenerate weight vector and xi at both ends of [0, 1)."""
    torch = _torch()
    from oracle.block_oracle import comb
    pr = Pair("c1", nw=nw, oracle=False)
    cfg = pr.cfg
    # one step so that the handle holds overlaps for these nw walkers
    W0 = torch.from_numpy(pr.walkers0).cuda()
    w0 = torch.ones(nw, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()              # the library runs on its own stream, torch on another
    pr.gpu.step(W0, w0, torch.from_numpy(pr.fields(0)).cuda(), cfg.dt)
    ov0 = torch.empty(nw, dtype=torch.complex128, device="cuda")
    pr.gpu.get_overlaps(ov0)
    pr.gpu.sync()
    Wh, ovh = W0.cpu().numpy(), ov0.cpu().numpy()
    for label, w in _weight_cases(nw):
        for xi in (0.0, 0.25, 0.637, np.nextafter(1.0, 0.0)):
            m_o, w_o = comb(w, xi)
            W = torch.from_numpy(Wh).cuda()
            wd = torch.from_numpy(w.copy()).cuda()
            xid = torch.tensor([xi], dtype=torch.float64, device="cuda")
            md = torch.empty(nw, dtype=torch.int32, device="cuda")
            torch.cuda.synchronize()
            pr.gpu.population_control(W, wd, xid, md)
            ov = torch.empty(nw, dtype=torch.complex128, device="cuda")
            pr.gpu.get_overlaps(ov)
            pr.gpu.sync()
            assert np.array_equal(md.cpu().numpy().astype(np.int64), m_o), (label, xi)
            assert np.array_equal(wd.cpu().numpy(), w_o, equal_nan=True), (label, xi)
            assert np.array_equal(W.cpu().numpy(), Wh[m_o]), (label, xi)
            assert np.array_equal(ov.cpu().numpy(), ovh[m_o]), (label, xi)
            ovh = ovh[m_o]                       # the handle's overlaps stay permuted
    # host pointers give the same thing
    w = _weight_cases(nw)[1][1]
    Wn, wn, mn = Wh.copy(), w.copy(), np.empty(nw, dtype=np.int32)
    pr.gpu.population_control(Wn, wn, np.array([0.4]), mn)
    m_o, w_o = comb(w, 0.4)
    assert np.array_equal(mn, m_o) and np.array_equal(wn, w_o) and np.array_equal(Wn, Wh[m_o])
    with pytest.raises(Exception):
        pr.gpu.population_control(Wn, wn, np.array([1.0]), mn)
    pr.close()


def test_estimators_match_the_oracle():
    torch = _torch()
    from oracle.block_oracle import estimators
    pr = Pair("c2", nw=100, oracle=False)
    r = np.random.default_rng(0)
    E = r.standard_normal((100, 3)) * 50 + 1j * r.standard_normal((100, 3))
    w = r.uniform(0, 2, 100); w[::7] = 0.0
    ref = estimators(w, E)
    out = torch.empty(4, dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    pr.gpu.estimators(torch.from_numpy(w).cuda(), torch.from_numpy(E).cuda(), out)
    pr.gpu.sync()
    sc = np.array([np.sum(w * np.abs(E[:, 0].real)), np.sum(w), np.sum(w * np.abs(E[:, 1].real)),
                   np.sum(w * np.abs(E[:, 2].real))])
    assert np.max(np.abs(out.cpu().numpy() - ref) / sc) < 1e-14
    outh = np.empty(4)
    pr.gpu.estimators(w, E, outh)
    assert np.array_equal(outh, out.cpu().numpy())
    pr.close()


@pytest.mark.parametrize("name,nw,n_steps,pop_every,ortho", [("c1", 16, 25, 5, 5), ("c2", 64, 10, 5, 5),
                                                             ("c1", 16, 7, 3, 2), ("c1", 16, 4, 0, 0)])
def test_run_block_matches_the_oracle_block_loop(name, nw, n_steps, pop_every, ortho):
    """A block as the paper times it (25 steps) with QR and the comb every 5
    steps: the comb's maps must come out identical (else walkers differ at O(1)), walkers,
    weights, overlaps, energies and the estimator sums to 1e-8 free-running."""
    torch = _torch()
    from oracle.block_oracle import run_block
    pr = Pair(name, nw=nw, ortho_every=ortho)
    cfg = pr.cfg
    x = np.stack([pr.fields(s) for s in range(n_steps)])
    n_pop = n_steps // pop_every if pop_every else 0
    xi = inputs.make_pop_uniforms(0, max(n_pop, 1))
    Wo, wo, ovo, Eo, est_o, maps = run_block(pr.oracle, pr.walkers0, np.ones(nw), x, xi, cfg.dt, pop_every)
    assert len(maps) == n_pop
    if n_pop:
        assert any(not np.array_equal(m, np.arange(nw)) for m in maps), "the comb should do something here"
    W = torch.from_numpy(pr.walkers0).cuda()
    w = torch.ones(nw, dtype=torch.float64, device="cuda")
    E = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")
    est = torch.empty(4, dtype=torch.float64, device="cuda")
    ov = torch.empty(nw, dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    pr.gpu.run_block(W, w, torch.from_numpy(x).cuda(), torch.from_numpy(xi).cuda() if n_pop else None, cfg.dt,
                     pop_every, E, est)
    pr.gpu.get_overlaps(ov)
    pr.gpu.sync()
    assert rel_fro(W.cpu().numpy(), Wo) < 1e-8
    assert rel_max(w.cpu().numpy(), wo) < 1e-8
    assert rel_max(ov.cpu().numpy(), ovo) < 1e-8
    sc = energy_scale(pr.oracle, Wo, Eo)
    for k in range(3):
        assert rel_max(E.cpu().numpy()[:, k], Eo[:, k], scale=sc) < 1e-8
    esc = np.array([np.sum(wo * sc), np.sum(wo), np.sum(wo * sc), np.sum(wo * sc)])
    assert np.max(np.abs(est.cpu().numpy() - est_o) / esc) < 1e-8
    # host buffers through the same call: bit-identical to the device-buffer call
    pr2 = Pair(name, nw=nw, ortho_every=ortho, oracle=False)
    Wn, wn = pr.walkers0.copy(), np.ones(nw)
    En, estn = np.empty((nw, 3), dtype=np.complex128), np.empty(4)
    pr2.gpu.run_block(Wn, wn, x, xi if n_pop else None, cfg.dt, pop_every, En, estn)
    assert np.array_equal(Wn, W.cpu().numpy()) and np.array_equal(wn, w.cpu().numpy())
    assert np.array_equal(En, E.cpu().numpy()) and np.array_equal(estn, est.cpu().numpy())
    pr2.close()
    pr.close()


@pytest.mark.parametrize("name,nw,ortho", [("c1", 16, 5), ("c2", 32, 3)])
def test_run_block_graph_replay_is_bit_identical_to_eager_launches(name, nw, ortho):
    """Third call on with the same buffers replays a CUDA graph of the whole block: same bits as
    the eager launches, including the phase of the QR schedule that the graph bakes in."""
    torch = _torch()
    pr = Pair(name, nw=nw, ortho_every=ortho, oracle=False)
    cfg = pr.cfg
    n_steps, pop_every = 10, 5          # 10 % 3 != 0 for c2: the ortho phase changes from block to block
    x = torch.from_numpy(np.stack([pr.fields(s) for s in range(n_steps)])).cuda()
    xi = torch.from_numpy(inputs.make_pop_uniforms(0, 2)).cuda()
    W0 = torch.from_numpy(pr.walkers0).cuda()
    W, w = torch.empty_like(W0), torch.empty(nw, dtype=torch.float64, device="cuda")
    E = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")
    est = torch.empty(4, dtype=torch.float64, device="cuda")

    def blocks(n):
        out = []
        for _ in range(n):
            W.copy_(W0); w.fill_(1.0)
            torch.cuda.synchronize()
            pr.gpu.run_block(W, w, x, xi, cfg.dt, pop_every, E, est)
            pr.gpu.sync()
            out.append((W.cpu().numpy(), w.cpu().numpy(), E.cpu().numpy(), est.cpu().numpy()))
        return out

    pr.gpu.set_block_graph(0)
    eager = blocks(6)
    assert pr.gpu.set_block_graph(-1) == 0
    pr2 = Pair(name, nw=nw, ortho_every=ortho, oracle=False)       # fresh handle: same QR phases
    gpu_keep = pr.gpu
    pr.gpu = pr2.gpu
    graphed = blocks(6)
    assert pr2.gpu.set_block_graph(-1) >= (1 if n_steps % ortho else 4)
    for a, b in zip(eager, graphed):
        for u, v in zip(a, b):
            assert np.array_equal(u, v)
    pr.gpu = gpu_keep
    pr2.close()
    pr.close()
