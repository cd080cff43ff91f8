"""GPU parity of the mixed-precision mode ("single precision is used for propagations and
double precision is used for local energy estimation"): the V_HS build runs in
emulated single precision on the tcgen05 tensor cores (bf16 x 3 operands, FP32 accumulation in tensor
memory), everything else in double.  The oracle stays the FP64 definition; the tolerances below are
single-precision ones derived in DESIGN.md (operand splitting keeps 24 bits; truncating FP32 accumulation
of n_chol / 16 updates of the large plane pair: 1e-7 .. 1e-6 relative on A at n_chol <= 540, 9e-6 at 4800;
times ||A|| ~ 0.4 on the walkers)."""
from __future__ import annotations

import numpy as np
import pytest

from tests.gpu_util import Pair, energy_scale, planar_to_complex, rel_fro, rel_max

pytestmark = pytest.mark.gpu

TOL_A = 5e-6          # ||A_mixed - A||_F / ||A||_F per walker (measured <= 1.0e-6 in these cases)
TOL_STEP = 2e-6       # walkers after one step (measured <= 2.7e-7)
TOL_OVLP = 1e-5       # overlaps (determinants of Nocc x Nocc blocks: errors add over the columns) and weights
TOL_RUN = 5e-5        # after 10 free-running steps
TOL_A_FULL = 3e-5     # n_chol = 3500 / 4800 (measured 6.4e-6 / 8.7e-6)
TOL_STEP_FULL = 1e-5  # (measured 1.6e-6 / 2.1e-6)


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def _mixed(pr, nw, **kw):
    from paper_2406_16238_b200 import afqmc
    cfg = pr.cfg
    return afqmc.AFQMC(pr.h1, pr.L_dev, pr.trial, M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta, n_chol=cfg.n_chol,
                       max_walkers=nw, walker_kind=cfg.walker_kind, taylor_order=cfg.taylor_order,
                       mixed_precision=True, **kw)


def _step(g, walkers, weights, x, dt):
    torch = _torch()
    W = torch.from_numpy(np.ascontiguousarray(walkers)).cuda()
    wt = torch.from_numpy(np.ascontiguousarray(weights)).cuda()
    xd = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    ov = torch.empty(W.shape[0], dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    g.step(W, wt, xd, dt)
    g.get_overlaps(ov)
    g.sync()
    return W.cpu().numpy(), wt.cpu().numpy(), ov.cpu().numpy()


# tile shapes: M below one q tile (24), ragged q tiles (38, 108), several row tiles (nw = 70 -> 140 rows),
# n_chol not a multiple of the 64-gamma stage (54, 300, 540)
CASES = [("c1", 16, {}), ("c2", 24, {}), ("c1", 5, dict(M=38, n_alpha=7, n_beta=7, n_chol=54)),
         ("c3", 70, dict(n_chol=300))]


@pytest.mark.parametrize("name,nw,over", CASES)
def test_vhs_and_one_step(name, nw, over):
    _torch()
    pr = Pair(name, nw=nw, ortho_every=0, **over)
    o, cfg = pr.oracle, pr.cfg
    g = _mixed(pr, nw)
    x = pr.fields(0)
    w0 = np.linspace(0.5, 1.5, nw)
    new_o, info = o.propagate(pr.walkers0, x, cfg.dt)
    Wg, wg, ovg = _step(g, pr.walkers0, w0, x, cfg.dt)
    A = planar_to_complex(g.debug_read(1), (nw, cfg.M, cfg.M))
    err = rel_fro(A, info["A"])
    assert err < TOL_A
    assert err > 1e-9                                         # it really is the single-precision route
    assert np.array_equal(A, A.transpose(0, 2, 1))            # mirrored stores: exactly symmetric
    assert rel_fro(Wg, new_o) < TOL_STEP
    _, w_o, ov_o = o.step(pr.walkers0, w0, x, cfg.dt)
    assert rel_max(ovg, ov_o) < TOL_OVLP
    assert rel_max(wg, w_o, scale=np.maximum(np.abs(w_o), 1e-3)) < TOL_OVLP
    g.close()
    pr.close()


def test_local_energy_stays_in_double():
    """The energy of given walkers does not go through the single-precision kernel: 1e-11 as the double path."""
    torch = _torch()
    pr = Pair("c2", nw=24)
    g = _mixed(pr, 24)
    W = torch.from_numpy(pr.walkers0).cuda()
    E = torch.empty((24, 3), dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    g.local_energy(W, E)
    g.sync()
    Eo = pr.oracle.local_energy(pr.walkers0)
    sc = energy_scale(pr.oracle, pr.walkers0, Eo)
    for k in range(3):
        assert rel_max(E.cpu().numpy()[:, k], Eo[:, k], scale=sc) < 1e-11
    g.close()
    pr.close()


@pytest.mark.parametrize("name,nw,ortho", [("c1", 16, 0), ("c2", 64, 5)])
def test_free_running(name, nw, ortho):
    torch = _torch()
    pr = Pair(name, nw=nw, ortho_every=ortho)
    o, cfg = pr.oracle, pr.cfg
    g = _mixed(pr, nw, ortho_every=ortho)
    Wo, wo = pr.walkers0, np.ones(nw)
    Wg, wg = Wo.copy(), wo.copy()
    for s in range(10):
        x = pr.fields(s)
        Wg, wg, ovg = _step(g, Wg, wg, x, cfg.dt)
        Wo, wo, ovo = o.step(Wo, wo, x, cfg.dt)
    assert rel_fro(Wg, Wo) < TOL_RUN
    assert rel_max(wg, wo, scale=np.maximum(np.abs(wo), 1e-3)) < TOL_RUN
    assert rel_max(ovg, ovo) < TOL_RUN
    E = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")
    Wd = torch.from_numpy(Wg).cuda()
    torch.cuda.synchronize()
    g.local_energy(Wd, E)
    g.sync()
    Eo = o.local_energy(Wo)
    sc = energy_scale(o, Wo, Eo)
    assert rel_max(E.cpu().numpy()[:, 0], Eo[:, 0], scale=sc) < TOL_RUN
    g.close()
    pr.close()


def test_mixed_precision_in_a_group_of_two():
    """Distributed Hamiltonian + mixed precision: the tcgen05 epilogue stores into the owners' slots."""
    torch = _torch()
    from oracle.afqmc_oracle import AFQMCOracle
    from paper_2406_16238_b200 import afqmc, inputs, sharded
    nw = 6
    cfg, h1, L, trial, walkers = inputs.make_problem_host("c1", nw=2 * nw)
    sl = sharded.gamma_slices(cfg.n_chol, 2)
    members = [afqmc.AFQMC(h1, torch.from_numpy(np.ascontiguousarray(L[a:b])).cuda(), trial, M=cfg.M, n_alpha=cfg.n_alpha,
                           n_beta=cfg.n_beta, n_chol=b - a, max_walkers=nw, walker_kind=cfg.walker_kind,
                           group_size=2, group_rank=r, mixed_precision=True) for r, (a, b) in enumerate(sl)]
    total = members[0].shard_setup_partial() + members[1].shard_setup_partial()
    addrs = np.stack([m.shard_get_buffers() for m in members])
    for m in members:
        m.shard_setup_finish(total)
        m.shard_set_peers(addrs)
    x = inputs.make_aux_fields(cfg, 0, 0, 2 * nw)
    W = [torch.from_numpy(np.ascontiguousarray(walkers[r * nw:(r + 1) * nw])).cuda() for r in range(2)]
    wt = [torch.ones(nw, dtype=torch.float64, device="cuda") for _ in range(2)]
    xs = [torch.from_numpy(np.ascontiguousarray(x[:, a:b])).cuda() for a, b in sl]
    torch.cuda.synchronize()
    for m, w in zip(members, W):
        m.shard_theta(w)
    for m in members:
        m.sync()
    for m, xx in zip(members, xs):
        m.shard_vhs(xx, cfg.dt, nw)
    for m in members:
        m.sync()
    for m, w, t in zip(members, W, wt):
        m.shard_propagate(w, t, cfg.dt)
    for m in members:
        m.sync()
    o = AFQMCOracle(h1, L, trial, cfg.n_alpha, cfg.n_beta, cfg.walker_kind, taylor_order=cfg.taylor_order)
    Wo, wo, _ = o.step(walkers, np.ones(2 * nw), x, cfg.dt)
    Wg = np.concatenate([w.cpu().numpy() for w in W])
    err = rel_fro(Wg, Wo)
    assert 1e-10 < err < TOL_STEP
    assert rel_max(np.concatenate([t.cpu().numpy() for t in wt]), wo) < TOL_OVLP
    for m in members:
        m.close()


def test_mixed_precision_argument_checks():
    torch = _torch()
    from paper_2406_16238_b200 import afqmc, inputs
    cfg, h1, L, trial, _ = inputs.make_problem_host("c1", nw=4, M=37, n_alpha=7, n_beta=7, n_chol=53)
    Ld = torch.from_numpy(L).cuda()
    kw = dict(M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta, n_chol=cfg.n_chol, max_walkers=4, walker_kind=0)
    with pytest.raises(afqmc.AfqmcError) as e:
        afqmc.AFQMC(h1, Ld, trial, mixed_precision=True, **kw)
    assert e.value.code == -6
    cfg, h1, L, trial, _ = inputs.make_problem_host("c1", nw=4)
    Ld = torch.from_numpy(L).cuda()
    kw = dict(M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta, n_chol=cfg.n_chol, max_walkers=4, walker_kind=0)
    with pytest.raises(afqmc.AfqmcError) as e:
        afqmc.AFQMC(h1, Ld, trial, mixed_precision=True, pack_chol=True, **kw)
    assert e.value.code == -1


@pytest.mark.parametrize("name,with_oracle", [("c4", True), ("c5", False)])
def test_full_size(name, with_oracle):
    """BASELINE.json's large configs in the launch configuration bench.py --mixed-precision times (whole batch
    per call: 256 rows = two 128-row blocks at c4, 5700 tiles at c5): one step on every walker against the
    double-precision CUDA path (itself held to the oracle at these sizes by tests/test_gpu_parity.py), and at
    c4 against the oracle on two sampled walkers."""
    torch = _torch()
    pr = Pair(name, device_L=True, oracle=with_oracle)
    cfg, nw = pr.cfg, pr.nw
    g = _mixed(pr, nw)
    x = pr.fields(0)
    w0 = np.linspace(0.5, 1.5, nw)
    Wm, wm, ovm = _step(g, pr.walkers0, w0, x, cfg.dt)
    for rep in range(12):                  # thousands of pipeline stages per SM and call: same bits every time
        W2, w2, _ = _step(g, pr.walkers0, w0, x, cfg.dt)
        assert W2.tobytes() == Wm.tobytes() and w2.tobytes() == wm.tobytes(), rep
    Wd, wd, ovd = _step(pr.gpu, pr.walkers0, w0, x, cfg.dt)
    for rep in range(12):                  # and the double path likewise
        W2, w2, _ = _step(pr.gpu, pr.walkers0, w0, x, cfg.dt)
        assert W2.tobytes() == Wd.tobytes() and w2.tobytes() == wd.tobytes(), rep
    err = rel_fro(Wm, Wd)
    assert 1e-10 < err < TOL_STEP_FULL
    # The tensor core adds into its FP32 accumulator with truncation, not round-to-nearest: the 300 updates of
    # the large (hh) accumulator at n_chol = 4800 leave a ONE-SIGNED relative error of ~1e-5 on A, which the
    # determinant of the N_occ x N_occ overlap collects: weights and |overlaps| come out larger by a factor
    # 1 + 2.2e-5 at c5 (1.8e-5 at c4) that is COMMON to all walkers (it cancels in every weighted average)
    # with a walker-to-walker spread of 9e-6.  DESIGN.md section 5.
    ratio = wm / wd
    assert abs(np.median(ratio) - 1.0) < 1.5e-4
    assert ratio.max() - ratio.min() < 4e-5
    assert rel_max(ovm, ovd) < 1.5e-4
    A = g.debug_read(1).reshape(nw, 2, cfg.M, cfg.M)
    Ad = pr.gpu.debug_read(1).reshape(nw, 2, cfg.M, cfg.M)
    assert rel_fro(A, Ad) < TOL_A_FULL
    del A, Ad
    if with_oracle:
        idx = np.array([0, nw - 1])
        Wo, wo, ovo = pr.oracle.step(pr.walkers0[idx], w0[idx], x[idx], cfg.dt)
        assert rel_fro(Wm[idx], Wo) < TOL_STEP_FULL
        assert rel_max(wm[idx], wo) < 1.5e-4
    g.close()
    pr.close()


def _random_cases(n, seed):
    """Seeded random shapes: even M and n_chol (TMA strides), RHF and UHF, occupied blocks 1..48, 1..140 rows."""
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(n):
        M = 2 * int(rng.integers(12, 80))
        uhf = bool(rng.integers(0, 2))
        na = int(rng.integers(1, min(48, M // 2)))
        nb = int(rng.integers(1, na + 1)) if uhf else na
        nchol = 2 * int(rng.integers(5, 120))
        nw = int(rng.integers(1, 71))
        out.append(("c2" if uhf else "c1", nw, dict(M=M, n_alpha=na, n_beta=nb, n_chol=nchol)))
    return out


@pytest.mark.parametrize("name,nw,over", _random_cases(10, 20240607) + [
    ("c2", 3, dict(M=160, n_alpha=64, n_beta=50, n_chol=40)),     # N2 = 228 > 128: one accumulator set in TMEM
    ("c2", 2, dict(M=150, n_alpha=40, n_beta=33, n_chol=30)),     # N2 = 146
])
def test_random_shapes(name, nw, over):
    """Tile edges of the tcgen05 kernels: ragged 8 x 16 tiles, odd tile counts (a pair with one tile), gamma and
    k padding, 1..140 rows, N2 from 2 to 228 columns."""
    _torch()
    pr = Pair(name, nw=nw, ortho_every=0, **over)
    o, cfg = pr.oracle, pr.cfg
    g = _mixed(pr, nw)
    x = pr.fields(0)
    w0 = np.linspace(0.5, 1.5, nw)
    new_o, info = o.propagate(pr.walkers0, x, cfg.dt)
    Wg, wg, ovg = _step(g, pr.walkers0, w0, x, cfg.dt)
    A = planar_to_complex(g.debug_read(1), (nw, cfg.M, cfg.M))
    assert rel_fro(A, info["A"]) < TOL_A
    X = planar_to_complex(g.debug_read(0), (nw, cfg.n_chol))
    assert rel_fro(X, info["X"]) < TOL_A
    assert rel_fro(Wg, new_o) < TOL_STEP
    _, w_o, ov_o = o.step(pr.walkers0, w0, x, cfg.dt)
    assert rel_max(ovg, ov_o) < TOL_OVLP
    assert rel_max(wg, w_o, scale=np.maximum(np.abs(w_o), 1e-3)) < TOL_OVLP
    g.close()
    pr.close()


@pytest.mark.parametrize("mixed", [False, True])
def test_bitwise_reproducible(mixed):
    """No atomics, fixed-order reductions, hardware-ordered pipelines: the same call gives the same bits.  A
    race in a shared-memory ring or in the tensor-memory hand-over would show up here as a flipped bit
    (the WAR race of DESIGN.md section 7 was found this way at full size)."""
    torch = _torch()
    pr = Pair("c3", nw=40, oracle=False, n_chol=600)
    cfg = pr.cfg
    g = _mixed(pr, 40) if mixed else pr.gpu
    x = torch.from_numpy(pr.fields(0)).cuda()
    ref = None
    for rep in range(25):
        W = torch.from_numpy(pr.walkers0).cuda()
        wt = torch.ones(40, dtype=torch.float64, device="cuda")
        E = torch.empty((40, 3), dtype=torch.complex128, device="cuda")
        torch.cuda.synchronize()
        g.step(W, wt, x, cfg.dt)
        g.local_energy(W, E)
        g.sync()
        out = (W.cpu().numpy().tobytes(), wt.cpu().numpy().tobytes(), E.cpu().numpy().tobytes())
        if ref is None:
            ref = out
        assert out == ref, rep
    if mixed:
        g.close()
    pr.close()
