"""GPU parity of the distributed-Hamiltonian mode: a group of
G members, each holding a gamma slice of L and its own walkers, must reproduce the oracle that
sees the whole tensor.  Same tolerances as tests/test_gpu_parity.py.

All members live on the ONE GPU of the box: in one process (LocalGroup, phases executed member
after member, so no kernel ever waits on another) and in two processes that exchange CUDA IPC
handles (DistGroup over gloo, host barriers between the phases)."""
from __future__ import annotations

import os
import subprocess
import sys

import numpy as np
import pytest

from paper_2406_16238_b200 import inputs
from tests.gpu_util import energy_scale, rel_fro, rel_max

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
TOL_STEP = 1e-10
TOL_RUN = 1e-8


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


class ShardedPair:
    """The oracle on the whole problem and a LocalGroup on its gamma slices."""

    def __init__(self, name, G, nw, seed=0, ortho_every=0, pack_chol=False, uneven=False, **over):
        torch = _torch()
        from oracle.afqmc_oracle import AFQMCOracle
        from paper_2406_16238_b200 import sharded
        cfg = inputs.get_config(name, **over)
        self.cfg, self.G, self.nw, self.seed = cfg, G, nw, seed
        self.h1 = inputs.make_h1(cfg, seed)
        self.trial = inputs.make_trial(cfg, self.h1, seed)
        self.L = inputs.make_L_host(cfg, seed)
        self.slices = sharded.gamma_slices(cfg.n_chol, G)
        if uneven and G == 2:                       # a deliberately lopsided split (even sizes)
            cut = 2 * max(1, cfg.n_chol // 6)
            self.slices = [(0, cut), (cut, cfg.n_chol)]
        self.L_dev = [torch.from_numpy(np.ascontiguousarray(self.L[a:b])).cuda() for a, b in self.slices]
        self.group = sharded.LocalGroup(self.h1, self.L_dev, self.trial, M=cfg.M, n_alpha=cfg.n_alpha,
                                        n_beta=cfg.n_beta, max_walkers=nw, walker_kind=cfg.walker_kind,
                                        taylor_order=cfg.taylor_order, ortho_every=ortho_every,
                                        pack_chol=pack_chol)
        self.oracle = AFQMCOracle(self.h1, self.L, self.trial, cfg.n_alpha, cfg.n_beta, cfg.walker_kind,
                                  taylor_order=cfg.taylor_order, ortho_every=ortho_every)
        self.walkers0 = inputs.make_walkers(cfg, self.trial, seed, G * nw)       # owner-major

    def fields(self, step):
        return inputs.make_aux_fields(self.cfg, self.seed, step, self.G * self.nw)

    def split(self, a):
        return [np.ascontiguousarray(a[r * self.nw:(r + 1) * self.nw]) for r in range(self.G)]

    def gpu_step(self, walkers, weights, x, dt):
        torch = _torch()
        W = [torch.from_numpy(w).cuda() for w in self.split(walkers)]
        wt = [torch.from_numpy(w).cuda() for w in self.split(weights)]
        xs = [torch.from_numpy(v).cuda() for v in self.split(x)]
        self.group.step(W, wt, xs, dt)
        ov = []
        for m in self.group.members:
            o = torch.empty(self.nw, dtype=torch.complex128, device="cuda")
            m.get_overlaps(o)
            m.sync()
            ov.append(o.cpu().numpy())
        return (np.concatenate([w.cpu().numpy() for w in W]), np.concatenate([w.cpu().numpy() for w in wt]),
                np.concatenate(ov))

    def gpu_energy(self, walkers):
        torch = _torch()
        W = [torch.from_numpy(w).cuda() for w in self.split(walkers)]
        E = [torch.empty((self.nw, 3), dtype=torch.complex128, device="cuda") for _ in range(self.G)]
        self.group.local_energy(W, E)
        return np.concatenate([e.cpu().numpy() for e in E])

    def close(self):
        self.group.close()
        self.L_dev = None


CASES = [("c1", 2, 8, {}), ("c1", 3, 5, {}), ("c2", 2, 12, {}),
         ("c1", 4, 3, dict(M=38, n_alpha=7, n_beta=7, n_chol=54)),
         ("c2", 2, 4, dict(M=40, n_alpha=9, n_beta=2, n_chol=70))]


@pytest.mark.parametrize("name,G,nw,over", CASES)
def test_setup_sums_match_the_oracle(name, G, nw, over):
    sp = ShardedPair(name, G, nw, **over)
    o = sp.oracle
    for m in sp.group.members:
        c = m.constants()
        assert abs(c["E_const"] - o.E_const) <= 1e-12 * abs(o.E_const)
        assert abs(c["e_trial"] - o.e_shift) <= 1e-11 * abs(o.e_shift)
        hm = m.debug_read(3).reshape(sp.cfg.M, sp.cfg.M)
        assert rel_fro(hm[None], o.h_mod[None]) < 1e-12
    # every member holds the same bits
    h0 = sp.group.members[0].debug_read(3)
    for m in sp.group.members[1:]:
        assert np.array_equal(h0, m.debug_read(3))
    sp.close()


@pytest.mark.parametrize("name,G,nw,over", CASES)
def test_per_step_parity_reseeded(name, G, nw, over):
    """Each step from the oracle's walkers: walkers, weights, overlaps to 1e-10; then energies."""
    sp = ShardedPair(name, G, nw, uneven=(G == 2 and name == "c1"), **over)
    o, cfg = sp.oracle, sp.cfg
    Wo, wo = sp.walkers0, np.linspace(0.5, 1.5, G * nw)
    for s in range(3):
        x = sp.fields(s)
        Wg, wg, ovg = sp.gpu_step(Wo, wo, x, cfg.dt)
        Wo, wo, ovo = o.step(Wo, wo, x, cfg.dt)
        assert rel_fro(Wg, Wo) < TOL_STEP, s
        assert rel_max(wg, wo, scale=np.maximum(np.abs(wo), 1e-3)) < TOL_STEP, s
        assert rel_max(ovg, ovo) < TOL_STEP, s
    Eo = o.local_energy(Wo)
    Eg = sp.gpu_energy(Wo)
    sc = energy_scale(o, Wo, Eo)
    for k in range(3):
        assert rel_max(Eg[:, k], Eo[:, k], scale=sc) < 1e-11
    sp.close()


@pytest.mark.parametrize("name,G,nw,steps,ortho,pack", [("c1", 2, 8, 10, 0, False), ("c2", 2, 16, 10, 5, False),
                                                         ("c1", 3, 4, 6, 2, True)])
def test_free_running_parity(name, G, nw, steps, ortho, pack):
    """N free-running steps (QR on schedule, pack_chol slices): weights, overlaps, energies to 1e-8."""
    sp = ShardedPair(name, G, nw, ortho_every=ortho, pack_chol=pack)
    o, cfg = sp.oracle, sp.cfg
    Wo, wo = sp.walkers0, np.ones(G * nw)
    Wg, wg = Wo.copy(), wo.copy()
    for s in range(steps):
        x = sp.fields(s)
        Wg, wg, ovg = sp.gpu_step(Wg, wg, x, cfg.dt)
        Wo, wo, ovo = o.step(Wo, wo, x, cfg.dt)
    assert rel_max(wg, wo, scale=np.maximum(np.abs(wo), 1e-3)) < TOL_RUN
    assert rel_max(ovg, ovo) < TOL_RUN
    assert rel_fro(Wg, Wo) < TOL_RUN
    Eo, Eg = o.local_energy(Wo), sp.gpu_energy(Wg)
    sc = energy_scale(o, Wo, Eo)
    assert rel_max(Eg[:, 0], Eo[:, 0], scale=sc) < TOL_RUN
    sp.close()


def test_group_of_slices_equals_single_handle():
    """The same walkers through one handle with the whole tensor and through a group of 2:
    sums over gamma are only re-associated, so the two GPU paths agree far below 1e-10."""
    torch = _torch()
    from paper_2406_16238_b200 import afqmc
    sp = ShardedPair("c2", 2, 10)
    cfg = sp.cfg
    one = afqmc.AFQMC(sp.h1, torch.from_numpy(sp.L).cuda(), sp.trial, M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta,
                      n_chol=cfg.n_chol, max_walkers=20, walker_kind=cfg.walker_kind, taylor_order=cfg.taylor_order)
    x = sp.fields(0)
    wt0 = np.linspace(0.7, 1.3, 20)
    Wg, wg, _ = sp.gpu_step(sp.walkers0, wt0, x, cfg.dt)
    W1 = torch.from_numpy(sp.walkers0).cuda()
    w1 = torch.from_numpy(wt0.copy()).cuda()
    xd = torch.from_numpy(x).cuda()
    E1 = torch.empty((20, 3), dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    one.step(W1, w1, xd, cfg.dt)
    one.local_energy(W1, E1)
    one.sync()
    assert rel_fro(Wg, W1.cpu().numpy()) < 1e-12
    assert rel_max(wg, w1.cpu().numpy()) < 1e-11
    Eg = sp.gpu_energy(W1.cpu().numpy())
    assert rel_max(Eg[:, 1], E1.cpu().numpy()[:, 1]) < 1e-12
    assert np.max(np.abs(Eg[:, 0] - E1.cpu().numpy()[:, 0])) < 1e-11 * np.max(np.abs(E1.cpu().numpy()[:, 1]))
    one.close()
    sp.close()


def test_error_codes():
    torch = _torch()
    from paper_2406_16238_b200 import afqmc
    cfg, h1, L, trial, walkers = inputs.make_problem_host("c1", nw=4)
    Ld = torch.from_numpy(np.ascontiguousarray(L[:48])).cuda()
    kw = dict(M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta, n_chol=48, max_walkers=4, walker_kind=0)
    with pytest.raises(afqmc.AfqmcError) as e:
        afqmc.AFQMC(h1, Ld, trial, group_size=9, group_rank=0, **kw)
    assert e.value.code == -6
    with pytest.raises(afqmc.AfqmcError) as e:
        afqmc.AFQMC(h1, Ld, trial, group_size=2, group_rank=2, **kw)
    assert e.value.code == -1
    m = afqmc.AFQMC(h1, Ld, trial, group_size=2, group_rank=0, **kw)
    W = torch.from_numpy(walkers).cuda()
    wt = torch.ones(4, dtype=torch.float64, device="cuda")
    x = torch.zeros((4, 48), dtype=torch.float64, device="cuda")
    with pytest.raises(afqmc.AfqmcError) as e:      # whole-step calls are refused on a member
        m.step(W, wt, x, 0.005)
    assert e.value.code == -6
    with pytest.raises(afqmc.AfqmcError) as e:      # phases need the setup sums and the peers first
        m.shard_theta(W)
    assert e.value.code == -1
    m.shard_setup_finish(m.shard_setup_partial())
    with pytest.raises(afqmc.AfqmcError) as e:
        m.shard_theta(W)
    assert e.value.code == -1
    addrs = np.stack([m.shard_get_buffers(), m.shard_get_buffers()])
    m.shard_set_peers(addrs)
    with pytest.raises(afqmc.AfqmcError) as e:      # the group batch must be full
        m.shard_theta(W[:2], nw=2)
    assert e.value.code == -2
    plain = afqmc.AFQMC(h1, Ld, trial, **kw)
    with pytest.raises(afqmc.AfqmcError) as e:      # and a plain handle has no phases
        plain.shard_theta(W)
    assert e.value.code == -1
    plain.close()
    m.close()


def test_two_processes_over_cuda_ipc(tmp_path):
    """One process per member (DistGroup): buffers exchanged as CUDA IPC handles, gloo for the
    setup sums, the field routing and the barriers.  Both processes use the box's one GPU; the
    phases are separated by host barriers, so no kernel waits on another process."""
    _torch()
    out = tmp_path / "result.npz"
    env = dict(os.environ, PYTHONPATH=ROOT + os.pathsep + os.environ.get("PYTHONPATH", ""))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node=2",
           "--master-addr", "127.0.0.1", "--master-port", "29517",
           os.path.join(ROOT, "tests", "shard_worker.py"), str(out)]
    r = subprocess.run(cmd, capture_output=True, text=True, env=env, timeout=600, cwd=ROOT)
    assert r.returncode == 0, r.stdout[-3000:] + r.stderr[-3000:]
    from oracle.afqmc_oracle import AFQMCOracle
    d = np.load(out)
    cfg, h1, L, trial, walkers = inputs.make_problem_host("c1", nw=12)
    o = AFQMCOracle(h1, L, trial, cfg.n_alpha, cfg.n_beta, cfg.walker_kind, taylor_order=cfg.taylor_order)
    Wo, wo = walkers, np.ones(12)
    for s in range(int(d["steps"])):
        Wo, wo, ovo = o.step(Wo, wo, inputs.make_aux_fields(cfg, 0, s, 12), cfg.dt)
    Eo = o.local_energy(Wo)
    assert rel_fro(d["W"], Wo) < TOL_RUN
    assert rel_max(d["wt"], wo) < TOL_RUN
    sc = energy_scale(o, Wo, Eo)
    assert rel_max(d["E"][:, 0], Eo[:, 0], scale=sc) < TOL_RUN
