"""GPU parity: the CUDA path (through the C ABI, via the ctypes binding) against the CPU oracle,
element by element on the same seeded inputs.  Tolerances are BASELINE.json north_star's:
1e-10 relative per step (walkers re-seeded from the oracle each step), 1e-8 relative on
weights, overlaps and local energies after the stated number of free-running steps.
Setup quantities and single contractions are held to 1e-12."""
from __future__ import annotations

import numpy as np
import pytest

from paper_2406_16238_b200 import inputs
from tests.gpu_util import Pair, energy_scale, planar_to_complex, rel_fro, rel_max

pytestmark = pytest.mark.gpu

TOL_STAGE = 1e-12
TOL_STEP = 1e-10
TOL_RUN = 1e-8


def _torch():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    return torch


def gpu_step(pr, walkers, weights, x, dt):
    """One afqmc_step on device buffers; returns host copies (walkers, weights, overlaps)."""
    torch = _torch()
    W = torch.from_numpy(np.ascontiguousarray(walkers)).cuda()
    wt = torch.from_numpy(np.ascontiguousarray(weights)).cuda()
    xd = torch.from_numpy(np.ascontiguousarray(x)).cuda()
    ov = torch.empty(W.shape[0], dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    pr.gpu.step(W, wt, xd, dt)
    pr.gpu.get_overlaps(ov)
    pr.gpu.sync()
    return W.cpu().numpy(), wt.cpu().numpy(), ov.cpu().numpy()


def gpu_energy(pr, walkers):
    torch = _torch()
    W = torch.from_numpy(np.ascontiguousarray(walkers)).cuda()
    E = torch.empty((W.shape[0], 3), dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    pr.gpu.local_energy(W, E)
    pr.gpu.sync()
    return E.cpu().numpy()


# --------------------------------------------------------------------------- setup (row a0)
@pytest.mark.parametrize("name,nw,over", [("c1", 16, {}), ("c2", 8, {}),
                                          ("c1", 4, dict(M=37, n_alpha=7, n_beta=7, n_chol=53))])
def test_setup_quantities(name, nw, over):
    _torch()
    pr = Pair(name, nw=nw, **over)
    o, g, cfg = pr.oracle, pr.gpu, pr.cfg
    assert rel_max(g.debug_read(4), o.m, scale=np.abs(o.m).max()) < TOL_STAGE
    hm = g.debug_read(3).reshape(cfg.M, cfg.M)
    assert rel_fro(hm[None], o.h_mod[None]) < TOL_STAGE
    lr = g.debug_read(5).reshape(cfg.n_chol, cfg.Nt, cfg.M)
    lr_o = np.concatenate(o.Lrot, axis=1)
    assert rel_fro(lr[None], lr_o[None]) < TOL_STAGE
    c = g.constants()
    assert abs(c["E_const"] - o.E_const) <= TOL_STAGE * abs(o.E_const)
    assert abs(c["e_trial"] - o.e_shift) <= 1e-11 * abs(o.e_shift)
    # E1 = expm(-dt/2 h_mod): library = scaling-and-squaring Taylor, oracle = eigendecomposition
    gpu_step(pr, pr.walkers0, np.ones(pr.nw), pr.fields(0), cfg.dt)
    E1 = g.debug_read(2).reshape(cfg.M, cfg.M)
    assert rel_fro(E1[None], o.one_body_propagator(cfg.dt)[None]) < TOL_STAGE
    pr.close()


# --------------------------------------------------------------------------- stages a1-a9
@pytest.mark.parametrize("name,nw,over", [("c1", 16, {}), ("c2", 24, {}),
                                          ("c1", 5, dict(M=37, n_alpha=7, n_beta=7, n_chol=53)),
                                          ("c2", 3, dict(M=41, n_alpha=9, n_beta=1, n_chol=70))])
def test_one_step_stage_by_stage(name, nw, over):
    _torch()
    pr = Pair(name, nw=nw, ortho_every=0, **over)
    o, g, cfg = pr.oracle, pr.gpu, pr.cfg
    x = pr.fields(0)
    w0 = np.linspace(0.5, 1.5, nw)
    new_o, info = o.propagate(pr.walkers0, x, cfg.dt)
    Wg, wg, ovg = gpu_step(pr, pr.walkers0, w0, x, cfg.dt)
    X = planar_to_complex(g.debug_read(0), (nw, cfg.n_chol))
    assert rel_fro(X, info["X"]) < TOL_STAGE
    A = planar_to_complex(g.debug_read(1), (nw, cfg.M, cfg.M))
    assert rel_fro(A, info["A"]) < 1e-11
    assert rel_fro(Wg, new_o) < TOL_STEP
    o.n_steps_done = 0
    _, w_o, ov_o = o.step(pr.walkers0, w0, x, cfg.dt)
    assert rel_max(ovg, ov_o) < TOL_STEP
    assert rel_max(wg, w_o, scale=np.maximum(np.abs(w_o), 1e-3)) < TOL_STEP
    pr.close()


# --------------------------------------------------------------------------- local energy a11
@pytest.mark.parametrize("name,nw,over", [
    ("c1", 16, {}), ("c2", 24, {}),
    ("c1", 3, dict(M=37, n_alpha=7, n_beta=7, n_chol=53)),
    ("c2", 3, dict(M=41, n_alpha=9, n_beta=1, n_chol=70)),
    ("c1", 2, dict(M=70, n_alpha=24, n_beta=24, n_chol=40)),
    ("c1", 2, dict(M=70, n_alpha=33, n_beta=33, n_chol=41)),
    ("c1", 2, dict(M=90, n_alpha=42, n_beta=42, n_chol=39)),
    ("c1", 2, dict(M=90, n_alpha=50, n_beta=50, n_chol=37)),
    ("c1", 2, dict(M=80, n_alpha=64, n_beta=64, n_chol=21)),
    ("c2", 2, dict(M=80, n_alpha=57, n_beta=43, n_chol=21)),
])
def test_local_energy(name, nw, over):
    """Every exchange tile shape (occupied block 1..64 columns), odd M, ragged gamma groups."""
    _torch()
    pr = Pair(name, nw=nw, **over)
    E_o = pr.oracle.local_energy(pr.walkers0)
    E_g = gpu_energy(pr, pr.walkers0)
    sc = energy_scale(pr.oracle, pr.walkers0, E_o)
    for k in range(3):
        assert rel_max(E_g[:, k], E_o[:, k], scale=sc) < TOL_STAGE * 10
    pr.close()


# --------------------------------------------------------------------------- N steps
def _run(pr, steps, reseed):
    """Returns the worst per-step errors (walkers, weights, overlaps) and final states."""
    o, cfg, nw = pr.oracle, pr.cfg, pr.nw
    Wo, wo = pr.walkers0.copy(), np.ones(nw)
    Wg, wg = pr.walkers0.copy(), np.ones(nw)
    worst = dict(walkers=0.0, weights=0.0, ovlp=0.0)
    for s in range(steps):
        x = pr.fields(s)
        if reseed:
            Wg, wg = Wo.copy(), wo.copy()
        Wg, wg, ovg = gpu_step(pr, Wg, wg, x, cfg.dt)
        Wo, wo, ovo = o.step(Wo, wo, x, cfg.dt)
        worst["walkers"] = max(worst["walkers"], rel_fro(Wg, Wo))
        worst["weights"] = max(worst["weights"], rel_max(wg, wo, scale=np.maximum(np.abs(wo), 1e-3)))
        worst["ovlp"] = max(worst["ovlp"], rel_max(ovg, ovo))
    return worst, (Wg, wg, ovg), (Wo, wo, ovo)


@pytest.mark.parametrize("name,nw", [("c1", 16), ("c2", 64)])
def test_per_step_parity_reseeded(name, nw):
    _torch()
    pr = Pair(name, nw=nw)
    worst, _, _ = _run(pr, pr.cfg.steps, reseed=True)
    assert worst["walkers"] < TOL_STEP, worst
    assert worst["weights"] < TOL_STEP, worst
    assert worst["ovlp"] < TOL_STEP, worst
    pr.close()


@pytest.mark.parametrize("name,nw", [("c1", 16), ("c2", 640), ("c3", 16)])
def test_free_running_parity(name, nw):
    """The stated number of steps without re-seeding (c2: QR every 5 steps), then the local
    energy: weights, overlaps, energies to 1e-8."""
    _torch()
    pr = Pair(name, nw=nw)
    worst, (Wg, wg, ovg), (Wo, wo, ovo) = _run(pr, pr.cfg.steps, reseed=False)
    assert worst["weights"] < TOL_RUN, worst
    assert worst["ovlp"] < TOL_RUN, worst
    assert worst["walkers"] < TOL_RUN, worst
    assert np.all(wo > 0), "synthetic recipe should keep every walker alive"
    E_o = pr.oracle.local_energy(Wo)
    E_g = gpu_energy(pr, Wg)
    sc = energy_scale(pr.oracle, Wo, E_o)
    for k in range(3):
        assert rel_max(E_g[:, k], E_o[:, k], scale=sc) < TOL_RUN
    pr.close()


# --------------------------------------------------------------------------- the one-kernel path at its limits
@pytest.mark.parametrize("over,fused", [
    # the frontier of small_path_fits (hard limits M <= 64, block <= 16, Nt <= 32, n_chol <= 2048 AND a walker's
    # working set within 200 KB of shared memory): the largest M that still fits for each shape
    (dict(M=61, n_alpha=16, n_beta=16, n_chol=2048, walker_kind=0), True),      # widest RHF block, longest gamma loop
    (dict(M=47, n_alpha=16, n_beta=16, n_chol=2048, walker_kind=1), True),      # Nt = 32: widest Gauss-Jordan
    (dict(M=57, n_alpha=16, n_beta=3, n_chol=2047, walker_kind=1), True),       # odd n_chol: the direct-load branch
    (dict(M=64, n_alpha=5, n_beta=5, n_chol=96, walker_kind=0), True),          # largest M
    (dict(M=62, n_alpha=16, n_beta=16, n_chol=2048, walker_kind=0), False),     # one past the shared-memory frontier
    (dict(M=48, n_alpha=16, n_beta=16, n_chol=2048, walker_kind=1), False),     # the same for UHF
    (dict(M=66, n_alpha=5, n_beta=5, n_chol=96, walker_kind=0), False),         # past M
    (dict(M=64, n_alpha=17, n_beta=17, n_chol=96, walker_kind=0), False),       # one past the occupied block
    (dict(M=48, n_alpha=16, n_beta=16, n_chol=2050, walker_kind=0), False),     # past n_chol
])
def test_one_kernel_path_at_and_past_its_limits(over, fused):
    """fused_small.cu serves M <= 64, occupied blocks <= 16, Nt <= 32, n_chol <= 2048 as far as a walker's working
    set fits one CTA's shared memory (M = 64 only with narrow blocks; 16 columns at n_chol = 2048 up to M = 61, UHF
    16 + 16 up to M = 47).  At that frontier - the full-width warp-level Gauss-Jordan, the gamma-chunked
    staging of the energy kernel, the bulk-copy ring with many chunks - a step with QR and the local energy against
    the oracle; one past each limit the launch count shows that the multi-kernel path took over, same parity."""
    _torch()
    nw = 5
    pr = Pair("c1", nw=nw, ortho_every=1, **over)
    _run(pr, 1, reseed=True)                        # the first step also builds E1 = expm(-dt/2 h_mod): not counted
    pr.oracle.n_steps_done = 0
    l0 = pr.gpu.launch_count()
    worst, (Wg, wg, ovg), (Wo, wo, ovo) = _run(pr, 2, reseed=True)
    l1 = pr.gpu.launch_count()
    assert worst["walkers"] < TOL_STEP and worst["weights"] < TOL_STEP and worst["ovlp"] < TOL_STEP, worst
    per_step = (l1 - l0) / 2
    if fused:
        assert per_step <= 4, per_step               # the step kernel + the QR kernels
    else:
        assert per_step >= 10, per_step
    E_o = pr.oracle.local_energy(Wo)
    l2 = pr.gpu.launch_count()
    E_g = gpu_energy(pr, Wo)
    assert (pr.gpu.launch_count() - l2 == 1) == fused
    sc = energy_scale(pr.oracle, Wo, E_o)
    for k in range(3):
        assert rel_max(E_g[:, k], E_o[:, k], scale=sc) < TOL_STAGE * 10
    pr.close()


# --------------------------------------------------------------------------- stream-K where every walker is checked
@pytest.mark.parametrize("name,nw,over", [("c2", 640, {})])
def test_forced_stream_k_every_walker(name, nw, over):
    """The library switches stream-K on (gemm_ws.cu: tiles cut at chunk boundaries, first parts parked in global
    memory, cross-CTA flags) only where its cost rule expects a gain - c4 / c5, where the oracle can only check a few
    sampled walkers.  tuning_flags bit 0 forces it wherever the tile count leaves a partial wave: c2's 640 walkers
    (640 tiles of 7 k-steps on 148 SMs).  (c3's shape with 64 walkers was tried too: the forced handle returned the
    plain kernel's bits there, i.e. the launcher's other conditions kept stream-K off - not a case.)  Every walker, weight and
    overlap of two re-seeded steps against the oracle; against the unforced handle the walkers agree to rounding but
    NOT bit for bit (the cut tiles add their two parts in another order - which shows the forced path really ran);
    and 25 repeats of one step are bit-identical (fixed-order sums, no dependence on which CTA arrives first)."""
    _torch()
    pr = Pair(name, nw=nw, tuning_flags=1, ortho_every=0, **over)
    worst, _, _ = _run(pr, 2, reseed=True)
    assert worst["walkers"] < TOL_STEP and worst["weights"] < TOL_STEP and worst["ovlp"] < TOL_STEP, worst
    plain = Pair(name, nw=nw, oracle=False, ortho_every=0, **over)
    x, w0, dt = pr.fields(0), np.ones(nw), pr.cfg.dt
    Wf, wf, ovf = gpu_step(pr, pr.walkers0, w0, x, dt)
    Wp, wp, ovp = gpu_step(plain, pr.walkers0, w0, x, dt)
    assert rel_fro(Wf, Wp) < 1e-13 and rel_max(wf, wp) < 1e-12
    assert not np.array_equal(Wf, Wp), "forced stream-K gave the plain kernel's bits: it did not run"
    for _ in range(25):
        Wr, wr, ovr = gpu_step(pr, pr.walkers0, w0, x, dt)
        assert np.array_equal(Wr, Wf) and np.array_equal(wr, wf) and np.array_equal(ovr, ovf)
    plain.close()
    pr.close()


# --------------------------------------------------------------------------- the other kernel paths at even M
@pytest.mark.parametrize("path", [1, 2, 3])
@pytest.mark.parametrize("name,nw,over", [("c1", 16, {}), ("c2", 24, {}),
                                          ("c1", 3, dict(M=90, n_alpha=42, n_beta=42, n_chol=38))])
def test_kernel_paths_at_even_M(name, nw, over, path):
    """afqmc_params.kernel_path: 1 = the cp.async kernels (what odd M runs), 2 = the one-kernel overlap / Theta
    route, both at EVEN M where the default is the TMA path; 3 = the multi-kernel path for a system small enough for
    the one-kernel step / local energy that the default (0) picks (c1): a step with QR and the local energy against
    the oracle, and against the default path to rounding."""
    _torch()
    pr = Pair(name, nw=nw, ortho_every=1, kernel_path=path, **over)
    ref = Pair(name, nw=nw, ortho_every=1, oracle=False, **over)
    cfg = pr.cfg
    x = pr.fields(0)
    w0 = np.linspace(0.5, 1.5, nw)
    Wg, wg, ovg = gpu_step(pr, pr.walkers0, w0, x, cfg.dt)
    Wr, wr, ovr = gpu_step(ref, pr.walkers0, w0, x, cfg.dt)
    Wo, wo, ovo = pr.oracle.step(pr.walkers0, w0, x, cfg.dt)
    assert rel_fro(Wg, Wo) < TOL_STEP and rel_max(wg, wo) < TOL_STEP and rel_max(ovg, ovo) < TOL_STEP
    assert rel_fro(Wg, Wr) < 1e-12 and rel_max(wg, wr) < 1e-12
    E_o = pr.oracle.local_energy(Wo)
    sc = energy_scale(pr.oracle, Wo, E_o)
    E_g = gpu_energy(pr, Wo)
    for k in range(3):
        assert rel_max(E_g[:, k], E_o[:, k], scale=sc) < TOL_STAGE * 10
    pr.close()
    ref.close()


# --------------------------------------------------------------------------- random shapes
def _random_cases(n, seed):
    rng = np.random.default_rng(seed)
    out = []
    for _ in range(n):
        M = int(rng.integers(8, 150))
        uhf = bool(rng.integers(0, 2))
        na = int(rng.integers(1, min(60, M)))
        nb = int(rng.integers(1, na + 1)) if uhf else na
        nchol = int(rng.integers(3, 200))
        nw = int(rng.integers(1, 40))
        out.append(("c2" if uhf else "c1", nw, dict(M=M, n_alpha=na, n_beta=nb, n_chol=nchol)))
    return out


@pytest.mark.parametrize("name,nw,over", _random_cases(14, 20240611))
def test_random_shapes(name, nw, over):
    """Seeded random shapes (odd and even M and n_chol, RHF and UHF, 1..59 occupied columns): one step and the
    local energy, stage tolerances as above.  Odd M / n_chol take the cp.async kernels, even ones the TMA kernels."""
    _torch()
    pr = Pair(name, nw=nw, ortho_every=0, **over)
    o, g, cfg = pr.oracle, pr.gpu, pr.cfg
    x = pr.fields(0)
    w0 = np.linspace(0.5, 1.5, nw)
    new_o, info = o.propagate(pr.walkers0, x, cfg.dt)
    Wg, wg, ovg = gpu_step(pr, pr.walkers0, w0, x, cfg.dt)
    assert rel_fro(planar_to_complex(g.debug_read(0), (nw, cfg.n_chol)), info["X"]) < TOL_STAGE * 10
    assert rel_fro(planar_to_complex(g.debug_read(1), (nw, cfg.M, cfg.M)), info["A"]) < 1e-11
    assert rel_fro(Wg, new_o) < TOL_STEP
    _, w_o, ov_o = o.step(pr.walkers0, w0, x, cfg.dt)
    assert rel_max(ovg, ov_o) < TOL_STEP
    assert rel_max(wg, w_o, scale=np.maximum(np.abs(w_o), 1e-3)) < TOL_STEP
    E_o = o.local_energy(new_o)
    E_g = gpu_energy(pr, new_o)
    sc = energy_scale(o, new_o, E_o)
    for k in range(3):
        assert rel_max(E_g[:, k], E_o[:, k], scale=sc) < TOL_STAGE * 10
    pr.close()


# --------------------------------------------------------------------------- full sizes
@pytest.mark.parametrize("name,idx,device_L", [("c3", (0, 1, 2, 3, 64, 65, 127, 128, 129, 130, 191, 200, 252, 253, 254, 255), False),
                                               ("c4", (0, 77, 127), True),
                                               ("c5", (0, 37, 63), True)])
def test_full_size_sampled_walkers(name, idx, device_L):
    """BASELINE.json's full sizes in the launch configuration bench.py times (the whole batch of
    Nw walkers per call, same handle parameters), checked on SAMPLED walkers: walkers are
    independent given (h1, L, trial), so the oracle run on walkers `idx` alone gives exactly what
    it would give for them inside the full batch.  Per step (sampled walkers of a copy of the
    batch re-seeded from the oracle): 1e-10; free-running over the stated number of steps, then
    the local energy: 1e-8."""
    torch = _torch()
    pr = Pair(name, device_L=device_L)
    o, cfg, nw = pr.oracle, pr.cfg, pr.nw
    assert cfg.ortho_every == 0          # two GPU steps per oracle step below: keep QR out of it
    idx = np.asarray(idx)
    ti = torch.from_numpy(idx).cuda()
    Wg = torch.from_numpy(pr.walkers0).cuda()
    wg = torch.ones(nw, dtype=torch.float64, device="cuda")
    ov = torch.empty(nw, dtype=torch.complex128, device="cuda")
    Wo, wo = pr.walkers0[idx].copy(), np.ones(len(idx))
    step_err = dict(walkers=0.0, weights=0.0, ovlp=0.0)
    run_err = dict(walkers=0.0, weights=0.0, ovlp=0.0)

    def upd(d, W, w, v, Wref, wref, vref):
        d["walkers"] = max(d["walkers"], rel_fro(W, Wref))
        d["weights"] = max(d["weights"], rel_max(w, wref, scale=np.maximum(np.abs(wref), 1e-3)))
        d["ovlp"] = max(d["ovlp"], rel_max(v, vref))

    for s in range(cfg.steps):
        x = pr.fields(s)
        xd = torch.from_numpy(x).cuda()
        Wr, wr = Wg.clone(), wg.clone()
        Wr[ti] = torch.from_numpy(Wo).cuda()
        wr[ti] = torch.from_numpy(wo).cuda()
        torch.cuda.synchronize()          # the library runs on its own stream, torch on another
        pr.gpu.step(Wr, wr, xd, cfg.dt)
        pr.gpu.get_overlaps(ov)
        pr.gpu.sync()
        re_s = (Wr[ti].cpu().numpy(), wr[ti].cpu().numpy(), ov[ti].cpu().numpy())
        pr.gpu.step(Wg, wg, xd, cfg.dt)
        pr.gpu.get_overlaps(ov)
        pr.gpu.sync()
        Wo, wo, ovo = o.step(Wo, wo, x[idx], cfg.dt)
        upd(step_err, *re_s, Wo, wo, ovo)
        upd(run_err, Wg[ti].cpu().numpy(), wg[ti].cpu().numpy(), ov[ti].cpu().numpy(), Wo, wo, ovo)
        del Wr, wr
    assert max(step_err.values()) < TOL_STEP, step_err
    assert max(run_err.values()) < TOL_RUN, run_err
    assert np.all(wo > 0)
    assert bool(torch.all(torch.isfinite(wg))) and bool(torch.all(wg >= 0))
    E = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")
    torch.cuda.synchronize()
    pr.gpu.local_energy(Wg, E)
    pr.gpu.sync()
    E_g = E[ti].cpu().numpy()
    E_o = o.local_energy(Wo)
    sc = energy_scale(o, Wo, E_o)
    for k in range(3):
        assert rel_max(E_g[:, k], E_o[:, k], scale=sc) < TOL_RUN
    # every walker of the batch, not only the sampled ones, has a finite energy near the trial's
    Ea = E.cpu().numpy()
    assert np.all(np.isfinite(Ea.view(np.float64)))
    pr.close()


# --------------------------------------------------------------------------- packed Cholesky tensor
@pytest.mark.parametrize("name,nw,over", [("c1", 16, {}), ("c2", 24, {}),
                                          ("c1", 5, dict(M=70, n_alpha=9, n_beta=9, n_chol=54)),
                                          ("c1", 3, dict(M=130, n_alpha=12, n_beta=12, n_chol=50))])
def test_pack_chol_gives_the_same_bits_and_releases_L(name, nw, over):
    """pack_chol: the handle keeps a tile-packed copy of the upper triangles and no
    longer reads the caller's dense tensor after afqmc_create (it is overwritten with NaN here);
    steps and energies are bit-identical to the dense-tensor handle and match the oracle."""
    torch = _torch()
    dense = Pair(name, nw=nw, kernel_path=3, **over)      # the multi-kernel path also at c1 (same V_HS kernel as packed)
    packed = Pair(name, nw=nw, oracle=False, pack_chol=True, **over)
    packed.L_dev.fill_(float("nan"))
    torch.cuda.synchronize()
    cfg = dense.cfg
    Wd, wd = dense.walkers0.copy(), np.ones(nw)
    Wp, wp = dense.walkers0.copy(), np.ones(nw)
    Wo, wo = dense.walkers0.copy(), np.ones(nw)
    for s in range(3):
        x = dense.fields(s)
        Wd, wd, ovd = gpu_step(dense, Wd, wd, x, cfg.dt)
        Wp, wp, ovp = gpu_step(packed, Wp, wp, x, cfg.dt)
        assert np.array_equal(dense.gpu.debug_read(1), packed.gpu.debug_read(1))      # A = V_HS
        assert np.array_equal(Wd, Wp) and np.array_equal(wd, wp) and np.array_equal(ovd, ovp)
        Wo, wo, ovo = dense.oracle.step(Wo, wo, x, cfg.dt)
    assert rel_fro(Wp, Wo) < TOL_RUN and rel_max(wp, wo) < TOL_RUN and rel_max(ovp, ovo) < TOL_RUN
    assert np.array_equal(gpu_energy(dense, Wd), gpu_energy(packed, Wp))
    dense.close()
    packed.close()


def test_pack_chol_needs_even_dimensions():
    torch = _torch()
    from paper_2406_16238_b200 import afqmc
    with pytest.raises(afqmc.AfqmcError) as e:
        Pair("c1", nw=2, oracle=False, pack_chol=True, M=37, n_alpha=7, n_beta=7, n_chol=53)
    assert e.value.code == -6


# --------------------------------------------------------------------------- boundary behaviour
def test_host_pointers_equal_device_pointers():
    torch = _torch()
    pr = Pair("c1", nw=16, oracle=False)
    x = pr.fields(0)
    Wd, wd, ovd = gpu_step(pr, pr.walkers0, np.ones(16), x, pr.cfg.dt)
    Wh, wh = pr.walkers0.copy(), np.ones(16)
    pr.gpu.step(Wh, wh, x, pr.cfg.dt)
    ovh = np.empty(16, dtype=np.complex128)
    pr.gpu.get_overlaps(ovh)
    assert np.array_equal(Wh, Wd) and np.array_equal(wh, wd) and np.array_equal(ovh, ovd)
    Eh = np.empty((16, 3), dtype=np.complex128)
    pr.gpu.local_energy(Wh, Eh)
    assert np.array_equal(Eh, gpu_energy(pr, Wd))
    pr.close()


def test_fewer_walkers_than_max_and_single_walker():
    _torch()
    pr = Pair("c1", nw=16)
    x = pr.fields(0)
    Wa, wa, ova = gpu_step(pr, pr.walkers0, np.ones(16), x, pr.cfg.dt)
    for n in (1, 5):
        Wn, wn, ovn = gpu_step(pr, pr.walkers0[:n], np.ones(n), x[:n], pr.cfg.dt)
        assert rel_fro(Wn, Wa[:n]) < 1e-13 and rel_max(wn, wa[:n]) < 1e-13
        assert rel_max(gpu_energy(pr, Wn)[:, 0], gpu_energy(pr, Wa)[:n, 0]) < 1e-13
    pr.close()


def test_walker_equals_trial():
    """Overlap 1, E = trial energy, force bias zero: X = m."""
    _torch()
    pr = Pair("c1", nw=2)
    cfg = pr.cfg
    W = np.repeat(pr.trial[None].astype(np.complex128), 2, axis=0)
    E = gpu_energy(pr, W)
    c = pr.gpu.constants()
    assert np.max(np.abs(E[:, 0] - c["e_trial"])) < 1e-12 * abs(c["e_trial"])
    gpu_step(pr, W, np.ones(2), np.zeros((2, cfg.n_chol)), cfg.dt)
    X = planar_to_complex(pr.gpu.debug_read(0), (2, cfg.n_chol))
    assert np.max(np.abs(X - pr.oracle.m[None])) < 1e-12 * np.abs(pr.oracle.m).max()
    pr.close()


def test_dead_walkers_get_zero_weight():
    """Reading S10: zero overlap or cos(theta) <= 0 gives weight exactly 0, no error.  Every walker's weight is
    compared with the oracle's.  Walker 1 has an overlap that is pure rounding noise (1e-17): its ratio
    ovlp'/ovlp is defined by that noise, so only finiteness is comparable there; walker 4 has an EXACT zero overlap
    (a zero column: the pivot search finds an exactly zero column on both sides) and must give exactly 0 on both;
    walker 5 has a small but representable overlap (det O = 0.03, overlap 9e-4; its force bias is already 30 times
    the usual one and its weight jumps to ~1.5e3, |c_fb| = 4.9) and must agree to cond * eps.  (A walker with
    det O = 1e-6 is no test: its force bias is 1e6 times the usual one, Taylor-6 blows up to overlaps of 1e193
    and the oracle itself returns weight 0.)"""
    _torch()
    pr = Pair("c1", nw=6)
    cfg = pr.cfg
    W = pr.walkers0.copy()
    # walker 1: first column replaced by an unoccupied eigenvector of h1 -> overlap ~ rounding noise
    lam, v = np.linalg.eigh(pr.h1)
    W[1] = pr.trial.astype(np.complex128)
    W[1][:, 0] = v[:, cfg.M - 1]
    W[2] = np.nan
    W[4][:, 2] = 0.0
    W[5] = pr.trial.astype(np.complex128)
    W[5][:, 0] = v[:, cfg.M - 1] + 3e-2 * pr.trial[:, 0]
    x = pr.fields(0, nw=6)
    Wg, wg, ovg = gpu_step(pr, W, np.ones(6), x, cfg.dt)
    _, wo, ovo = pr.oracle.step(W, np.ones(6), x, cfg.dt)
    assert wg[2] == 0.0 and wo[2] == 0.0
    assert wg[4] == 0.0 and wo[4] == 0.0
    assert wg[0] > 0 and wg[3] > 0
    assert rel_max(wg[[0, 3]], wo[[0, 3]]) < TOL_STEP
    assert np.isfinite(wg[1]) and wg[1] >= 0.0 and np.isfinite(wo[1]) and wo[1] >= 0.0
    # cond(O) ~ 30 and xbar 30 times the usual one: 1e-10 per step times that amplification
    assert wo[5] > 100 and abs(wg[5] - wo[5]) < 1e-8 * wo[5], (wg[5], wo[5])
    assert abs(ovg[5] - ovo[5]) < 1e-9 * abs(ovo[5]), (ovg[5], ovo[5])
    pr.close()


# --------------------------------------------------------------------------- literal amplitudes (stress case)
def _literal_stress(xbar_bound=0.0, ehyb_bound=0.0):
    """SURVEY 8(d) R1 / BASELINE.md 5: c1 with BASELINE.json's LITERAL N(0,1) exp(-g/24) amplitudes (no global
    rescale).  ||A||_2 = 2..9, |xbar| up to 50, Taylor-6 is no exponential there and every weight is exactly 0
    by step 7 - but one step is still a deterministic map, so per-step parity (GPU re-seeded from the oracle
    each step) must hold to 1e-10 on walkers and overlaps, and the weights must agree INCLUDING the exact
    zeros of the phaseless cut: oracle zero => GPU zero unless |cos theta| < 1e-9 (SURVEY 8c "Parity metric").
    Tolerance of a non-zero weight: w' = w |e^{c_fb + c_mf} ovlp'/ovlp ...| and the exponential has condition number
    |c_fb| + |c_mf| (2.2e3 at step 7 here, where |xbar| reaches 50): 1e-10 relative on the exponent's terms is
    1e-10 max(1, |c_fb| + |c_mf|) relative on the weight."""
    _torch()
    pr = Pair("c1", literal=True, xbar_bound=xbar_bound, ehyb_bound=ehyb_bound)
    o, cfg, nw = pr.oracle, pr.cfg, pr.nw
    Wo, wo = pr.walkers0.copy(), np.ones(nw)
    zeros_seen = 0
    borderline = []
    stats = dict(xbar_hits=0, ehyb_hits=0, xbar_max=0.0)
    for s in range(cfg.steps):
        x = pr.fields(s)
        _, info = o.propagate(Wo, x, cfg.dt)
        nA = max(np.linalg.norm(info["A"][w], 2) for w in range(nw))
        if s == 0:
            assert nA > 1.5                                   # this IS the stress regime
        cos = info["S"].real / np.abs(info["S"])
        stats["xbar_max"] = max(stats["xbar_max"], float(np.abs(info["xbar"]).max()))
        if xbar_bound > 0:
            raw = 1j * np.sqrt(cfg.dt) * (info["X"] - o.m[None, :])
            stats["xbar_hits"] += int((np.abs(raw) > xbar_bound).sum())
        if ehyb_bound > 0:
            with np.errstate(all="ignore"):
                D = -np.log(np.abs(info["I"])) / cfg.dt
            stats["ehyb_hits"] += int((np.abs(D) > ehyb_bound).sum())
        w_in = wo.copy() if s > 0 else np.ones(nw)
        w_in = np.where(w_in > 0, w_in, 1.0)                  # keep every walker's weight rule exercised
        Wg, wg, ovg = gpu_step(pr, Wo, w_in, x, cfg.dt)
        o.n_steps_done = 0
        Wn, wn, ovn = o.step(Wo, w_in, x, cfg.dt)
        # Conditioning of the stress regime (values from the oracle): the blown-up walkers have nearly dependent
        # columns, cond(O) = cond(psi^T phi) grows from 1 to 3e6 over the ten steps.  Theta = phi O^-1 (hence xbar, A
        # and the propagated walker) amplifies FP64 rounding by cond(O_old), a determinant by cond of its matrix.
        # With 1e-14 (a hundred ulps) as the agreement of two FP64 evaluations in different summation orders the
        # bars are 1e-10 max(1, 1e-4 cond): the plain 1e-10 up to cond = 1e4.
        blk = slice(0, cfg.n_alpha)
        c_old = np.array([np.linalg.cond(pr.trial[:, blk].T @ Wo[k][:, blk]) for k in range(nw)])
        c_new = np.array([np.linalg.cond(pr.trial[:, blk].T @ Wn[k][:, blk]) for k in range(nw)])
        a_old = np.maximum(1.0, 1e-4 * c_old)
        a_new = np.maximum(1.0, 1e-4 * (c_old + c_new))
        dW = np.linalg.norm((Wg - Wn).reshape(nw, -1), axis=1) / np.linalg.norm(Wn.reshape(nw, -1), axis=1)
        assert np.all(dW < TOL_STEP * a_old), (s, dW.max(), c_old.max())
        assert np.all(np.abs(ovg - ovn) < TOL_STEP * a_new * np.abs(ovn)), (s, c_new.max())
        for k in range(nw):
            if abs(cos[k]) < 1e-9:
                borderline.append((s, k))
                continue
            if wn[k] == 0.0:
                assert wg[k] == 0.0, (s, k, wg[k], cos[k])
                zeros_seen += 1
            else:
                amp = max(1.0, abs(info["c_fb"][k]) + abs(info["c_mf"][k])) * a_new[k]
                assert abs(wg[k] - wn[k]) < TOL_STEP * amp * wn[k], (s, k, wg[k], wn[k], amp)
        _, wo, _ = Wn, wo * (wn / w_in), ovn
        Wo = Wn
    pr.close()
    assert not borderline, borderline
    return zeros_seen, wo, stats




def test_c1_literal_amplitudes():
    """The literal c1 inputs without bounds: see _literal_stress."""
    zeros_seen, wo, _ = _literal_stress()
    assert zeros_seen >= 10, zeros_seen                       # the phaseless cut really fired
    assert np.all(wo == 0.0)                                  # R1: all 16 walkers are dead by the last step


def test_bounds_trigger_on_literal_amplitudes():
    """SURVEY 8f NEXT-1 / DESIGN.md S8b (oracle pin P17): the optional force-bias and hybrid-energy bounds, on inputs
    where both DO trigger (literal c1 amplitudes: raw |xbar| up to 50, hybrid energies far outside +-sqrt(2/dt)).
    Same per-step parity as above; with the bounds the shifts stay <= 1 and the weights stay finite."""
    dt = 0.005
    zeros_seen, wo, st = _literal_stress(xbar_bound=1.0, ehyb_bound=float(np.sqrt(2.0 / dt)))
    assert st["xbar_hits"] > 50 and st["ehyb_hits"] > 5, st
    assert st["xbar_max"] <= 1.0 + 1e-12
    assert np.all(np.isfinite(wo))


@pytest.mark.parametrize("kernel_path", [0, 3])
def test_overflowed_importance_function_is_a_dead_walker_even_with_the_bound(kernel_path):
    """Reading S10 comes before reading S8b: a walker whose |I| is not finite (here exp(-dt (E_const - E_shift))
    overflows through an absurd caller-supplied E_shift) gets weight exactly 0; the hybrid-energy bound clips finite
    values only and must not turn inf into exp(dt b).  Both weight kernels (one-kernel step, kernel_path 0 at c1;
    weight_update_kernel, kernel_path 3) against the oracle, which judges isfinite(I) before it clips."""
    torch = _torch()
    from oracle.afqmc_oracle import AFQMCOracle
    from paper_2406_16238_b200 import afqmc
    cfg = inputs.get_config("c1")
    nw, dt = 6, cfg.dt
    h1 = inputs.make_h1(cfg, 0)
    trial = inputs.make_trial(cfg, h1, 0)
    L = inputs.make_L_host(cfg, 0, False)
    W0 = inputs.make_walkers(cfg, trial, 0, nw)
    x = inputs.make_aux_fields(cfg, 0, 0, nw)
    bound = float(np.sqrt(2.0 / dt))
    for e_shift, dead in ((1.0e6, True), (0.0, False)):           # dt * 1e6 = 5000 > log(DBL_MAX) = 709.8
        o = AFQMCOracle(h1, L, trial, cfg.n_alpha, cfg.n_beta, cfg.walker_kind, taylor_order=cfg.taylor_order,
                        e_shift=e_shift, ehyb_bound=bound)
        Ld = torch.from_numpy(L).cuda()
        g = afqmc.AFQMC(h1, Ld, trial, M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta, n_chol=cfg.n_chol,
                        max_walkers=nw, walker_kind=cfg.walker_kind, taylor_order=cfg.taylor_order,
                        e_shift=e_shift, ehyb_bound=bound, kernel_path=kernel_path)
        Wd = torch.from_numpy(W0.copy()).cuda()
        wd = torch.ones(nw, dtype=torch.float64, device="cuda")
        xd = torch.from_numpy(x).cuda()
        torch.cuda.synchronize()
        g.step(Wd, wd, xd, dt)
        g.sync()
        _, w_o, _ = o.step(W0, np.ones(nw), x, dt)
        w_g = wd.cpu().numpy()
        if dead:
            assert np.all(w_o == 0.0) and np.all(w_g == 0.0), (w_o, w_g)
        else:
            assert np.all(w_o > 0.0) and rel_max(w_g, w_o) < TOL_STEP
        g.close()


# --------------------------------------------------------------------------- every exchange-kernel instantiation
_INSTS = [(8, 5, 7, 3), (8, 7, 5, 3), (8, 6, 6, 3), (12, 4, 7, 3), (12, 7, 4, 3), (12, 5, 5, 3), (12, 5, 4, 3),
          (12, 4, 5, 3), (8, 5, 7, 7), (8, 7, 5, 7), (8, 6, 6, 7)]


@pytest.mark.parametrize("name,nw,over", [("c1", 7, dict(M=90, n_alpha=42, n_beta=42, n_chol=41)),
                                          ("c2", 9, dict(M=60, n_alpha=16, n_beta=14, n_chol=50)),
                                          ("c1", 5, dict(M=64, n_alpha=5, n_beta=5, n_chol=77))])
def test_every_exchange_plan_gives_the_same_energy(name, nw, over):
    """The local energy must not depend on the exchange kernel's tile plan (afqmc_exchange_plan_pin): for every
    instantiation (consumer warps, rectangle bound, epilogue warps), every warp grid and a spread of tile sizes -
    full and ragged tiles in both directions, one and several epilogue passes, compile-time and predicated warp
    rectangles - the energies equal the oracle's.  (The tuned plans of the configs only ever run a few of these.)"""
    _torch()
    from paper_2406_16238_b200 import afqmc
    base = Pair(name, nw=nw, **over)
    cfg, o = base.cfg, base.oracle
    W = base.walkers0
    E_o = o.local_energy(W)
    sc = energy_scale(o, W, E_o)
    base.close()
    blocks = [cfg.n_alpha] if cfg.walker_kind == 0 else [cfg.n_alpha, cfg.n_beta]
    tried = 0
    for (ncw, mi, ni, ew) in _INSTS:
        for wm in [d for d in range(1, ncw + 1) if ncw % d == 0]:
            for G, Wn in ((1, 1), (2, 3), (3, 2), (5, 4), (9, 7), (13, 2)):
                ok = [afqmc.exchange_plan_pin(ns, cfg.M, False, ncw, mi, ni, wm, G, Wn, ew) for ns in blocks]
                if not all(ok):
                    continue
                pr = Pair(name, nw=nw, oracle=False, kernel_path=3, **over)
                E_g = gpu_energy(pr, W)
                pr.close()
                for k in range(3):
                    assert rel_max(E_g[:, k], E_o[:, k], scale=sc) < TOL_STAGE * 10, (ncw, mi, ni, ew, wm, G, Wn, k)
                tried += 1
    assert tried >= 20, tried
    # a plan pinned AFTER a handle was created would make the kernel write another number of partial-sum rows than
    # the handle allocated and sums: the library refuses instead
    pr = Pair(name, nw=nw, oracle=False, kernel_path=3, **over)
    ns0 = blocks[0]
    _, before = afqmc.exchange_plan(ns0, cfg.M)
    G_now = int(before.split(" G ")[1].split()[0])
    for (ncw, mi, ni, ew) in _INSTS:
        done = False
        for wm in [d for d in range(1, ncw + 1) if ncw % d == 0]:
            if afqmc.exchange_plan_pin(ns0, cfg.M, False, ncw, mi, ni, wm, 1 if G_now != 1 else 2, 1, ew):
                done = True
                break
        if done:
            break
    assert done
    with pytest.raises(afqmc.AfqmcError):
        gpu_energy(pr, W)
    pr.close()
    # leave no pinned plan behind: later tests in this process get the library's own plans, whatever the order
    afqmc.exchange_plan_unpin()
    pr = Pair(name, nw=nw, oracle=False, kernel_path=3, **over)
    E_g = gpu_energy(pr, W)
    pr.close()
    for k in range(3):
        assert rel_max(E_g[:, k], E_o[:, k], scale=sc) < TOL_STAGE * 10, k


# --------------------------------------------------------------------------- a10 on ill-conditioned walkers
def _reortho_gpu(pr, W):
    torch = _torch()
    Wd = torch.from_numpy(np.ascontiguousarray(W)).cuda()
    nblk = 1 if pr.cfg.walker_kind == 0 else 2
    dR = torch.empty((W.shape[0], nblk), dtype=torch.float64, device="cuda")
    torch.cuda.synchronize()
    pr.gpu.reorthonormalise(Wd, dR)
    pr.gpu.sync()
    return Wd.cpu().numpy(), dR.cpu().numpy()


def _check_qr(pr, W, Q, dR, kappa):
    """Q against the definition (orthonormal, same span, R = Q^H phi upper triangular with a real positive diagonal)
    to rounding, and against the oracle's Householder QR to the FORWARD accuracy the factorisation allows: Q and R of
    a matrix with condition number kappa are only determined to ~kappa * eps by ANY backward-stable algorithm, so the
    1e-10 of the well-conditioned case widens to max(1e-10, 50 kappa eps)."""
    cfg = pr.cfg
    blocks = [(0, cfg.n_alpha)] if cfg.walker_kind == 0 else [(0, cfg.n_alpha), (cfg.n_alpha, cfg.n_alpha + cfg.n_beta)]
    Qo, detRo = pr.oracle.reorthonormalise(W)
    tol = max(1e-10, 50 * kappa * 2.2e-16)
    for w in range(W.shape[0]):
        for b, (a0, a1) in enumerate(blocks):
            q, phi = Q[w][:, a0:a1], W[w][:, a0:a1]
            n = a1 - a0
            assert np.abs(q.conj().T @ q - np.eye(n)).max() < 1e-13
            R = q.conj().T @ phi
            assert np.linalg.norm(phi - q @ R) < 1e-13 * np.linalg.norm(phi)
            assert np.abs(np.tril(R, -1)).max() < 1e-13 * np.abs(R).max()
            d = np.diag(R)
            assert np.all(d.real > 0) and np.abs(d.imag).max() < 1e-13 * np.abs(R).max()
            assert abs(np.prod(d.real) / dR[w, b] - 1.0) < tol * 10
            assert np.linalg.norm(q - Qo[w][:, a0:a1]) < tol * np.sqrt(n)
        det_g = dR[w, 0] ** 2 if cfg.walker_kind == 0 else dR[w, 0] * dR[w, 1]
        assert abs(det_g / detRo[w] - 1.0) < tol * 20


@pytest.mark.parametrize("name,nw", [("c1", 6), ("c2", 6)])
@pytest.mark.parametrize("kappa", [1e4, 1e8, 1e12])
def test_reortho_ill_conditioned(name, nw, kappa):
    """Row a10 on walkers with nearly parallel columns: phi = U diag(sigma) V^H with singular
    values from 1 down to 1 / kappa.  Cholesky-QR alone breaks down at kappa ~ 1e8 (Gram matrix not positive
    definite in FP64); the kernel's shifted pass must take over (and only then)."""
    _torch()
    pr = Pair(name, nw=nw)
    cfg = pr.cfg
    r = np.random.default_rng(int(np.log10(kappa)))
    W = np.empty((nw, cfg.M, cfg.Nt), dtype=np.complex128)
    blocks = [(0, cfg.n_alpha)] if cfg.walker_kind == 0 else [(0, cfg.n_alpha), (cfg.n_alpha, cfg.n_alpha + cfg.n_beta)]
    for w in range(nw):
        for a0, a1 in blocks:
            n = a1 - a0
            U = np.linalg.qr(r.standard_normal((cfg.M, n)) + 1j * r.standard_normal((cfg.M, n)))[0]
            V = np.linalg.qr(r.standard_normal((n, n)) + 1j * r.standard_normal((n, n)))[0]
            sig = kappa ** (-np.arange(n) / (n - 1.0))
            W[w][:, a0:a1] = (U * sig) @ V.conj().T
    n0 = pr.gpu.qr_shifted_passes()
    Q, dR = _reortho_gpu(pr, W)
    _check_qr(pr, W, Q, dR, kappa)
    shifted = pr.gpu.qr_shifted_passes() - n0
    assert (shifted == 0) if kappa <= 1e4 else (shifted >= nw), shifted
    pr.close()


def test_reortho_after_long_free_projection():
    """300 c1 steps without any re-orthonormalisation, then ONE QR: the library against the oracle's QR of the very
    same walkers; the stored overlaps are divided by (det R)^2 and must equal the overlaps recomputed from Q."""
    torch = _torch()
    pr = Pair("c1", ortho_every=0)
    cfg, nw = pr.cfg, pr.nw
    Wd = torch.from_numpy(pr.walkers0.copy()).cuda()
    wd = torch.ones(nw, dtype=torch.float64, device="cuda")
    for s in range(300):
        xd = torch.from_numpy(pr.fields(s)).cuda()
        torch.cuda.synchronize()
        pr.gpu.step(Wd, wd, xd, cfg.dt)
    pr.gpu.sync()
    W = Wd.cpu().numpy()
    assert np.all(np.isfinite(W))
    kappa = max(np.linalg.cond(W[k]) for k in range(nw))
    dR = torch.empty((nw, 1), dtype=torch.float64, device="cuda")
    ov = torch.empty(nw, dtype=torch.complex128, device="cuda")
    pr.gpu.reorthonormalise(Wd, dR)
    pr.gpu.get_overlaps(ov)
    pr.gpu.sync()
    Q = Wd.cpu().numpy()
    _check_qr(pr, W, Q, dR.cpu().numpy(), kappa)
    assert rel_max(ov.cpu().numpy(), pr.oracle.overlap(Q)) < 1e-10 * max(1.0, 1e-4 * kappa)
    pr.close()


def test_error_codes():
    torch = _torch()
    from paper_2406_16238_b200 import afqmc, inputs
    cfg = inputs.get_config("c1")
    h1 = inputs.make_h1(cfg)
    tr = inputs.make_trial(cfg, h1)
    Lh = inputs.make_L_host(cfg)
    Ld = torch.from_numpy(Lh).cuda()
    kw = dict(M=cfg.M, n_alpha=5, n_beta=5, n_chol=cfg.n_chol, max_walkers=4, walker_kind=0)

    def code(**over):
        args = dict(kw)
        L = over.pop("L", Ld)
        t = over.pop("trial", tr)
        args.update(over)
        with pytest.raises(afqmc.AfqmcError) as e:
            afqmc.AFQMC(h1, L, t, **args)
        return e.value.code

    assert code(n_beta=4) == -2
    assert code(taylor_order=17) == -6
    assert code(L=Lh) == -1
    assert code(trial=tr * 1.001) == -5
    assert code(n_alpha=cfg.M + 1, n_beta=cfg.M + 1) == -2
    g = afqmc.AFQMC(h1, Ld, tr, **kw)
    W = torch.zeros((5, cfg.M, 5), dtype=torch.complex128, device="cuda")
    with pytest.raises(afqmc.AfqmcError) as e:
        g.step(W, torch.ones(5, dtype=torch.float64, device="cuda"),
               torch.zeros((5, cfg.n_chol), dtype=torch.float64, device="cuda"), 0.005)
    assert e.value.code == -2
    with pytest.raises(afqmc.AfqmcError) as e:
        g.step(W[:2], torch.ones(2, dtype=torch.float64, device="cuda"),
               torch.zeros((2, cfg.n_chol), dtype=torch.float64, device="cuda"), -1.0)
    assert e.value.code == -1
    g.close()
