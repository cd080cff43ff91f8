"""Seeded synthetic inputs shaped like the paper's molecules.

This module serves BOTH the CUDA path and the oracle (tests/bench hand its arrays to
each).  It holds none of the method's arithmetic: only random draws, symmetrisation,
one analytic amplitude factor, an eigen/QR call for the trial orbitals.  It imports
neither `oracle/` nor the CUDA binding.

The paper's workloads are molecules (benzene dimer, [Cu2O2]2+) whose
integrals are not available; BASELINE.json's five configs take their shapes.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

__all__ = ["Config", "CONFIGS", "get_config", "make_h1", "make_trial", "make_walkers",
           "make_aux_fields", "make_pop_uniforms", "chol_scale", "make_L_slab", "make_L_host", "make_L_device",
           "device_slab_provider", "make_problem_host"]


@dataclass(frozen=True)
class Config:
    name: str
    M: int
    n_alpha: int
    n_beta: int
    n_chol: int
    nw: int
    walker_kind: int      # 0 RHF restricted walkers, 1 UHF [alpha|beta]
    decay: float          # s_g = exp(-g / decay)
    steps: int
    ortho_every: int
    trial: str            # "eig" (lowest eigenvectors of h1) or "qr" (QR of random blocks)
    dt: float = 0.005
    taylor_order: int = 6

    @property
    def Nt(self):
        return self.n_alpha if self.walker_kind == 0 else self.n_alpha + self.n_beta


# BASELINE.json `configs`, in order.
CONFIGS = {
    "c1": Config("c1", 24, 5, 5, 96, 16, 0, 24.0, 10, 0, "eig"),
    "c2": Config("c2", 108, 16, 14, 540, 640, 1, 100.0, 20, 5, "qr"),
    "c3": Config("c3", 300, 50, 50, 1500, 256, 0, 300.0, 10, 0, "eig"),
    "c4": Config("c4", 700, 40, 40, 3500, 128, 0, 700.0, 5, 0, "eig"),
    "c5": Config("c5", 1200, 42, 42, 4800, 64, 0, 960.0, 3, 0, "eig"),
}


def get_config(name, **overrides):
    c = CONFIGS[name]
    if overrides:
        d = {f: getattr(c, f) for f in c.__dataclass_fields__}
        d.update(overrides)
        c = Config(**d)
    return c


def _rng(seed, stream, sub=0):
    return np.random.Generator(np.random.Philox(key=[int(seed) * 4096 + int(stream), int(sub)]))


def _sym_from_upper(g):
    """Mirror the upper triangle (incl. diagonal) of the last two axes: exactly symmetric."""
    u = np.triu(g)
    return u + np.swapaxes(np.triu(g, 1), -1, -2)


def make_h1(cfg, seed=0):
    """h1: upper triangle ~ N(0, std 0.5) mirrored, plus diag(linspace(-2, 0, M))."""
    g = _rng(seed, 1).standard_normal((cfg.M, cfg.M)) * 0.5
    return _sym_from_upper(g) + np.diag(np.linspace(-2.0, 0.0, cfg.M))


def make_trial(cfg, h1, seed=0):
    """[M, Nt] real orthonormal columns, alpha block first."""
    if cfg.trial == "eig":
        _, v = np.linalg.eigh(h1)
        blocks = [v[:, :cfg.n_alpha]]
        if cfg.walker_kind == 1:
            blocks.append(v[:, :cfg.n_beta])
    else:
        r = _rng(seed, 2)
        na = r.standard_normal((cfg.M, cfg.n_alpha))
        blocks = [np.linalg.qr(na)[0]]
        if cfg.walker_kind == 1:
            nb = r.standard_normal((cfg.M, cfg.n_beta))
            blocks.append(np.linalg.qr(nb)[0])
    return np.ascontiguousarray(np.concatenate(blocks, axis=1))


def make_walkers(cfg, trial, seed=0, nw=None, noise=1e-2):
    """[nw, M, Nt] complex128 = trial + noise * (N(0,1) + i N(0,1)), independent per walker."""
    nw = cfg.nw if nw is None else nw
    r = _rng(seed, 3)
    pert = r.standard_normal((nw, cfg.M, cfg.Nt)) + 1j * r.standard_normal((nw, cfg.M, cfg.Nt))
    return np.ascontiguousarray(trial[None].astype(np.complex128) + noise * pert)


def make_aux_fields(cfg, seed, step, nw=None):
    """x[w, g] ~ N(0, 1) float64 for one step; host-drawn, fed identically to both paths."""
    nw = cfg.nw if nw is None else nw
    return _rng(seed, 1000, step).standard_normal((nw, cfg.n_chol))


def make_pop_uniforms(seed, n, block=0):
    """xi[j] ~ U[0, 1) float64, one per population-control call of a block; host-drawn, fed
    identically to both paths (the library draws no random numbers)."""
    return _rng(seed, 2000, block).random(n)


def chol_scale(cfg, literal=False):
    """One global factor c so that E[sum_g (c s_g G_g)^2] = c^2 M sum_g s_g^2 * 1 = 10 * 1
    (G_g symmetric with unit-variance entries).  This is DESIGN.md reading R1: BASELINE's
    amplitudes fix the profile over g, the global scale is fixed analytically so that
    ||A||_2 ~ 2 sqrt(10 dt) ~ 0.45.  literal=True returns 1 (the stress case)."""
    if literal:
        return 1.0
    s2 = np.exp(-2.0 * np.arange(cfg.n_chol) / cfg.decay).sum()
    return float(np.sqrt(10.0 / (cfg.M * s2)))


def make_L_slab(cfg, seed, g0, g1, literal=False):
    """Host recipe: L[g] = c * exp(-g/decay) * sym(N(0,1)), one Philox stream per g."""
    c = chol_scale(cfg, literal)
    out = np.empty((g1 - g0, cfg.M, cfg.M))
    for g in range(g0, g1):
        gm = _rng(seed, 7, g).standard_normal((cfg.M, cfg.M))
        out[g - g0] = _sym_from_upper(gm) * (c * np.exp(-g / cfg.decay))
    return out


def make_L_host(cfg, seed=0, literal=False):
    return make_L_slab(cfg, seed, 0, cfg.n_chol, literal)


def make_L_device(cfg, seed=0, device="cuda", slab=32, literal=False):
    """Device recipe for the large configs (13.7 GB / 55 GB): same distribution and
    profile as the host recipe, drawn with torch's device generator slab by slab (the
    VALUES differ from the host recipe; a test that uses this hands the oracle a copy
    of these very slabs through `device_slab_provider`)."""
    import torch
    c = chol_scale(cfg, literal)
    M = cfg.M
    L = torch.empty((cfg.n_chol, M, M), dtype=torch.float64, device=device)
    gen = torch.Generator(device=device)
    for g0 in range(0, cfg.n_chol, slab):
        g1 = min(cfg.n_chol, g0 + slab)
        gen.manual_seed(int(seed) * 1000003 + g0)
        g = torch.randn((g1 - g0, M, M), dtype=torch.float64, device=device, generator=gen)
        u = torch.triu(g)
        s = u + torch.triu(g, 1).transpose(-1, -2)
        amp = c * torch.exp(-torch.arange(g0, g1, dtype=torch.float64, device=device) / cfg.decay)
        L[g0:g1] = s * amp[:, None, None]
        del g, u, s
    return L


def device_slab_provider(L_dev, slab=64):
    """Zero-argument callable yielding (g0, host ndarray) copies of a device tensor."""
    def it():
        n = L_dev.shape[0]
        for g0 in range(0, n, slab):
            yield g0, L_dev[g0:g0 + slab].cpu().numpy()
    return it


def make_problem_host(name, seed=0, nw=None, literal=False, **overrides):
    """Everything for the small configs on the host: (cfg, h1, L, trial, walkers)."""
    cfg = get_config(name, **overrides)
    h1 = make_h1(cfg, seed)
    L = make_L_host(cfg, seed, literal)
    trial = make_trial(cfg, h1, seed)
    walkers = make_walkers(cfg, trial, seed, nw)
    return cfg, h1, L, trial, walkers


def make_complex_problem(M, n_alpha, n_beta, n_pairs, walker_kind, seed=0, nw=4, noise=1e-2, complex_trial=False):
    """Complex Cholesky vectors: complex Hermitian h1, vectors {C_k, C_k^+} (a set closed under
    the adjoint factorises a (ps|qr) = (qr|ps) symmetric tensor), k < n_pairs, i.e. n_chol = 2 n_pairs vectors and
    4 n_pairs auxiliary fields; real trial = lowest eigenvectors of Re h1 (complex_trial: complex128 lowest
    eigenvectors of the Hermitian h1 itself); walkers = trial + complex noise.  The amplitude follows
    reading R1: E[sum_g |L_g|^2] such that ||A||_2 ~ 0.4 at dt = 0.005.
    Returns (h1, L [2 n_pairs, M, M] complex, trial [M, Nt], walkers [nw, M, Nt])."""
    r = _rng(seed, 11)
    h = (r.standard_normal((M, M)) + 1j * r.standard_normal((M, M))) * 0.35
    h = 0.5 * (h + h.conj().T) + np.diag(np.linspace(-2.0, 0.0, M))
    amp = np.sqrt(10.0 / (M * 4.0 * n_pairs))
    C = (r.standard_normal((n_pairs, M, M)) + 1j * r.standard_normal((n_pairs, M, M))) * amp
    L = np.ascontiguousarray(np.concatenate([C, C.conj().transpose(0, 2, 1)], axis=0))
    _, v = np.linalg.eigh(h if complex_trial else h.real)   # lowest eigenvectors (as c1's recipe)
    blocks = [v[:, :n_alpha]]
    if walker_kind == 1:
        blocks.append(v[:, :n_beta])
    trial = np.ascontiguousarray(np.concatenate(blocks, axis=1))
    Nt = trial.shape[1]
    pert = r.standard_normal((nw, M, Nt)) + 1j * r.standard_normal((nw, M, Nt))
    walkers = np.ascontiguousarray(trial[None].astype(np.complex128) + noise * pert)
    return np.ascontiguousarray(h), L, trial, walkers


def make_complex_fields(seed, step, nw, n_fields):
    return _rng(seed, 1100, step).standard_normal((nw, n_fields))
