"""Helpers shared by the GPU parity tests: build one problem for BOTH sides from the seeded
generators (paper_2406_16238_b200.inputs), create the CUDA handle and the oracle, and the
comparison metrics of DESIGN.md "Parity metric".  No method arithmetic lives here."""
from __future__ import annotations

import numpy as np

from paper_2406_16238_b200 import inputs


def rel_fro(a, b):
    """max over the leading (walker) axis of ||a - b||_F / ||b||_F."""
    a = np.asarray(a)
    b = np.asarray(b)
    n = a.shape[0]
    d = np.linalg.norm((a - b).reshape(n, -1), axis=1)
    s = np.linalg.norm(b.reshape(n, -1), axis=1)
    return float(np.max(d / np.maximum(s, 1e-300)))


def rel_max(a, b, scale=None):
    a = np.asarray(a)
    b = np.asarray(b)
    s = np.abs(b) if scale is None else np.asarray(scale)
    return float(np.max(np.abs(a - b) / np.maximum(s, 1e-300)))


def planar_to_complex(buf, shape):
    """[nw][2][...] planar doubles -> complex [nw][...]."""
    nw = shape[0]
    p = np.asarray(buf).reshape(nw, 2, *shape[1:])
    return p[:, 0] + 1j * p[:, 1]


class Pair:
    """One synthetic problem on both sides.  `L_dev` is the device tensor the library borrows;
    the oracle gets either the very same host array or a slab provider over the device tensor."""

    def __init__(self, name, nw=None, seed=0, device_L=False, literal=False, oracle=True,
                 ortho_every=None, pack_chol=False, kernel_path=0, xbar_bound=0.0, ehyb_bound=0.0, tuning_flags=0, **overrides):
        import torch
        from oracle.afqmc_oracle import AFQMCOracle
        from paper_2406_16238_b200 import afqmc

        cfg = inputs.get_config(name, **overrides)
        self.cfg = cfg
        self.nw = cfg.nw if nw is None else nw
        self.seed = seed
        self.h1 = inputs.make_h1(cfg, seed)
        self.trial = inputs.make_trial(cfg, self.h1, seed)
        if device_L:
            self.L_dev = inputs.make_L_device(cfg, seed, literal=literal)
            L_for_oracle = inputs.device_slab_provider(self.L_dev)
        else:
            L_host = inputs.make_L_host(cfg, seed, literal)
            self.L_dev = torch.from_numpy(L_host).cuda()
            L_for_oracle = L_host
        oe = cfg.ortho_every if ortho_every is None else ortho_every
        self.gpu = afqmc.AFQMC(self.h1, self.L_dev, self.trial, M=cfg.M, n_alpha=cfg.n_alpha,
                               n_beta=cfg.n_beta, n_chol=cfg.n_chol, max_walkers=self.nw,
                               walker_kind=cfg.walker_kind, taylor_order=cfg.taylor_order,
                               ortho_every=oe, pack_chol=pack_chol, kernel_path=kernel_path,
                               xbar_bound=xbar_bound, ehyb_bound=ehyb_bound, tuning_flags=tuning_flags)
        self.oracle = None
        if oracle:
            self.oracle = AFQMCOracle(self.h1, L_for_oracle, self.trial, cfg.n_alpha, cfg.n_beta,
                                      cfg.walker_kind, taylor_order=cfg.taylor_order,
                                      ortho_every=oe, xbar_bound=xbar_bound, ehyb_bound=ehyb_bound)
        self.walkers0 = inputs.make_walkers(cfg, self.trial, seed, self.nw)

    def fields(self, step, nw=None):
        return inputs.make_aux_fields(self.cfg, self.seed, step, self.nw if nw is None else nw)

    def close(self):
        self.gpu.close()
        self.L_dev = None


def energy_scale(o, walkers, E):
    """|E1b| + |E_C| + |E_X| per walker (E_C and E_X cancel heavily)."""
    X = o.force_bias_X(o.theta(walkers))
    ec = 0.5 * np.sum(X * X, axis=1)
    ex = E[:, 2] - ec
    return np.abs(E[:, 1]) + np.abs(ec) + np.abs(ex)
