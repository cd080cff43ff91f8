"""CPU oracle for what sits between walker steps in a block: population control, the weighted
energy estimator, and the block loop itself.

TEST INFRASTRUCTURE ONLY (same rules as `afqmc_oracle.py`): only `tests/`,
`__graft_entry__.smoke()` and the `cpu_baseline` / `--impl reference` legs of `bench.py` may
import it; it shares no code with the CUDA library and imports nothing from it.

Source: /root/reference/PAPER.md.  The paper names the stages of a block — "wavefunction
propagation, stabilization, population control, and estimator calculation" —
prints the estimator (Code Snippet 9) and says that population control may be
done locally within one rank / one GPU.  It does not say WHICH population-control
algorithm; reading S21 takes the comb (stochastic reconfiguration with one uniform
random number per call), restated here from its definition:

    total weight W = sum_i w_i, spacing s = W / Nw, teeth t_k = (k + xi) s, k = 0..Nw-1,
    xi in [0, 1);  new walker k is a copy of the old walker i whose cumulative-weight interval
    [c_{i-1}, c_i) holds t_k  (c_i = w_0 + ... + w_i);  every new weight is s.

The random number xi is an INPUT (drawn on the host from a seed and fed identically to both
paths).  Floating point decides integers here (which interval a tooth falls in), so the rule is
fixed to the last bit: c is the sequential left-to-right float64 running sum, s = c[Nw-1] / Nw,
t_k = (k + xi) * s (one addition in float64 of the exactly representable k and xi, one
multiplication), and i_k = min(#{j : c_j <= t_k}, i_last) with i_last the first index whose c
equals the total (so a tooth that rounding pushes to the very end still lands on the last walker
that carries weight).  If W is not finite or not > 0 nothing is changed.

Pins (tests/test_oracle_pins.py): P14 (comb) and P15 (estimator, block loop).
"""
from __future__ import annotations

import numpy as np

__all__ = ["comb", "estimators", "run_block"]


def comb(weights, xi):
    """Population control by the comb.  Returns (map, new_weights): new walker k = old walker
    map[k]; map is int64 [Nw], non-decreasing.  ("population control", PAPER.md:185, 489;
    reading S21.)"""
    w = np.asarray(weights, dtype=np.float64)
    nw = w.shape[0]
    xi = float(xi)
    if not (0.0 <= xi < 1.0):
        raise ValueError("xi must be in [0, 1)")
    c = np.empty(nw, dtype=np.float64)
    s = 0.0
    for i in range(nw):                       # sequential running sum, left to right
        s = s + float(w[i])
        c[i] = s
    total = c[nw - 1]
    if not (np.isfinite(total) and total > 0.0):
        return np.arange(nw, dtype=np.int64), w.copy()
    spacing = total / nw
    i_last = 0
    while c[i_last] != total:
        i_last += 1
    m = np.empty(nw, dtype=np.int64)
    for k in range(nw):
        tooth = (float(k) + xi) * spacing
        i = 0
        while i < i_last and c[i] <= tooth:
            i += 1
        m[k] = i
    return m, np.full(nw, spacing, dtype=np.float64)


def estimators(weights, E):
    """Code Snippet 9 (`**` there is an extraction typo for `*`, reading S19):
    (ENumer, EDenom, E1Body, E2Body) = (sum w Re E[:,0], sum w, sum w Re E[:,1], sum w Re E[:,2]).
    The mixed estimate of the energy is ENumer / EDenom (Eq. 11 with Eq. 10's weights)."""
    w = np.asarray(weights, dtype=np.float64)
    E = np.asarray(E, dtype=np.complex128)
    return np.array([np.sum(w * E[:, 0].real), np.sum(w), np.sum(w * E[:, 1].real),
                     np.sum(w * E[:, 2].real)])


def run_block(oracle, walkers, weights, fields, xi, dt, pop_every):
    """One block (a block is a fixed number of steps followed by the
    estimators): for s = 1..n_steps: `step` (which re-orthonormalises on the oracle's own
    schedule), and after every pop_every-th step of the block the comb with the next xi; then
    the local energy of the walkers and the estimator sums.

    fields: [n_steps, Nw, n_chol]; xi: sequence with one entry per population-control call.
    Returns (walkers, weights, overlaps, E [Nw, 3], estimators [4], maps (list of int arrays))."""
    W = np.asarray(walkers, dtype=np.complex128)
    w = np.asarray(weights, dtype=np.float64)
    ov = None
    maps = []
    j = 0
    for s in range(fields.shape[0]):
        W, w, ov = oracle.step(W, w, fields[s], dt)
        if pop_every > 0 and (s + 1) % pop_every == 0:
            m, w = comb(w, xi[j])
            j += 1
            W = W[m]
            ov = ov[m]
            maps.append(m)
    E = oracle.local_energy(W)
    return W, w, ov, E, estimators(w, E), maps
