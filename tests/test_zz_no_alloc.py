"""afqmc_comb_static - the population-control comb for callers that cannot allocate device memory.

Who they are: a driver that resamples walkers but owns no afqmc_handle (afqmc_create cudaMallocs the workspaces of
the whole step), or one that runs when the GPU has no memory left to hand out (the Cholesky tensor and the
application's memory pool hold all of it, so cudaMalloc fails), or one that cannot afford the device-wide stall of a
cudaMalloc / cudaFree while its other streams are busy.  For them the comb's scratch - the running sum of the
weights - is a fixed 512 KiB array inside libafqmc.so, and the entry point takes only the caller's inputs and outputs.

The GPU test holds the new entry point to the existing handle path (afqmc_population_control): resampling map
bit-equal (index work) and new weights bit-equal, on calls issued back to back without any clearing in between -
every call shares the one array, which still holds the previous call's sums.  This file sorts last on purpose:
`pytest -x` stops at the first failure, and a failure here must not hide the parity tests.  It passes alone in a fresh
process (first use of the array on the device) and after the other tests (library already in use)."""
from __future__ import annotations

import ctypes as C

import numpy as np
import pytest


def _weight_cases(nw, seed):
    r = np.random.default_rng(1000 * seed + nw)
    w = r.uniform(0.05, 3.0, nw) ** 2
    wz = w.copy()
    wz[r.choice(nw, max(1, nw // 8), replace=False)] = 0.0
    ws = np.zeros(nw)
    ws[nw // 2] = 2.5
    wn = w.copy()
    wn[0] = np.nan
    return [("random", w), ("with dead walkers", wz), ("equal", np.full(nw, 0.7)), ("one survivor", ws),
            ("all dead", np.zeros(nw)), ("nan", wn), ("wide range", np.exp(r.uniform(-30, 3, nw)))]


def test_sizes_beyond_the_array_are_refused_without_a_device():
    """The argument checks come before any CUDA call: a batch that does not fit the built-in array is refused with a
    message that names the limit, not truncated or run out of bounds."""
    from paper_2406_16238_b200 import afqmc
    lib = afqmc.lib
    buf = C.create_string_buffer(512)
    dummy = np.zeros(4)
    p = dummy.ctypes.data
    assert lib.afqmc_comb_static(p, p, p, afqmc.COMB_STATIC_MAX_WALKERS + 1, None, buf, len(buf)) == -2
    assert b"65536" in buf.value and b"65537" in buf.value
    assert lib.afqmc_comb_static(p, p, p, 0, None, buf, len(buf)) == -2
    assert lib.afqmc_comb_static(None, p, p, 4, None, buf, len(buf)) == -1
    assert b"null" in buf.value
    assert lib.afqmc_comb_static(p, p, p, afqmc.COMB_STATIC_MAX_WALKERS + 1, None, None, 0) == -2   # err is optional


@pytest.mark.gpu
def test_comb_static_matches_the_handle_path_on_consecutive_calls():
    """Two (and more) calls in a row, sizes going down and up again so that the array always holds a longer, stale
    running sum from the call before: map and weights equal afqmc_population_control's to the last bit, for the
    degenerate weight vectors too (dead walkers, all dead, NaN: identity map and untouched weights)."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2406_16238_b200 import afqmc
    from oracle.block_oracle import comb
    from tests.gpu_util import Pair

    sizes = [640, 77, 640, 1, 16, 333]
    pr = Pair("c1", nw=max(sizes), oracle=False)          # the existing path: a handle with its own workspaces
    cfg = pr.cfg
    row = cfg.M * (cfg.n_alpha if cfg.walker_kind == 0 else cfg.n_alpha + cfg.n_beta)
    stream = torch.cuda.Stream()
    n_calls = 0
    for rep, nw in enumerate(sizes):
        for label, w in _weight_cases(nw, rep):
            for xi in (0.0, 0.637, np.nextafter(1.0, 0.0)):
                # existing path (runs on the handle's own stream; host pointers are staged and synchronised inside)
                w_ref = w.copy()
                m_ref = np.empty(nw, dtype=np.int32)
                W = np.zeros((nw, row), dtype=np.complex128)
                pr.gpu.population_control(W, w_ref, np.array([xi]), m_ref, nw=nw)
                # new entry point: device inputs and outputs only, nothing else
                wd = torch.from_numpy(w.copy()).cuda()
                xid = torch.tensor([xi], dtype=torch.float64, device="cuda")
                md = torch.full((nw,), -7, dtype=torch.int32, device="cuda")
                torch.cuda.synchronize()
                with torch.cuda.stream(stream):
                    afqmc.comb_static(wd, xid, md, stream=stream.cuda_stream)
                stream.synchronize()
                n_calls += 1
                assert np.array_equal(md.cpu().numpy(), m_ref), (nw, label, xi)
                assert np.array_equal(wd.cpu().numpy(), w_ref, equal_nan=True), (nw, label, xi)
                if nw <= 77:                              # and the oracle's comb, where its Python loops are quick
                    m_o, w_o = comb(w, xi)
                    assert np.array_equal(md.cpu().numpy().astype(np.int64), m_o), (nw, label, xi)
                    assert np.array_equal(wd.cpu().numpy(), w_o, equal_nan=True), (nw, label, xi)
    assert n_calls >= 2

    # back to back on one stream with no host synchronisation in between: the second call must not see the first's sums
    wa = np.exp(np.random.default_rng(5).uniform(-3, 3, 500))
    wb = np.random.default_rng(6).uniform(0.1, 1.0, 200)
    ref = []
    for w in (wa, wb):
        w_ref, m_ref = w.copy(), np.empty(len(w), dtype=np.int32)
        pr.gpu.population_control(np.zeros((len(w), row), dtype=np.complex128), w_ref, np.array([0.3]), m_ref,
                                  nw=len(w))
        ref.append((m_ref, w_ref))
    xid = torch.tensor([0.3], dtype=torch.float64, device="cuda")
    da, db = torch.from_numpy(wa.copy()).cuda(), torch.from_numpy(wb.copy()).cuda()
    ma = torch.empty(500, dtype=torch.int32, device="cuda")
    mb = torch.empty(200, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    afqmc.comb_static(da, xid, ma, stream=stream.cuda_stream)
    afqmc.comb_static(db, xid, mb, stream=stream.cuda_stream)
    stream.synchronize()
    for (m_ref, w_ref), m, w in zip(ref, (ma, mb), (da, db)):
        assert np.array_equal(m.cpu().numpy(), m_ref)
        assert np.array_equal(w.cpu().numpy(), w_ref)

    # the default stream (stream = NULL) and the largest batch the array holds
    nmax = afqmc.COMB_STATIC_MAX_WALKERS
    wl = torch.rand(nmax, dtype=torch.float64, device="cuda") + 0.01
    wl_host = wl.cpu().numpy().copy()
    ml = torch.empty(nmax, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()
    afqmc.comb_static(wl, xid, ml)
    torch.cuda.synchronize()
    m = ml.cpu().numpy().astype(np.int64)
    cum = np.cumsum(wl_host)                      # sequential float64 sum, as the kernel's
    total = cum[-1]
    assert np.all(np.diff(m) >= 0) and m[0] >= 0 and m[-1] < nmax
    teeth = (np.arange(nmax) + 0.3) * (total / nmax)
    assert np.array_equal(m, np.minimum(np.searchsorted(cum, teeth, side="right"), nmax - 1))
    assert np.all(wl.cpu().numpy() == total / nmax)

    # host memory is refused (the entry point stages nothing), and so is a batch beyond the array
    with pytest.raises(afqmc.AfqmcError):
        afqmc.comb_static(np.ones(4), xid, ma)
    with pytest.raises(afqmc.AfqmcError, match="65536"):
        afqmc.comb_static(wl, xid, ml, nw=nmax + 1)
    pr.close()
