"""CPU check of the arithmetic claim behind the mixed-precision kernels (vhs_tc.cu / taylor_tc.cu, DESIGN.md
section 5): a double split into three bfloat16 numbers h + m + l keeps 24 significant bits, and the six
partial products of order <= 2 (hh, hm, mh, hl, lh, mm), each exact in FP32, reproduce the product of two
such numbers to ~2^-23.  The bfloat16 rounding is emulated on float32 bit patterns (round to nearest even),
the same operation as __float2bfloat16_rn; nothing here touches the CUDA path or the oracle."""
from __future__ import annotations

import numpy as np


def bf16_rn(x):
    """float32 array -> nearest bfloat16 (ties to even), returned as float32."""
    u = np.asarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32)


def split3(x):
    x = np.asarray(x, dtype=np.float64)
    h = bf16_rn(x.astype(np.float32))
    r1 = x - h.astype(np.float64)
    m = bf16_rn(r1.astype(np.float32))
    r2 = r1 - m.astype(np.float64)
    l = bf16_rn(r2.astype(np.float32))
    return h, m, l


def test_three_bfloat16_keep_24_bits():
    rng = np.random.default_rng(0)
    x = rng.standard_normal(200000) * np.exp(rng.uniform(-20, 20, 200000))
    h, m, l = split3(x)
    err = np.abs(x - (h.astype(np.float64) + m + l)) / np.abs(x)
    assert err.max() <= 2.0 ** -24
    # each plane is a bfloat16 number (8 significant bits): the lower 16 bits of its float32 pattern are zero
    for p in (h, m, l):
        assert not np.any(p.view(np.uint32) & 0xFFFF)
    # the planes decay by ~2^-8 each (what makes dropping ml, lm, ll a 2^-24 effect)
    assert np.median(np.abs(m) / np.abs(h)) < 2.0 ** -8 and np.median(np.abs(l) / np.abs(h)) < 2.0 ** -16


def test_six_plane_pairs_reproduce_the_product():
    rng = np.random.default_rng(1)
    a = rng.standard_normal(100000)
    b = rng.standard_normal(100000)
    ah, am, al = (p.astype(np.float64) for p in split3(a))
    bh, bm, bl = (p.astype(np.float64) for p in split3(b))
    six = ah * bh + ah * bm + am * bh + ah * bl + al * bh + am * bm
    err = np.abs(six - a * b) / np.abs(a * b)
    assert err.max() < 2.0 ** -22
    # every bf16 x bf16 product has at most 16 significant bits: exact in float32
    for u, v in ((ah, bh), (am, bm), (al, bh)):
        assert np.array_equal((u.astype(np.float32) * v.astype(np.float32)).astype(np.float64), u * v)


def test_a_float32_is_exactly_three_bfloat16():
    """What the Taylor epilogue relies on when it writes the next term's planes from an FP32 value."""
    rng = np.random.default_rng(2)
    t = (rng.standard_normal(100000) * np.exp(rng.uniform(-10, 10, 100000))).astype(np.float32)
    h = bf16_rn(t)
    r1 = t - h
    m = bf16_rn(r1)
    l = bf16_rn(r1 - m)
    assert np.array_equal(h.astype(np.float64) + m + l, t.astype(np.float64))
