"""CPU-side checks of the boundary: the library builds, loads, exports every symbol that
include/afqmc.h declares, the ctypes struct matches the C struct, and argument validation
that needs no device works.  No compute calls here."""
from __future__ import annotations

import ctypes as C
import os
import re
import subprocess

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "afqmc.h")


def _declared():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(afqmc_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import __graft_entry__ as ge
    ge.build()
    from paper_2406_16238_b200 import afqmc
    names = _declared()
    assert len(names) >= 10
    for n in names:
        assert hasattr(afqmc.lib, n), n
    assert sorted(afqmc.EXPORTS) == names


def test_params_struct_layout_matches_c(tmp_path):
    """sizeof and the offset of EVERY field of afqmc_params, as gcc lays the header's struct out, against the
    ctypes mirror (same names, same order)."""
    from paper_2406_16238_b200 import afqmc
    P = afqmc.AfqmcParams
    names = [f[0] for f in P._fields_]
    hdr = re.sub(r"/\*.*?\*/", "", open(HEADER).read(), flags=re.S)
    body = hdr[hdr.index("typedef struct {"):hdr.index("} afqmc_params;")]
    assert re.findall(r"\b(\w+);", body) == names
    src = tmp_path / "sz.c"
    offs = ", ".join(f"offsetof(afqmc_params, {n})" for n in names)
    src.write_text('#include <stdio.h>\n#include <stddef.h>\n#include "afqmc.h"\n'
                   'int main(){size_t v[] = {sizeof(afqmc_params), ' + offs + '};\n'
                   'for (unsigned i = 0; i < sizeof(v) / sizeof(v[0]); ++i) printf("%zu ", v[i]);return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()
    assert [int(v) for v in out] == [C.sizeof(P)] + [getattr(P, n).offset for n in names]


def test_header_is_plain_c():
    r = subprocess.run(["gcc", "-std=c99", "-pedantic", "-Werror", "-fsyntax-only", "-x", "c", HEADER],
                       capture_output=True, text=True)
    assert r.returncode == 0, r.stderr


def test_null_and_bad_arguments_are_rejected_without_a_device():
    from paper_2406_16238_b200 import afqmc
    lib = afqmc.lib
    h = C.c_void_p()
    p = afqmc.AfqmcParams()
    assert lib.afqmc_create(None, None, None, C.byref(p), C.byref(h)) == -1
    a = np.zeros(4)
    p.struct_size = 3
    assert lib.afqmc_create(a.ctypes.data, a.ctypes.data, a.ctypes.data, C.byref(p), C.byref(h)) == -1
    assert b"struct_size" in lib.afqmc_last_error(None)
    assert lib.afqmc_step(None, None, None, None, 0.005, 1) == -1
    assert lib.afqmc_local_energy(None, None, None, 1) == -1
    assert lib.afqmc_sync(None) == -1
    assert lib.afqmc_launch_count(None) == -1
    lib.afqmc_destroy(None)


def test_no_cpu_fallback_in_the_product_path():
    """The package never imports or executes anything under oracle/."""
    pk = os.path.join(ROOT, "paper_2406_16238_b200")
    pat = re.compile(r"^\s*(from|import)\s+oracle\b|oracle[./]afqmc_oracle", re.M)
    for d, _, fs in os.walk(pk):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(d, f)).read()), f


def test_library_reads_no_environment_variables():
    """The kernel path is chosen by afqmc_params.kernel_path only: a user's environment cannot change it."""
    pk = os.path.join(ROOT, "paper_2406_16238_b200", "csrc")
    for f in os.listdir(pk):
        assert "getenv" not in open(os.path.join(pk, f)).read(), f


def test_shard_setup_reduce_adds_in_member_order():
    """afqmc_shard_setup_reduce is a plain host loop (no device): left-to-right sum over the members."""
    from paper_2406_16238_b200 import afqmc
    r = np.random.default_rng(3)
    parts = r.standard_normal((5, 11)) * 10.0 ** r.integers(-8, 8, size=(5, 11))
    out = afqmc.AFQMC.shard_setup_reduce(parts)
    ref = parts[0].copy()
    for k in range(1, 5):
        ref = ref + parts[k]
    assert np.array_equal(out, ref)
    assert afqmc.lib.afqmc_shard_setup_reduce(None, 2, 3, None) == -1


def test_exchange_plan_exists_for_every_block_size():
    """Host logic of the exchange kernel's tile plan (exchange_ws.cu: make_plan): every occupied-block size the
    library accepts (1..64), short and long K loops, real and pair mode gets a plan that fits shared memory and wastes
    less than half of the issued DMMA blocks; the shapes of BASELINE.json's configs take their tuned entries."""
    from paper_2406_16238_b200 import afqmc
    for pair in (False, True):
        for M in (64, 108, 300, 1200):
            for ns in range(1, 65):
                if ns > M:
                    continue
                eff, desc = afqmc.exchange_plan(ns, M, pair)
                smem = int(re.search(r"smem (\d+)", desc).group(1))
                assert 0.5 < eff <= 1.0 + 1e-9, (ns, M, pair, desc)
                assert smem <= 232448, (ns, M, pair, desc)
    assert "warps 12+3" in afqmc.exchange_plan(42, 1200)[1] and "tile 126x168" in afqmc.exchange_plan(42, 1200)[1]
    assert "warps 8+7" in afqmc.exchange_plan(50, 300)[1] and "tile 150x100" in afqmc.exchange_plan(50, 300)[1]
    assert "warps 8+7" in afqmc.exchange_plan(16, 108)[1]
    # pinning: a candidate that cannot exist is refused, one that exists replaces the plan
    own = afqmc.exchange_plan(50, 302)[1]
    own2 = afqmc.exchange_plan(42, 90)[1]
    assert not afqmc.exchange_plan_pin(50, 300, False, 12, 4, 7, 4, 30, 30)
    assert afqmc.exchange_plan_pin(50, 302, False, 12, 4, 7, 6, 3, 1)
    assert "grid 6x2" in afqmc.exchange_plan(50, 302)[1] and "grid 6x2" not in own
    # ... and unpinning gives the library's own choice back (nothing pinned is left behind for later tests)
    afqmc.exchange_plan_unpin(50, 302)
    assert afqmc.exchange_plan(50, 302)[1] == own
    assert afqmc.exchange_plan_pin(50, 302, False, 12, 4, 7, 6, 3, 1)
    assert any(afqmc.exchange_plan_pin(42, 90, False, 12, 4, 7, wm, 1, 1) for wm in (1, 2, 3, 4, 6, 12))
    assert afqmc.exchange_plan(42, 90)[1] != own2
    afqmc.exchange_plan_unpin()                               # ns = 0: every pin
    assert afqmc.exchange_plan(42, 90)[1] == own2 and afqmc.exchange_plan(50, 302)[1] == own
    assert afqmc.lib.afqmc_exchange_plan_unpin(65, 100, 0) == -1
