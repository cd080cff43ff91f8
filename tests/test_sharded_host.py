"""Host logic of the distributed-Hamiltonian drivers (paper_2406_16238_b200/sharded.py) on CPU:
the gamma partition and the routing of the auxiliary fields to the member that holds the matching
slice, in one process and across world_size-2 gloo ranks.  No device is needed."""
from __future__ import annotations

import json
import os
import socket
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _sharded():
    import __graft_entry__ as ge
    ge.build()
    from paper_2406_16238_b200 import sharded
    return sharded


@pytest.mark.parametrize("n,G", [(96, 2), (96, 3), (54, 4), (4800, 8), (70, 2), (16, 8)])
def test_gamma_slices_partition(n, G):
    sl = _sharded().gamma_slices(n, G)
    assert len(sl) == G and sl[0][0] == 0 and sl[-1][1] == n
    for (a, b), (c, d) in zip(sl, sl[1:]):
        assert b == c
    sizes = [b - a for a, b in sl]
    assert all(s > 0 and s % 2 == 0 for s in sizes)
    assert max(sizes) - min(sizes) <= 2


def test_gamma_slices_rejects_bad_input():
    sh = _sharded()
    for n, G in [(95, 2), (6, 4), (10, 0)]:
        with pytest.raises(ValueError):
            sh.gamma_slices(n, G)


def test_fields_for_member_is_the_column_block_of_the_group_batch():
    sh = _sharded()
    rng = np.random.default_rng(0)
    G, nw, n = 3, 5, 24
    x = rng.standard_normal((G * nw, n))
    per_owner = [x[r * nw:(r + 1) * nw] for r in range(G)]
    for a, b in sh.gamma_slices(n, G):
        got = sh.fields_for_member(per_owner, (a, b)).numpy()
        assert np.array_equal(got, x[:, a:b])


WORKER = r"""
import sys, json
sys.path.insert(0, {root!r})
import numpy as np, torch, torch.distributed as dist
from paper_2406_16238_b200 import sharded
dist.init_process_group("gloo")
rank, G = dist.get_rank(), dist.get_world_size()
nw, n = 4, 20
x = np.random.default_rng(7).standard_normal((G * nw, n))          # the whole group's fields
slices = sharded.gamma_slices(n, G)
mine = torch.from_numpy(np.ascontiguousarray(x[rank * nw:(rank + 1) * nw]))
got = sharded.exchange_fields(mine, slices).numpy()
a, b = slices[rank]
ok = bool(np.array_equal(got, x[:, a:b]))
# setup sums: all-reduce gives every member the same bits
part = torch.from_numpy(np.random.default_rng(rank).standard_normal(9))
dist.all_reduce(part)
print("RESULT " + json.dumps(dict(rank=rank, ok=ok, shape=list(got.shape), s=part.numpy().tolist())), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_exchange_fields_world_size_2_gloo(tmp_path):
    _sharded()
    script = tmp_path / "worker.py"
    script.write_text(WORKER.format(root=ROOT))
    port = _free_port()
    procs = []
    for r in range(2):
        env = dict(os.environ, RANK=str(r), LOCAL_RANK=str(r), WORLD_SIZE="2",
                   MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
        procs.append(subprocess.Popen([sys.executable, str(script)], env=env, stdout=subprocess.PIPE,
                                      stderr=subprocess.PIPE, text=True))
    res = {}
    for p in procs:
        out, err = p.communicate(timeout=300)
        assert p.returncode == 0, err[-2000:]
        d = json.loads([l for l in out.splitlines() if l.startswith("RESULT ")][0][7:])
        res[d["rank"]] = d
    assert res[0]["ok"] and res[1]["ok"]
    assert res[0]["shape"] == [8, 10] and res[1]["shape"] == [8, 10]
    assert res[0]["s"] == res[1]["s"]
