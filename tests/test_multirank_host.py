"""N > 1 host logic of bench.py (replicas only, no data-path collective)
on CPU with the gloo backend, world_size 2: every rank gets the slowest rank's time, the job value
counts all replicas, replicas draw different walkers/fields but the same Hamiltonian, and the
reference arm runs on rank 0 only."""
from __future__ import annotations

import os
import socket
import subprocess
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))

WORKER = r"""
import os, sys, json
sys.path.insert(0, {root!r})
import torch.distributed as dist
import bench
from paper_2406_16238_b200 import inputs
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
ms = [120.0, 80.0][rank]
tmax = bench.max_over_ranks(ms, dist, "cpu")
cfg = inputs.get_config("c1")
seed = bench.replica_seed(rank)
h1 = inputs.make_h1(cfg, 0)
tr = inputs.make_trial(cfg, h1, 0)
W = inputs.make_walkers(cfg, tr, seed, 4)
x = inputs.make_aux_fields(cfg, seed, 0, 4)
out = dict(rank=rank, world=world, tmax=tmax, value=bench.job_value(world, 16, 5, tmax),
           h1=float(h1.sum()), w=float(abs(W).sum()), x=float(x.sum()))
dist.barrier()
print("RESULT " + json.dumps(out), flush=True)
dist.destroy_process_group()
"""


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def test_world_size_2_gloo(tmp_path):
    import json
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
        line = [l for l in out.splitlines() if l.startswith("RESULT ")][0]
        d = json.loads(line[7:])
        res[d["rank"]] = d
    assert res[0]["world"] == res[1]["world"] == 2
    assert res[0]["tmax"] == res[1]["tmax"] == 120.0          # slowest rank decides
    assert np.isclose(res[0]["value"], 2 * 16 * 5 / 0.120)    # whole-job aggregate, weak scaling
    assert res[0]["h1"] == res[1]["h1"]                        # same Hamiltonian
    assert res[0]["w"] != res[1]["w"] and res[0]["x"] != res[1]["x"]   # own walkers and fields


def test_reference_arm_runs_on_rank_0_only():
    """`bench.py --impl reference` under torchrun: ranks > 0 exit 0 without work or output."""
    env = dict(os.environ, RANK="1", LOCAL_RANK="1", WORLD_SIZE="2", MASTER_ADDR="127.0.0.1",
               MASTER_PORT=str(_free_port()))
    r = subprocess.run([sys.executable, os.path.join(ROOT, "bench.py"), "--impl", "reference", "--gpus", "2",
                        "--workload", "c1", "--steps", "1", "--warmup", "0"], env=env, capture_output=True,
                       text=True, timeout=300)
    assert r.returncode == 0, r.stderr[-2000:]
    assert r.stdout.strip() == ""
