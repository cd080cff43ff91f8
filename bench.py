"""bench.py - walker-steps/s of the ph-AFQMC hot path (one step = afqmc_step + afqmc_local_energy
over one batch of Nw synthetic walkers) on B200, with the roofline of the dominant kernel and
the CPU oracle timed beside it.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload c5] [--impl reference]

Multi-GPU (torchrun, one rank per GPU): replicas only - every rank holds its own copy of the
Hamiltonian and its own Nw walkers, no data-path collective; the value
is N * Nw * K / max-over-ranks time, scaling "weak".

Timed region of `value`: inputs resident in HBM (walkers, weights, all aux fields pre-staged),
K x (afqmc_step, afqmc_local_energy) on one stream, CUDA events on that stream.  `e2e`: the
same K steps through the same C-ABI calls with pinned HOST buffers (the library stages H2D /
D2H inside each call).  The Cholesky tensor (13.7 GB at c4, 55 GB at c5) is far larger than the
126 MB L2, so no explicit L2 flush is needed between iterations (config.l2: "inputs > L2").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "walker-steps/s (propagate + local energy)"
UNIT = "walker-steps/s"


def ncu_traffic(workload, stage):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of a stage's kernel from profiles/ncu_traffic.json
    (one `ncu --set full` capture per entry; the file names the capture and the commit it was taken on), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            e = json.load(f).get(f"{workload}:{stage}")
        return None if e is None else {"bytes": e["bytes"], "capture": e.get("capture"), "commit": e.get("commit")}
    except (OSError, ValueError, KeyError):
        return None


def flops_model(cfg, nw, complex_fields=0):
    """Algorithmic real FP64 flops per launch of each contraction stage.
    complex_fields > 0: complex Cholesky vectors with that many Hermitian matrices (complex x complex products,
    8 real flops per multiply-add; the exchange stage runs ONE pass over the two planes of Lrot)."""
    M, ng, K = cfg.M, cfg.n_chol, cfg.taylor_order
    blocks = [cfg.n_alpha] if cfg.walker_kind == 0 else [cfg.n_alpha, cfg.n_beta]
    Nt = sum(blocks)
    if complex_fields:
        nf = complex_fields
        return {
            "exchange": nw * sum(8.0 * nf * ns * ns * M + 8.0 * nf * ns * ns for ns in blocks),
            # two runs of the symmetric-half kernel: Re planes (symmetric sum), Im planes (antisymmetric sum)
            "vhs": nw * 4.0 * nf * M * (M + 1),
            "taylor": nw * 8.0 * K * M * M * Nt,
            "force_bias": nw * 8.0 * nf * Nt * M,
            "one_body": 2 * nw * 8.0 * M * M * Nt,
        }
    return {
        "exchange": nw * sum(4.0 * ng * ns * ns * M + 8.0 * ng * ns * ns for ns in blocks),
        # symmetric half of A only (L_g = L_g^T; SURVEY 8a row a5 "packed-symmetric minimum")
        "vhs": nw * 2.0 * ng * M * (M + 1),
        "vhs_dense_equivalent": nw * 4.0 * ng * M * M,
        "taylor": nw * 8.0 * K * M * M * Nt,
        "force_bias": nw * 4.0 * ng * Nt * M,
        "one_body": 2 * nw * 4.0 * M * M * Nt,
    }


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "200"],
                                      stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            pass

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        rows = [r.split(",") for r in self.f.read().strip().splitlines() if r.count(",") >= 6]
        self.f.close()
        os.unlink(self.f.name)
        if not rows:
            return out
        sm = [float(r[0]) for r in rows]
        out["sm_mhz"] = float(np.median(sm))
        out["sm_max_mhz"] = float(rows[0][1])
        out["power_w_max"] = max(float(r[2]) for r in rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        out["reasons"] = [n for i, n in enumerate(names) if any("Not" not in r[3 + i] for r in rows)]
        out["samples"] = len(rows)
        return out


def oracle_sample(cfg, h1, L_host, trial, nw_s, steps, warmup, seed=0):
    """Times the oracle as it stands on `nw_s` walkers: `steps` x (step + local energy).
    Returns (walker-steps/s, seconds per sample step, threads)."""
    from oracle.afqmc_oracle import AFQMCOracle
    from paper_2406_16238_b200 import inputs
    o = AFQMCOracle(h1, L_host, trial, cfg.n_alpha, cfg.n_beta, cfg.walker_kind,
                    taylor_order=cfg.taylor_order, ortho_every=cfg.ortho_every)
    W = inputs.make_walkers(cfg, trial, seed, nw_s)
    wt = np.ones(nw_s)
    ts = []
    for s in range(warmup + steps):
        x = inputs.make_aux_fields(cfg, seed, s, nw_s)
        t0 = time.perf_counter()
        W, wt, _ = o.step(W, wt, x, cfg.dt)
        o.local_energy(W)
        ts.append(time.perf_counter() - t0)
    t = float(np.sum(ts[warmup:]))
    try:
        import threadpoolctl
        thr = max([p["num_threads"] for p in threadpoolctl.threadpool_info()] + [1])
    except Exception:
        thr = os.cpu_count()
    return nw_s * steps / t, t / steps, thr


def sample_walkers(cfg):
    """Bounded oracle sample: about 10-30 s of CPU work per bench run."""
    return {"c1": 16, "c2": 64, "c3": 8, "c4": 4, "c5": 4}.get(cfg.name, 4)


def make_L(cfg, seed, want_host, want_dev):
    """(L_dev or None, L_host or None): host recipe for small configs, device recipe beyond 1 GB."""
    import torch
    from paper_2406_16238_b200 import inputs
    big = cfg.n_chol * cfg.M * cfg.M * 8 > (1 << 30)
    if big and torch.cuda.is_available():
        Ld = inputs.make_L_device(cfg, seed)
        Lh = Ld.cpu().numpy() if want_host else None
        return (Ld if want_dev else None), Lh
    Lh = inputs.make_L_host(cfg, seed)
    Ld = torch.from_numpy(Lh).cuda() if want_dev else None
    return Ld, (Lh if want_host else None)


def time_blocks(g, cfg, stream, walkers_h, seed, nw, reps, n_steps=25, pop_every=5):
    """Secondary figure: afqmc_run_block = 25 steps with the comb every 5 steps, the
    handle's QR schedule, ONE local energy + estimator sums per block.  Timed eagerly and as the
    CUDA-graph replay (third call on with the same buffers).  Every block restarts from the same
    walkers (the reset copy is outside the event bracket)."""
    import torch
    from paper_2406_16238_b200 import inputs
    with torch.cuda.stream(stream):
        W0 = torch.from_numpy(walkers_h).cuda()
        W = torch.empty_like(W0)
        w = torch.empty(nw, dtype=torch.float64, device="cuda")
        x = torch.from_numpy(np.stack([inputs.make_aux_fields(cfg, seed, 1000 + s, nw)
                                       for s in range(n_steps)])).cuda()
        xi = torch.from_numpy(inputs.make_pop_uniforms(seed, n_steps // pop_every)).cuda()
        E = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")
        est = torch.empty(4, dtype=torch.float64, device="cuda")

        def run(n, timed):
            tot = 0.0
            for _ in range(n):
                W.copy_(W0)
                w.fill_(1.0)
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(stream)
                g.run_block(W, w, x, xi, cfg.dt, pop_every, E, est)
                e1.record(stream)
                torch.cuda.synchronize()
                tot += e0.elapsed_time(e1)
            return tot / n if timed else None

        l0 = g.launch_count()
        g.set_block_graph(0)
        run(1, False)
        l_block = g.launch_count() - l0
        ms_eager = run(reps, True)
        est_eager = est.cpu().numpy().copy()
        r0 = g.set_block_graph(1)
        run(2, False)                      # eager (key first seen) + capture
        ms_graph = run(reps, True)
        replays = g.set_block_graph(-1) - r0
        est_graph = est.cpu().numpy()
    return {"steps_per_block": n_steps, "pop_every": pop_every, "ortho_every": cfg.ortho_every,
            "local_energy": "once per block", "launches_per_block": int(l_block),
            "ms_per_block_eager": ms_eager, "ms_per_block_graph": ms_graph,
            "walker_steps_per_s": nw * n_steps / (ms_graph * 1e-3), "graph_launches": int(replays),
            "E_mixed": float(est_graph[0] / est_graph[1]),
            "graph_equals_eager": bool(np.array_equal(est_eager, est_graph))}


def time_sharded(cfg, h1, Ld, trial, G, K, Wm, seed):
    """Secondary figure (--group G): the distributed-Hamiltonian route with all G
    members on THIS one GPU, each holding a gamma slice of the same tensor (views, no copy) and
    Nw / G walkers, so the group does the same work as the plain step.  A phase is issued member
    after member on the members' own streams (their persistent kernels share the SMs; no kernel
    waits on another), barriers are stream synchronisations; the figure is the cost of the slot
    traffic and the owner-side sums, not of NVLink."""
    import torch
    from paper_2406_16238_b200 import inputs, sharded
    nw = cfg.nw // G
    slices = sharded.gamma_slices(cfg.n_chol, G)
    grp = sharded.LocalGroup(h1, [Ld[a:b] for a, b in slices], trial, M=cfg.M, n_alpha=cfg.n_alpha,
                             n_beta=cfg.n_beta, max_walkers=nw, walker_kind=cfg.walker_kind,
                             taylor_order=cfg.taylor_order, ortho_every=cfg.ortho_every)
    walkers = inputs.make_walkers(cfg, trial, seed, G * nw)
    W = [torch.from_numpy(np.ascontiguousarray(walkers[r * nw:(r + 1) * nw])).cuda() for r in range(G)]
    wt = [torch.ones(nw, dtype=torch.float64, device="cuda") for _ in range(G)]
    E = [torch.empty((nw, 3), dtype=torch.complex128, device="cuda") for _ in range(G)]
    xs = []
    for s in range(Wm + K):
        x = inputs.make_aux_fields(cfg, seed, s, G * nw)
        xs.append([torch.from_numpy(np.ascontiguousarray(x[r * nw:(r + 1) * nw])).cuda() for r in range(G)])

    def one(s):
        grp.step(W, wt, xs[s], cfg.dt)
        grp.local_energy(W, E)

    for s in range(Wm):
        one(s)
    l0 = sum(m.launch_count() for m in grp.members)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for s in range(Wm, Wm + K):
        one(s)
    torch.cuda.synchronize()
    t = time.perf_counter() - t0
    launches = sum(m.launch_count() for m in grp.members) - l0
    Em = float(np.mean(np.concatenate([e.cpu().numpy()[:, 0].real for e in E])))
    grp.close()
    return {"members_on_this_gpu": G, "walkers_per_member": nw, "gamma_per_member": [b - a for a, b in slices],
            "ms_per_group_step": t / K * 1e3, "walker_steps_per_s": G * nw * K / t, "timing": "host clock around "
            "K x (group step + group local energy), stream synchronisations as group barriers",
            "launches": int(launches), "E_mean_real": Em}


def replica_seed(rank):
    """Every replica draws its own walkers and fields; the Hamiltonian (seed 0) is the same."""
    return int(rank)


def max_over_ranks(ms, dist, device):
    """Slowest rank's time: all-reduce MAX over the process group (NCCL on the GPU box, gloo in
    the CPU test); the identity without a group."""
    if dist is None:
        return float(ms)
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_value(world, nw_per_rank, steps, t_ms):
    """Whole-job walker-steps/s of `world` replicas of nw_per_rank walkers (weak scaling)."""
    return world * nw_per_rank * steps / (t_ms * 1e-3)


def run_reference(args, cfg, rank):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the workload."""
    if rank != 0:
        return
    from paper_2406_16238_b200 import inputs
    h1 = inputs.make_h1(cfg, 0)
    trial = inputs.make_trial(cfg, h1, 0)
    _, Lh = make_L(cfg, 0, True, False)
    nw_s = sample_walkers(cfg)
    v, sec, thr = oracle_sample(cfg, h1, Lh, trial, nw_s, args.steps, args.warmup)
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic",
        "config": {"workload": cfg.name, "M": cfg.M, "n_alpha": cfg.n_alpha, "n_beta": cfg.n_beta,
                   "n_chol": cfg.n_chol, "n_walkers": nw_s, "dt": cfg.dt,
                   "taylor_order": cfg.taylor_order},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": thr, "kind": "oracle",
                         "sample": f"{nw_s} of {cfg.nw} walkers x {args.steps} steps (step + local energy)"},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c5", choices=["c1", "c2", "c3", "c4", "c5"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--pack-chol", action="store_true",
                    help="handle keeps the tile-packed upper triangles of L (PAPER.md:205); the dense tensor is "
                         "freed after afqmc_create")
    ap.add_argument("--mixed-precision", action="store_true",
                    help="V_HS build in emulated single precision on tcgen05 (afqmc_params.mixed_precision); "
                         "not the headline configuration (north_star: complex128 throughout)")
    ap.add_argument("--complex-chol", action="store_true",
                    help="complex Cholesky vectors (afqmc_params.complex_chol) on the workload's shapes: "
                         "n_chol / 2 complex vectors = n_chol Hermitian matrices = n_chol fields (c1-c3)")
    ap.add_argument("--complex-trial", action="store_true",
                    help="with --complex-chol: complex trial (afqmc_params.complex_trial), the lowest eigenvectors of "
                         "the complex Hermitian h1")
    ap.add_argument("--min-seconds", type=float, default=0.0,
                    help="raise K until the timed region lasts at least this long (small workloads: the clock "
                         "sampler needs >= 1 s for its five samples); the line reports the K that was timed")
    ap.add_argument("--no-block", action="store_true", help="skip the 25-step block timing")
    ap.add_argument("--block-reps", type=int, default=3)
    ap.add_argument("--group", type=int, default=0,
                    help="also time the distributed-Hamiltonian route with this many members on the one GPU")
    ap.add_argument("--profiler-range", action="store_true",
                    help="cudaProfilerStart/Stop around the timed steps (ncu --profile-from-start off)")
    args = ap.parse_args()

    import torch
    from paper_2406_16238_b200 import inputs
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = inputs.get_config(args.workload)
    if args.impl == "reference":
        run_reference(args, cfg, rank)
        return

    from paper_2406_16238_b200 import afqmc
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()

    K, Wm, nw = args.steps, args.warmup, cfg.nw
    seed = replica_seed(rank)
    h1 = inputs.make_h1(cfg, 0)
    trial = inputs.make_trial(cfg, h1, 0)
    want_cpu = (rank == 0 and world == 1 and not args.no_cpu_baseline)
    stream = torch.cuda.Stream()
    cx = None
    if args.complex_chol:
        if cfg.n_chol * cfg.M * cfg.M * 8 > (2 << 30):
            raise SystemExit("--complex-chol: workloads c1-c3 only (the tensor is generated on the host)")
        hc, Lc, trial, walkers_c = inputs.make_complex_problem(cfg.M, cfg.n_alpha, cfg.n_beta, cfg.n_chol // 4,
                                                               cfg.walker_kind, seed, nw,
                                                               complex_trial=args.complex_trial)
        cx = dict(h=hc, L=Lc, walkers=walkers_c, nf=2 * Lc.shape[0])
        h1 = hc
        Ld = torch.from_numpy(Lc).cuda()
        g = afqmc.AFQMC(hc, Ld, trial, M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta, n_chol=Lc.shape[0],
                        max_walkers=nw, walker_kind=cfg.walker_kind, taylor_order=cfg.taylor_order,
                        ortho_every=cfg.ortho_every, stream=stream.cuda_stream, complex_chol=True,
                        complex_trial=args.complex_trial)
        args.no_block = True
    else:
        Ld, _ = make_L(cfg, 0, False, True)
        g = afqmc.AFQMC(h1, Ld, trial, M=cfg.M, n_alpha=cfg.n_alpha, n_beta=cfg.n_beta,
                        n_chol=cfg.n_chol, max_walkers=nw, walker_kind=cfg.walker_kind,
                        taylor_order=cfg.taylor_order, ortho_every=cfg.ortho_every,
                        stream=stream.cuda_stream, pack_chol=args.pack_chol,
                        mixed_precision=args.mixed_precision)
    if args.pack_chol or args.mixed_precision or args.complex_chol:
        Ld = None
        torch.cuda.empty_cache()
    hbm_resident_gb = (torch.cuda.mem_get_info()[1] - torch.cuda.mem_get_info()[0]) / 1e9
    peak_dmma, peak_dfma, _ = afqmc.measure_fp64_peak(200.0)
    # the same issue loop held for 2 s: the rate the SMs sustain once the power management has settled, which is the
    # fair denominator for a kernel timed inside a seconds-long step loop (the 200 ms figure is the burst rate)
    peak_dmma_sustained = afqmc.measure_fp64_peak(2000.0)[0] if rank == 0 else None

    if cx:
        walkers_h = cx["walkers"]
        xs_h = np.stack([inputs.make_complex_fields(seed, s, nw, cx["nf"]) for s in range(Wm + K)])
    else:
        walkers_h = inputs.make_walkers(cfg, trial, seed, nw)
        xs_h = np.stack([inputs.make_aux_fields(cfg, seed, s, nw) for s in range(Wm + K)])
    with torch.cuda.stream(stream):
        W = torch.from_numpy(walkers_h).cuda()
        wt = torch.ones(nw, dtype=torch.float64, device="cuda")
        xs = torch.from_numpy(xs_h).cuda()
        E = torch.empty((nw, 3), dtype=torch.complex128, device="cuda")

        NX = xs.shape[0]                   # fields of Wm + args.steps steps, reused cyclically beyond that

        def one(s):
            g.step(W, wt, xs[s % NX], cfg.dt)
            g.local_energy(W, E)

        for s in range(Wm):
            one(s)
        g.sync()
        if args.min_seconds > 0.0:
            # size the timed region from a short untimed probe (same on every rank: the max is taken)
            q0, q1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            nprobe = max(3, Wm)
            q0.record(stream)
            for s in range(nprobe):
                one(s)
            q1.record(stream)
            torch.cuda.synchronize()
            est = max_over_ranks(q0.elapsed_time(q1) / nprobe, dist, "cuda")
            K = max(K, int(np.ceil(args.min_seconds * 1e3 / max(est, 1e-4))))
            W.copy_(torch.from_numpy(walkers_h))
            wt.fill_(1.0)
            torch.cuda.synchronize()
        l0 = g.launch_count()
        barrier()
        torch.cuda.synchronize()
        clk = ClockSampler(local)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        if args.profiler_range:
            torch.cuda.profiler.start()
        e0.record(stream)
        for s in range(Wm, Wm + K):
            one(s)
        e1.record(stream)
        torch.cuda.synchronize()
        if args.profiler_range:
            torch.cuda.profiler.stop()
        barrier()
        clocks = clk.stop()
        ms = e0.elapsed_time(e1)
        launches = g.launch_count() - l0
        E_last = E.cpu().numpy()
        wt_last = wt.cpu().numpy()
        # the per-stage breakdown (roofline of the dominant kernel) comes from a SEPARATE pass over the same K
        # steps with the library's event brackets on, so that `value` above carries no event-record overhead
        Wb = torch.from_numpy(walkers_h).cuda()
        wb = torch.ones(nw, dtype=torch.float64, device="cuda")
        g.set_profiling(True)
        g.stage_times(reset=True)
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        Kp = min(K, max(args.steps, 200))       # a raised K (--min-seconds) is not needed for the breakdown
        p0.record(stream)
        for s in range(Wm, Wm + Kp):
            g.step(Wb, wb, xs[s % NX], cfg.dt)
            g.local_energy(Wb, E)
        p1.record(stream)
        torch.cuda.synchronize()
        ms_prof = p0.elapsed_time(p1) * K / Kp   # scaled to K steps: everything below divides by K
        stages = g.stage_times(reset=True)
        g.set_profiling(False)
        del Wb, wb

    tmax = max_over_ranks(ms, dist, "cuda")
    value = job_value(world, nw, K, tmax)

    # ---- the paper's own timed unit: a block of 25 steps, energy once per block --
    block = None
    if not args.no_block and rank == 0:
        block = time_blocks(g, cfg, stream, walkers_h, seed, nw, args.block_reps)

    # ---- end to end through the C ABI with pinned host buffers ---------------------------------
    e2e = None
    if not args.no_e2e:
        Wp = torch.from_numpy(walkers_h.copy()).pin_memory()
        wp = torch.ones(nw, dtype=torch.float64).pin_memory()
        xp = torch.from_numpy(xs_h).pin_memory()
        Ep = torch.empty((nw, 3), dtype=torch.complex128).pin_memory()
        Wn, wn, En = Wp.numpy(), wp.numpy(), Ep.numpy()

        def one_host(s):
            g.step(Wn, wn, xp[s % NX].numpy(), cfg.dt)
            g.local_energy(Wn, En)

        for s in range(min(Wm, 2)):
            one_host(s)
        barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for s in range(Wm, Wm + K):
            one_host(s)
        g.sync()
        t_e2e = time.perf_counter() - t0
        barrier()
        t_e2e = max_over_ranks(t_e2e, dist, "cuda")
        wbytes = Wn.nbytes
        e2e = {"value": job_value(world, nw, K, t_e2e * 1e3), "unit": UNIT,
               "h2d_bytes_per_step": int(2 * wbytes + wn.nbytes + xp[0].numpy().nbytes),
               "d2h_bytes_per_step": int(wbytes + wn.nbytes + En.nbytes)}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel -------------------------------------------------------
    fl = flops_model(cfg, nw, cx["nf"] if cx else 0)
    per_stage = {k: {"ms_per_step": v[0] / Kp, "launches": v[1]} for k, v in stages.items() if v[1]}
    for k, f in fl.items():
        if k in per_stage and per_stage[k]["ms_per_step"] > 0:
            tf = f / (per_stage[k]["ms_per_step"] * 1e-3) / 1e12
            per_stage[k]["tflops"] = tf
            per_stage[k]["frac_of_dmma_peak"] = tf / peak_dmma
    if args.mixed_precision and "vhs" in per_stage:
        # bf16 x 3 on tcgen05: HBM bound (the split upper-triangle tiles are streamed once per step)
        ntile = sum(1 for pb in range((cfg.M + 7) // 8) for qb in range((cfg.M + 15) // 16) if qb * 16 + 15 >= pb * 8)
        gp = (cfg.n_chol + 63) // 64 * 64
        by = ntile * 3 * 128 * gp * 2 + nw * 2 * cfg.M * cfg.M * 8
        v = per_stage["vhs"]
        v.pop("frac_of_dmma_peak", None)
        v["tflops"] = 6 * fl["vhs"] / (v["ms_per_step"] * 1e-3) / 1e12      # bf16 flops issued: 6 plane pairs
        v["algorithmic_bytes"] = by
        v["gbytes_per_s"] = by / (v["ms_per_step"] * 1e-3) / 1e9
        v["note"] = "emulated single precision (bf16 x 3, FP32 accumulate in TMEM); bound: hbm"
        for k, note in (("taylor", "split of A + one launch per order"), ("force_bias", "split of Theta^T + one launch"),
                        ("one_body", "split of the walkers + one launch per half step")):
            if k in per_stage:
                t = per_stage[k]
                t.pop("frac_of_dmma_peak", None)
                t["tflops"] = 6 * fl[k] / (t["ms_per_step"] * 1e-3) / 1e12      # bf16 flops issued
                t["note"] = "emulated single precision on tcgen05 (" + note + ")"
    dom = max(per_stage, key=lambda k: per_stage[k]["ms_per_step"])
    nl = {"exchange": 1 if cfg.walker_kind == 0 else 2, "taylor": cfg.taylor_order, "one_body": 2}.get(dom, 1)
    roof = {"kernel": dom, "bound": "tensor", "unit": "TFLOP/s", "peak": peak_dmma,
            "peak_source": "FP64 DMMA issue rate measured on this GPU by afqmc_measure_fp64_peak "
                           "(register-only mma.sync.m8n8k4.f64 loop, 200 ms); MEASURED_PEAKS.json has "
                           "no FP64 entry",
            "achieved": per_stage[dom].get("tflops"), "frac": per_stage[dom].get("frac_of_dmma_peak"),
            "peak_sustained": peak_dmma_sustained,
            "frac_sustained": (per_stage[dom]["tflops"] / peak_dmma_sustained
                               if per_stage[dom].get("tflops") and peak_dmma_sustained else None),
            "peak_sustained_source": "the same loop held for 2 s (power management settled)",
            "flops_per_launch": fl.get(dom, 0.0) / nl,
            "ms_per_launch": per_stage[dom]["ms_per_step"] / nl,
            "share_of_step": per_stage[dom]["ms_per_step"] / (ms_prof / K),
            "timing": "CUDA events of the library's own stage brackets on the launch stream, in a separate pass "
                      "over the same K steps (%.3f ms per step with the brackets on, %.3f without)" % (ms_prof / K, ms / K),
            "traffic": None}
    tr = ncu_traffic(cfg.name + ("+complex" if cx else ""), dom)
    if tr:
        roof["traffic"] = tr["bytes"]
        roof["traffic_source"] = f"{tr['capture']} (commit {tr['commit']})"
    # the profiling guide's rule for a dtype without a measured peak: another dtype's measured peak x the
    # nominal ratio (bf16 burst figure of MEASURED_PEAKS.json x 40 / 2250 for FP64); a weaker denominator
    # than the DMMA rate measured above, kept beside it for comparison
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            mp = json.load(f)
        rule = float(mp["bf16_tflops"]) * 40.0 / 2250.0
        roof["peak_by_guide_rule"] = rule
        roof["frac_by_guide_rule"] = (roof["achieved"] / rule) if roof["achieved"] else None
        roof["hbm_gbs_measured"] = mp.get("hbm_gbs")
        # north_star: achieved HBM GB/s of the streaming kernels against the measured copy bandwidth.  Algorithmic
        # bytes only (each array once): a4 reads X (complex) and x and writes the shifted fields (complex);
        # the energy reduction reads X of the energy pass (complex) and the exchange kernel's partial sums
        # [n_chol / G][nw] (complex) per spin block.  Both are launch-latency sized at these shapes.
        nf_ = cx["nf"] if cx else cfg.n_chol
        plan_G = [int(t.split(" G ")[1].split()[0]) if " G " in t else 1
                  for t in (afqmc.exchange_plan(ns, cfg.M, bool(cx))[1] for ns in
                            ([cfg.n_alpha] if cfg.walker_kind == 0 else [cfg.n_alpha, cfg.n_beta]))]
        stream_bytes = {"field_shift": 40.0 * nf_ * nw,
                        "e_reduce": 16.0 * nf_ * nw + sum(16.0 * ((nf_ + G_ - 1) // G_) * nw for G_ in plan_G)}
        for k_, by_ in stream_bytes.items():
            if k_ in per_stage and per_stage[k_]["ms_per_step"] > 0 and mp.get("hbm_gbs"):
                gbs = by_ / (per_stage[k_]["ms_per_step"] * 1e-3) / 1e9
                per_stage[k_].update({"bound": "hbm", "algorithmic_bytes": by_, "gbytes_per_s": gbs,
                                      "frac_of_hbm_peak": gbs / float(mp["hbm_gbs"])})
    except (OSError, KeyError, ValueError):
        pass

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": tmax / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg.name, "M": cfg.M, "n_alpha": cfg.n_alpha, "n_beta": cfg.n_beta,
                   "n_chol": cfg.n_chol, "n_walkers_per_gpu": nw, "dt": cfg.dt,
                   "taylor_order": cfg.taylor_order, "ortho_every": cfg.ortho_every,
                   "local_energy": "every step", "parallelism": f"replicas x{world}",
                   "pack_chol": bool(args.pack_chol), "mixed_precision": bool(args.mixed_precision),
                   "complex_chol": bool(args.complex_chol), "complex_trial": bool(args.complex_trial),
                   "exchange_plan": [afqmc.exchange_plan(ns, cfg.M, bool(cx))[1] for ns in
                                     ([cfg.n_alpha] if cfg.walker_kind == 0 else [cfg.n_alpha, cfg.n_beta])],
                   "hbm_resident_gb": round(hbm_resident_gb, 1),
                   "steps_requested": args.steps, "min_seconds": args.min_seconds,
                   "l2": "inputs > L2 (Cholesky tensor %.1f GB)" % (cfg.n_chol * cfg.M * cfg.M * 8 / 1e9)},
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches),
        "roofline": roof, "stages": per_stage, "block": block,
        "fp64_peaks_measured": {"dmma_tflops": peak_dmma, "dfma_tflops": peak_dfma},
        "check": {"E_mean_real": float(np.mean(E_last[:, 0].real)), "weights_min": float(wt_last.min()),
                  "weights_max": float(wt_last.max())},
    }

    if args.group > 1 and world == 1 and not cx:
        if Ld is None:
            Ld, _ = make_L(cfg, 0, False, True)
        line["distributed_hamiltonian"] = time_sharded(cfg, h1, Ld, trial, args.group, K, Wm, seed)

    if want_cpu and cx:
        from oracle.complex_chol_oracle import ComplexCholOracle
        g.close()
        nw_s = 2
        t0 = time.perf_counter()
        o = ComplexCholOracle(cx["h"], cx["L"], trial, cfg.n_alpha, cfg.n_beta, cfg.walker_kind,
                              taylor_order=cfg.taylor_order, check=False)
        Wn, wn, _ = o.step(cx["walkers"][:nw_s], np.ones(nw_s), xs_h[0][:nw_s], cfg.dt)      # warm-up, untimed
        t1 = time.perf_counter()
        Wn, wn, _ = o.step(Wn, wn, xs_h[1 % len(xs_h)][:nw_s], cfg.dt)
        o.local_energy(Wn)
        sec = time.perf_counter() - t1
        line["cpu_baseline"] = {"value": nw_s / sec, "unit": UNIT, "cores": os.cpu_count(), "kind": "oracle",
                                "sample": f"{nw_s} of {nw} walkers x 1 step after 1 warm-up step (step + local energy), {sec:.1f} s "
                                          f"(+ {t1 - t0:.1f} s setup), oracle/complex_chol_oracle.py"}
        want_cpu = False
    if want_cpu:
        g.close()
        if Ld is None:
            Ld, _ = make_L(cfg, 0, False, True)
        Lh = Ld.cpu().numpy()
        del Ld
        torch.cuda.empty_cache()
        nw_s = sample_walkers(cfg)
        # one untimed warm-up step (first-touch page faults of the host tensor, BLAS thread start-up), two timed
        v, sec, thr = oracle_sample(cfg, h1, Lh, trial, nw_s, 2, 1)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": thr, "kind": "oracle",
                                "sample": f"{nw_s} of {nw} walkers x 2 steps after 1 warm-up step (step + local "
                                          f"energy), {sec:.1f} s per step; the oracle's V_HS and setup stream the whole "
                                          f"Cholesky tensor for these {nw_s} walkers, the GPU arm amortises that stream "
                                          f"over {nw}: the oracle's walker-steps/s at full batch would be higher"}
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
