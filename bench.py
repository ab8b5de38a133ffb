#!/usr/bin/env python
"""bench.py — SCAPE step throughput on B200 (BASELINE.json `metric`): params/s, step ms and
achieved HBM GB/s against the measured peak.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload llama1p8b] [--impl reference]

A "step" is one pass of the whole hot path (scape_step: stages 1-6 of the north star) over one
seeded synthetic gradient set of the workload's shape.  The default workload is the Llama-1.8B-
shaped shard (R = 4 bf16 gradient buffers, 99 % sparsity), the configuration the headline bar
is quoted on; it fits one GPU.  Inputs (~50 GB) are far larger than L2, so no flush is needed
between steps.  The path does not shard across GPUs ("replicas only"):
with --gpus N each rank runs an independent replica of the same workload, no collective on the
data path; `value` = params all ranks processed / max-over-ranks device time ("weak").

Prints ONE JSON line (rank 0).  `--impl reference` times the CPU oracle instead (a deliberately
plain program: the ratio against it is not the headline; parity and roofline.frac are).
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "scape_step_params_per_s"
UNIT = "params/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="llama1p8b",
                    help="pr1 | gpt345m | llama500m | llama1p8b | llama1p8b_literal | sweep:<log2n>:<sparsity>:<R>")
    ap.add_argument("--div", type=int, default=1, help="shrink every tensor by this factor")
    ap.add_argument("--sparsity", type=float, default=None)
    ap.add_argument("--sets", type=int, default=4, help="distinct consecutive gradient sets kept resident and cycled")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-div", type=int, default=64, help="oracle sample: every tensor this many times smaller")
    ap.add_argument("--cpu-steps", type=int, default=3)
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--layers", action="store_true",
                    help="per-layer refresh (scape_set_layers: one top-k per tensor of the workload, PAPER.md:89, :138) instead of "
                         "the north star's flat top-k")
    ap.add_argument("--workers", action="store_true",
                    help="workers mode (include/scape.h 'Workers', not the north-star path): every rank holds the whole shard and its "
                         "own R gradient buffers, per-layer refresh split over the ranks, NCCL all-reduce of the k local sums and of the "
                         "mask words between scape_step_local and scape_step_apply")
    ap.add_argument("--sweep", default=None, metavar="CSV",
                    help="run BASELINE.json config 5 (sizes 2^20..2^30 x sparsity x R, Gaussian grads) and write one CSV row per point")
    ap.add_argument("--sweep-log2n", default="20,21,22,23,24,25,26,27,28,29,30")
    ap.add_argument("--sweep-sparsity", default="0,0.9,0.99,0.999")
    ap.add_argument("--sweep-R", default="1,2,4,8")
    ap.add_argument("--no-also", action="store_true",
                    help="skip `also_measured` (the other BASELINE.json configs timed after the headline region, N = 1 only)")
    ap.add_argument("--also-steps", type=int, default=10)
    ap.add_argument("--plumbing-only", action="store_true",
                    help="launcher / rendezvous / barrier / max-over-ranks / JSON line WITHOUT the CUDA step, on the gloo backend: "
                         "what tests/test_multirank_cpu.py runs on a CPU box; the line says so and carries no measurement")
    return ap.parse_args()


def get_workload(args):
    from paper_2607_01678_b200 import synth
    if args.workload.startswith("sweep:"):
        _, l2, s, r = args.workload.split(":")
        return synth.sweep_point(int(l2), float(s), int(r))
    return synth.workload(args.workload, div=args.div, sparsity=args.sparsity)


# ---------------------------------------------------------------------------------------------
# algorithmic bytes
# ---------------------------------------------------------------------------------------------
def grad_bytes(w):
    return 2 if w.grad_dtype == "bf16" else 4


def bytes_per_param_fused(w, k, N):
    """Fused streaming kernel, steady state (sparse mask in, m stored sparsely): reads theta, g^r,
    e^r, the bits + rank128 of the current and the previous mask, the previous packed mean (= m);
    writes theta, e^r, b^r, b-bar (= new m) and the certainly-selected bits of the next mask.
    With sparsity 0 every step is dense: m is read and written densely, nothing is packed."""
    G, R, d = grad_bytes(w), w.R, k / N
    if k == N:
        return (G + 8) * R + 16
    return (G + 8) * R + 8 + 4 * d * (R + 2) + 2 * (1 / 8 + 4 / 128) + 1 / 8


def bytes_per_param_step(w, k, N):
    """Whole step, the method's own minimum traffic (SURVEY.md §8(d) B_alg: m stored sparsely)."""
    G, R, d = grad_bytes(w), w.R, k / N
    if k == N:
        return (G + 8) * R + 16
    return (G + 8) * R + 8 + 16 * d + 4 * d * R + 3 / 8


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(p) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def recorded_traffic(workload_name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the fused kernel from the committed
    `ncu --set full` captures (profiles/traffic.csv: workload, kernel, bytes, source), or None."""
    import csv
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.csv"), newline="") as f:
            for row in csv.DictReader(f):
                if row["workload"] == workload_name:
                    return int(row["fused_dram_bytes_per_launch"])
    except Exception:
        pass
    return None


# ---------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md recipe)
# ---------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        self.p = None

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100", "-i", str(self.index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.p is None:
            return out
        time.sleep(0.15)
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        for line in self.f.read().splitlines():
            c = [x.strip() for x in line.split(",")]
            if len(c) < 9:
                continue
            try:
                sm.append(float(c[1])); mx.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.f.name)
        if sm:
            sm.sort()
            out.update(sm_mhz=sm[len(sm) // 2], sm_max_mhz=max(mx), reasons=sorted(reasons), samples=len(sm))
        return out


# ---------------------------------------------------------------------------------------------
# the CPU oracle as a timed baseline (bounded sample)
# ---------------------------------------------------------------------------------------------
def time_oracle(args, steps, warmup, div):
    """Runs oracle/ as it stands, single-threaded, on the same workload with every tensor `div`
    times smaller.  Returns (params_per_s, ms_per_step, sample description, N_sample)."""
    import numpy as np
    import torch
    from oracle.scape_oracle import ScapeOracle
    from paper_2607_01678_b200 import synth
    wl = args.workload
    if wl.startswith("sweep:"):
        w = get_workload(args)
    else:
        w = synth.workload(wl, div=max(div, args.div), sparsity=args.sparsity)
    gs = synth.GradStream(w, device="cpu", seed=args.seed)
    th = gs.theta0().numpy().copy()
    ora = ScapeOracle(w.numel, w.R, w.sparsity, **w.hyper)
    # the first step of Alg. 1 is dense (M_0 = 1); it is always part of the warm-up
    total = 0.0
    for i in range(1 + warmup + steps):
        grads = [g.to(torch.float32).numpy() for g in gs.next()]
        t0 = time.perf_counter()
        ora.step(th, grads)
        dt = time.perf_counter() - t0
        if i >= 1 + warmup:
            total += dt
    ms = 1e3 * total / steps
    desc = (f"{w.name}: N={w.numel} (every tensor /{max(div, args.div)}), R={w.R}, sparsity={w.sparsity}, "
            f"{steps} steady-state steps after {1 + warmup} warm-up (incl. the dense first step); "
            f"oracle/scape_oracle.cpp -O2 -ffp-contract=off, 1 thread")
    return w.numel * steps / total, ms, desc, w.numel


def run_reference(args):
    """--impl reference: the oracle on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = get_workload(args)
    pps, ms, desc, n = time_oracle(args, steps=max(1, args.steps), warmup=max(0, args.warmup), div=args.cpu_div)
    line = {
        "impl": "reference", "metric": METRIC, "value": pps, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic (seeded)",
        "config": {"workload": w.name, "R": w.R, "sparsity": w.sparsity, "grad_dtype": w.grad_dtype,
                   "sample": desc},
        "cpu_baseline": {"value": pps, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
                         "host_cores": os.cpu_count()},
        "e2e": {"value": pps, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def run_sweep(args):
    """BASELINE.json config 5: 3 warm-up + 10 timed steps per point (after the dense first step),
    i.i.d. Gaussian gradients std 1e-3, fixed seed, a fresh gradient set every step.  Points whose footprint fits the 126 MB L2 run
    above the DRAM roofline and are labelled l2_resident."""
    import torch
    from paper_2607_01678_b200 import binding, synth
    torch.cuda.set_device(0)
    peak, _ = measured_peak()
    rows = ["log2n,N,sparsity,R,k,ms_per_step,params_per_s,step_gbs_alg,frac_of_measured_peak,footprint_mib,l2_resident,kernel,select_fast,select_general"]
    for l2 in [int(x) for x in args.sweep_log2n.split(",")]:
        for sp in [float(x) for x in args.sweep_sparsity.split(",")]:
            for R in [int(x) for x in args.sweep_R.split(",")]:
                w = synth.sweep_point(l2, sp, R)
                N = w.numel
                gs = synth.GradStream(w, device="cuda", seed=args.seed)
                theta = gs.theta0()
                # A fresh gradient set for every step (1 dense + 3 warm-up + 10 timed), drawn on the device between
                # the steps, as in training, where a gradient never repeats.  (Cycling a few resident sets, as round 1
                # did, makes the top-k threshold resonate with the error feedback -- period = number of sets -- and the
                # select's predicted bracket three times wider than on non-repeating inputs: DESIGN.md §5.2.)  Each
                # timed step has its own CUDA-event pair; the time between the pairs (the draw) is not counted.
                sc = binding.Scape(N, R, sp, **w.hyper)
                k = sc.k
                for i in range(4):
                    grads = gs.next()
                    sc.step(theta, grads)
                    del grads
                torch.cuda.synchronize()
                f0, g0 = sc.select_stats() if k < N else (0, 0)
                evs = []
                for i in range(10):
                    grads = gs.next()
                    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    a.record()
                    sc.step(theta, grads)
                    b.record()
                    evs.append((a, b))
                    del grads
                torch.cuda.synchronize()
                ms = sum(a.elapsed_time(b) for a, b in evs) / 10
                del gs
                f1, g1 = sc.select_stats() if k < N else (0, 0)
                gbs = bytes_per_param_step(w, k, N) * N / (ms * 1e-3) / 1e9
                foot = (8 + 8 * R) * N / 2**20
                rows.append(f"{l2},{N},{sp},{R},{k},{ms:.5f},{N / (ms * 1e-3):.4e},{gbs:.1f},{gbs / peak:.4f},{foot:.1f},"
                            f"{int(foot < 126)},{sc.last_kernel},{f1 - f0},{g1 - g0}")
                print(rows[-1], flush=True)
                sc.close()
                del sc, theta
                torch.cuda.empty_cache()
    with open(args.sweep, "w") as f:
        f.write("\n".join(rows) + "\n")


def max_over_ranks_ms(ms, world, device):
    """Device time of the slowest rank (every multi-GPU number is the max over ranks)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(n_params, steps, elapsed_ms, world):
    """params/s of the whole job: every rank processed n_params * steps in elapsed_ms (replicas only)."""
    return world * n_params * steps / (elapsed_ms * 1e-3)


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher around it: start the N ranks here, exactly as the
    driver's own command line does (torch.distributed.run, one node, 127.0.0.1), and hand on their
    output and exit code.  Under torchrun (WORLD_SIZE set) this is never reached."""
    import socket
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def run_plumbing_only(args):
    """The N > 1 host logic with no GPU: rendezvous, barrier, max over ranks, whole-job aggregate, one
    JSON line from rank 0.  Every rank pretends its region took (10 + 5 rank) ms."""
    import torch
    import torch.distributed as dist
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if world > 1:
        dist.init_process_group("gloo")
        dist.barrier()
    K = args.steps
    ms = max_over_ranks_ms(10.0 + 5.0 * rank, world, torch.device("cpu"))
    if world > 1:
        dist.barrier()
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": args.warmup,
                          "ms_per_step": None, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                          "plumbing_only": {"note": "no CUDA step was run (CPU test of the launcher)", "max_over_ranks_ms": ms,
                                            "aggregate_of_fake_region": whole_job_value(1000, K, ms, world)},
                          "gpu_launches": 0}), flush=True)
    if world > 1:
        dist.destroy_process_group()


def timed_region(step, theta, ring, first, K):
    """K back-to-back steps, one CUDA event before each and one after the last (all on torch's current
    stream, the one the step is enqueued on).  -> (elapsed ms of the whole region, per-step ms list)."""
    import torch
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
    n_sets = len(ring)
    for i in range(K):
        ev[i].record()
        step(theta, ring[(first + i) % n_sets])
    ev[K].record()
    torch.cuda.synchronize()
    per = [ev[i].elapsed_time(ev[i + 1]) for i in range(K)]
    return ev[0].elapsed_time(ev[K]), per


def step_stats(per):
    s = sorted(per)
    return {"ms_median": s[len(s) // 2] if len(s) % 2 else 0.5 * (s[len(s) // 2 - 1] + s[len(s) // 2]),
            "ms_min": s[0], "ms_max": s[-1]}


def measure_also(name, w, theta, ring, K, W, peak, layers=False):
    """One more workload timed like the headline (dense first step, W warm-up steps, K timed steps
    with per-step events), reported in `also_measured`."""
    import torch
    from paper_2607_01678_b200 import binding
    N, R = w.numel, w.R
    sc = binding.Scape(N, R, w.sparsity, **w.hyper)
    if layers:
        sc.set_layers(w.offsets(), w.compress_flags())
    k = sc.k
    n_sets = len(ring)
    sc.step(theta, ring[0])
    for i in range(W):
        sc.step(theta, ring[(1 + i) % n_sets])
    torch.cuda.synchronize()
    sc.profile(True)
    f0, g0 = sc.select_stats()
    l0 = sc.launches
    elapsed, per = timed_region(sc.step, theta, ring, 1 + W, K)
    fused_ms, select_ms, psteps = sc.profile_read()
    sc.profile(False)
    f1, g1 = sc.select_stats()
    ms = elapsed / K
    kms = fused_ms / max(1, psteps)
    fb = bytes_per_param_fused(w, k, N) * N
    sb = bytes_per_param_step(w, k, N) * N
    out = {"workload": name, "shard_numel": N, "R": R, "grad_dtype": w.grad_dtype, "sparsity": w.sparsity, "k": k,
           "refresh": "per layer (one top-k per tensor)" if layers else "flat top-k over the shard",
           "steps": K, "warmup": W, "ms_per_step": ms, **step_stats(per), "params_per_s": N / (ms * 1e-3),
           "kernel": sc.last_kernel, "kernel_ms": kms, "kernel_share_of_step": kms / ms,
           "kernel_gbs": fb / (kms * 1e-3) / 1e9, "kernel_frac_of_peak": fb / (kms * 1e-3) / 1e9 / peak,
           "select_ms": select_ms / max(1, psteps), "step_gbs": sb / (ms * 1e-3) / 1e9,
           "step_frac_of_peak": sb / (ms * 1e-3) / 1e9 / peak,
           "select_fast": f1 - f0, "select_general": g1 - g0, "gpu_launches": sc.launches - l0,
           "l2_resident": (8 + (grad_bytes(w) + 4) * R) * N < 126e6}
    assert bool(torch.isfinite(theta).all())
    sc.close()
    return out


def measure_fresh(name, w, K, W, peak, seed, layers=False):
    """The same step with a FRESH gradient set every step, drawn on the device between the steps (as in training, where
    a gradient never repeats; the draw is not timed: every timed step has its own CUDA-event pair).  The resident sets the
    headline cycles keep the select's predicted brackets wide (the threshold resonates with the error feedback, period =
    number of sets): this line shows the select stage on non-repeating inputs."""
    import torch
    from paper_2607_01678_b200 import binding, synth
    N, R = w.numel, w.R
    gs = synth.GradStream(w, device="cuda", seed=seed)
    theta = gs.theta0()
    sc = binding.Scape(N, R, w.sparsity, **w.hyper)
    if layers:
        sc.set_layers(w.offsets(), w.compress_flags())
    k = sc.k
    for _ in range(1 + W):
        grads = gs.next()
        sc.step(theta, grads)
        del grads
    torch.cuda.synchronize()
    sc.profile(True)
    f0, g0 = sc.select_stats()
    evs = []
    for _ in range(K):
        grads = gs.next()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        sc.step(theta, grads)
        b.record()
        evs.append((a, b))
        del grads
    torch.cuda.synchronize()
    per = [a.elapsed_time(b) for a, b in evs]
    fused_ms, select_ms, psteps = sc.profile_read()
    sc.profile(False)
    f1, g1 = sc.select_stats()
    ms = sum(per) / K
    kms = fused_ms / max(1, psteps)
    fb = bytes_per_param_fused(w, k, N) * N
    sb = bytes_per_param_step(w, k, N) * N
    out = {"workload": name, "gradients": "fresh every step (drawn on the device between the timed steps; per-step CUDA events)",
           "shard_numel": N, "R": R, "grad_dtype": w.grad_dtype, "sparsity": w.sparsity, "k": k,
           "refresh": "per layer (one top-k per tensor)" if layers else "flat top-k over the shard",
           "steps": K, "warmup": W, "ms_per_step": ms, **step_stats(per), "params_per_s": N / (ms * 1e-3),
           "kernel": sc.last_kernel, "kernel_ms": kms, "kernel_share_of_step": kms / ms,
           "kernel_gbs": fb / (kms * 1e-3) / 1e9, "kernel_frac_of_peak": fb / (kms * 1e-3) / 1e9 / peak,
           "select_ms": select_ms / max(1, psteps), "step_gbs": sb / (ms * 1e-3) / 1e9,
           "step_frac_of_peak": sb / (ms * 1e-3) / 1e9 / peak,
           "select_fast": f1 - f0, "select_general": g1 - g0, "l2_resident": False}
    assert bool(torch.isfinite(theta).all())
    sc.close()
    del gs, theta
    torch.cuda.empty_cache()
    return out


# ---------------------------------------------------------------------------------------------
def main():
    args = parse()
    if args.impl == "reference":
        return run_reference(args)
    if args.sweep:
        return run_sweep(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        sys.exit(spawn_ranks(args))
    if args.plumbing_only:
        return run_plumbing_only(args)

    import torch
    import torch.distributed as dist
    from paper_2607_01678_b200 import binding, synth

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU fallback")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    elif args.workers:                      # a world of one: the same NCCL calls, nothing to wait for
        dist.init_process_group("nccl", init_method="file://" + tempfile.mktemp(prefix="scape_pg_"), rank=0, world_size=1,
                                device_id=torch.device("cuda", local))
    binding.lib()

    w = get_workload(args)
    N, R = w.numel, w.R
    K, W = args.steps, max(args.warmup, 3)
    dev = torch.device("cuda", local)

    # ---- inputs resident in HBM before the timed region --------------------------------
    gs = synth.GradStream(w, device=dev, seed=args.seed + rank)
    theta = gs.theta0()
    if args.workers and world > 1:          # every worker holds the same parameters
        theta = synth.GradStream(w, device=dev, seed=args.seed).theta0()
    n_sets = max(1, min(args.sets, K + W + 1))
    ring = [gs.next() for _ in range(n_sets)]
    del gs
    torch.cuda.empty_cache()

    sc = binding.Scape(N, R, w.sparsity, **w.hyper)
    step = sc.step
    if args.layers and not args.workers:
        sc.set_layers(w.offsets(), w.compress_flags())
    if args.workers:
        from paper_2607_01678_b200 import workers as wk
        sc.set_layers(w.offsets(), w.compress_flags())          # per-layer refresh, one layer per tensor
        sc.set_workers(world, rank, wk.balance_layers([n for _, n in w.tensors], world))
        # the exchange runs inside the library (scape_step_exchange) over two NCCL communicators of its own:
        # the sums on the caller's stream, the mask portions on the handle's stream
        ids = [binding.scape_nccl_unique_id(), binding.scape_nccl_unique_id()] if rank == 0 else [None, None]
        if world > 1:
            dist.broadcast_object_list(ids, src=0)
        comms = [binding.scape_nccl_comm_create(world, rank, i) for i in ids]
        step = lambda th, g: sc.step_workers(th, g, comm=comms[0], mask_comm=comms[1])    # noqa: E731
    k = sc.k
    # the first step of Alg. 1 is dense (M_0 = 1): always warm-up, reported separately
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); step(theta, ring[0]); e1.record(); torch.cuda.synchronize()
    first_step_ms = e0.elapsed_time(e1)
    for i in range(W):
        step(theta, ring[(1 + i) % n_sets])
    torch.cuda.synchronize()

    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = ClockSampler(local)
    if rank == 0:
        clocks.start()
    sc.profile(True)
    launches0 = sc.launches
    fast0, general0 = sc.select_stats()
    elapsed_ms, per_step = timed_region(step, theta, ring, 1 + W, K)
    fused_ms, select_ms, psteps = sc.profile_read()
    kernel_name = sc.last_kernel
    sc.profile(False)
    gpu_launches = sc.launches - launches0
    fast1, general1 = sc.select_stats()
    clk = clocks.stop() if rank == 0 else None
    elapsed_ms = max_over_ranks_ms(elapsed_ms, world, dev)
    if world > 1:
        dist.barrier()
    assert bool(torch.isfinite(theta).all()), "theta is not finite after the timed steps"
    mask_count = sc.count_next()
    assert mask_count == k, (mask_count, k)

    ms_per_step = elapsed_ms / K
    # replicas: every rank updates its own copy of the shard; workers: the ranks update ONE shard together
    value = whole_job_value(N, K, elapsed_ms, 1 if args.workers else world)

    # ---- roofline of the dominant kernel -------------------------------------------------
    peak, peak_src = measured_peak()
    fused_avg_ms = fused_ms / max(1, psteps)
    fb = bytes_per_param_fused(w, k, N) * N
    achieved = fb / (fused_avg_ms * 1e-3) / 1e9
    sb = bytes_per_param_step(w, k, N) * N
    roofline = {
        "bound": "hbm", "kernel": kernel_name, "achieved": achieved, "peak": peak, "unit": "GB/s",
        "frac": achieved / peak, "traffic": recorded_traffic(w.name),
        "peak_source": peak_src, "algorithmic_bytes_per_launch": fb, "kernel_ms": fused_avg_ms,
        "kernel_share_of_step": fused_avg_ms / ms_per_step,
        "select_ms": select_ms / max(1, psteps),
        "select_steps_fast": fast1 - fast0, "select_steps_general": general1 - general0,
        "step_algorithmic_bytes": sb, "step_gbs": sb / (ms_per_step * 1e-3) / 1e9,
        "step_frac_of_peak": sb / (ms_per_step * 1e-3) / 1e9 / peak,
        "step_frac_of_8TBs_nominal": sb / (ms_per_step * 1e-3) / 1e9 / 8000.0,
    }

    # ---- asynchronous refresh (scape_set_async_refresh): what a step costs the caller's
    # stream when other work (a stand-in for the forward / backward: ~5 ms of bf16 GEMMs, library calls) follows it
    async_line = None
    if world == 1 and not args.workers and not args.no_also and k < N:
        big = torch.randn(8192, 8192, device=dev, dtype=torch.bfloat16)
        big2 = torch.empty_like(big)
        small = torch.randn(1024, 1024, device=dev, dtype=torch.bfloat16)
        small2 = torch.empty_like(small)

        def busy_full():                         # six GEMMs that each fill every SM for ~0.7 ms
            for _ in range(6):
                torch.matmul(big, big, out=big2)

        # 600 GEMMs of 64 tiles each, replayed as one CUDA graph (no launch gaps): the stream is busy, most SMs are not
        torch.matmul(small, small, out=small2)
        torch.cuda.synchronize()
        g_small = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g_small):
            for _ in range(600):
                torch.matmul(small, small, out=small2)

        def busy_partial():
            g_small.replay()

        def loop(n, with_step, busy):
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a.record()
            for i in range(n):
                if with_step:
                    step(theta, ring[i % n_sets])
                busy()
            b.record()
            torch.cuda.synchronize()
            return a.elapsed_time(b) / n
        async_line = {"streaming_kernel_ms": fused_avg_ms, "select_ms": select_ms / max(1, psteps),
                      "note": "10 iterations of [scape_step; other work on the same stream]; step_cost = iteration - other work alone; "
                              "async: stage 2 on the handle's own high-priority stream.  Work that fills every SM leaves nothing to "
                              "overlap with; work that keeps the stream busy but not the SMs hides the refresh"}
        for name, busy in (("other_work_fills_all_sms", busy_full), ("other_work_leaves_sms_idle", busy_partial)):
            busy()
            busy_ms = loop(10, False, busy)
            res = {}
            for mode in (False, True):
                sc.set_async_refresh(mode)
                loop(3, True, busy)
                res[mode] = loop(10, True, busy)
            sc.set_async_refresh(False)
            sc.join_refresh()
            torch.cuda.synchronize()
            async_line[name] = {"other_work_ms": busy_ms, "step_cost_in_stream_ms": res[False] - busy_ms,
                                "step_cost_async_ms": res[True] - busy_ms}
        del g_small, big, big2, small, small2

    # ---- Algorithm 2's parameter side on the same shard: the owner packs
    # theta on the mask the last step used, a non-owner applies it to its FP32 copy and refreshes the bf16 compute copy
    alg2_line = None
    if world == 1 and not args.workers and not args.no_also and k < N:
        w_copy = theta.clone()
        w_hat = torch.empty(N, dtype=torch.bfloat16, device=dev)
        kk = sc.count_last()
        pay = sc.param_pack(theta, dtype=torch.bfloat16)
        sc.param_apply(w_copy, pay, w_hat)
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(3)]
        torch.cuda.synchronize()
        reps = 5
        ev[0].record()
        for _ in range(reps):
            sc.param_pack(theta, dtype=torch.bfloat16, out=pay)
        ev[1].record()
        for _ in range(reps):
            sc.param_apply(w_copy, pay, w_hat)
        ev[2].record()
        torch.cuda.synchronize()
        pack_ms, apply_ms = ev[0].elapsed_time(ev[1]) / reps, ev[1].elapsed_time(ev[2]) / reps
        apply_bytes = N * (4 + 4 + 2 + 1 / 8 + 8 / 128) + 2 * kk          # w in / out, w^ out, bits + rk, bf16 payload
        alg2_line = {"k": kk, "payload": "bf16", "param_pack_ms": pack_ms, "param_apply_ms": apply_ms,
                     "param_apply_algorithmic_bytes": apply_bytes, "param_apply_gbs": apply_bytes / (apply_ms * 1e-3) / 1e9,
                     "param_apply_frac_of_peak": apply_bytes / (apply_ms * 1e-3) / 1e9 / peak,
                     "param_pack_entries_per_s": kk / (pack_ms * 1e-3)}
        del w_copy, w_hat, pay

    sc.close()
    del sc

    # ---- the rest of `metric` ("at 90 %/99 % sparsity", the other model shapes), same run, N = 1 only
    also = None
    if world == 1 and not args.no_also and not args.workers and not args.layers and w.name == "llama1p8b":
        Ka, Wa = max(1, args.also_steps), 6
        also = [measure_also("llama1p8b --layers", w, theta, ring, Ka, Wa, peak, layers=True)]
        del ring, theta
        torch.cuda.empty_cache()
        for lay in (False, True):                    # the headline shard on non-repeating gradients
            also.append(measure_fresh("llama1p8b, fresh gradients" + (" --layers" if lay else ""), w, Ka, 12, peak, args.seed, layers=lay))
        cache = {}                                   # llama500m at 99 % re-uses the inputs drawn for 90 %
        for nm, sp in (("llama500m", 0.9), ("llama500m", None), ("gpt345m", None), ("pr1", None)):
            wa = synth.workload(nm, sparsity=sp)
            if nm not in cache:
                cache.clear()
                torch.cuda.empty_cache()
                ga = synth.GradStream(wa, device=dev, seed=args.seed)
                th0 = ga.theta0()
                # as many distinct gradient sets as the timed run needs, if ~100 GB hold them (else they are cycled)
                set_bytes = wa.numel * wa.R * grad_bytes(wa)
                n_also = int(max(2, min(1 + Wa + Ka, (100e9 - (12 + 4 * wa.R) * wa.numel) // set_bytes)))
                cache[nm] = (th0, [ga.next() for _ in range(n_also)])
                del ga, th0
            also.append(measure_also(nm, wa, cache[nm][0].clone(), cache[nm][1], Ka, Wa, peak))
        cache.clear()
        # BASELINE.json config 5 at the shape of the paper's deployment (one gradient per worker):
        # N = 2^28, R = 1, i.i.d. Gaussian gradients that never repeat inside the run
        for sp in (0.9, 0.99):
            torch.cuda.empty_cache()
            wa = synth.sweep_point(28, sp, 1)
            ga = synth.GradStream(wa, device=dev, seed=args.seed)
            th0 = ga.theta0()
            sets = [ga.next() for _ in range(1 + Wa + Ka)]
            del ga
            also.append(measure_also(f"sweep:28:{sp}:1", wa, th0, sets, Ka, Wa, peak))
            del th0, sets
    else:
        del ring, theta
    torch.cuda.empty_cache()

    # ---- end to end through the C-ABI with HOST buffers ---------------------------------------
    e2e = None
    if not args.no_e2e and not args.workers:
        gs = synth.GradStream(w, device=dev, seed=args.seed + rank)
        th_h = gs.theta0().cpu().pin_memory()
        g_h = [g.cpu().pin_memory() for g in gs.next()]
        del gs
        torch.cuda.empty_cache()
        sh = binding.Scape(N, R, w.sparsity, **w.hyper)
        for _ in range(2):                       # dense first step + one sparse step: warm-up
            sh.step_host(th_h, g_h)
        n_e2e = max(1, args.e2e_steps)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for _ in range(n_e2e):
            sh.step_host(th_h, g_h)
        b.record()
        torch.cuda.synchronize()
        e2e_ms = a.elapsed_time(b)
        e2e_ms = max_over_ranks_ms(e2e_ms, world, dev)
        gbytes = N * grad_bytes(w) * R
        e2e = {"value": whole_job_value(N, n_e2e, e2e_ms, world), "unit": UNIT,
               "h2d_bytes_per_step": 4 * N + gbytes, "d2h_bytes_per_step": 4 * N,
               "steps": n_e2e, "ms_per_step": e2e_ms / n_e2e,
               "api": "scape_step_host (pinned host param + R gradient buffers in, param out)"}
        sh.close()
        del sh, th_h, g_h

    # ---- the oracle on the host cores, bounded sample (rank 0, N = 1 only) --------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        pps, cms, desc, _ = time_oracle(args, steps=args.cpu_steps, warmup=1, div=args.cpu_div)
        cpu = {"value": pps, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
               "ms_per_step_on_sample": cms, "host_cores": os.cpu_count()}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": W,
            "ms_per_step": ms_per_step, **step_stats(per_step), "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic (seeded; shapes and distributions of BASELINE.json configs)",
            "config": {"workload": w.name, "shard_numel": N, "R": R, "sparsity": w.sparsity, "k": k,
                       "grad_dtype": w.grad_dtype, "dist": w.dist, "ar1_rho": w.rho, "hyper": w.hyper,
                       "gradient_sets_cycled": n_sets, "l2": "inputs (tens of GB) exceed the 126 MB L2; no flush needed",
                       "parallelism": (f"workers: {world} rank(s) x {R} replicas, per-layer refresh split over the ranks, NCCL all-reduce "
                                       f"of {k} fp32 sums + {(N + 31) // 32} mask words per step") if args.workers else
                                      "replicas only (no sharding, no collective)" if world > 1 else "single GPU",
                       "refresh": "per layer (one top-k per tensor)" if (args.layers or args.workers) else "flat top-k over the shard",
                       "first_dense_step_ms": first_step_ms},
            "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": gpu_launches, "clocks": clk,
            "also_measured": also, "async_refresh": async_line, "alg2_param_side": alg2_line,
        }
        print(json.dumps(line), flush=True)
    if world > 1 or args.workers:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
