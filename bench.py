#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path on BASELINE.json's
headline workload: configs[2], N = 1,048,576 uniformly filled ellipsoid, mean gamma 30, n = 6,
leaf 256, theta = 0.5, FP64, KD tree.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config I] [--tree kd|morton]
    python bench.py --config 5        error-versus-time sweep of BASELINE.json configs[4] (+ the all-pairs ceiling)
    python bench.py --config 9        the paper's own (n, eta) sweep: N = 1.28e6 cube, N0 = (n+1)^3
    python bench.py --probe-fp64      FP64 pipe micro-benchmarks (operand patterns; profiles/r02_fp64_pipe_microbench.md)

One "step" = one pass of Alg 5.12 over one bunch: mean momentum, tree order,
bounding boxes, dual tree traversal -> CSR lists, P2M, M2M, M2L, L2L, P2P, L2P, prefactors, scatter.
`value` = particles / s with the inputs resident in HBM; `e2e` = the same through fmm_field_host
with pinned HOST buffers (H2D of positions / momenta and D2H of E, B inside the timed region).
The path does not shard (north_star: one GPU, no collectives): --gpus N runs N independent replicas
("replicas only") and reports their aggregate.  --impl reference times the CPU oracle.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2302_07567_b200 import workloads  # noqa: E402

STAGE_KEYS = ("ms_tree", "ms_lists", "ms_p2m", "ms_m2m", "ms_m2l", "ms_l2l", "ms_p2p", "ms_l2p")
METRIC = "fmm_E+B_particles_per_s"
UNIT = "particles/s"
FLOP_PER_EVAL = 34          # algorithmic flop per kernel evaluation (fma = 2, rsqrt = 1)
FP64_LANES_PER_SM = 64      # B200: 148 SMs x 64 FP64 FMA lanes
SM_COUNT = 148


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json configs[i-1] (1-based)")
    ap.add_argument("--tree", default="kd", choices=["kd", "morton"])
    ap.add_argument("--kernel", default="mean_gamma", choices=["mean_gamma", "source_momentum"],
                    help="near-field kernel: eq. (3.2) with gamma_bar (default) or the G6 alternative (SURVEY 8(f) rank 2)")
    ap.add_argument("--method", default="fmm", choices=["fmm", "treecode"],
                    help="Alg 5.12 (default) or the particle-cluster treecode variant (SURVEY 8(f) rank 3)")
    ap.add_argument("--overlap", action="store_true", help="run P2P on a second stream beside the far-field chain (fmm_plan_set_overlap)")
    ap.add_argument("--plan-step", default="update", choices=["update", "refit", "keep_lists"],
                    help="what a timed step does before fmm_eval: fmm_plan_update (a0-a3, the default and the headline), fmm_plan_refit "
                         "(order kept: a0, a2, a3) or fmm_plan_refit_keep_lists (order and lists kept: a0, a2); SURVEY.md 8(f) rank 4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample-leaves", type=int, default=0,
                    help="target leaves the oracle evaluates per step (0 = all of them: a whole, unscaled step)")
    ap.add_argument("--probe-fp64", action="store_true", help="print the FP64 pipe micro-benchmark table and exit")
    ap.add_argument("--sweep-targets", type=int, default=4096, help="sampled targets of the error column of the sweeps")
    return ap.parse_args()


def workload_config(w, args):
    """The same dictionary on both arms (the driver compares them)."""
    cfg = {"workload": w.name, "N": w.N, "order_n": w.order_n, "leaf_size": w.leaf_size, "theta": w.theta,
           "tree": args.tree, "seed": w.seed, "precision": "fp64", "kernel": args.kernel, "method": args.method,
           "l2": "L2 flushed (256 MiB write) before every timed step; flush not timed"}
    if getattr(args, "plan_step", "update") != "update":
        cfg["plan_step"] = args.plan_step   # (not the headline: the tree order / the lists of an earlier build are reused)
    return cfg


# ------------------------------------------------------------------------------------------------
# CPU oracle timing (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------------
def oracle_step(w, tree, sample_leaves):
    """One bounded-sample pass of the oracle's serial FMM (OpenMP over targets): full tree + lists +
    upward pass, then near + far field for `sample_leaves` evenly spaced target leaves; the leaf part is
    scaled by leaves / sample to a whole-bunch time.  Returns (seconds_extrapolated, seconds_spent, info)."""
    import oracle
    t0 = time.perf_counter()
    op = oracle.Plan(*w.arrays(), w.q, order_n=w.order_n, leaf_size=w.leaf_size, theta=w.theta,
                     tree_mode=oracle.TREE_KD if tree == "kd" else oracle.TREE_MORTON_MEDIAN)
    t1 = time.perf_counter()
    op.upward()
    t2 = time.perf_counter()
    if sample_leaves <= 0 or sample_leaves >= op.leaves:   # the whole step, nothing scaled
        op.eval()
        t3 = time.perf_counter()
        info = {"plan_s": round(t1 - t0, 3), "upward_s": round(t2 - t1, 3), "sample_eval_s": round(t3 - t2, 3),
                "sample_leaves": int(op.leaves), "leaves": int(op.leaves)}
        op.close()
        return t3 - t0, t3 - t0, info
    S = max(1, min(sample_leaves, op.leaves))
    # the sample is 8 evenly spaced runs of contiguous leaves (whole sub-trees): the M2L work of their ancestor chains
    # then scales with the sample like the leaf work does (single evenly spaced leaves would pull in almost every
    # upper-level node and overstate the extrapolated time)
    runs = min(8, S)
    per = S // runs
    S = per * runs
    starts = (np.arange(runs) * op.leaves) // runs
    sel = (op.leaves + (starts[:, None] + np.arange(per)[None, :]).ravel()).astype(np.int64)
    op.eval(leaves=sel)
    t3 = time.perf_counter()
    full = (t1 - t0) + (t2 - t1) + (t3 - t2) * (op.leaves / S)
    info = {"plan_s": round(t1 - t0, 3), "upward_s": round(t2 - t1, 3), "sample_eval_s": round(t3 - t2, 3),
            "sample_leaves": int(S), "leaves": int(op.leaves)}
    op.close()
    return full, t3 - t0, info


def cpu_baseline(w, tree, sample_leaves):
    import oracle
    full, spent, info = oracle_step(w, tree, sample_leaves)
    whole = info["sample_leaves"] == info["leaves"]
    return {"value": w.N / full, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "extrapolated": not whole,
            "sample": (f"serial-FMM oracle (gcc -O2, OpenMP over targets): one whole step (tree + lists + upward pass + all "
                       f"{info['leaves']} target leaves), {spent:.1f} s of CPU work" if whole else
                       f"serial-FMM oracle (gcc -O2, OpenMP over targets): full tree + lists + upward pass, then "
                       f"{info['sample_leaves']} of {info['leaves']} target leaves evaluated (near + far) and scaled by "
                       f"leaves/sample; {spent:.1f} s of CPU work"),
            "detail": info}


def run_reference(args):
    """The reference arm of this tier: the CPU oracle as it stands, whole steps (every target leaf) unless
    --cpu-sample-leaves asks for a bounded sample, in which case the line says "extrapolated": true and ms_per_step is the
    MEASURED time of a step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    w = workloads.config(args.config)
    for _ in range(min(args.warmup, 1)):
        oracle_step(w, args.tree, max(8, (args.cpu_sample_leaves or 64) // 4))
    tot, spent_tot, info = 0.0, 0.0, None
    for _ in range(args.steps):
        full, spent, info = oracle_step(w, args.tree, args.cpu_sample_leaves)
        tot += full
        spent_tot += spent
    whole = info["sample_leaves"] == info["leaves"]
    value = w.N * args.steps / tot
    sample = (f"each step: one whole oracle step (tree, lists, upward pass, all {info['leaves']} target leaves), "
              f"{spent_tot / args.steps:.1f} s CPU per step" if whole else
              f"each step: oracle tree + lists + upward pass in full, {info['sample_leaves']} of {info['leaves']} "
              f"target leaves evaluated; value scales the leaf part by leaves/sample, ms_per_step is the measured time "
              f"({spent_tot / args.steps:.1f} s CPU per step)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * spent_tot / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(w, args),
            "extrapolated": not whole,
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------------
# clocks during the timed region (B200_PROFILING.md "clocks line")
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.index = [], None, index

    def __enter__(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None
        return self

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def __exit__(self, *exc):
        if self.proc:
            time.sleep(0.15)
            self.proc.terminate()
            self.thread.join(timeout=2)

    def summary(self):
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); smax.append(float(r[1])); power.append(float(r[2]))
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except (ValueError, IndexError):
                continue
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(smax)), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": float(max(power))}


# ------------------------------------------------------------------------------------------------
# N > 1: replicas only.  The only cross-rank traffic is the barrier and this MAX.
# ------------------------------------------------------------------------------------------------
def max_over_ranks(ms, world, device=None):
    """Slowest rank's device time in ms (all_reduce MAX over the default process group when world > 1)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device if device is not None else "cpu")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(world, n_per_rank, steps, ms_total):
    """Whole-job particles/s: every rank evaluates its own replica of n_per_rank particles `steps` times."""
    return world * n_per_rank * steps / (ms_total * 1e-3)


def ncu_capture(w, tree):
    """Per-launch ncu counters of the committed capture of this workload (profiles/ncu_traffic.csv; the .md beside it
    names the command and the commit).  {kernel or stage: {...}}; empty if the capture is of another workload."""
    out = {}
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["workload"] == w.name and row["tree"] == tree:
                    out[row["kernel"]] = {"dram_bytes": int(row["dram_bytes_read"]) + int(row["dram_bytes_write"]),
                                          "launches": int(row.get("launches") or 1), "capture": row.get("capture", "")}
    except Exception:
        pass
    return out


PROBE_PATTERNS = [
    (0, "DFMA, one register source (v = fma(v, a, b), a and b kernel parameters)", "inst"),
    (1, "DFMA, three distinct register sources (v_k = fma(x_k, y_k, v_k))", "inst"),
    (2, "DFMA, three register sources of which one repeats in the neighbour (operand reuse)", "inst"),
    (3, "DMUL / DADD, two distinct register sources", "inst"),
    (4, "MUFU.RSQ64H", "inst"),
    (5, "one-sided near-field evaluation (25 FP64 instructions)", "eval"),
    (6, "mutual near-field pair = two evaluations (34 FP64 instructions)", "eval"),
]


def probe_fp64(pattern=0):
    """Thread-level instructions (or kernel evaluations) per second of one pattern of libfmm_probe.so."""
    import ctypes as C
    import torch
    from paper_2302_07567_b200 import build
    lib = C.CDLL(str(build.build_probe()))
    lib.fmm_probe_fp64.restype = C.c_int
    lib.fmm_probe_fp64.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double), C.c_void_p]
    rate, ms = C.c_double(), C.c_double()
    rc = lib.fmm_probe_fp64(pattern, C.byref(rate), C.byref(ms), C.c_void_p(torch.cuda.current_stream().cuda_stream))
    if rc != 0:
        raise RuntimeError(f"fmm_probe_fp64({pattern}) failed: {rc}")
    return float(rate.value)


def run_probe(args):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --probe-fp64 needs a CUDA device")
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    lanes = SM_COUNT * FP64_LANES_PER_SM * sm_max * 1e6   # thread-level FP64 instructions per second at one per lane and clock
    rows = []
    print(f"| pattern | rate | of {SM_COUNT} SMs x {FP64_LANES_PER_SM} lanes x {sm_max:.0f} MHz |")
    print("|---|---|---|")
    for k, name, unit in PROBE_PATTERNS:
        r = probe_fp64(k)
        if unit == "inst":
            print(f"| {name} | {r / 1e12:.2f} T inst/s | {100 * r / lanes:.1f} % |")
        else:
            print(f"| {name} | {r / 1e9:.1f} G evaluations/s = {r * FLOP_PER_EVAL / 1e12:.2f} TFLOP/s (34 flop) | "
                  f"{100 * r * FLOP_PER_EVAL / (2 * lanes):.1f} % of peak, {lanes / r:.1f} lane-cycles per evaluation |")
        rows.append({"pattern": k, "name": name, "rate": r})
    print(json.dumps({"probe_fp64": rows, "lanes_per_s": lanes}))


def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2302_07567_b200 import binding as fmm, build

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback; use --impl reference for the oracle)")
    if rank == 0:
        build.build_library()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
        dist.barrier()
    fmm.load_library()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = workloads.config(args.config)
    flags = fmm.FMM_TREE_KD if args.tree == "kd" else fmm.FMM_TREE_MORTON_MEDIAN
    if args.kernel == "source_momentum":
        flags |= fmm.FMM_KERNEL_SOURCE_MOMENTUM
    if args.method == "treecode":
        flags |= fmm.FMM_METHOD_TREECODE
    d_in = [torch.as_tensor(a).to(dev) for a in w.arrays()]
    out = torch.empty((6, w.N), dtype=torch.float64, device=dev)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)
    prm = dict(order_n=w.order_n, leaf_size=w.leaf_size, theta=w.theta, flags=flags, device=dev)

    plan = fmm.fmm_plan_create(*d_in, w.q, **prm)
    overlap = args.overlap
    plan.set_overlap(overlap)
    plan.set_timing(not overlap)   # per-stage events force the serial order: with overlap they are taken in a second pass

    plan_step = {"update": plan.update, "refit": plan.refit, "keep_lists": plan.refit_keep_lists}[args.plan_step]

    def step():
        plan_step(*d_in, w.q)       # a0-a3 (refit: without the sort; keep_lists: without the sort and the traversal)
        plan.eval(out)              # a4-a10

    for _ in range(args.warmup):
        step()
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    stage_ms = {}
    l0 = fmm.fmm_launch_count()
    with ClockSampler(local) as clk:
        for k in range(args.steps):
            flush.fill_(k & 0xff)
            ev[k][0].record()
            step()
            ev[k][1].record()
            st = plan.stats()
            if not overlap:
                for key in STAGE_KEYS:
                    stage_ms.setdefault(key, []).append(st[key])
        barrier()
        launches = fmm.fmm_launch_count() - l0
        ms_serial = None
        if overlap:
            # stage pass: the same K steps again, stages in serial order with CUDA events around every kernel group
            # (fmm_plan_set_timing); these are the per-kernel durations the roofline object uses
            plan.set_timing(True)
            sev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
            for k in range(args.steps):
                flush.fill_(k & 0xff)
                sev[k][0].record()
                step()
                sev[k][1].record()
                st = plan.stats()
                for key in STAGE_KEYS:
                    stage_ms.setdefault(key, []).append(st[key])
            barrier()
            ms_serial = sum(a.elapsed_time(b) for a, b in sev) / args.steps
            plan.set_timing(False)
    ms_total = max_over_ranks(sum(a.elapsed_time(b) for a, b in ev), world, dev)
    value = aggregate_throughput(world, w.N, args.steps, ms_total)
    clocks = clk.summary()

    # ---- end to end through the host entry point (pinned host buffers, copies inside the timed region)
    h_in = [torch.as_tensor(a).pin_memory() for a in w.arrays()]
    h_out = torch.empty((6, w.N), dtype=torch.float64).pin_memory()
    for _ in range(min(args.warmup, 2)):
        fmm.fmm_field_host(*h_in, w.q, out=h_out, **prm)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        fmm.fmm_field_host(*h_in, w.q, out=h_out, **prm)
    e1.record()
    barrier()
    e2e_value = aggregate_throughput(world, w.N, args.steps, max_over_ranks(e0.elapsed_time(e1), world, dev))

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel (live CUDA-event times from the library's own stage timers)
    stages = {k[3:]: float(np.mean(v)) for k, v in stage_ms.items()}
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    sm_max = float(peaks.get("sm_max_mhz", 1965.0))
    nominal = SM_COUNT * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    measured_dfma = 2.0 * probe_fp64(0) / 1e12
    dom = "p2p" if stages["p2p"] >= stages["m2l"] else "m2l"
    evals = {"p2p": st["p2p_pairs"], "m2l": st["m2l_pairs"]}
    ach = {k: evals[k] * FLOP_PER_EVAL / (stages[k] * 1e-3) / 1e12 for k in ("p2p", "m2l")}
    cap = ncu_capture(w, args.tree)
    dom_kernel = ("p2p_mutual_kernel" if st["p2p_mutual"] else "p2p_kernel") if dom == "p2p" else "m2l_kernel"
    roofline = {"bound": "alu", "kernel": dom_kernel, "achieved": ach[dom], "peak": nominal, "unit": "TFLOP/s",
                "frac": ach[dom] / nominal, "traffic": cap.get(dom_kernel, {}).get("dram_bytes"),
                "traffic_source": ("bytes per launch, ncu dram__bytes_read.sum + dram__bytes_write.sum of the committed capture "
                                   + cap.get(dom_kernel, {}).get("capture", "(none for this workload)") + " (profiles/ncu_traffic.md), "
                                   "not of this run"),
                "peak_source": f"FP64 vector pipe: {SM_COUNT} SMs x {FP64_LANES_PER_SM} lanes x 2 flop x {sm_max:.0f} MHz (DESIGN.md); "
                               "MEASURED_PEAKS.json has no FP64 entry",
                "measured_dfma_tflops": measured_dfma, "frac_of_measured_dfma": ach[dom] / measured_dfma,
                "flop_per_eval": FLOP_PER_EVAL,
                "p2p": {"evals": evals["p2p"], "ms": stages["p2p"], "tflops": ach["p2p"], "frac": ach["p2p"] / nominal,
                        "mutual": bool(st["p2p_mutual"])},
                "m2l": {"evals": evals["m2l"], "ms": stages["m2l"], "tflops": ach["m2l"], "frac": ach["m2l"] / nominal}}
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    # HBM-side rooflines of the tree / interpolation stages (north_star): ALGORITHMIC bytes (every array a
    # stage must read or write once) over the stage's CUDA-event time, against the measured copy bandwidth; beside them the
    # DRAM bytes ncu counted for the stage's kernels in the committed capture.  These stages are launch- and latency-bound
    # at N = 2^20 (a few MB to a few hundred MB per stage), so the fractions are small by nature.
    Pn = (w.order_n + 1) ** 3
    nodes, leaves_n = st["nodes"], st["leaves"]
    stage_bytes = {
        "tree": 128 * w.N,                                              # read x, p (48 B) + write tree-ordered x, weights, perm (60 B) + slack
        "lists": 8 * (st["n_p2p"] + st["n_m2l"]) * 3,                   # 64-bit pair keys: emit, deal to rows, CSR
        "p2m": 56 * w.N + 32 * Pn * leaves_n,
        "m2m": 32 * Pn * ((nodes - 1) + (nodes - leaves_n)),             # read every child once, write every parent once
        "l2l": 48 * Pn * (nodes - 1) * 2 + 48 * Pn * (nodes - leaves_n),  # read parent + child, write child
        # leaf expansions + positions, the near-field partial sums and reaction segments, perm, the six outputs
        "l2p": 48 * Pn * leaves_n + (24 + 48 * st["p2p_split"] + 4 + 48) * w.N + 48 * st["react_particles"],
    }
    stage_roof = {}
    for k, b in stage_bytes.items():
        if stages.get(k, 0) > 0:
            stage_roof[k] = {"bytes": int(b), "gbs": round(b / (stages[k] * 1e-3) / 1e9, 1),
                             "frac_of_hbm_peak": round(b / (stages[k] * 1e-3) / 1e9 / hbm, 4),
                             "ncu_dram_bytes": cap.get("stage:" + k, {}).get("dram_bytes")}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(w, args),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 6 * 8 * w.N, "d2h_bytes_per_step": 6 * 8 * w.N},
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
            "stages_ms": {k: round(v, 4) for k, v in stages.items()},
            "stages_hbm": stage_roof,
            "stage_timing": ("per-stage CUDA events of a second pass of the same K steps in serial stage order "
                             f"({ms_serial:.3f} ms/step); the timed region runs P2P on a second stream beside P2M/M2M/M2L/L2L"
                             if ms_serial is not None else "per-stage CUDA events inside the timed region (serial stage order)"),
            "lists": {"n_p2p": st["n_p2p"], "n_m2l": st["n_m2l"], "kappa": st["kappa"], "gamma_bar": st["gamma_bar"],
                      "p2p_split": st["p2p_split"], "m2l_split": st["m2l_split"]},
            "hbm_peak_gbs": hbm, "parallelism": "replicas only" if world > 1 else "single GPU"}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w, args.tree, args.cpu_sample_leaves)
        line["paper_context"] = "paper: GPU 57-197x over one CPU core (A100/V100/P100, PAPER.md:664); not the target"
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


# ------------------------------------------------------------------------------------------------
# error-versus-time sweeps (BASELINE.json configs[4]; the paper's Fig. 2 / Fig. 3)
# ------------------------------------------------------------------------------------------------
def run_sweep(args):
    """--config 5: N = 2^20 Gaussian bunch, n = 2..8 x theta in {0.3, 0.5, 0.7}, N0 = 256, plus the all-pairs direct sum at
    N = 262,144 (the FP64 ceiling of configs[4]).  --config 9: the paper's own sweep, N = 1.28e6 uniform cube, identical
    momenta (gamma = 50), n in {2, 4, 6, 8, 10} x eta in {0.3, 0.4, 0.5}, N0 = (n+1)^3.
    For every point: tree + lists (fmm_plan_update) and one evaluation (fmm_eval), both timed on the device (best of
    --steps repetitions after --warmup); the error is eq. (6.1) of the FMM result against direct summation
    (fmm_direct, a11) on a seeded sample of targets.  theta = 0.7 lies outside the range where Alg 5.6 / 5.7 guarantee
    disjoint boxes (G11): those rows are reported, nothing is expected of their accuracy.
    One JSON line: value = particles/s of the n = 6, theta = 0.5 point (config 9: n = 4, eta = 0.5); the table is in `sweep`."""
    import torch
    from paper_2302_07567_b200 import binding as fmm, build
    if int(os.environ.get("RANK", "0")) != 0:
        return
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA path has no CPU fallback)")
    build.build_library()
    fmm.load_library()
    dev = torch.device("cuda", int(os.environ.get("LOCAL_RANK", "0")))
    torch.cuda.set_device(dev)
    paper = args.config == 9
    if paper:
        w = workloads.paper_cube(N=1_280_000)
        orders, thetas, head = [2, 4, 6, 8, 10], [0.3, 0.4, 0.5], (4, 0.5)
    else:
        w = workloads.config(5)
        orders, thetas, head = [2, 3, 4, 5, 6, 7, 8], [0.3, 0.5, 0.7], (6, 0.5)
    flags = fmm.FMM_TREE_KD if args.tree == "kd" else fmm.FMM_TREE_MORTON_MEDIAN
    d_in = [torch.as_tensor(a).to(dev) for a in w.arrays()]
    tg = np.sort(np.random.default_rng(5005).choice(w.N, size=min(args.sweep_targets, w.N), replace=False)).astype(np.int64)
    tgd = torch.as_tensor(tg, device=dev)
    out = torch.empty((6, w.N), dtype=torch.float64, device=dev)
    reps = max(1, min(args.steps, 5))

    def timed(fn):
        best = None
        for _ in range(reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); fn(); e1.record(); e1.synchronize()
            ms = e0.elapsed_time(e1)
            best = ms if best is None else min(best, ms)
        return best

    rows, ref, value, head_ms = [], None, None, None
    with ClockSampler(dev.index or 0) as clk:
        for theta in thetas:
            for n in orders:
                N0 = (n + 1) ** 3 if paper else 256
                plan = fmm.fmm_plan_create(*d_in, w.q, order_n=n, leaf_size=N0, theta=theta, flags=flags, device=dev)
                plan.set_timing(True)
                for _ in range(min(args.warmup, 2)):
                    plan.update(*d_in, w.q); plan.eval(out)
                ms_plan = timed(lambda: (plan.update(*d_in, w.q), plan.stats()))
                ms_eval = timed(lambda: plan.eval(out))
                st = plan.stats()
                if ref is None:   # gamma_bar is a property of the bunch: one direct reference for the whole sweep
                    ref = fmm.fmm_direct(*d_in, w.q, gamma_bar=st["gamma_bar"], targets=tg, device=dev)
                errs = [float(torch.sqrt(((a - b) ** 2).sum() / (b ** 2).sum())) for a, b in ((out[:3, tgd], ref[0]), (out[3:, tgd], ref[1]))]
                nominal = SM_COUNT * FP64_LANES_PER_SM * 2 * 1.965e9
                row = dict(n=n, theta=theta, N0=N0, n_p2p=st["n_p2p"], n_m2l=st["n_m2l"], p2p_pairs=st["p2p_pairs"],
                           m2l_pairs=st["m2l_pairs"], ms_plan=round(ms_plan, 3), ms_eval=round(ms_eval, 3),
                           ms_p2p=round(st["ms_p2p"], 3), ms_m2l=round(st["ms_m2l"], 3),
                           p2p_frac=round(st["p2p_pairs"] * FLOP_PER_EVAL / max(st["ms_p2p"], 1e-6) / 1e-3 / nominal, 3),
                           m2l_frac=round(st["m2l_pairs"] * FLOP_PER_EVAL / max(st["ms_m2l"], 1e-6) / 1e-3 / nominal, 3),
                           particles_per_s=w.N / ((ms_plan + ms_eval) * 1e-3), err=max(errs), err_E=errs[0], err_B=errs[1])
                rows.append(row)
                if (n, theta) == head:
                    value, head_ms = row["particles_per_s"], ms_plan + ms_eval
                print(f"| {n} | {theta} | {N0} | {st['p2p_pairs']:.3e} | {st['m2l_pairs']:.3e} | {ms_plan:.2f} | {ms_eval:.2f} | "
                      f"{row['particles_per_s']:.3e} | {100 * row['p2p_frac']:.1f} % | {100 * row['m2l_frac']:.1f} % | {max(errs):.2e} |",
                      file=sys.stderr, flush=True)
                plan.close()
        allpairs = None
        if not paper:
            wa = workloads.config(6)
            a_in = [torch.as_tensor(a).to(dev) for a in wa.arrays()]
            fmm.fmm_direct(*a_in, wa.q, gamma_bar=10.0, device=dev)
            ms = timed(lambda: fmm.fmm_direct(*a_in, wa.q, gamma_bar=10.0, device=dev))
            tf = float(wa.N) ** 2 * FLOP_PER_EVAL / (ms * 1e-3) / 1e12
            allpairs = {"N": wa.N, "ms": ms, "tflops": tf, "frac_of_fp64_peak": tf / (SM_COUNT * FP64_LANES_PER_SM * 2 * 1.965e9 / 1e12)}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": 1, "steps": reps, "warmup": min(args.warmup, 2),
            "ms_per_step": head_ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": dict(workload_config(w, args), order_n=head[0], theta=head[1], sweep=True,
                                               l2="no flush: every point runs once per repetition, best of the repetitions"),
            "clocks": clk.summary(), "sweep": rows, "allpairs": allpairs,
            "sweep_columns": "n, theta, N0, list lengths, kernel evaluations, ms (tree+lists / evaluation / P2P / M2L), "
                             "fraction of FP64 peak (34 flop per evaluation), particles/s, eq. (6.1) error vs fmm_direct on "
                             f"{len(tg)} sampled targets"}
    print(json.dumps(line))


def main():
    args = parse_args()
    if args.probe_fp64:
        run_probe(args)
    elif args.impl == "reference":
        run_reference(args)
    elif args.config in (5, 9):
        run_sweep(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
