#!/usr/bin/env python
"""bench.py -- throughput of the whole hot path on BASELINE.json's
headline workload: configs[2], N = 1,048,576 uniformly filled ellipsoid, mean gamma 30, n = 6,
leaf 256, theta = 0.5, FP64, KD tree.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config I] [--tree kd|morton]

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
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-sample-leaves", type=int, default=4096,
                    help="target leaves the oracle evaluates in the cpu_baseline leg (the reference arm uses 1/8 of it per step)")
    return ap.parse_args()


def workload_config(w, tree):
    return {"workload": w.name, "N": w.N, "order_n": w.order_n, "leaf_size": w.leaf_size, "theta": w.theta,
            "tree": tree, "seed": w.seed, "precision": "fp64",
            "l2": "L2 flushed (256 MiB write) before every timed step; flush not timed"}


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
    return {"value": w.N / full, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
            "sample": (f"serial-FMM oracle (gcc -O2, OpenMP over targets): full tree + lists + upward pass, then "
                       f"{info['sample_leaves']} of {info['leaves']} target leaves evaluated (near + far) and scaled by "
                       f"leaves/sample; {spent:.1f} s of CPU work"),
            "detail": info}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    w = workloads.config(args.config)
    per_step = max(8, args.cpu_sample_leaves // 8)   # bounded sample: K steps must end within minutes
    for _ in range(min(args.warmup, 1)):
        oracle_step(w, args.tree, max(8, per_step // 4))
    tot, spent_tot, info = 0.0, 0.0, None
    for _ in range(args.steps):
        full, spent, info = oracle_step(w, args.tree, per_step)
        tot += full
        spent_tot += spent
    value = w.N * args.steps / tot
    sample = (f"each step: oracle tree + lists + upward pass in full, {info['sample_leaves']} of {info['leaves']} "
              f"target leaves evaluated and scaled by leaves/sample ({spent_tot / args.steps:.1f} s CPU per step)")
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": workload_config(w, args.tree),
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


def ncu_traffic(kernel, w, tree):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed `ncu --set full`
    capture (profiles/ncu_traffic.csv; the .md beside it names the command).  None if the capture is of another workload."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            for row in csv.DictReader(f):
                if row["kernel"] == kernel and row["workload"] == w.name and row["tree"] == tree:
                    return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
    except Exception:
        pass
    return None


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

    def step():
        plan.update(*d_in, w.q)     # a0-a3
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
    measured_dfma = fmm.fmm_probe_fp64_peak()
    dom = "p2p" if stages["p2p"] >= stages["m2l"] else "m2l"
    evals = {"p2p": st["p2p_pairs"], "m2l": st["m2l_pairs"]}
    ach = {k: evals[k] * FLOP_PER_EVAL / (stages[k] * 1e-3) / 1e12 for k in ("p2p", "m2l")}
    roofline = {"bound": "alu", "kernel": dom + "_kernel", "achieved": ach[dom], "peak": nominal, "unit": "TFLOP/s",
                "frac": ach[dom] / nominal, "traffic": ncu_traffic(dom + "_kernel", w, args.tree),
                "traffic_unit": "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum, profiles/ncu_traffic.csv)",
                "peak_source": f"FP64 vector pipe: {SM_COUNT} SMs x {FP64_LANES_PER_SM} lanes x 2 flop x {sm_max:.0f} MHz (DESIGN.md); "
                               "MEASURED_PEAKS.json has no FP64 entry",
                "measured_dfma_tflops": measured_dfma, "frac_of_measured_dfma": ach[dom] / measured_dfma,
                "flop_per_eval": FLOP_PER_EVAL,
                "p2p": {"evals": evals["p2p"], "ms": stages["p2p"], "tflops": ach["p2p"], "frac": ach["p2p"] / nominal},
                "m2l": {"evals": evals["m2l"], "ms": stages["m2l"], "tflops": ach["m2l"], "frac": ach["m2l"] / nominal}}
    hbm = float(peaks.get("hbm_gbs", 6650.0))
    # HBM-side rooflines of the tree / interpolation stages (north_star): ALGORITHMIC bytes (every array a
    # stage must read or write once) over the stage's CUDA-event time, against the measured copy bandwidth.  These stages are
    # launch- and latency-bound at N = 2^20 (a few MB to a few hundred MB per stage), so the fractions are small by nature.
    Pn = (w.order_n + 1) ** 3
    nodes, leaves_n = st["nodes"], st["leaves"]
    stage_bytes = {
        "tree": 128 * w.N,                                              # read x, p (48 B) + write tree-ordered x, weights, perm (60 B) + slack
        "lists": 8 * (st["n_p2p"] + st["n_m2l"]) * 3,                   # 64-bit pair keys: emit, sort, CSR
        "p2m": 56 * w.N + 32 * Pn * leaves_n,
        "m2m": 32 * Pn * ((nodes - 1) + (nodes - leaves_n)),             # read every child once, write every parent once
        "l2l": 48 * Pn * (nodes - 1) * 2 + 48 * Pn * (nodes - leaves_n),  # read parent + child, write child
        "l2p": 48 * Pn * leaves_n + (24 + 48 * st.get("p2p_split", 1) + 4 + 48) * w.N,
    }
    stage_roof = {k: {"bytes": int(b), "gbs": round(b / (stages[k] * 1e-3) / 1e9, 1), "frac_of_hbm_peak": round(b / (stages[k] * 1e-3) / 1e9 / hbm, 4)}
                  for k, b in stage_bytes.items() if stages.get(k, 0) > 0}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": dict(workload_config(w, args.tree), kernel=args.kernel, method=args.method),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 6 * 8 * w.N, "d2h_bytes_per_step": 6 * 8 * w.N},
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
            "stages_ms": {k: round(v, 4) for k, v in stages.items()},
            "stages_hbm": stage_roof,
            "stage_timing": ("per-stage CUDA events of a second pass of the same K steps in serial stage order "
                             f"({ms_serial:.3f} ms/step); the timed region runs P2P on a second stream beside P2M/M2M/M2L/L2L"
                             if ms_serial is not None else "per-stage CUDA events inside the timed region (serial stage order)"),
            "lists": {"n_p2p": st["n_p2p"], "n_m2l": st["n_m2l"], "kappa": st["kappa"], "gamma_bar": st["gamma_bar"]},
            "hbm_peak_gbs": hbm, "parallelism": "replicas only" if world > 1 else "single GPU"}
    if world == 1 and not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(w, args.tree, args.cpu_sample_leaves)
        line["paper_context"] = "paper: GPU 57-197x over one CPU core (A100/V100/P100, PAPER.md:664); not the target"
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_cuda(args)


if __name__ == "__main__":
    main()
