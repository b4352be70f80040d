"""Error-versus-time sweep of the FMM (BASELINE.json configs[4]; the paper's Fig. 2).

    python -m paper_2302_07567_b200.sweep [--N 1048576] [--orders 2 3 4 5 6 7 8] [--thetas 0.3 0.5 0.7]
                                          [--leaf 256 | --paper-leaf] [--workload gaussian|paper_cube]
                                          [--targets 4096] [--allpairs 262144] [--json out.jsonl]

For every (n, theta): tree + lists (fmm_plan_update) and one evaluation (fmm_eval), both timed on the device;
the error is eq. (6.1) of the FMM result against direct summation (fmm_direct, a11) on a seeded
sample of target particles.  theta = 0.7 lies outside the range where Alg 5.6/5.7 guarantee disjoint boxes
(reading G11): those rows are reported, nothing is expected of their accuracy.
--allpairs times the all-pairs direct sum (configs[4]'s "FP64 roofline ceiling", N = 262,144).
Everything runs on cuda:0 through the C ABI; there is no CPU path.
"""
from __future__ import annotations

import argparse
import json

import numpy as np
import torch

from . import binding as fmm
from . import workloads

FLOP_PER_EVAL = 34
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12


def err61(f, fref):
    """eq. (6.1): max over E, B of the relative l2 error over the sample; f = (E[3,k], B[3,k])."""
    out = []
    for a, b in zip(f, fref):
        out.append(float(torch.sqrt(((a - b) ** 2).sum() / (b ** 2).sum())))
    return max(out), out


def timed(fn):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    r = fn()
    e1.record()
    e1.synchronize()
    return r, e0.elapsed_time(e1)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--N", type=int, default=1_048_576)
    ap.add_argument("--orders", type=int, nargs="+", default=[2, 3, 4, 5, 6, 7, 8])
    ap.add_argument("--thetas", type=float, nargs="+", default=[0.3, 0.5, 0.7])
    ap.add_argument("--leaf", type=int, default=256)
    ap.add_argument("--paper-leaf", action="store_true", help="N0 = (n+1)^3 as in the paper (PAPER.md:517)")
    ap.add_argument("--workload", default="gaussian", choices=["gaussian", "paper_cube"])
    ap.add_argument("--targets", type=int, default=4096)
    ap.add_argument("--allpairs", type=int, default=262_144)
    ap.add_argument("--json", default=None)
    args = ap.parse_args()

    dev = torch.device("cuda", 0)
    fmm.load_library()
    if args.workload == "gaussian":
        w = workloads.config(5, N=args.N)
    else:
        w = workloads.paper_cube(N=args.N)
    d_in = [torch.as_tensor(a).to(dev) for a in w.arrays()]
    tg = np.sort(np.random.default_rng(5005).choice(w.N, size=min(args.targets, w.N), replace=False)).astype(np.int64)
    rows = []
    ref = None
    print(f"# workload {w.name} N={w.N} seed={w.seed}; error on {len(tg)} sampled targets vs fmm_direct")
    print("| n | theta | N0 | P2P pairs | M2L pairs | plan ms | eval ms | particles/s (plan+eval) | err (6.1) | err E | err B |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    for theta in args.thetas:
        for n in args.orders:
            N0 = (n + 1) ** 3 if args.paper_leaf else args.leaf
            plan = fmm.fmm_plan_create(*d_in, w.q, order_n=n, leaf_size=N0, theta=theta, device=dev)
            _, ms_plan = timed(lambda: plan.update(*d_in, w.q))
            plan.eval()                                        # warm-up (first launch of this order's kernels)
            (E, B), ms_eval = timed(lambda: plan.eval())
            st = plan.stats()
            if ref is None:                                    # gamma_bar is a property of the bunch: one reference
                ref = fmm.fmm_direct(*d_in, w.q, gamma_bar=st["gamma_bar"], targets=tg, device=dev)
            tgd = torch.as_tensor(tg, device=dev)
            e, (eE, eB) = err61((E[:, tgd], B[:, tgd]), ref)
            row = dict(n=n, theta=theta, N0=N0, n_p2p=st["n_p2p"], n_m2l=st["n_m2l"], p2p_pairs=st["p2p_pairs"],
                       m2l_pairs=st["m2l_pairs"], ms_plan=ms_plan, ms_eval=ms_eval, particles_per_s=w.N / ((ms_plan + ms_eval) * 1e-3),
                       err=e, err_E=eE, err_B=eB, workload=w.name, N=w.N)
            rows.append(row)
            print(f"| {n} | {theta} | {N0} | {st['p2p_pairs']:.3e} | {st['m2l_pairs']:.3e} | {ms_plan:.2f} | {ms_eval:.2f} | "
                  f"{row['particles_per_s']:.3e} | {e:.2e} | {eE:.2e} | {eB:.2e} |", flush=True)
            plan.close()
    if args.allpairs > 0:
        wa = workloads.config(6, N=args.allpairs)
        a_in = [torch.as_tensor(a).to(dev) for a in wa.arrays()]
        fmm.fmm_direct(*a_in, wa.q, gamma_bar=10.0, device=dev)
        _, ms = timed(lambda: fmm.fmm_direct(*a_in, wa.q, gamma_bar=10.0, device=dev))
        evals = float(wa.N) ** 2
        tf = evals * FLOP_PER_EVAL / (ms * 1e-3) / 1e12
        print(f"\nall-pairs direct sum N={wa.N}: {ms:.2f} ms, {evals / (ms * 1e-3):.3e} evaluations/s, "
              f"{tf:.2f} TFLOP/s (34 flop/evaluation) = {100 * tf / FP64_NOMINAL_TFLOPS:.1f} % of {FP64_NOMINAL_TFLOPS:.2f} TFLOP/s")
        rows.append(dict(allpairs_N=wa.N, ms=ms, tflops=tf, frac=tf / FP64_NOMINAL_TFLOPS))
    if args.json:
        with open(args.json, "w") as f:
            for r in rows:
                f.write(json.dumps(r) + "\n")


if __name__ == "__main__":
    main()
