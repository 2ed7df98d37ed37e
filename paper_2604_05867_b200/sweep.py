"""Harness for BASELINE.json configs[2]: iterate until max_x D - I(p) < tol (R8: the stop test lives in the
harness, not in the library), for one or several d.  Marshalling only -- every BA step runs in libba.

    python -m paper_2604_05867_b200.sweep --n 20 --d 0.64 0.70 0.75 0.80 0.85 0.90 0.95 --tol 1e-6 --mode fast

Reports, per d: iterations, I(p), the current U = max_x D, the running minimum min_s U_s (R10: every U_s is a
valid upper bound), the paper's stop statistic U - log2 Z and (1/n) U / (1-d).
"""
import argparse
import json

import numpy as np

from . import (BA_MODE_ENUM, BA_MODE_FAST, ba_bounds, ba_create, ba_destroy, ba_get_history, ba_iterate,
               ba_set_mode)


def run_until_gap(n, d, tol=1e-6, max_iters=20000, chunk=100, mode=BA_MODE_FAST, device="cuda:0"):
    """Chunks of `chunk` iterations until U - I < tol or max_iters (G8: may not be reached within a cap)."""
    ctx = ba_create(n, d, device=device)
    try:
        ba_set_mode(ctx, mode)
        done, min_u, I, U, lz = 0, float("inf"), float("nan"), float("nan"), float("nan")
        while done < max_iters:
            k = min(chunk, max_iters - done)
            ba_iterate(ctx, k)
            done += k
            hist = ba_get_history(ctx, k)
            min_u = min(min_u, float(hist[:, 1].min()))
            I, U = ba_bounds(ctx)
            lz = float(hist[-1, 2])
            if U - I < tol:
                break
        return {"n": n, "d": d, "iterations": done, "I_lower": I, "maxD_upper": U, "running_min_upper": min_u,
                "gap": U - I, "gap_running_min": min_u - I, "stop_statistic_U_minus_log2Z": U - lz,
                "upper_over_n": min_u / n, "upper_over_n_over_1_minus_d": (min_u / n) / (1.0 - d) if d < 1 else None,
                "converged": bool(U - I < tol)}
    finally:
        ba_destroy(ctx)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--n", type=int, default=20)
    ap.add_argument("--d", type=float, nargs="+", default=[0.64, 0.70, 0.75, 0.80, 0.85, 0.90, 0.95])
    ap.add_argument("--tol", type=float, default=1e-6)
    ap.add_argument("--max-iters", type=int, default=20000)
    ap.add_argument("--chunk", type=int, default=100)
    ap.add_argument("--mode", choices=["enum", "fast"], default="fast")
    args = ap.parse_args()
    mode = BA_MODE_ENUM if args.mode == "enum" else BA_MODE_FAST
    for d in args.d:
        print(json.dumps(run_until_gap(args.n, d, args.tol, args.max_iters, args.chunk, mode)), flush=True)


if __name__ == "__main__":
    main()
