"""The paper's own workload through libba: capacities C_{n,k} of the exact deletion channels BDC_{n,k} for k = 1..n
(P:107-115), each run stopped on the paper's rule, and their combination into upper bounds on C_n(d) and C(d) for
every deletion probability d from ONE set of runs (Lemma 2; Lemma 1; the reason the paper
works with BDC_{n,k}).

    python -m paper_2604_05867_b200.exact --n 16 [--a 0.005] [--d 0.5 0.64 0.7 ...] [--mode enum|fast] [--symmetry]

Only argument marshalling and the harness arithmetic of Lemma 2 live here; every BA step runs in the CUDA kernels
(ba_set_exact, ba_iterate).  Stop rule (R8): iterate until U_t - log2 Z_t < a, then the paper reports
"rate + a"; here both rigorous brackets are kept: I_t <= C_{n,k} <= min_s U_s.
"""
import argparse
import json
from math import comb

from . import (BA_MODE_ENUM, BA_MODE_FAST, ba_bounds, ba_create, ba_destroy, ba_get_history, ba_iterate, ba_set_exact,
               ba_set_mode, ba_set_symmetry, ba_stats)


def capacity_nk(n, k, a=0.005, max_iters=20000, chunk=50, mode=BA_MODE_ENUM, symmetry=False, device="cuda:0"):
    """BA on BDC_{n,k} from the uniform start until U - log2 Z < a or max_iters.
    Returns dict(k, I_lower, U_upper (running minimum of U), stop_statistic, iterations, converged)."""
    ctx = ba_create(n, 0.5, device=device)                      # d is irrelevant once the exact channel is selected
    try:
        ba_set_mode(ctx, mode)
        ba_set_exact(ctx, k)
        if symmetry:
            ba_set_symmetry(ctx, 1)
        done, min_u, stat, I = 0, float("inf"), float("inf"), 0.0
        while done < max_iters:
            step = min(chunk, max_iters - done)
            ba_iterate(ctx, step)
            done += step
            hist = ba_get_history(ctx, step)                    # {I_t, U_t, log2 Z_t} of the chunk
            min_u = min(min_u, float(hist[:, 1].min()))
            I, U = ba_bounds(ctx)
            lz, _ = ba_stats(ctx)
            stat = U - lz                                       # max_x log2(p_{t+1}(x) / p_t(x))
            if stat < a:
                break
        return dict(k=k, I_lower=I, U_upper=min_u, stop_statistic=stat, iterations=done, converged=stat < a)
    finally:
        ba_destroy(ctx)


def lemma2_bound(n, d, upper):
    """Lemma 2: C_n(d) <= sum_{k=1..n} C(n,k) d^{n-k} (1-d)^k C_{n,k}, with upper[k] >= C_{n,k}."""
    return sum(comb(n, k) * d ** (n - k) * (1.0 - d) ** k * upper[k] for k in range(1, n + 1))


def run(n, a=0.005, ds=(0.1, 0.2, 0.3, 0.4, 0.5, 0.6, 0.64, 0.7, 0.8, 0.9), mode=BA_MODE_ENUM, symmetry=False,
        max_iters=20000, device="cuda:0"):
    """All C_{n,k}, k = 1..n, and the bounds on C_n(d), C(d) <= C_n(d)/n (Lemma 1) for every d of `ds`."""
    rows = [capacity_nk(n, k, a=a, max_iters=max_iters, mode=mode, symmetry=symmetry and n >= 9, device=device)
            for k in range(1, n + 1)]
    upper = {r["k"]: r["U_upper"] for r in rows}
    lower = {r["k"]: r["I_lower"] for r in rows}
    bounds = []
    for d in ds:
        ub = lemma2_bound(n, d, upper)
        bounds.append(dict(d=d, Cn_upper=ub, Cd_upper=ub / n, Cd_upper_over_1_minus_d=ub / n / (1.0 - d) if d < 1 else None,
                           lemma2_with_lower_brackets=lemma2_bound(n, d, lower)))
    return dict(n=n, a=a, capacities=rows, bounds=bounds)


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--n", type=int, default=12)
    ap.add_argument("--a", type=float, default=0.005, help="tolerance of the paper's stop rule (P:600)")
    ap.add_argument("--d", type=float, nargs="*", default=[0.1, 0.2, 0.3, 0.4, 0.5, 0.6, 0.64, 0.7, 0.8, 0.9])
    ap.add_argument("--mode", choices=["enum", "fast"], default="enum")
    ap.add_argument("--symmetry", action="store_true", help="complement symmetry (ENUM mode, n >= 9)")
    ap.add_argument("--max-iters", type=int, default=20000)
    args = ap.parse_args()
    res = run(args.n, a=args.a, ds=args.d, mode=BA_MODE_ENUM if args.mode == "enum" else BA_MODE_FAST,
              symmetry=args.symmetry, max_iters=args.max_iters)
    for r in res["capacities"]:
        print(f"C_{{{args.n},{r['k']}}} in [{r['I_lower']:.6f}, {r['U_upper']:.6f}]  (U - log2 Z = {r['stop_statistic']:.2e} "
              f"after {r['iterations']} iterations{'' if r['converged'] else ', NOT converged'})")
    for b in res["bounds"]:
        print(f"d = {b['d']:.2f}:  C_n(d) <= {b['Cn_upper']:.6f}   C(d) <= C_n(d)/n <= {b['Cd_upper']:.6f}"
              f"   = {b['Cd_upper_over_1_minus_d']:.4f} (1-d)")
    print(json.dumps(res))


if __name__ == "__main__":
    main()
