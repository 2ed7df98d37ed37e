"""BASELINE.json configs[0] and configs[1] through the binding (marshalling only): prints I, max D, log2 Z after K
iterations for the uniform start and, for configs[1], the seeded Dirichlet(1) start, in both modes.

    python -m paper_2604_05867_b200.configs
"""
import json
import os
import sys

from . import ba_bounds, ba_create, ba_destroy, ba_get_history, ba_iterate, ba_set_mode, ba_set_p, ba_stats


def run(n, d, K, p0=None, mode=0):
    ctx = ba_create(n, d)
    try:
        ba_set_mode(ctx, mode)
        if p0 is not None:
            ba_set_p(ctx, p0)
        ba_iterate(ctx, K)
        I, U = ba_bounds(ctx)
        lz, _ = ba_stats(ctx)
        h = ba_get_history(ctx, K)
        return dict(n=n, d=d, K=K, mode=mode, I=I, U=U, log2Z=lz, min_U=float(h[:, 1].min()), I0=float(h[0, 0]), U0=float(h[0, 1]))
    finally:
        ba_destroy(ctx)


def main():
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import synthetic_inputs as si                           # seeded starts shared with the tests (no method arithmetic)
    out = {}
    for mode in (0, 1):
        out[f"configs[0] uniform mode{mode}"] = run(8, 0.5, 200, None, mode)
        out[f"configs[1] uniform mode{mode}"] = run(14, 0.64, 500, None, mode)
        out[f"configs[1] dirichlet seed 0 mode{mode}"] = run(14, 0.64, 500, si.dirichlet_p0(14, 0), mode)
    print(json.dumps(out, indent=1))


if __name__ == "__main__":
    main()
