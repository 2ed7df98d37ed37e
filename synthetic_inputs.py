"""Seeded synthetic inputs shared by the oracle-side tests and the CUDA-side tests / bench.

Holds none of the method's arithmetic: only the starting distributions p0 that
BASELINE.json's configs name, so that both sides start from
bit-identical float64 arrays.  The workload of this paper is fully determined by (n, d, p0);
no public dataset or benchmark suite is involved.
"""
import numpy as np

# BASELINE.json configs[0..4] as (n, d) pairs; configs[2] sweeps d.
CONFIGS = {
    "config1": dict(n=8, d=0.5, K=200),
    "config2": dict(n=14, d=0.64, K=500),
    "config3": dict(n=20, d_sweep=(0.64, 0.70, 0.75, 0.80, 0.85, 0.90, 0.95)),
    "config4": dict(n=24, d=0.70, warmup=5, K=100),
    "config5": dict(n=28, d=0.80, K=20),
}


def uniform_p0(n):
    """p0(x) = 1/2^n (BASELINE.json configs[0..4]; P:138 'a common choice')."""
    return np.full(1 << n, 1.0 / (1 << n), dtype=np.float64)


def dirichlet_p0(n, seed=0):
    """Seeded Dirichlet(1) start over {0,1}^n (BASELINE.json configs[1], seed 0)."""
    return np.random.default_rng(seed).dirichlet(np.ones(1 << n)).astype(np.float64)


def random_positive_p(n, seed):
    """A strictly positive normalised vector with a wide dynamic range (log-uniform over
    ~12 decades), mimicking the spread p develops under BA."""
    rng = np.random.default_rng(seed)
    v = np.exp(rng.uniform(-28.0, 0.0, size=1 << n))
    v /= v.sum()
    # renormalise once more in float64 so that |sum-1| is at rounding level
    return (v / v.sum()).astype(np.float64)
