"""Test-local CPU routines used beyond the dense oracle's reach: independent restatements
of the definitions, each pinned on CPU against oracle/ (tests/test_oracle_pins.py::test_cpu_routines_*) before the
GPU tests rely on them.  Test infrastructure only: nothing here is imported by the product."""
import numpy as np


def column_by_dp(yval, k, n):
    """emb(y, x) for all x in [0,2^n) at once: textbook DP over the positions of x (e[r] = #embeddings of y[0:r]
    in the scanned prefix), vectorised over x.  uint32[2^n]."""
    X = np.arange(1 << n, dtype=np.uint32)
    e = [np.ones(1 << n, dtype=np.uint32)] + [np.zeros(1 << n, dtype=np.uint32) for _ in range(k)]
    for i in range(n):
        xb = (X >> np.uint32(n - 1 - i)) & np.uint32(1)
        for r in range(min(k, i + 1), 0, -1):
            yb = (yval >> (k - r)) & 1
            e[r] += np.where(xb == yb, e[r - 1], np.uint32(0))
    return e[k]


def weights(n, d):
    """w_k = (1-d)^k d^(n-k) with 0^0 = 1 (R7), as python floats."""
    return [(1.0 - d) ** k * d ** (n - k) if 0 < d < 1 else float((k == n) if d == 0 else (k == 0)) for k in range(n + 1)]


def bit_reverse_table(n):
    """rev[x] = x with its n bits reversed (the paper's rev), int64[2^n]."""
    X = np.arange(1 << n, dtype=np.int64)
    rev = np.zeros(1 << n, dtype=np.int64)
    for i in range(n):
        rev |= ((X >> i) & 1) << (n - 1 - i)
    return rev
