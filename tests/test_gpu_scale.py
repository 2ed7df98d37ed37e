"""GPU tests beyond the dense oracle's reach: trajectory parity at n=14,
and at n=20 / n=24 (the bench configuration) closed forms, invariants and sampled rows / columns recomputed
by independent CPU routines written here from the definitions (P:109 emb, P:140-158 BA step).
"""
import math
from math import comb

import numpy as np
import pytest

import synthetic_inputs as si
from oracle import oracle as orc

pytestmark = pytest.mark.gpu

REL_QD = 1e-12
ABS_U = 1e-10


@pytest.fixture(scope="module")
def ba():
    import paper_2604_05867_b200 as ba_mod
    ba_mod.load()
    return ba_mod


# ------------------------------------------------------------------ independent CPU routines (test-local)

def row_by_prefix_dp(x, n):
    """{code(y): emb(y,x)} for every distinct subsequence y of x: scan x left to right, every known y
    spawns y.b (cnt[y.b] += cnt[y]).  code(y) = 1<<|y| | val(y)."""
    cnt = {1: 1}
    for i in range(n):
        b = (x >> (n - 1 - i)) & 1
        add = {}
        for cy, e in cnt.items():
            c2 = (cy << 1) | b
            add[c2] = add.get(c2, 0) + e
        for c2, e in add.items():
            cnt[c2] = cnt.get(c2, 0) + e
    return cnt


def column_by_dp(yval, k, n):
    """emb(y, x) for all x in [0,2^n) at once: textbook DP over the positions of x, vectorised over x."""
    X = np.arange(1 << n, dtype=np.uint32)
    e = [np.ones(1 << n, dtype=np.uint32)] + [np.zeros(1 << n, dtype=np.uint32) for _ in range(k)]
    for i in range(n):
        xb = (X >> np.uint32(n - 1 - i)) & np.uint32(1)
        for r in range(min(k, i + 1), 0, -1):
            yb = (yval >> (k - r)) & 1
            e[r] += np.where(xb == yb, e[r - 1], np.uint32(0))
    return e[k]


def weights(n, d):
    return [(1.0 - d) ** k * d ** (n - k) if 0 < d < 1 else float((k == n) if d == 0 else (k == 0)) for k in range(n + 1)]


def D_row(x, n, d, q):
    w = weights(n, d)
    terms = []
    for cy, e in row_by_prefix_dp(x, n).items():
        k = cy.bit_length() - 1
        W = w[k] * e
        if W > 0.0:
            terms.append(W * (math.log2(W) - math.log2(q[cy - 1])))
    return math.fsum(terms), len(terms)


# ------------------------------------------------------------------ T5 config 2

@pytest.mark.parametrize("start", ["uniform", "dirichlet"])
def test_T5_trajectory_config2(ba, start):
    n, d, K = 14, 0.64, 500
    p0 = si.uniform_p0(n) if start == "uniform" else si.dirichlet_p0(n, 0)
    ref = orc.ba_run(orc.channel(n, d), p0, K)
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_set_p(ctx, p0)
        ba.ba_iterate(ctx, K)
        I, U = ba.ba_bounds(ctx)
        hist = ba.ba_get_history(ctx, K)
        p = ba.ba_get_p(ctx)
    finally:
        ba.ba_destroy(ctx)
    assert abs(U - ref["hist"][-1, 1]) <= ABS_U and abs(I - ref["hist"][-1, 0]) <= ABS_U
    assert np.max(np.abs(hist - ref["hist"])) <= ABS_U
    assert np.max(np.abs(p - ref["p"]) / ref["p"]) <= 1e-8
    assert np.all(np.diff(hist[:, 0]) >= -1e-13)              # I_t non-decreasing (Theorem 1)
    assert np.all(hist[:, 0] <= hist[:, 2] + 1e-13) and np.all(hist[:, 2] <= hist[:, 1] + 1e-13)   # I <= log2 Z <= U
    # R11: both starts bracket C_14(0.64) in [2.208857, 2.209342] (SURVEY P13 scratch, secondary)
    assert I <= 2.209342 + 1e-6 and U >= 2.208857 - 1e-6


# ------------------------------------------------------------------ T7 scale checks

def scale_checks(ba, n, d, n_rows, n_cols, seed):
    rng = np.random.default_rng(seed)
    NX = 1 << n
    w = weights(n, d)
    ctx = ba.ba_create(n, d)
    try:
        cnt = ba.ba_debug_count_terms(ctx)                    # P1/P2/P4 as device-side integer checksums
        assert cnt["in_terms"] == cnt["out_terms"] == ba.ba_terms_per_sweep(n)
        assert cnt["in_emb_sum"] == cnt["out_emb_sum"] == 4 ** n
        # ---- iteration 0 from uniform p: closed forms
        ba.ba_iterate(ctx, 1)
        q0, D0 = ba.ba_get_q(ctx), ba.ba_get_D(ctx)
        I0, U0 = ba.ba_bounds(ctx)
        for k in range(n + 1):                                # P6: q_0(y) = C(n,k) w_k / 2^k for every y
            want = comb(n, k) * w[k] / 2.0 ** k
            blk = q0[(1 << k) - 1:(2 << k) - 1]
            assert np.max(np.abs(blk - want)) <= REL_QD * want
        assert abs(D0[0] - n * (1 - d)) <= REL_QD * n and abs(D0[NX - 1] - n * (1 - d)) <= REL_QD * n   # P8
        assert abs(U0 - n * (1 - d)) <= REL_QD * n and I0 <= U0
        xs = [0b0101010101010101010101010101 & (NX - 1), 1, NX - 2] + [int(v) for v in rng.integers(0, NX, n_rows)]
        for x in xs:                                          # P8b / P14: sampled rows by an independent routine
            want, nt = D_row(x, n, d, q0)
            assert abs(D0[x] - want) <= REL_QD * abs(want), f"D0[{x}] ({nt} terms)"
        # ---- iteration 1 from the (non-uniform) p_1
        p1 = ba.ba_get_p(ctx)
        assert abs(math.fsum(p1) - 1.0) <= 1e-12
        ba.ba_iterate(ctx, 1)
        q1, D1 = ba.ba_get_q(ctx), ba.ba_get_D(ctx)
        I1, U1 = ba.ba_bounds(ctx)
        lz, its = ba.ba_stats(ctx)
        assert its == 2 and I0 <= I1 + 1e-13 and I1 <= lz + 1e-13 and lz <= U1 + 1e-13           # P10
        for k in range(n + 1):                                # P7: per-length mass
            want = comb(n, k) * w[k]
            assert abs(math.fsum(q1[(1 << k) - 1:(2 << k) - 1]) - want) <= 1e-12 * want
        rev = np.zeros(NX, dtype=np.int64)                    # P11: symmetry under cpl and rev (Theorem 4)
        X = np.arange(NX, dtype=np.int64)
        for i in range(n):
            rev |= ((X >> i) & 1) << (n - 1 - i)
        assert np.max(np.abs(D1 - D1[(NX - 1) - X])) <= 1e-11 and np.max(np.abs(D1 - D1[rev])) <= 1e-11
        assert np.max(np.abs(p1 - p1[rev]) / p1) <= 1e-11
        assert abs(U1 - D1.max()) <= 1e-15 and abs(I1 - math.fsum(p1 * D1)) <= 1e-12
        for x in xs[:max(4, n_rows // 2)]:                    # sampled rows with the downloaded q_1
            want, _ = D_row(x, n, d, q1)
            assert abs(D1[x] - want) <= REL_QD * abs(want), f"D1[{x}]"
        for _ in range(n_cols):                               # sampled columns with the downloaded p_1
            k = int(rng.integers(max(1, n // 2 - 3), n // 2 + 4))
            yv = int(rng.integers(0, 1 << k))
            e = column_by_dp(yv, k, n)
            want = w[k] * math.fsum((e.astype(np.float64) * p1)[e > 0])
            got = q1[(1 << k) - 1 + yv]
            assert abs(got - want) <= REL_QD * want, f"q1[y={yv:0{k}b}]"
            col = ba.ba_debug_emb_col(ctx, (1 << k) - 1 + yv)
            assert np.array_equal(col, e)                     # emb bit-exact along the whole column
        x = xs[3]
        row = ba.ba_debug_emb_row(ctx, x)                     # emb bit-exact along a whole row
        ref = row_by_prefix_dp(x, n)
        assert int(np.count_nonzero(row)) == len(ref)
        for cy, e in ref.items():
            assert row[cy - 1] == e
    finally:
        ba.ba_destroy(ctx)


def test_T7_scale_n20(ba):
    scale_checks(ba, 20, 0.80, n_rows=12, n_cols=3, seed=20)


def test_T7_scale_n24_bench_config(ba):
    # BASELINE.json configs[3]: n=24, d=0.70, uniform p0 -- the launch configuration bench.py times
    scale_checks(ba, 24, 0.70, n_rows=6, n_cols=2, seed=24)


# ------------------------------------------------------------------ T8 boundary errors that need a context

def test_T8_state_and_argument_errors(ba):
    n = 6
    ctx = ba.ba_create(n, 0.5)
    try:
        for fn in (ba.ba_bounds, ba.ba_get_q, ba.ba_get_D, ba.ba_last_timing):
            with pytest.raises(ba.BAError) as ei:
                fn(ctx)
            assert ei.value.code == ba.BA_ESTATE
        with pytest.raises(ba.BAError) as ei:
            ba.ba_iterate(ctx, -1)
        assert ei.value.code == ba.BA_EINVAL
        ba.ba_iterate(ctx, 0)
        assert ba.ba_iters_done(ctx) == 0
        with pytest.raises(ba.BAError) as ei:
            ba.ba_set_mode(ctx, 7)
        assert ei.value.code == ba.BA_EINVAL
        p = si.uniform_p0(n)
        for bad in (p * 1.001, np.where(np.arange(1 << n) == 3, 0.0, p), np.where(np.arange(1 << n) == 3, np.nan, p),
                    np.where(np.arange(1 << n) == 3, -p, p)):
            with pytest.raises(ba.BAError) as ei:
                ba.ba_set_p(ctx, bad)
            assert ei.value.code == ba.BA_EINVAL
        with pytest.raises(ba.BAError):
            ba.ba_debug_emb_row(ctx, 1 << n)
        with pytest.raises(ba.BAError):
            ba.ba_debug_emb_col(ctx, (2 << n) - 1)
        with pytest.raises(ba.BAError):
            ba.ba_get_history(ctx, 1)
        ba.ba_iterate(ctx, 3)
        assert ba.ba_get_history(ctx, 3).shape == (3, 3)
        assert np.array_equal(ba.ba_get_p(ctx) > 0, np.ones(1 << n, dtype=bool))
    finally:
        ba.ba_destroy(ctx)
    lib_ctx = ba.ba_create(n, 0.5, use_torch_memory=False)    # library-owned buffers and stream
    try:
        ba.ba_iterate(lib_ctx, 2)
        I, U = ba.ba_bounds(lib_ctx)
        assert 0 < I <= U
    finally:
        ba.ba_destroy(lib_ctx)


# ------------------------------------------------------------------ configs[2] harness (stop rule R8, bounds R10)

@pytest.mark.parametrize("mode", [0, 1])
def test_config3_harness_small(ba, mode):
    from paper_2604_05867_b200 import sweep
    r = sweep.run_until_gap(8, 0.5, tol=1e-6, max_iters=6000, chunk=250, mode=mode)
    assert r["converged"] and r["gap"] < 1e-6 and r["iterations"] <= 6000
    # C_8(0.5) = 2.123006166059 (secondary pin): I <= C <= running min U, both within the gap
    assert r["I_lower"] <= 2.123006166059 + 1e-9 <= r["running_min_upper"] + 2e-9
    assert r["running_min_upper"] - r["I_lower"] < 1e-6 and r["stop_statistic_U_minus_log2Z"] <= r["gap"] + 1e-12
    assert r["upper_over_n_over_1_minus_d"] == pytest.approx(r["running_min_upper"] / 8 / 0.5)


@pytest.mark.slow
def test_T7_scale_n28_config5(ba):
    # BASELINE.json configs[4]: n=28, d=0.80 (34 GB on the device, ~8 minutes on a B200, ~20 GB of host arrays).
    # Opt-in: BA_RUN_N28=1.  Result of the round-1 run: profiles/r01c_scale_n28.md.
    import os
    if os.environ.get("BA_RUN_N28") != "1":
        pytest.skip("set BA_RUN_N28=1 to run the n=28 scale check")
    scale_checks(ba, 28, 0.80, n_rows=3, n_cols=0, seed=28)


# ------------------------------------------------------------------ one-step parity at the oracle's reach, extreme d

@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("d,seed", [(0.95, None), (0.95, 3), (0.05, 4)])
def test_T3_T4_one_step_n14_extreme_d(ba, d, seed, mode):
    # configs[2] sweeps d up to 0.95: the hoisted logarithm must keep 1e-12 on D where D itself is small
    n = 14
    p = si.uniform_p0(n) if seed is None else si.random_positive_p(n, seed)
    ref = orc.ba_step(orc.channel(n, d), p)
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_set_mode(ctx, mode)
        ba.ba_set_p(ctx, p)
        ba.ba_iterate(ctx, 1)
        q, D = ba.ba_get_q(ctx), ba.ba_get_D(ctx)
        I, U = ba.ba_bounds(ctx)
    finally:
        ba.ba_destroy(ctx)
    assert np.max(np.abs(q - ref["q"]) / ref["q"]) <= REL_QD
    assert np.max(np.abs(D - ref["D"]) / np.abs(ref["D"])) <= REL_QD
    assert abs(I - ref["I"]) <= REL_QD * max(1.0, abs(ref["I"])) and abs(U - ref["U"]) <= REL_QD * max(1.0, abs(ref["U"]))
