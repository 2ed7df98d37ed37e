"""GPU tests beyond the dense oracle's reach: trajectory parity at n=14,
and at n=20 / n=24 (the bench configuration) / n=26 closed forms, invariants, 64 sampled rows recomputed by the oracle
itself (orc_emb_row / orc_D_row: P:109 keep-mask enumeration of one input), sampled columns by a DP pinned
on CPU against the dense oracle, and all-entries agreement of the enumerating path with the FAST path on an asymmetric p.
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


# ------------------------------------------------------------------ the oracle at full size, one row at a time

from tests.cpu_routines import column_by_dp, weights, bit_reverse_table     # pinned on CPU in tests/test_oracle_pins.py


def oracle_rows(n, xs):
    """{x: emb row of x} from oracle/ (orc_emb_row, keep-mask enumeration of one input); rows in parallel
    threads (the C call releases the GIL)."""
    from concurrent.futures import ThreadPoolExecutor
    import os
    xs = sorted(set(int(x) for x in xs))
    with ThreadPoolExecutor(max_workers=min(16, os.cpu_count() or 1)) as ex:
        rows = list(ex.map(lambda x: orc.emb_row(n, x), xs))
    return dict(zip(xs, rows))


def check_rows_against_oracle(n, d, rows, q, D, what):
    """D(x) of the device vs the oracle's plain definition (orc_D_row) on the device's own q."""
    worst = 0.0
    for x, row in rows.items():
        want, nt = orc.D_row(n, d, row, q)
        err = abs(D[x] - want) / abs(want)
        worst = max(worst, err)
        assert err <= REL_QD, f"{what}: D[{x}] = {D[x]!r}, oracle {want!r} ({nt} terms), rel {err:.3g}"
    return worst


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

def sample_inputs(n, n_rows, rng):
    NX = 1 << n
    alt = int("01" * n, 2) & (NX - 1)                          # alternating string: the most distinct subsequences
    fixed = [0, NX - 1, alt, alt ^ (NX - 1), 1, NX - 2, (1 << (n // 2)) - 1, int("0011" * n, 2) & (NX - 1)]
    return fixed + [int(v) for v in rng.integers(0, NX, max(0, n_rows - len(fixed)))]


def scale_checks(ba, n, d, n_rows, n_cols, seed, asym=True):
    rng = np.random.default_rng(seed)
    NX = 1 << n
    w = weights(n, d)
    xs = sample_inputs(n, n_rows, rng)
    rows = oracle_rows(n, xs)                                 # ~64 rows, from oracle/ itself
    ctx = ba.ba_create(n, d)
    try:
        cnt = ba.ba_debug_count_terms(ctx)                    # P1/P2/P4 as device-side integer checksums
        assert cnt["in_terms"] == cnt["out_terms"] == ba.ba_terms_per_sweep(n)
        assert cnt["in_emb_sum"] == cnt["out_emb_sum"] == 4 ** n
        for x in xs[:6]:                                      # emb bit-exact along whole rows (max-node row included)
            assert np.array_equal(ba.ba_debug_emb_row(ctx, x), rows[x]), f"emb row {x}"
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
        check_rows_against_oracle(n, d, rows, q0, D0, "iteration 0")
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
        rev = bit_reverse_table(n)                            # P11: symmetry under cpl and rev (Theorem 4)
        X = np.arange(NX, dtype=np.int64)
        assert np.max(np.abs(D1 - D1[(NX - 1) - X])) <= 1e-11 and np.max(np.abs(D1 - D1[rev])) <= 1e-11
        assert np.max(np.abs(p1 - p1[rev]) / p1) <= 1e-11
        assert abs(U1 - D1.max()) <= 1e-15 and abs(I1 - math.fsum(p1 * D1)) <= 1e-12
        check_rows_against_oracle(n, d, rows, q1, D1, "iteration 1")
        for _ in range(n_cols):                               # sampled columns with the downloaded p_1
            k = int(rng.integers(max(1, n // 2 - 3), n // 2 + 4))
            yv = int(rng.integers(0, 1 << k))
            e = column_by_dp(yv, k, n)
            want = w[k] * math.fsum((e.astype(np.float64) * p1)[e > 0])
            got = q1[(1 << k) - 1 + yv]
            assert abs(got - want) <= REL_QD * want, f"q1[y={yv:0{k}b}]"
            col = ba.ba_debug_emb_col(ctx, (1 << k) - 1 + yv)
            assert np.array_equal(col, e)                     # emb bit-exact along the whole column
        if not asym:
            return
        # ---- an ASYMMETRIC p (not uniform, not cpl/rev-symmetric): every entry of q, D, p_next of the enumerating
        # path against the FAST path (oracle-green at n <= 14, no size-dependent branch) on the same p, plus the
        # oracle rows on that same q; sampled columns by the pinned DP.  A mis-addressed gather cannot hide here.
        pa = si.random_positive_p(n, seed + 1000)
        res = {}
        for mode in (ba.BA_MODE_ENUM, ba.BA_MODE_FAST):
            ba.ba_set_mode(ctx, mode)
            ba.ba_set_p(ctx, pa)
            ba.ba_iterate(ctx, 1)
            res[mode] = (ba.ba_get_q(ctx), ba.ba_get_D(ctx), ba.ba_get_p(ctx), ba.ba_bounds(ctx), ba.ba_stats(ctx)[0])
        ba.ba_set_mode(ctx, ba.BA_MODE_ENUM)
        (qe, De, pe, be, lze), (qf, Df, pf, bf, lzf) = res[ba.BA_MODE_ENUM], res[ba.BA_MODE_FAST]
        assert np.max(np.abs(qe - qf) / qf) <= REL_QD, "q: ENUM vs FAST, all entries"
        assert np.max(np.abs(De - Df) / np.abs(Df)) <= REL_QD, "D: ENUM vs FAST, all entries"
        assert np.max(np.abs(pe - pf) / pf) <= 1e-11
        assert abs(be[0] - bf[0]) <= 1e-12 * max(1, abs(bf[0])) and abs(be[1] - bf[1]) <= 1e-12 * max(1, abs(bf[1])) and abs(lze - lzf) <= 1e-12
        check_rows_against_oracle(n, d, rows, qe, De, "asymmetric p")
        for _ in range(max(1, n_cols)):
            k = int(rng.integers(max(1, n // 2 - 3), n // 2 + 4))
            yv = int(rng.integers(0, 1 << k))
            e = column_by_dp(yv, k, n)
            want = w[k] * math.fsum((e.astype(np.float64) * pa)[e > 0])
            assert abs(qe[(1 << k) - 1 + yv] - want) <= REL_QD * want, f"q(asym)[y={yv:0{k}b}]"
        for k in range(n + 1):                                # P7 on the asymmetric p
            want = comb(n, k) * w[k]
            assert abs(math.fsum(qe[(1 << k) - 1:(2 << k) - 1]) - want) <= 1e-12 * want
    finally:
        ba.ba_destroy(ctx)


def test_T7_scale_n20(ba):
    scale_checks(ba, 20, 0.80, n_rows=64, n_cols=3, seed=20)


def test_T7_scale_n24_bench_config(ba):
    # BASELINE.json configs[3]: n=24, d=0.70, uniform p0 -- the launch configuration bench.py times
    scale_checks(ba, 24, 0.70, n_rows=64, n_cols=2, seed=24)


def test_T7_scale_n26(ba):
    # above the bench size, default on (h = 18: the last size whose alpha always fit 16 bits)
    scale_checks(ba, 26, 0.75, n_rows=16, n_cols=1, seed=26)


def test_T7_symmetry_and_exact_at_scale_n20(ba):
    # complement symmetry on vs off, and the exact channel's pruned ENUM sweeps vs the FAST transform, all entries
    n, d = 20, 0.70
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_iterate(ctx, 2)
        q, D, p = ba.ba_get_q(ctx), ba.ba_get_D(ctx), ba.ba_get_p(ctx)
    finally:
        ba.ba_destroy(ctx)
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_set_symmetry(ctx, 1)
        ba.ba_iterate(ctx, 2)
        qs, Ds, ps = ba.ba_get_q(ctx), ba.ba_get_D(ctx), ba.ba_get_p(ctx)
    finally:
        ba.ba_destroy(ctx)
    assert np.max(np.abs(qs - q) / q) <= 1e-11 and np.max(np.abs(Ds - D) / np.abs(D)) <= 1e-11 and np.max(np.abs(ps - p) / p) <= 1e-10
    for k in (3, 10, 17):                                     # k < h - ..., k ~ n/2, k > h + m: both prunings of the exact mode
        pa = si.random_positive_p(n, 500 + k)
        out = {}
        for mode in (ba.BA_MODE_ENUM, ba.BA_MODE_FAST):
            ctx = ba.ba_create(n, d)
            try:
                ba.ba_set_mode(ctx, mode)
                ba.ba_set_exact(ctx, k)
                ba.ba_set_p(ctx, pa)
                ba.ba_iterate(ctx, 1)
                out[mode] = (ba.ba_get_q(ctx), ba.ba_get_D(ctx), ba.ba_bounds(ctx))
            finally:
                ba.ba_destroy(ctx)
        (qe, De, be), (qf, Df, bf) = out[ba.BA_MODE_ENUM], out[ba.BA_MODE_FAST]
        nz = qf > 0
        assert np.array_equal(qe > 0, nz) and np.max(np.abs(qe[nz] - qf[nz]) / qf[nz]) <= REL_QD
        assert np.all(np.abs(De - Df) <= REL_QD * np.abs(Df) + 1e-15)
        assert abs(be[0] - bf[0]) <= 1e-12 and abs(be[1] - bf[1]) <= 1e-12


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
    # Opt-in: BA_RUN_N28=1.  Result of the last run: profiles/ (r02_scale_n28.md).
    import os
    if os.environ.get("BA_RUN_N28") != "1":
        pytest.skip("set BA_RUN_N28=1 to run the n=28 scale check")
    scale_checks(ba, 28, 0.80, n_rows=8, n_cols=0, seed=28, asym=False)


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


# ------------------------------------------------------------------ measurement entry points of the ABI

def test_measured_peaks_and_setup_time(ba):
    pk = ba.ba_measure_peaks()
    # B200: FP64 and the integer-multiply pipe issue one warp-instruction every 2 clocks per scheduler (2 per clock per
    # SM), a conflict-free LDS.64 moves 256 bytes (1 per clock per SM), FP32 FMA fills the issue slots (4 per clock per SM)
    assert 1.5 <= pk["dfma"] <= 2.1 and 1.8 <= pk["idp2a"] <= 2.1 and 0.8 <= pk["lds64"] <= 1.1 and 3.3 <= pk["ffma"] <= 4.1
    assert pk["sms"] >= 100 and 1000.0 <= pk["sm_mhz"] <= 2200.0
    ctx = ba.ba_create(16, 0.7)
    try:
        with pytest.raises(ba.BAError) as ei:
            ba.ba_setup_ms(ctx)                              # the Hc pass has not run yet
        assert ei.value.code == ba.BA_ESTATE
        ba.ba_iterate(ctx, 1)
        assert 0.0 < ba.ba_setup_ms(ctx) < 5000.0
    finally:
        ba.ba_destroy(ctx)


def test_history_ring_wraps_in_two_pieces(ba):
    # more iterations than the ring holds (65536): the last `count` entries come back oldest first across the wrap
    n, d, K = 2, 0.5, 65536 + 300
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_iterate(ctx, K)
        full = ba.ba_get_history(ctx, 65536)
        tail = ba.ba_get_history(ctx, 500)
        I, U = ba.ba_bounds(ctx)
        with pytest.raises(ba.BAError):
            ba.ba_get_history(ctx, 65537)
    finally:
        ba.ba_destroy(ctx)
    assert np.array_equal(full[-500:], tail) and tail[-1, 0] == I and tail[-1, 1] == U
    assert np.all(np.diff(full[:, 0]) >= -1e-15)              # I_t non-decreasing along the whole window (Theorem 1)
    assert abs(I - 0.8304820237218407) <= 1e-12               # C_2(0.5), closed form
