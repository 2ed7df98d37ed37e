"""GPU parity tests: libba (through the C ABI binding) against the CPU oracle on the same seeded
inputs (SURVEY.md section 8(c) protocol T1-T6).  Tolerances are BASELINE.json:north_star's:
emb bit-exact; q and D within 1e-12 relative; bounds within 1e-10 bits after the same K.
"""
import functools

import numpy as np
import pytest

import synthetic_inputs as si
from oracle import oracle as orc

pytestmark = pytest.mark.gpu

REL_QD = 1e-12      # north_star: "q and D within 1e-12 relative error in FP64"
ABS_U = 1e-10       # north_star: "the upper bound within 1e-10 bits after the same number of iterations"


@pytest.fixture(scope="module")
def ba():
    import paper_2604_05867_b200 as ba_mod
    ba_mod.load()
    return ba_mod


@functools.lru_cache(maxsize=None)
def E_of(n):
    return orc.emb_dense(n)


@functools.lru_cache(maxsize=None)
def W_of(n, d):
    return orc.channel(n, d, E_of(n))


def relerr(a, b):
    return np.max(np.abs(a - b) / np.abs(b))


# ------------------------------------------------------------------ T1 / T2: emb bit-exact

@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 9, 10])
def test_T1_emb_rows_bit_exact(ba, n):
    E = E_of(n)
    ctx = ba.ba_create(n, 0.5)
    try:
        for x in range(1 << n):
            row = ba.ba_debug_emb_row(ctx, x)
            assert np.array_equal(row, E[x]), f"row x={x}"
    finally:
        ba.ba_destroy(ctx)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7, 8, 9, 10])
def test_T2_emb_cols_bit_exact(ba, n):
    E = E_of(n)
    ctx = ba.ba_create(n, 0.5)
    try:
        for j in range((2 << n) - 1):
            col = ba.ba_debug_emb_col(ctx, j)
            assert np.array_equal(col, E[:, j]), f"col idx={j}"
    finally:
        ba.ba_destroy(ctx)


def test_T1_T2_emb_sampled_n14(ba):
    n = 14
    E = E_of(n)
    rng = np.random.default_rng(7)
    ctx = ba.ba_create(n, 0.64)
    try:
        xs = [0, (1 << n) - 1, 0b01010101010101, 0b00110011001100] + list(rng.integers(0, 1 << n, 60))
        for x in xs:
            assert np.array_equal(ba.ba_debug_emb_row(ctx, int(x)), E[int(x)])
        js = [0, 1, 2, (2 << n) - 2] + list(rng.integers(0, (2 << n) - 1, 60))
        for j in js:
            assert np.array_equal(ba.ba_debug_emb_col(ctx, int(j)), E[:, int(j)])
    finally:
        ba.ba_destroy(ctx)


@pytest.mark.parametrize("n", [3, 8, 11, 14])
def test_term_counts_match_lemma6(ba, n):
    # P4: both enumerators visit exactly T(n) terms; sum of emb = 4^n ... = sum_k C(n,k) 2^n
    ctx = ba.ba_create(n, 0.5)
    try:
        r = ba.ba_debug_count_terms(ctx)
        T = ba.ba_terms_per_sweep(n)
        assert T == int((E_of(n) > 0).sum()) if n <= 11 else True
        assert r["in_terms"] == T and r["out_terms"] == T
        assert r["in_emb_sum"] == 4 ** n and r["out_emb_sum"] == 4 ** n
    finally:
        ba.ba_destroy(ctx)


# ------------------------------------------------------------------ T3 / T4: one-step parity

def one_step_check(ba, n, d, p, mode):
    ref = orc.ba_step(W_of(n, d), p)
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_set_mode(ctx, mode)
        ba.ba_set_p(ctx, p)
        ba.ba_iterate(ctx, 1)
        q, D = ba.ba_get_q(ctx), ba.ba_get_D(ctx)
        I, U = ba.ba_bounds(ctx)
        lz, it = ba.ba_stats(ctx)
        pn = ba.ba_get_p(ctx)
    finally:
        ba.ba_destroy(ctx)
    assert it == 1
    nzq = ref["q"] > 0
    assert np.array_equal(q > 0, nzq)
    assert relerr(q[nzq], ref["q"][nzq]) <= REL_QD
    assert relerr(D, ref["D"]) <= REL_QD, f"max |dD|/|D| = {relerr(D, ref['D'])}"
    assert abs(I - ref["I"]) <= REL_QD * max(1.0, abs(ref["I"]))
    assert abs(U - ref["U"]) <= REL_QD * max(1.0, abs(ref["U"]))
    assert abs(lz - ref["log2Z"]) <= REL_QD * max(1.0, abs(ref["log2Z"]))
    assert relerr(pn, ref["p_next"]) <= 1e-11


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("n,d", [(1, 0.3), (2, 0.5), (5, 0.25), (8, 0.5), (9, 0.64), (10, 0.9), (12, 0.7)])
def test_T3_T4_one_step_uniform(ba, n, d, mode):
    one_step_check(ba, n, d, si.uniform_p0(n), mode)


@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("n,d,seed", [(6, 0.4, 11), (8, 0.5, 12), (11, 0.64, 13), (12, 0.85, 14)])
def test_T3_T4_one_step_random_p(ba, n, d, seed, mode):
    one_step_check(ba, n, d, si.random_positive_p(n, seed), mode)


@pytest.mark.parametrize("mode", [0, 1])
def test_T3_T4_one_step_from_oracle_iterates_config1(ba, mode):
    # p_t from the oracle at t in {0,1,10,K-1} loaded with ba_set_p (R9 (i))
    n, d, K = 8, 0.5, 200
    W = W_of(n, d)
    p = si.uniform_p0(n)
    wanted = {0, 1, 10, K - 1}
    for t in range(K):
        if t in wanted:
            one_step_check(ba, n, d, p.copy(), mode)
        p = orc.ba_step(W, p)["p_next"]


# ------------------------------------------------------------------ T5: trajectories

@pytest.mark.parametrize("mode", [0, 1])
def test_T5_trajectory_config1(ba, mode):
    n, d, K = 8, 0.5, 200
    ref = orc.ba_run(W_of(n, d), si.uniform_p0(n), K)
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_set_mode(ctx, mode)
        ba.ba_iterate(ctx, K)
        I, U = ba.ba_bounds(ctx)
        hist = ba.ba_get_history(ctx, K)
        p = ba.ba_get_p(ctx)
    finally:
        ba.ba_destroy(ctx)
    assert abs(U - ref["hist"][-1, 1]) <= ABS_U
    assert abs(I - ref["hist"][-1, 0]) <= ABS_U
    assert np.max(np.abs(hist - ref["hist"])) <= ABS_U
    assert relerr(p, ref["p"]) <= 1e-9
    # P13 secondary pins: I_199 = 2.1229915839401, U_199 = 2.1260407187234
    assert I == pytest.approx(2.1229915839401, abs=2e-13)
    assert U == pytest.approx(2.1260407187234, abs=2e-13)


# ------------------------------------------------------------------ T6: special cases

@pytest.mark.parametrize("mode", [0, 1])
def test_T6_special_cases(ba, mode):
    def run(n, d, K, p0=None):
        ctx = ba.ba_create(n, d)
        try:
            ba.ba_set_mode(ctx, mode)
            if p0 is not None:
                ba.ba_set_p(ctx, p0)
            ba.ba_iterate(ctx, K)
            return ba.ba_bounds(ctx), ba.ba_get_D(ctx)
        finally:
            ba.ba_destroy(ctx)

    for d in (0.0, 0.2, 0.64, 1.0):                          # C_1(d) = 1-d
        (I, U), _ = run(1, d, 1)
        assert I == pytest.approx(1 - d, abs=1e-14) and U == pytest.approx(1 - d, abs=1e-14)
    for n in (3, 9):                                          # C_n(0) = n; D = -log2 p (R7)
        (I, U), _ = run(n, 0.0, 1)
        assert I == pytest.approx(n, abs=1e-12) and U == pytest.approx(n, abs=1e-12)
        p = si.random_positive_p(n, 5)
        _, D = run(n, 0.0, 1, p)
        assert np.allclose(D, -np.log2(p), rtol=1e-13)
        (I, U), _ = run(n, 1.0, 1)                            # C_n(1) = 0
        assert abs(I) <= 1e-15 and abs(U) <= 1e-15
    d = 0.5                                                   # C_2(d) closed form
    (I, U), _ = run(2, d, 3000)
    assert I == pytest.approx(0.8304820237218407, abs=1e-12)
    assert U == pytest.approx(0.8304820237218407, abs=1e-9)


# ------------------------------------------------------------------ NEXT-3: the paper's exact channel BDC_{n,k}

def exact_W(n, k):
    # P_{n,k}(y|x) = emb(y,x)/C(n,k) on the outputs of length k, 0 elsewhere, in the dense q layout
    from math import comb
    W = np.zeros(E_of(n).shape, dtype=np.float64)
    sl = slice((1 << k) - 1, (2 << k) - 1)
    W[:, sl] = E_of(n)[:, sl].astype(np.float64) / comb(n, k)
    return W


# (11,1) (11,2) (12,3): k small with a high part, so whole prefixes / nodes are skipped because they cannot reach
# length k from below (klen < t); (11,10) (12,11) (14,13): k > t + 8, skipped from above.  Both prunings of the
# ENUM exact mode are therefore compared with the oracle here (mode 0), not only the FAST transform.
@pytest.mark.parametrize("mode", [0, 1])
@pytest.mark.parametrize("n,k", [(2, 1), (5, 3), (8, 1), (8, 4), (8, 8), (11, 6), (11, 1), (11, 2), (12, 3), (11, 10),
                                 (12, 11), (14, 13)])
def test_exact_channel_one_step_and_trajectory(ba, n, k, mode):
    W = exact_W(n, k)
    p = si.random_positive_p(n, 100 + n + k)
    ref1 = orc.ba_step(W, p)
    refK = orc.ba_run(W, p, 40)
    ctx = ba.ba_create(n, 0.5)
    try:
        ba.ba_set_mode(ctx, mode)
        ba.ba_set_exact(ctx, k)
        ba.ba_set_p(ctx, p)
        ba.ba_iterate(ctx, 1)
        q, D = ba.ba_get_q(ctx), ba.ba_get_D(ctx)
        nz = ref1["q"] > 0
        assert np.array_equal(q > 0, nz)
        assert relerr(q[nz], ref1["q"][nz]) <= REL_QD
        # D = Hc - sum emb c (hoisted logarithm) has an absolute error of a few ulp of Hc; on BDC_{n,k} an input whose
        # only output is nearly certain has D ~ 1e-7 bits, where that is 1e-10 relative:
        # 1e-12 relative with an absolute floor of 1e-15 bits
        assert np.all(np.abs(D - ref1["D"]) <= REL_QD * np.abs(ref1["D"]) + 1e-15)
        ba.ba_iterate(ctx, 39)
        I, U = ba.ba_bounds(ctx)
        assert abs(I - refK["hist"][-1, 0]) <= ABS_U and abs(U - refK["hist"][-1, 1]) <= ABS_U
        with pytest.raises(ba.BAError) as ei:
            ba.ba_set_exact(ctx, k)                          # only before the first iteration
        assert ei.value.code == ba.BA_ESTATE
    finally:
        ba.ba_destroy(ctx)


@pytest.mark.parametrize("n,k", [(11, 2), (12, 6), (12, 11)])
def test_exact_channel_with_complement_symmetry(ba, n, k):
    # the pruned ENUM exact mode under ba_set_symmetry(1): uniform start, K iterations, against the oracle
    K = 12
    ref = orc.ba_run(exact_W(n, k), si.uniform_p0(n), K)
    ctx = ba.ba_create(n, 0.5)
    try:
        ba.ba_set_exact(ctx, k)
        ba.ba_set_symmetry(ctx, 1)
        ba.ba_iterate(ctx, K)
        q, D, p = ba.ba_get_q(ctx), ba.ba_get_D(ctx), ba.ba_get_p(ctx)
        hist = ba.ba_get_history(ctx, K)
    finally:
        ba.ba_destroy(ctx)
    nz = ref["q"] > 0
    assert np.array_equal(q > 0, nz) and relerr(q[nz], ref["q"][nz]) <= 1e-11
    assert np.all(np.abs(D - ref["D"]) <= 1e-11 * np.abs(ref["D"]) + 1e-15) and relerr(p, ref["p"]) <= 1e-9
    assert np.max(np.abs(hist - ref["hist"])) <= ABS_U


def test_exact_channel_paper_values_and_lemma2(ba):
    from math import comb

    def run(n, k, K):
        ctx = ba.ba_create(n, 0.5)
        try:
            ba.ba_set_mode(ctx, 1)
            if k is not None:
                ba.ba_set_exact(ctx, k)
            ba.ba_iterate(ctx, K)
            I, U = ba.ba_bounds(ctx)
            return I, float(ba.ba_get_history(ctx, K)[:, 1].min())
        finally:
            ba.ba_destroy(ctx)

    assert run(2, 2, 10)[0] == pytest.approx(2.0, abs=1e-13)          # C_{2,2} = 2
    assert run(2, 1, 4000)[0] == pytest.approx(1.0, abs=1e-9)         # C_{2,1} = 1
    assert run(8, 8, 3)[0] == pytest.approx(8.0, abs=1e-12)           # C_{n,n} = n (Tables 1-2, last row)
    I1, U1 = run(8, 1, 4000)
    assert I1 == pytest.approx(1.0, abs=2e-3) and U1 >= 1.0 - 1e-12   # C_{n,1} = 1 (Tables 1-2, first row)
    # Lemma 2 with rigorous brackets at n=8, d=0.5: I(C_n(d)) <= sum_k Bin(k) U(C_{n,k})
    d, n = 0.5, 8
    left = run(n, None, 300)[0]
    right = sum(comb(n, k) * d ** (n - k) * (1 - d) ** k * run(n, k, 300)[1] for k in range(1, n + 1))
    assert left <= right and right == pytest.approx(2.3045, abs=5e-3) and left == pytest.approx(2.1230, abs=1e-4)


# ------------------------------------------------------------------ NEXT-2 (cpl half): complement symmetry

@pytest.mark.parametrize("n,d,K", [(9, 0.5, 30), (11, 0.64, 25), (12, 0.8, 20)])
def test_complement_symmetry_matches_oracle(ba, n, d, K):
    ref = orc.ba_run(W_of(n, d), si.uniform_p0(n), K)
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_set_symmetry(ctx, 1)
        ba.ba_iterate(ctx, K)
        I, U = ba.ba_bounds(ctx)
        q, D, p = ba.ba_get_q(ctx), ba.ba_get_D(ctx), ba.ba_get_p(ctx)
        hist = ba.ba_get_history(ctx, K)
        with pytest.raises(ba.BAError) as ei:               # an asymmetric p is refused while symmetry is on
            ba.ba_set_p(ctx, si.random_positive_p(n, 1))
        assert ei.value.code == ba.BA_EINVAL
    finally:
        ba.ba_destroy(ctx)
    assert np.max(np.abs(hist - ref["hist"])) <= ABS_U and abs(I - ref["hist"][-1, 0]) <= ABS_U and abs(U - ref["hist"][-1, 1]) <= ABS_U
    assert relerr(q, ref["q"]) <= 1e-11 and relerr(D, ref["D"]) <= 1e-11 and relerr(p, ref["p"]) <= 1e-9
    NX = 1 << n
    assert np.array_equal(p, p[::-1]) and np.array_equal(D, D[::-1])          # x -> ~x is index reversal of [0, 2^n)
    for k in range(1, n + 1):                                                  # q(~y) = q(y) within every length
        blk = q[(1 << k) - 1:(2 << k) - 1]
        assert np.array_equal(blk, blk[::-1])


def test_complement_symmetry_argument_errors(ba):
    ctx = ba.ba_create(8, 0.5)
    try:
        with pytest.raises(ba.BAError) as ei:
            ba.ba_set_symmetry(ctx, 1)                       # n = 8 has no high part
        assert ei.value.code == ba.BA_EINVAL
    finally:
        ba.ba_destroy(ctx)
    ctx = ba.ba_create(10, 0.5)
    try:
        ba.ba_set_p(ctx, si.random_positive_p(10, 2))
        with pytest.raises(ba.BAError) as ei:
            ba.ba_set_symmetry(ctx, 1)                       # current p is not symmetric
        assert ei.value.code == ba.BA_EINVAL
        ba.ba_set_symmetry(ctx, 0)
    finally:
        ba.ba_destroy(ctx)


# ------------------------------------------------------------------ G8: the floor of the update, on the device

@pytest.mark.parametrize("mode", [0, 1])
def test_floor_G8_on_device(ba, mode):
    # twin of tests/test_oracle_pins.py::test_floor_G8_fires_exactly_and_leaves_the_rest: n = 3, d = 0.9, one input at
    # 1e-305, so p 2^D / Z < 2^-1000 for that input only (reading G8)
    n, d = 3, 0.9
    p = si.uniform_p0(n).copy()
    p[5] = 1e-305
    p[2] += 1.0 / 8 - 1e-305
    ref = orc.ba_step(W_of(n, d), p)
    assert ref["p_next"][5] == 2.0 ** -1000                    # the oracle's floor fired (pinned on CPU)
    ctx = ba.ba_create(n, d)
    try:
        ba.ba_set_mode(ctx, mode)
        ba.ba_set_p(ctx, p)
        ba.ba_iterate(ctx, 1)
        pn, D = ba.ba_get_p(ctx), ba.ba_get_D(ctx)
        ba.ba_iterate(ctx, 1)                                  # and the iterate stays usable (no log2 0, no NaN)
        I, U = ba.ba_bounds(ctx)
    finally:
        ba.ba_destroy(ctx)
    assert pn[5] == 2.0 ** -1000                               # bit-exact
    keep = np.arange(1 << n) != 5
    assert relerr(pn[keep], ref["p_next"][keep]) <= 1e-12 and relerr(D, ref["D"]) <= REL_QD
    assert np.isfinite(I) and np.isfinite(U) and I <= U


# ------------------------------------------------------------------ contexts are independent (include/ba.h)

def test_two_contexts_of_different_tile_width_alive_together(ba):
    # an n >= 8 ctx (m = 8, the largest dynamic shared-memory request) and an n < 8 ctx (m = 4) interleaved:
    # creating the second must not shrink what the first may launch with
    big = ba.ba_create(12, 0.7)
    try:
        ba.ba_iterate(big, 1)
        small = ba.ba_create(4, 0.3)
        try:
            ba.ba_iterate(small, 2)
            ba.ba_iterate(big, 2)
            ba.ba_iterate(small, 1)
            Ib, Ub = ba.ba_bounds(big)
            Is, Us = ba.ba_bounds(small)
        finally:
            ba.ba_destroy(small)
        ba.ba_iterate(big, 1)
        assert np.array_equal(ba.ba_debug_emb_row(big, 0b010011010111), E_of(12)[0b010011010111])
    finally:
        ba.ba_destroy(big)
    rb = orc.ba_run(W_of(12, 0.7), si.uniform_p0(12), 3)["hist"][-1]
    rs = orc.ba_run(W_of(4, 0.3), si.uniform_p0(4), 3)["hist"][-1]
    assert abs(Ib - rb[0]) <= ABS_U and abs(Ub - rb[1]) <= ABS_U and abs(Is - rs[0]) <= ABS_U and abs(Us - rs[1]) <= ABS_U


def test_fast_mode_is_refused_while_symmetry_is_on(ba):
    ctx = ba.ba_create(10, 0.5)
    try:
        ba.ba_set_symmetry(ctx, 1)
        with pytest.raises(ba.BAError) as ei:
            ba.ba_set_mode(ctx, ba.BA_MODE_FAST)             # FAST iterations would break p(x) == p(~x) bit for bit
        assert ei.value.code == ba.BA_EINVAL
        ba.ba_set_symmetry(ctx, 0)
        ba.ba_set_mode(ctx, ba.BA_MODE_FAST)
        with pytest.raises(ba.BAError) as ei:
            ba.ba_set_symmetry(ctx, 1)
        assert ei.value.code == ba.BA_EINVAL
    finally:
        ba.ba_destroy(ctx)


# ------------------------------------------------------------------ NEXT-3: the paper's workload (all k, stop rule, Lemma 2)

@pytest.mark.parametrize("mode", [0, 1])
def test_exact_workflow_all_k_and_lemma2_against_oracle(ba, mode):
    from paper_2604_05867_b200 import exact
    n, a = 8, 0.005                                           # the paper's tolerance
    res = exact.run(n, a=a, ds=(0.3, 0.5, 0.64), mode=mode)
    assert [r["k"] for r in res["capacities"]] == list(range(1, n + 1)) and all(r["converged"] for r in res["capacities"])
    up = {}
    for r in res["capacities"]:                               # every bracket contains the oracle's own converged bracket
        k = r["k"]
        ref = orc.ba_run(exact_W(n, k), si.uniform_p0(n), 6000)["hist"]
        lo_ref, up_ref = ref[-1, 0], ref[:, 1].min()
        assert r["I_lower"] <= up_ref + 1e-9 and lo_ref <= r["U_upper"] + 1e-9 and r["I_lower"] <= r["U_upper"]
        assert r["stop_statistic"] < a and r["U_upper"] - r["I_lower"] < 2 * a + 0.05
        it = r["iterations"]                                  # same iterate as the oracle after the same number of steps
        assert abs(r["I_lower"] - ref[it - 1, 0]) <= ABS_U
        up[k] = r["U_upper"]
    assert res["capacities"][0]["U_upper"] >= 1.0 - 1e-12 and res["capacities"][-1]["I_lower"] == pytest.approx(float(n), abs=1e-12)   # C_{n,1} = 1, C_{n,n} = n (Tables 1-2)
    for b in res["bounds"]:                                   # Lemma 2 above the direct capacity C_n(d)
        direct = orc.ba_run(W_of(n, b["d"]), si.uniform_p0(n), 400)["hist"][-1, 0]
        assert direct <= b["Cn_upper"] + 1e-12
        assert b["Cn_upper"] == pytest.approx(exact.lemma2_bound(n, b["d"], up), rel=1e-15)
        assert b["Cd_upper"] == pytest.approx(b["Cn_upper"] / n)
