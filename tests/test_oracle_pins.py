"""Pins for the CPU oracle (oracle/ba_oracle.c): everything here is fixed by the paper or by
mathematics, never by the oracle itself or by the CUDA path.

Each test names the passage of PAPER.md ("P:line") or the closed form it checks.
"""
import functools
import math
import os
from math import comb

import numpy as np
import pytest

from oracle import oracle as orc
import synthetic_inputs as si

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "paper_values.txt")


@functools.lru_cache(maxsize=None)
def E_of(n):
    return orc.emb_dense(n)


def idx(length, val):
    return (1 << length) - 1 + val


def length_slices(n):
    return [slice((1 << k) - 1, (1 << (k + 1)) - 1) for k in range(n + 1)]


def paper_values():
    vals = {}
    with open(GOLDEN) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            name, value = line.split()[:2]
            vals[name] = float(value)
    return vals


# ----------------------------------------------------------------------------- emb (O3)

def emb_dp(x, n, y, k):
    """Independent textbook DP: e[r] = #embeddings of y[0:r] in the scanned prefix of x."""
    e = [1] + [0] * k
    for i in range(n):
        xb = (x >> (n - 1 - i)) & 1
        for r in range(k, 0, -1):
            if ((y >> (k - r)) & 1) == xb:
                e[r] += e[r - 1]
    return e[k]


def test_emb_hand_worked_n2():
    # n=2, by hand from the definition "#times y appears as a subsequence of x".
    # columns: eps, 0, 1, 00, 01, 10, 11
    expect = np.array([[1, 2, 0, 1, 0, 0, 0],    # x=00
                       [1, 1, 1, 0, 1, 0, 0],    # x=01
                       [1, 1, 1, 0, 0, 1, 0],    # x=10
                       [1, 0, 2, 0, 0, 0, 1]],   # x=11
                      dtype=np.uint32)
    assert np.array_equal(E_of(2), expect)


def test_emb_hand_worked_n3_row():
    # x=010: eps 1; 0:2, 1:1; 00:1, 01:1, 10:1, 11:0; 010:1 and nothing else of length 3
    row = E_of(3)[0b010]
    expect = np.zeros(15, dtype=np.uint32)
    expect[idx(0, 0)] = 1
    expect[idx(1, 0)] = 2
    expect[idx(1, 1)] = 1
    expect[idx(2, 0b00)] = 1
    expect[idx(2, 0b01)] = 1
    expect[idx(2, 0b10)] = 1
    expect[idx(3, 0b010)] = 1
    assert np.array_equal(row, expect)


@pytest.mark.parametrize("n", [1, 2, 3, 4, 5, 6, 7])
def test_emb_matches_independent_dp_all_pairs(n):
    # P3: brute-force mask count == textbook DP, every (x, y)
    E = E_of(n)
    for x in range(1 << n):
        for k in range(n + 1):
            for y in range(1 << k):
                assert E[x, idx(k, y)] == emb_dp(x, n, y, k)


def test_emb_matches_independent_dp_sampled_n10():
    E = E_of(10)
    rng = np.random.default_rng(123)
    for _ in range(3000):
        x = int(rng.integers(0, 1 << 10))
        k = int(rng.integers(0, 11))
        y = int(rng.integers(0, 1 << k))
        assert E[x, idx(k, y)] == emb_dp(x, 10, y, k)


@pytest.mark.parametrize("n", [1, 2, 5, 8, 10])
def test_emb_row_sums_are_binomials(n):
    # P1: sum_{|y|=k} emb(y,x) = C(n,k) for every x and k (C(n,k) equally likely subsets)
    E = E_of(n).astype(np.int64)
    for k, sl in enumerate(length_slices(n)):
        assert np.all(E[:, sl].sum(axis=1) == comb(n, k))


@pytest.mark.parametrize("n", [1, 2, 5, 8, 10])
def test_emb_column_counts_lemma6(n):
    # P2: #length-n supersequences of y is sum_{i<=n-k} C(n,i) (Lemma 6);
    #     sum_x emb(y,x) = C(n,k) 2^{n-k} (each keep-set times the free deleted bits)
    E = E_of(n).astype(np.int64)
    for k, sl in enumerate(length_slices(n)):
        nnz = (E[:, sl] > 0).sum(axis=0)
        assert np.all(nnz == sum(comb(n, i) for i in range(n - k + 1)))
        assert np.all(E[:, sl].sum(axis=0) == comb(n, k) * (1 << (n - k)))


def T_of(n):
    return sum((1 << k) * sum(comb(n, i) for i in range(n - k + 1)) for k in range(n + 1))


def distinct_subseq_count(x, n):
    """Classic recurrence: number of distinct subsequences (incl. empty) of x."""
    total, last = 1, {0: 0, 1: 0}
    for i in range(n):
        b = (x >> (n - 1 - i)) & 1
        new = 2 * total - last[b]
        last[b] = total
        total = new
    return total


@pytest.mark.parametrize("n", [1, 4, 8, 10])
def test_total_terms_T_n(n):
    # P4: nnz(E) = T(n) by Lemma 6, and per-row nnz = #distinct subsequences (classic recurrence)
    E = E_of(n)
    nnz_rows = (E > 0).sum(axis=1)
    assert int(nnz_rows.sum()) == T_of(n)
    for x in range(0, 1 << n, max(1, (1 << n) // 64)):
        assert nnz_rows[x] == distinct_subseq_count(x, n)
    assert T_of(8) == 12866 and T_of(14) == 9549554


def test_emb_max_is_central_binomial():
    # max emb = C(n, n/2) attained by y = 0^{n/2} in x = 0^n
    for n in (4, 8, 10):
        assert int(E_of(n).max()) == comb(n, n // 2)


# ----------------------------------------------------------------------------- channel (O4)

@pytest.mark.parametrize("n,d", [(1, 0.3), (5, 0.5), (8, 0.64), (10, 0.9), (6, 0.0), (6, 1.0)])
def test_channel_rows_sum_to_one(n, d):
    # P5 (north_star: "each row of W summing to 1")
    W = orc.channel(n, d, E_of(n))
    assert np.allclose(W.sum(axis=1), 1.0, rtol=0, atol=1e-14)
    assert np.all(W >= 0)


def test_weights_endpoints_and_values():
    # R7: 0^0 = 1
    assert np.array_equal(orc.weights(4, 0.0), [0, 0, 0, 0, 1])
    assert np.array_equal(orc.weights(4, 1.0), [1, 0, 0, 0, 0])
    w = orc.weights(5, 0.25)
    for k in range(6):
        assert w[k] == pytest.approx(0.75 ** k * 0.25 ** (5 - k), rel=1e-15)


def test_channel_entry_is_emb_times_weight():
    n, d = 6, 0.37
    E = E_of(n)
    W = orc.channel(n, d, E)
    for k, sl in enumerate(length_slices(n)):
        assert np.allclose(W[:, sl], E[:, sl] * ((1 - d) ** k * d ** (n - k)), rtol=1e-15, atol=0)


# ----------------------------------------------------------------------------- generic BA step on textbook channels

def h2(s):
    return 0.0 if s in (0.0, 1.0) else -s * math.log2(s) - (1 - s) * math.log2(1 - s)


def converge(W, p0, iters):
    return orc.ba_run(W, p0, iters)


def test_ba_on_bsc_bec_z_channels():
    # textbook capacities, independent of emb: BSC 1-h(e); BEC 1-e; Z-channel closed form
    e = 0.11
    bsc = np.array([[1 - e, e], [e, 1 - e]])
    r = converge(bsc, np.array([0.3, 0.7]), 200)
    assert r["hist"][-1, 0] == pytest.approx(1 - h2(e), abs=1e-12)
    assert r["hist"][-1, 1] == pytest.approx(1 - h2(e), abs=1e-12)
    assert np.allclose(r["p"], 0.5, atol=1e-9)

    bec = np.array([[1 - e, e, 0.0], [0.0, e, 1 - e]])
    r = converge(bec, np.array([0.5, 0.5]), 5)
    assert r["hist"][-1, 0] == pytest.approx(1 - e, abs=1e-14)
    assert r["hist"][-1, 1] == pytest.approx(1 - e, abs=1e-14)

    f = 0.5   # Z-channel, 1 -> 0 with prob f: C = log2(1 + (1-f) f^{f/(1-f)})
    z = np.array([[1.0, 0.0], [f, 1 - f]])
    r = converge(z, np.array([0.5, 0.5]), 3000)
    cz = math.log2(1 + (1 - f) * f ** (f / (1 - f)))
    assert r["hist"][-1, 0] == pytest.approx(cz, abs=1e-9)
    assert r["hist"][-1, 1] == pytest.approx(cz, abs=1e-6)


def test_ba_step_definitions_on_random_small_matrix():
    # one step against the BA definitions written with python floats / fractions
    rng = np.random.default_rng(5)
    W = rng.random((5, 7))
    W[rng.random((5, 7)) < 0.3] = 0.0
    W[:, 0] += 0.1
    W /= W.sum(axis=1, keepdims=True)
    p = rng.random(5)
    p /= p.sum()
    r = orc.ba_step(W, p)
    q = [math.fsum(p[x] * W[x, j] for x in range(5)) for j in range(7)]
    assert np.allclose(r["q"], q, rtol=1e-15)
    # W^(t)(x) = prod_y (p(x) W/q)^W  =>  D(x) = log2 W^(t)(x) - log2 p(x)
    for x in range(5):
        prod_form = 1.0
        for j in range(7):
            if W[x, j] > 0:
                prod_form *= (p[x] * W[x, j] / q[j]) ** W[x, j]
        assert r["D"][x] == pytest.approx(math.log2(prod_form) - math.log2(p[x]), abs=1e-13)
    Wt = p * np.exp2(r["D"])
    assert np.allclose(r["p_next"], Wt / Wt.sum(), rtol=1e-14)
    assert r["I"] == pytest.approx(float(np.dot(p, r["D"])), rel=1e-14)
    assert r["U"] == r["D"].max()
    assert r["log2Z"] == pytest.approx(math.log2(Wt.sum()), abs=1e-14)
    # stop statistic of the paper: max_x log(X'/X) = U - log2 Z
    assert np.max(np.log2(r["p_next"] / p)) == pytest.approx(r["U"] - r["log2Z"], abs=1e-13)


# ----------------------------------------------------------------------------- BA on BDC_d^n: closed forms

@pytest.mark.parametrize("n,d", [(5, 0.3), (8, 0.5), (10, 0.64)])
def test_q_at_uniform_closed_form(n, d):
    # P6: q_0(y) = C(n,k) (1-d)^k d^{n-k} / 2^k for |y| = k  (from P2)
    r = orc.ba_step(orc.channel(n, d, E_of(n)), si.uniform_p0(n))
    for k, sl in enumerate(length_slices(n)):
        expect = comb(n, k) * (1 - d) ** k * d ** (n - k) / 2 ** k
        assert np.allclose(r["q"][sl], expect, rtol=1e-13, atol=0)


@pytest.mark.parametrize("n,d,seed", [(6, 0.4, 1), (9, 0.7, 2)])
def test_q_per_length_mass_any_p(n, d, seed):
    # P7: sum_{|y|=k} q(y) = C(n,k) (1-d)^k d^{n-k} for every normalised p (from P1)
    p = si.random_positive_p(n, seed)
    r = orc.ba_step(orc.channel(n, d, E_of(n)), p)
    for k, sl in enumerate(length_slices(n)):
        assert r["q"][sl].sum() == pytest.approx(comb(n, k) * (1 - d) ** k * d ** (n - k), rel=1e-12)


@pytest.mark.parametrize("n,d", [(4, 0.2), (8, 0.5), (10, 0.64)])
def test_D0_closed_forms(n, d):
    # P8:  D_0(0^n) = D_0(1^n) = n(1-d)  (W(0^k|0^n)/q_0(0^k) = 2^k)
    # P8b: D_0(x) = sum_k w_k S_k(x) + sum_k C(n,k) w_k (k - log2 C(n,k)), S_k = sum emb log2 emb
    E = E_of(n)
    r = orc.ba_step(orc.channel(n, d, E), si.uniform_p0(n))
    assert r["D"][0] == pytest.approx(n * (1 - d), rel=1e-13)
    assert r["D"][-1] == pytest.approx(n * (1 - d), rel=1e-13)
    Ef = E.astype(np.float64)
    ElogE = np.where(E > 0, Ef * np.log2(np.maximum(Ef, 1.0)), 0.0)
    const = 0.0
    Dx = np.zeros(1 << n)
    for k, sl in enumerate(length_slices(n)):
        wk = (1 - d) ** k * d ** (n - k)
        Dx += wk * ElogE[:, sl].sum(axis=1)
        const += comb(n, k) * wk * (k - math.log2(comb(n, k)))
    assert np.allclose(r["D"], Dx + const, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("d", [0.0, 0.1, 0.5, 0.64, 0.9, 1.0])
def test_C1_is_one_minus_d_at_iteration_zero(d):
    # P9 / P:59: n = 1 gives C(d) <= 1-d, i.e. C_1(d) = 1-d; uniform p is optimal so I_0 = U_0
    r = orc.ba_step(orc.channel(1, d, E_of(1)), si.uniform_p0(1))
    scale = paper_values()["C_1_over_1mind"]
    assert r["I"] == pytest.approx(scale * (1 - d), abs=1e-15)
    assert r["U"] == pytest.approx(scale * (1 - d), abs=1e-15)


@pytest.mark.parametrize("n", [1, 3, 6, 9])
def test_Cn_at_d0_is_n_and_at_d1_is_0(n):
    # P9 (north_star: C_n(0) = n): noiseless channel, uniform p optimal
    r = orc.ba_step(orc.channel(n, 0.0, E_of(n)), si.uniform_p0(n))
    assert r["I"] == pytest.approx(n, abs=1e-13) and r["U"] == pytest.approx(n, abs=1e-13)
    p = si.random_positive_p(n, 3)
    r = orc.ba_step(orc.channel(n, 0.0, E_of(n)), p)
    assert np.allclose(r["D"], -np.log2(p), rtol=1e-14)               # R7: D(x) = -log2 p(x)
    r = orc.ba_step(orc.channel(n, 1.0, E_of(n)), si.uniform_p0(n))
    assert r["I"] == 0.0 and r["U"] == 0.0


def C2_closed_form(d):
    # P9: by symmetry p(00)=p(11)=(1-s)/2, p(01)=p(10)=s/2,
    # C_2(d) = 2d(1-d)(1-s) + (1-d)^2 (1+h(s)),  s = 1/(1+2^{2d/(1-d)})
    s = 1.0 / (1.0 + 2.0 ** (2 * d / (1 - d)))
    return 2 * d * (1 - d) * (1 - s) + (1 - d) ** 2 * (1 + h2(s))


@pytest.mark.parametrize("d", [0.1, 0.5, 0.64, 0.9])
def test_C2_closed_form(d):
    r = orc.ba_run(orc.channel(2, d, E_of(2)), si.uniform_p0(2), 3000)
    assert r["hist"][-1, 0] == pytest.approx(C2_closed_form(d), abs=1e-12)
    assert r["hist"][-1, 1] == pytest.approx(C2_closed_form(d), abs=1e-9)
    if d == 0.5:
        assert C2_closed_form(d) == pytest.approx(0.8304820237218407, abs=1e-15)


def C2_by_grid_search(d):
    """Independent of BA: maximise I(X;Y) over the symmetric family on a fine grid."""
    E = E_of(2).astype(np.float64)
    w = [d * d, (1 - d) * d, (1 - d) ** 2]
    W = E * np.array([w[0]] + [w[1]] * 2 + [w[2]] * 4)
    best = 0.0
    for s in np.linspace(0.0, 1.0, 20001)[1:-1]:
        p = np.array([(1 - s) / 2, s / 2, s / 2, (1 - s) / 2])
        q = p @ W
        with np.errstate(divide="ignore", invalid="ignore"):
            t = np.where(W > 0, W * np.log2(W / q), 0.0)
        best = max(best, float(p @ t.sum(axis=1)))
    return best


def test_C2_against_grid_search():
    for d in (0.3, 0.64):
        r = orc.ba_run(orc.channel(2, d, E_of(2)), si.uniform_p0(2), 2000)
        assert r["hist"][-1, 0] == pytest.approx(C2_by_grid_search(d), abs=1e-8)


# ----------------------------------------------------------------------------- BA invariants (P10-P12)

@pytest.mark.parametrize("n,d,K", [(6, 0.5, 60), (8, 0.5, 200), (9, 0.8, 80)])
def test_bounds_order_and_monotone_I(n, d, K):
    # P10: I_t <= log2 Z_t <= U_t; I_t non-decreasing (Theorem 1); gap shrinks overall
    r = orc.ba_run(orc.channel(n, d, E_of(n)), si.uniform_p0(n), K)
    I, U, LZ = r["hist"][:, 0], r["hist"][:, 1], r["hist"][:, 2]
    assert np.all(I <= LZ + 1e-14) and np.all(LZ <= U + 1e-14)
    assert np.all(np.diff(I) >= -1e-14)
    assert (U[-1] - I[-1]) < 0.05 * (U[0] - I[0])
    assert U.min() <= n * (1 - d) + 1e-12                               # C_n(d) <= n(1-d)
    assert r["p"].sum() == pytest.approx(1.0, abs=1e-13)


def test_config1_secondary_values():
    # P13 (SURVEY scratch values; secondary pins produced by two independent throw-away codes)
    n, d, K = 8, 0.5, 200
    r = orc.ba_run(orc.channel(n, d, E_of(n)), si.uniform_p0(n), K)
    h = r["hist"]
    assert h[0, 0] == pytest.approx(1.4659436104746, abs=2e-13)
    assert h[0, 1] == pytest.approx(4.0, abs=1e-14)
    assert h[-1, 0] == pytest.approx(2.1229915839401, abs=2e-13)
    assert h[-1, 1] == pytest.approx(2.1260407187234, abs=2e-13)
    assert h[-1, 2] == pytest.approx(2.1229916758545, abs=2e-13)


def test_capacity_sequence_and_subadditivity():
    # P13: C_n(0.5), n=1..8 (scratch); P10: C_{n+m} <= C_n + C_m; C_n/n above the paper's
    # Table 3 bound on C(0.5) (soft sanity: C(d) <= C_n(d)/n)
    expect = [0.5, 0.830482023722, 1.095807177237, 1.329365012828,
              1.543920898143, 1.745649427607, 1.937970453523, 2.123006166059]
    C = []
    for n in range(1, 9):
        r = orc.ba_run(orc.channel(n, 0.5, E_of(n)), si.uniform_p0(n), 6000)
        lo, up = r["hist"][-1, 0], r["hist"][:, 1].min()
        assert up - lo < 2e-6
        assert lo - 1e-9 <= expect[n - 1] <= up + 1e-9
        C.append((lo, up))
    for a in range(1, 8):
        for b in range(1, 9 - a):
            assert C[a + b - 1][0] <= C[a - 1][1] + C[b - 1][1] + 1e-9
    bound = paper_values()["Cd_bound_d050"]
    assert all(C[n - 1][1] / n >= bound - 5e-5 for n in range(1, 9))


def cpl(x, n):
    return x ^ ((1 << n) - 1)


def rev(x, n):
    return int(format(x, f"0{n}b")[::-1], 2) if n else 0


@pytest.mark.parametrize("n,d", [(7, 0.5), (9, 0.7)])
def test_symmetry_theorem4(n, d):
    # P11 / Theorem 4: uniform start => p_t, q_t invariant under cpl and rev
    r = orc.ba_run(orc.channel(n, d, E_of(n)), si.uniform_p0(n), 25)
    p, q = r["p"], r["q"]
    for x in range(1 << n):
        assert p[x] == pytest.approx(p[cpl(x, n)], rel=1e-12)
        assert p[x] == pytest.approx(p[rev(x, n)], rel=1e-12)
    for k in range(n + 1):
        for y in range(1 << k):
            assert q[idx(k, y)] == pytest.approx(q[idx(k, cpl(y, k))], rel=1e-12)
            assert q[idx(k, y)] == pytest.approx(q[idx(k, rev(y, k))], rel=1e-12)


def test_start_independence():
    # P12 / R11: Dirichlet(1) and uniform starts bracket a common point
    n, d = 8, 0.64
    W = orc.channel(n, d, E_of(n))
    a = orc.ba_run(W, si.uniform_p0(n), 400)["hist"]
    b = orc.ba_run(W, si.dirichlet_p0(n, 0), 400)["hist"]
    lo = max(a[-1, 0], b[-1, 0])
    up = min(a[:, 1].min(), b[:, 1].min())
    assert lo <= up + 1e-12
    assert abs(a[-1, 0] - b[-1, 0]) < max(a[-1, 1] - a[-1, 0], b[-1, 1] - b[-1, 0])


# ----------------------------------------------------------------------------- exact channels BDC_{n,k} and Lemma 2

def exact_channel(n, k):
    # P_{n,k}(y|x) = emb(y,x)/C(n,k)
    return E_of(n)[:, length_slices(n)[k]].astype(np.float64) / comb(n, k)


def test_exact_channel_small_values_from_paper():
    # C_{2,1} = 1, C_{2,2} = 2;  Tables 1-2: C_{n,1} = 1, C_{n,n} = n
    pv = paper_values()
    r = orc.ba_run(exact_channel(2, 1), si.uniform_p0(2), 4000)
    assert r["hist"][-1, 0] == pytest.approx(pv["C_2_1"], abs=1e-9)
    r = orc.ba_run(exact_channel(2, 2), si.uniform_p0(2), 10)
    assert r["hist"][-1, 0] == pytest.approx(pv["C_2_2"], abs=1e-13)
    r = orc.ba_run(exact_channel(8, 1), si.uniform_p0(8), 4000)
    assert r["hist"][-1, 0] == pytest.approx(pv["C_n_1"], abs=2e-3)
    assert r["hist"][:, 1].min() >= pv["C_n_1"] - 1e-12
    r = orc.ba_run(exact_channel(8, 8), si.uniform_p0(8), 3)
    assert r["hist"][-1, 0] == pytest.approx(8 * pv["C_n_n_over_n"], abs=1e-13)


def test_lemma2_convex_combination():
    # Lemma 2: C_n(d) <= sum_k C(n,k) d^{n-k} (1-d)^k C_{n,k}; checked with rigorous
    # brackets: lower bound I on the left, upper bounds U_k on the right (2.3045 >= 2.1230)
    n, d = 8, 0.5
    left = orc.ba_run(orc.channel(n, d, E_of(n)), si.uniform_p0(n), 300)["hist"][-1, 0]
    right = 0.0
    for k in range(1, n + 1):
        Uk = orc.ba_run(exact_channel(n, k), si.uniform_p0(n), 300)["hist"][:, 1].min()
        right += comb(n, k) * d ** (n - k) * (1 - d) ** k * Uk
    assert left <= right
    assert right == pytest.approx(2.3045, abs=5e-3)
    assert left == pytest.approx(2.1230, abs=1e-4)


# ----------------------------------------------------------------------------- G8 floor of the update (P:154-158 + reading G8)

def test_floor_G8_fires_exactly_and_leaves_the_rest():
    # Reading G8: p' = max(p 2^D / Z, 2^-1000).  A 3-bit channel with one input at 1e-305 and d = 0.9:
    # D(x) holds (1-d)^n log2(1/p(x)) = 1e-3 * 1013 ~ 1 bit (G8), so p 2^D / Z ~ 1e-305 * 2^2 < 2^-1000 = 9.33e-302:
    # that entry must come out as 2^-1000 exactly, and every other entry must be the plain P:154-158 update
    # (the floor is not a renormalisation).  (At d = 0.5 the same p regrows to 8e-268 in one step: no floor.)
    n, d = 3, 0.9
    W = orc.channel(n, d, E_of(n))
    p = si.uniform_p0(n).copy()
    p[5] = 1e-305
    p[2] += 1.0 / 8 - 1e-305
    r = orc.ba_step(W, p)
    assert r["p_next"][5] == 2.0 ** -1000                              # exact: a power of two
    Z = 2.0 ** r["log2Z"]
    plain = p * np.exp2(r["D"]) / Z
    assert plain[5] < 2.0 ** -1000 and plain[5] > 0.0                  # the floor really was the binding branch
    keep = np.arange(8) != 5
    assert np.allclose(r["p_next"][keep], plain[keep], rtol=1e-14, atol=0)
    assert np.all(r["p_next"][keep] > 1e-3)                            # untouched by the floor
    # a p sitting exactly at the floor stays there, one just above it follows P:156
    p2 = si.uniform_p0(n).copy()
    p2[1] = 2.0 ** -1000
    p2[6] = 2.0 ** -990
    p2[0] += 2.0 / 8 - p2[1] - p2[6]
    r2 = orc.ba_step(W, p2)
    assert r2["p_next"][1] == 2.0 ** -1000 or r2["p_next"][1] == pytest.approx(p2[1] * 2 ** r2["D"][1] / 2 ** r2["log2Z"], rel=1e-13)
    assert r2["p_next"][6] == pytest.approx(p2[6] * 2 ** r2["D"][6] / 2 ** r2["log2Z"], rel=1e-13)
    assert r2["p_next"][6] > 2.0 ** -1000


def test_floor_G8_generic_matrix():
    # same on a generic 2-input channel (no emb involved): BSC with a collapsed input
    e = 0.2
    W = np.array([[1 - e, e], [e, 1 - e]])
    p = np.array([1.0 - 1e-306, 1e-306])
    r = orc.ba_step(W, p)
    assert r["p_next"][1] == 2.0 ** -1000
    assert r["p_next"][0] == pytest.approx(1.0, rel=1e-15)


# ----------------------------------------------------------------------------- single-row oracle (beyond the dense reach)

def test_emb_row_equals_dense_rows():
    # orc_emb_row is the same keep-mask count as orc_emb_dense for one x: every row, n <= 8; sampled n = 10
    for n in (1, 2, 3, 5, 8):
        E = E_of(n)
        for x in range(1 << n):
            assert np.array_equal(orc.emb_row(n, x), E[x])
    E = E_of(10)
    for x in np.random.default_rng(9).integers(0, 1 << 10, 64):
        assert np.array_equal(orc.emb_row(10, int(x)), E[int(x)])


def test_emb_row_hand_worked_and_invariants_large_n():
    row = orc.emb_row(3, 0b010)                                        # the hand-worked row of test_emb_hand_worked_n3_row
    expect = np.zeros(15, dtype=np.uint32)
    for (k, y, e) in [(0, 0, 1), (1, 0, 2), (1, 1, 1), (2, 0b00, 1), (2, 0b01, 1), (2, 0b10, 1), (3, 0b010, 1)]:
        expect[idx(k, y)] = e
    assert np.array_equal(row, expect)
    n = 18                                                             # beyond the dense reach: invariants fixed by mathematics
    for x in (0, (1 << n) - 1, 0b010101010101010101, 0b001101011100101101):
        row = orc.emb_row(n, x).astype(np.int64)
        for k, sl in enumerate(length_slices(n)):
            assert int(row[sl].sum()) == comb(n, k)                    # P1
        assert int(np.count_nonzero(row)) == distinct_subseq_count(x, n)   # classic recurrence (P4)
    assert int(np.count_nonzero(orc.emb_row(n, 0b010101010101010101))) == 10945   # Fib(21): alternating string has the most
    rng = np.random.default_rng(4)
    x = int(rng.integers(0, 1 << n))
    row = orc.emb_row(n, x)
    for _ in range(200):                                               # P3: independent textbook DP on sampled entries
        k = int(rng.integers(0, n + 1))
        y = int(rng.integers(0, 1 << k))
        assert row[idx(k, y)] == emb_dp(x, n, y, k)
    with pytest.raises(ValueError):
        orc.emb_row(8, 256)


@pytest.mark.parametrize("n,d", [(5, 0.3), (9, 0.64), (10, 0.9)])
def test_D_row_matches_definition_and_closed_forms(n, d):
    # orc_D_row is P:189-193 for one x.  (i) closed form P8 with the closed-form q_0 of P6 (no BA step involved):
    # D_0(0^n) = n(1-d);  (ii) python-float restatement of the definition on a random q;  (iii) the full step.
    q0 = np.empty((2 << n) - 1)
    for k, sl in enumerate(length_slices(n)):
        q0[sl] = comb(n, k) * (1 - d) ** k * d ** (n - k) / 2.0 ** k
    for x in (0, (1 << n) - 1):
        D, nt = orc.D_row(n, d, orc.emb_row(n, x), q0)
        assert D == pytest.approx(n * (1 - d), rel=1e-13) and nt == n + 1
    rng = np.random.default_rng(n)
    q = rng.random((2 << n) - 1) + 0.01
    x = int(rng.integers(0, 1 << n))
    row = orc.emb_row(n, x)
    terms = []
    for j in np.flatnonzero(row):
        k = (int(j) + 1).bit_length() - 1
        Wv = float(row[j]) * (1 - d) ** k * d ** (n - k)
        terms.append(Wv * (math.log2(Wv) - math.log2(q[j])))
    D, nt = orc.D_row(n, d, row, q)
    assert D == pytest.approx(math.fsum(terms), rel=1e-13, abs=1e-15) and nt == len(terms)
    p = si.random_positive_p(n, 77)
    r = orc.ba_step(orc.channel(n, d, E_of(n)), p)
    for x in rng.integers(0, 1 << n, 16):
        D, _ = orc.D_row(n, d, orc.emb_row(n, int(x)), r["q"])
        assert D == pytest.approx(r["D"][int(x)], rel=1e-14)


def test_D_row_endpoints_of_d():
    # R7: d = 0 keeps only y = x (D = -log2 q(idx(x))); d = 1 keeps only the empty output (D = -log2 q(0))
    n = 6
    q = np.random.default_rng(1).random((2 << n) - 1) + 0.1
    x = 0b101101
    row = orc.emb_row(n, x)
    assert orc.D_row(n, 0.0, row, q)[0] == pytest.approx(-math.log2(q[idx(n, x)]), rel=1e-15)
    assert orc.D_row(n, 1.0, row, q)[0] == pytest.approx(-math.log2(q[0]), rel=1e-15)


# ----------------------------------------------------------------------------- pins of the test-local CPU routines (tests/cpu_routines.py)

def test_cpu_routines_column_dp_equals_oracle_columns():
    from tests import cpu_routines as cr
    for n in (1, 4, 7, 10):
        E = E_of(n)
        rng = np.random.default_rng(n)
        cols = [(k, y) for k in range(n + 1) for y in range(1 << k)]
        if n == 10:
            cols = [cols[i] for i in rng.integers(0, len(cols), 200)] + [(0, 0), (10, 1023), (10, 0), (5, 0b10101)]
        for (k, y) in cols:
            assert np.array_equal(cr.column_by_dp(y, k, n), E[:, idx(k, y)])


def test_cpu_routines_weights_and_rev():
    from tests import cpu_routines as cr
    for (n, d) in [(5, 0.25), (7, 0.0), (7, 1.0), (12, 0.64)]:
        assert np.allclose(cr.weights(n, d), orc.weights(n, d), rtol=1e-15, atol=0)
    t = cr.bit_reverse_table(5)
    assert [int(t[x]) for x in (0b00001, 0b10110, 0b11111)] == [0b10000, 0b01101, 0b11111]
    assert all(int(t[x]) == rev(x, 5) for x in range(32))
