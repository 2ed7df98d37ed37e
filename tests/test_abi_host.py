"""CPU-side checks of the C ABI (include/ba.h): the library loads, exports every declared symbol, and the
entry points that need no device behave as the header says (host part)."""
import ctypes
import os
import re
from math import comb

import pytest

import paper_2604_05867_b200 as ba

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "ba.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(ba_[a-z_A-Z0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    L = ba.load()
    syms = declared_symbols()
    assert "ba_create" in syms and "ba_iterate" in syms and "ba_bounds" in syms and "ba_get_p" in syms
    for s in syms:
        assert hasattr(L, s), f"libba.so does not export {s}"
    assert set(ba.EXPORTS) == set(syms)


def test_terms_per_sweep_is_lemma6_sum():
    # T(n) = sum_k 2^k sum_{i<=n-k} C(n,i)   (Lemma 6); values of SURVEY 8(a)
    for n, want in [(8, 12866), (14, 9549554), (20, 6972520226), (24, 564842295746), (28, 45753316474466)]:
        assert ba.ba_terms_per_sweep(n) == want
        assert want == sum((1 << k) * sum(comb(n, i) for i in range(n - k + 1)) for k in range(n + 1))
    for bad in (0, -3, ba.BA_NMAX + 1):
        with pytest.raises(ba.BAError):
            ba.ba_terms_per_sweep(bad)


def test_scratch_bytes():
    assert ba.ba_scratch_bytes(0) == 0 and ba.ba_scratch_bytes(ba.BA_NMAX + 1) == 0
    prev = 0
    for n in (1, 4, 8, 12, 20, 24, 28):
        b = ba.ba_scratch_bytes(n)
        assert b > prev and b % 256 == 0
        prev = b
    # c (2^{n+1} doubles) and Hc (2^n doubles) alone need 24 * 2^n bytes
    assert ba.ba_scratch_bytes(24) >= 24 << 24
    assert ba.ba_scratch_bytes(28) < 40e9                      # fits a 180 GB B200 many times over


def test_create_rejects_bad_arguments_without_touching_the_device():
    L = ba.load()
    h = ctypes.c_void_p()
    for n, d in [(0, 0.5), (-1, 0.5), (ba.BA_NMAX + 1, 0.5), (8, -0.1), (8, 1.5), (8, float("nan"))]:
        assert L.ba_create(n, d, ctypes.byref(h)) == ba.BA_EINVAL
        assert not h.value
    assert L.ba_create(8, 0.5, None) == ba.BA_EINVAL
    assert L.ba_create_ext(8, 0.5, None, None, None, None, 0, None, ctypes.byref(h)) == ba.BA_EINVAL
    # null context: every entry point returns BA_EINVAL and ba_last_error gives a static string
    assert L.ba_iterate(None, 1) == ba.BA_EINVAL
    assert L.ba_bounds(None, None, None) == ba.BA_EINVAL
    assert L.ba_get_p(None, None) == ba.BA_EINVAL
    assert L.ba_set_mode(None, 0) == ba.BA_EINVAL
    assert b"context" in L.ba_last_error(None)
    L.ba_destroy(None)                                          # no-op


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("CUDA device present")
    with pytest.raises(ba.BAError):
        ba.ba_create(8, 0.5)


@pytest.mark.parametrize("m", [1, 2, 3, 5, 8])
def test_pair_tables_cover_every_pair_once(m):
    # the class tables + riders of the ENUM kernels partition the pairs (v, z != empty) of the m-bit channel:
    # 16 classes x (T(m) - 2^m) pairs (Lemma 6), with the B_s of an independent DP
    rc, st = ba.ba_debug_check_tables(m)
    assert rc == ba.BA_OK
    T = sum((1 << k) * sum(comb(m, i) for i in range(m - k + 1)) for k in range(m + 1))
    assert st[0] + st[1] == 16 * (T - (1 << m)) == st[2] + st[3]
    if m == 8:
        assert 0 < st[1] < 0.05 * (st[0] + st[1]) and st[1] == st[3]      # riders: the 3.4 % deep pairs
    assert ba.ba_debug_check_tables(0)[0] == ba.BA_EINVAL and ba.ba_debug_check_tables(9)[0] == ba.BA_EINVAL


def test_lemma2_combiner_arithmetic():
    # Lemma 2: sum_k C(n,k) d^(n-k) (1-d)^k C_{n,k}.  With C_{n,k} = k (the noiseless value, an upper bound
    # of every C_{n,k}) the sum is the mean of Binomial(n, 1-d): n (1-d), the easy bound C_n(d) <= n (1-d).
    from paper_2604_05867_b200 import exact
    for n, d in [(8, 0.5), (12, 0.64), (29, 0.3)]:
        assert exact.lemma2_bound(n, d, {k: float(k) for k in range(1, n + 1)}) == pytest.approx(n * (1 - d), rel=1e-12)
    assert exact.lemma2_bound(2, 0.5, {1: 1.0, 2: 2.0}) == pytest.approx(2 * 0.25 * 1.0 + 0.25 * 2.0)   # C_{2,1} = 1, C_{2,2} = 2
