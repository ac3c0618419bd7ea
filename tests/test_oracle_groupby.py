"""Pins for the CPU oracle's GROUP BY / exact NDV / min-max (no GPU).

Each test checks the oracle against something other than itself: a hand-worked
closed form (tests/golden/groupby_closed_form.txt), O(n^2) brute force written
from the relational definition, invariants, special cases that
reduce to numpy routines, and metamorphic relations.
"""
import math

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import oracle
from oracle import SUM, COUNT, MIN, MAX

ALL4 = [(SUM, 0), (COUNT, 0), (MIN, 0), (MAX, 0)]


def brute_force(keys, vals, aggs):
    """For each row, scan all rows with the same key (O(n^2)); pure Python ints / floats."""
    cols = [list(map(int, k)) for k in keys]
    n = len(cols[0])
    tup = [tuple(c[i] for c in cols) for i in range(n)]
    out = {}
    for i in range(n):
        if tup[i] in out:
            continue
        rows = [r for r in range(n) if tup[r] == tup[i]]
        res = []
        for op, c in aggs:
            if op == COUNT:
                res.append(len(rows))
                continue
            xs = [vals[c][r] for r in rows]
            if vals[c].dtype == np.float64:
                xs = [float(x) for x in xs]
                res.append({SUM: math.fsum(xs), MIN: min(xs), MAX: max(xs)}[op])
            else:
                xs = [int(x) for x in xs]
                s = sum(xs) & ((1 << 64) - 1)
                s = s - (1 << 64) if s >= (1 << 63) else s
                res.append({SUM: s, MIN: min(xs), MAX: max(xs)}[op])
        out[tup[i]] = res
    return out


def as_dict(res):
    d = {}
    for g in range(res.n_groups):
        d[tuple(int(k[g]) for k in res.keys)] = [a[g].item() for a in res.aggs]
    return d


def test_closed_form_golden(golden):
    n, D = 10, 3
    i = np.arange(n, dtype=np.int64)
    res = oracle.groupby(i % D, [i], [(COUNT, 0), (SUM, 0), (MIN, 0), (MAX, 0)])
    rows = golden("groupby_closed_form.txt")
    assert res.n_groups == len(rows)
    for g, row in enumerate(rows):
        key, cnt, s, lo, hi = map(int, row)
        assert int(res.keys[0][g]) == key
        assert [int(a[g]) for a in res.aggs] == [cnt, s, lo, hi]


@pytest.mark.parametrize("n,D", [(1, 1), (7, 7), (1000, 13), (100003, 1000), (1 << 20, 4099)])
def test_closed_form_general(n, D):
    i = np.arange(n, dtype=np.int64)
    res = oracle.groupby((i % D).astype(np.int32), [i], [(COUNT, 0), (SUM, 0), (MIN, 0), (MAX, 0)])
    assert res.n_groups == min(n, D)
    for g in range(res.n_groups):
        k = int(res.keys[0][g])
        c = -((k - n) // D)  # ceil((n-k)/D)
        assert k == g
        assert int(res.aggs[0][g]) == c
        assert int(res.aggs[1][g]) == c * k + D * c * (c - 1) // 2
        assert int(res.aggs[2][g]) == k
        assert int(res.aggs[3][g]) == k + D * (c - 1)


@pytest.mark.parametrize("seed", range(6))
def test_brute_force_int(seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(1, 65))
    keys = rng.integers(-5, 6, size=n).astype(np.int64)
    v0 = rng.integers(-1000, 1001, size=n).astype(np.int64)
    v1 = rng.integers(-(1 << 62), 1 << 62, size=n).astype(np.int64)   # wraps in SUM
    aggs = [(SUM, 0), (COUNT, 0), (MIN, 0), (MAX, 0), (SUM, 1), (MIN, 1), (MAX, 1)]
    got = as_dict(oracle.groupby(keys, [v0, v1], aggs))
    assert got == brute_force([keys], [v0, v1], aggs)


@pytest.mark.parametrize("seed", range(4))
def test_brute_force_two_keys_and_f64(seed):
    rng = np.random.default_rng(100 + seed)
    n = int(rng.integers(1, 65))
    k0 = rng.integers(0, 3, size=n).astype(np.int8)
    k1 = rng.integers(-1, 2, size=n).astype(np.int8)
    f = (rng.integers(0, 1 << 53, size=n).astype(np.float64)) * 2.0 ** -53
    aggs = [(SUM, 0), (COUNT, 0), (MIN, 0), (MAX, 0)]
    want = brute_force([k0, k1], [f], aggs)
    for exact in (False, True):
        got = as_dict(oracle.groupby([k0, k1], [f], aggs, exact_f64_sum=exact))
        assert got.keys() == want.keys()
        for k in want:
            if exact:   # math.fsum is the correctly rounded exact sum
                assert got[k] == want[k]
            else:
                assert got[k][1:] == want[k][1:]
                assert got[k][0] == pytest.approx(want[k][0], rel=1e-13)


@settings(max_examples=60, deadline=None)
@given(st.lists(st.tuples(st.integers(-(1 << 63), (1 << 63) - 1), st.integers(-(1 << 63), (1 << 63) - 1)),
                min_size=0, max_size=40),
       st.integers(1, 4))
def test_brute_force_hypothesis(rows, fold):
    keys = np.array([r[0] % fold if fold < 4 else r[0] for r in rows], dtype=np.int64)
    vals = np.array([r[1] for r in rows], dtype=np.int64)
    got = as_dict(oracle.groupby(keys, [vals], ALL4))
    assert got == (brute_force([keys], [vals], ALL4) if len(rows) else {})


def test_exact_f64_sum_is_correctly_rounded_for_large_groups():
    # 2^20 copies of (1 - 2^-53): exact sum = 2^20 - 2^-33, representable
    n = 1 << 20
    v = np.full(n, 1.0 - 2.0 ** -53)
    res = oracle.groupby(np.zeros(n, dtype=np.int64), [v], [(SUM, 0)], exact_f64_sum=True)
    assert res.aggs[0][0] == 2.0 ** 20 - 2.0 ** -33
    # a sum needing more than 64 integer bits: 3 * 2^11 values of (2^53-1) 2^-53 stay exact via fsum
    v = ((np.arange(5000) * 1802201963 % (1 << 53)).astype(np.float64)) * 2.0 ** -53
    res = oracle.groupby(np.zeros(5000, dtype=np.int64), [v], [(SUM, 0)], exact_f64_sum=True)
    assert res.aggs[0][0] == math.fsum(v.tolist())


def test_exact_f64_precondition_is_enforced():
    with pytest.raises(ValueError):
        oracle.groupby(np.zeros(2, dtype=np.int64), [np.array([0.5, 1.5])], [(SUM, 0)], exact_f64_sum=True)


def test_invariants_and_ndv():
    rng = np.random.default_rng(7)
    n = 200_000
    keys = rng.integers(-3000, 3000, size=n).astype(np.int32)
    vals = rng.integers(-10**9, 10**9, size=n).astype(np.int64)
    res = oracle.groupby(keys, [vals], ALL4)
    assert int(res.aggs[1].sum()) == n                                   # sum COUNT = n
    assert int(res.aggs[0].sum()) == int(vals.sum())                     # sum of SUMs = total
    assert int(res.aggs[2].min()) == int(vals.min())
    assert int(res.aggs[3].max()) == int(vals.max())
    assert res.n_groups == oracle.exact_ndv(keys) == len(np.unique(keys))
    assert np.all(np.diff(res.keys[0]) > 0)                              # distinct, sorted
    lo, hi = oracle.minmax(keys)
    assert (lo, hi) == (int(keys.min()), int(keys.max()))
    assert res.keys[0][0] == lo and res.keys[0][-1] == hi


def test_special_cases_reduce_to_numpy():
    rng = np.random.default_rng(8)
    v = rng.integers(-50, 50, size=1000).astype(np.int64)
    one = oracle.groupby(np.full(1000, 42, dtype=np.int64), [v], ALL4)   # all keys equal
    assert one.n_groups == 1 and int(one.keys[0][0]) == 42
    assert [int(a[0]) for a in one.aggs] == [int(v.sum()), 1000, int(v.min()), int(v.max())]
    perm = rng.permutation(1000).astype(np.int64)                        # all keys distinct
    each = oracle.groupby(perm, [v], ALL4)
    assert each.n_groups == 1000
    inv = np.argsort(perm)
    for j in (0, 2, 3):
        assert np.array_equal(each.aggs[j], v[inv])
    assert np.all(each.aggs[1] == 1)


def test_metamorphic():
    rng = np.random.default_rng(9)
    n = 5000
    keys = rng.integers(0, 300, size=n).astype(np.int64)
    vals = rng.integers(-10**6, 10**6, size=n).astype(np.int64)
    base = oracle.groupby(keys, [vals], ALL4)
    p = rng.permutation(n)                                               # row order is irrelevant
    shuf = oracle.groupby(keys[p], [vals[p]], ALL4)
    assert all(np.array_equal(a, b) for a, b in zip(base.aggs, shuf.aggs))
    dbl = oracle.groupby(np.concatenate([keys, keys]), [np.concatenate([vals, vals])], ALL4)
    assert np.array_equal(dbl.aggs[0], 2 * base.aggs[0]) and np.array_equal(dbl.aggs[1], 2 * base.aggs[1])
    assert np.array_equal(dbl.aggs[2], base.aggs[2]) and np.array_equal(dbl.aggs[3], base.aggs[3])
    bij = oracle.groupby(-7 * keys + 11, [vals], ALL4)                   # order-reversing bijection
    assert np.array_equal(bij.keys[0][::-1], -7 * base.keys[0] + 11)
    assert all(np.array_equal(a[::-1], b) for a, b in zip(bij.aggs, base.aggs))


def test_only_restriction_matches_full():
    rng = np.random.default_rng(10)
    keys = rng.integers(0, 100, size=3000).astype(np.int64)
    vals = rng.integers(0, 1000, size=3000).astype(np.int64)
    full = as_dict(oracle.groupby(keys, [vals], ALL4))
    some = as_dict(oracle.groupby(keys, [vals], ALL4, only=np.array([3, 50, 99, 1234])))
    assert set(some) == {(3,), (50,), (99,)} and all(full[k] == some[k] for k in some)


def test_empty_and_extremes():
    e = oracle.groupby(np.zeros(0, dtype=np.int64), [np.zeros(0, dtype=np.int64)], ALL4)
    assert e.n_groups == 0
    assert oracle.minmax(np.zeros(0, dtype=np.int64)) == ((1 << 63) - 1, -(1 << 63))
    assert oracle.exact_ndv(np.zeros(0, dtype=np.int64)) == 0
    k = np.array([-(1 << 63), (1 << 63) - 1, -(1 << 63), 0], dtype=np.int64)
    r = oracle.groupby(k, [np.array([1, 2, 3, 4], dtype=np.int64)], [(SUM, 0), (COUNT, 0)])
    assert r.keys[0].tolist() == [-(1 << 63), 0, (1 << 63) - 1]
    assert r.aggs[0].tolist() == [4, 4, 2] and r.aggs[1].tolist() == [2, 1, 1]


# ---- multi-key group-by (§4.3): 3 and 4 key columns ---------------------------

@pytest.mark.parametrize("nk,seed", [(3, 0), (3, 1), (4, 2), (4, 3), (4, 4)])
def test_brute_force_multi_key(nk, seed):
    rng = np.random.default_rng(700 + seed)
    n = int(rng.integers(1, 81))
    dts = [np.int8, np.int32, np.int64, np.int32]
    spans = [(-2, 2), (1 << 20, (1 << 20) + 3), (-(1 << 40), -(1 << 40) + 2), (-1, 2)]
    keys = [rng.integers(lo, hi, size=n).astype(dt) for (lo, hi), dt in list(zip(spans, dts))[:nk]]
    v = rng.integers(-(1 << 62), 1 << 62, size=n).astype(np.int64)
    got = as_dict(oracle.groupby(keys, [v], ALL4))
    assert got == brute_force(keys, [v], ALL4)
    assert oracle.exact_ndv(keys) == len(got)


def test_multi_key_closed_form_crt():
    """keys (i mod 3, i mod 5, i mod 7, i mod 11), i < 2 * 1155: by the Chinese remainder
    theorem every one of the 3*5*7*11 = 1155 residue tuples occurs exactly twice, as rows
    i0 and i0 + 1155 (i0 = the tuple's CRT solution), so SUM(i) = 2 * i0 + 1155."""
    M = [3, 5, 7, 11]
    P = 1155
    i = np.arange(2 * P, dtype=np.int64)
    keys = [(i % m).astype(np.int32) for m in M]
    res = oracle.groupby(keys, [i], [(COUNT, 0), (SUM, 0), (MIN, 0), (MAX, 0)])
    assert res.n_groups == P and oracle.exact_ndv(keys) == P
    # sorted lexicographically, first column most significant
    tup = [tuple(int(k[g]) for k in res.keys) for g in range(P)]
    assert tup == sorted(tup) and tup[0] == (0, 0, 0, 0) and tup[-1] == (2, 4, 6, 10)
    for g in (0, 1, 17, 500, P - 1):
        i0 = next(x for x in range(P) if all(x % m == r for m, r in zip(M, tup[g])))
        assert [int(a[g]) for a in res.aggs] == [2, 2 * i0 + P, i0, i0 + P]


def test_multi_key_column_order_matters_and_unused_columns_do_not():
    rng = np.random.default_rng(9)
    a = rng.integers(0, 4, size=500).astype(np.int64)
    b = rng.integers(0, 4, size=500).astype(np.int64)
    c = rng.integers(0, 4, size=500).astype(np.int64)
    v = rng.integers(-100, 100, size=500).astype(np.int64)
    r_abc = as_dict(oracle.groupby([a, b, c], [v], ALL4))
    r_cab = as_dict(oracle.groupby([c, a, b], [v], ALL4))
    assert {(k[1], k[2], k[0]): x for k, x in r_cab.items()} == r_abc
    # a constant extra column changes nothing but the key tuple
    z = np.full(500, 7, dtype=np.int64)
    r_abcz = as_dict(oracle.groupby([a, b, c, z], [v], ALL4))
    assert {k[:3]: x for k, x in r_abcz.items()} == r_abc and all(k[3] == 7 for k in r_abcz)
    # the `only` restriction on tuples
    some = sorted(r_abc)[::5]
    only = [np.array([k[j] for k in some], dtype=np.int64) for j in range(3)]
    r_only = as_dict(oracle.groupby([a, b, c], [v], ALL4, only=only))
    assert r_only == {k: r_abc[k] for k in some}
