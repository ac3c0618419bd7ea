"""Pins for the oracle's order-preserving dictionary encoding (Algorithm 1):
the brute-force definition (code = number of distinct smaller values), a worked example, and the
properties the paper asks of it (order preserved - "it must preserve the order of the keys in the
encoded values", PAPER.md:223 - and dictionary[code] == key)."""
import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import oracle


def brute(keys):
    distinct = []
    for k in keys:
        if k not in distinct:
            distinct.append(k)
    return [sum(1 for d in distinct if d < k) for k in keys], sorted(distinct)


def test_worked_example():
    # keys 30 10 30 20 10 -> distinct {10, 20, 30} -> codes 2 0 2 1 0
    codes, d, ndv = oracle.dict_encode(np.array([30, 10, 30, 20, 10], dtype=np.int64))
    assert codes.tolist() == [2, 0, 2, 1, 0] and d.tolist() == [10, 20, 30] and ndv == 3


@settings(max_examples=200, deadline=None)
@given(st.lists(st.integers(min_value=-(1 << 63), max_value=(1 << 63) - 1), min_size=0, max_size=40),
       st.lists(st.integers(min_value=-3, max_value=3), min_size=0, max_size=40))
def test_matches_brute_force(wide, narrow):
    for keys in (wide, narrow, wide + narrow):
        codes, d, ndv = oracle.dict_encode(np.array(keys, dtype=np.int64))
        bc, bd = brute(keys)
        assert codes.tolist() == bc and d.tolist() == bd and ndv == len(bd)


@pytest.mark.parametrize("dtype", [np.int8, np.int32, np.int64])
def test_order_and_round_trip(dtype):
    rng = np.random.default_rng(3)
    info = np.iinfo(dtype)
    keys = rng.integers(info.min, info.max, size=20000, endpoint=True).astype(dtype)
    keys[:5] = [info.min, info.max, 0, info.min, info.max]
    codes, d, ndv = oracle.dict_encode(keys)
    assert ndv == np.unique(keys).size and np.all(d[1:] > d[:-1])           # strictly increasing dictionary
    assert np.array_equal(d[codes], keys.astype(np.int64))                      # round trip
    i, j = rng.integers(0, keys.size, size=(2, 5000))
    assert np.array_equal(keys[i] < keys[j], codes[i] < codes[j])               # order preserved
    assert codes.min() == 0 and codes.max() == ndv - 1
    assert oracle.exact_ndv(keys) == ndv                                        # agrees with the independent counter


def test_degenerate_cases():
    codes, d, ndv = oracle.dict_encode(np.zeros(0, dtype=np.int64))
    assert ndv == 0 and codes.size == 0 and d.size == 0
    codes, d, ndv = oracle.dict_encode(np.full(100, -7, dtype=np.int64))
    assert ndv == 1 and not codes.any() and d.tolist() == [-7]
    keys = np.arange(1000, dtype=np.int64)[::-1] * 3
    codes, d, ndv = oracle.dict_encode(keys)
    assert ndv == 1000 and np.array_equal(codes, np.arange(1000)[::-1])         # all distinct: code = rank
