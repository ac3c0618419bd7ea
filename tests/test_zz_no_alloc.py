"""eiger_groupby_direct_static - the entry point that allocates nothing (its accumulator array is a
static __device__ array inside the library) - against the ordinary path (eiger_groupby, EIGER_AUTO),
bit for bit (integer keys, wrapping int64 SUM, COUNT), on two calls in a row.  The second call uses
fewer keys over a smaller range than the first, so anything the first call left in the shared array
would show up as extra groups or wrong sums.  Collected last on purpose (file name)."""
import pytest
import torch

import datagen
import paper_2607_04489_b200 as eiger

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _keys_vals(seed, n, lo, ndv, dtype):
    i = torch.arange(n, dtype=torch.int64, device=DEV)
    keys = (datagen.uniform_int(seed, 0, i, 0, ndv - 1) + lo).to(dtype)
    vals = datagen.uniform_int(seed, 1, i, -(1 << 30), (1 << 30) - 2) * 1025 + 7      # about +-2^40
    return keys.contiguous(), vals.contiguous()


def _existing_path(keys, vals):
    r = eiger.groupby([keys], [vals], [(eiger.SUM, 0), (eiger.COUNT, 0)]).sorted()
    return r.keys[0], r.aggs[0], r.aggs[1]


def _static_path(keys, vals, lo, hi, cap):
    ok = torch.full((cap,), -7, dtype=keys.dtype, device=DEV)
    osum = torch.full((cap,), -7, dtype=torch.int64, device=DEV)
    ocnt = torch.full((cap,), -7, dtype=torch.int64, device=DEV)
    g = eiger.groupby_direct_static(keys, vals, lo, hi, ok, osum, ocnt)
    order = torch.argsort(ok[:g])
    return g, ok[:g][order], osum[:g][order], ocnt[:g][order]


def _compare(keys, vals, lo, hi, cap):
    g, k, s, c = _static_path(keys, vals, lo, hi, cap)
    wk, ws, wc = _existing_path(keys, vals)
    assert g == wk.numel()
    assert torch.equal(k, wk) and torch.equal(s, ws) and torch.equal(c, wc)
    return g


def test_static_scratch_entry_point_matches_the_existing_path_twice_in_a_row():
    top = eiger.static_max_slots()
    assert top == 65536
    # call 1: the full range of the static array, every slot used, int32 keys from a negative base
    k1, v1 = _keys_vals(101, 3_000_001, -12345, top, torch.int32)
    assert _compare(k1, v1, -12345, -12345 + top - 1, top) == top
    # call 2, straight after: 1000 keys inside a 5000-wide range - stale slots of call 1 must not appear
    k2, v2 = _keys_vals(202, 777_777, 40, 1000, torch.int64)
    assert _compare(k2, v2, 0, 4999, 5000) == 1000
    # and once more with int8 keys and sums that wrap modulo 2^64
    k3 = (torch.arange(100_000, device=DEV) % 200 - 100).to(torch.int8)
    v3 = torch.full((100_000,), (1 << 62) + 3, dtype=torch.int64, device=DEV)
    assert _compare(k3, v3, -128, 127, 256) == 200


def test_static_scratch_entry_point_limits_and_errors():
    top = eiger.static_max_slots()
    k, v = _keys_vals(303, 10_000, 0, 100, torch.int32)
    out = lambda n, dt=torch.int64: torch.empty(n, dtype=dt, device=DEV)
    with pytest.raises(eiger.EigerError) as e:                    # a range beyond the array: refused, nothing launched
        eiger.groupby_direct_static(k, v, 0, top, out(8, torch.int32), out(8), out(8))
    assert e.value.code == eiger.ERR_STATIC_LIMIT and "EIGER_STATIC_MAX_SLOTS" in str(e.value)
    with pytest.raises(eiger.EigerError) as e:                    # bounds that do not hold
        eiger.groupby_direct_static(k, v, 0, 49, out(128, torch.int32), out(128), out(128))
    assert e.value.code == eiger.ERR_STATS
    with pytest.raises(eiger.EigerError) as e:                    # too few output rows
        eiger.groupby_direct_static(k, v, 0, 99, out(10, torch.int32), out(10), out(10))
    assert e.value.code == eiger.ERR_OUT_CAPACITY
    # an empty input is zero groups; the call after the failures above is clean again
    assert eiger.groupby_direct_static(k[:0], v[:0], 0, 9, out(4, torch.int32), out(4), out(4)) == 0
    assert _compare(k, v, 0, 99, 100) == 100
