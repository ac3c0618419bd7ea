"""ORACLE — test infrastructure, not product code.

ctypes front end of ``oracle/eiger_oracle.cpp`` (plain single-threaded C++17; see
that file's header for what each function follows in the paper and how it is
pinned).  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s
``cpu_baseline`` / ``--impl reference`` legs may import this package; the product
package ``paper_2607_04489_b200`` never does, and this package never imports it.

Argument marshalling only: keys are widened to int64 (exact), value columns are
passed as int64 or float64; all arithmetic happens in the C++ file.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "eiger_oracle.cpp")
_LIB = os.path.join(_HERE, "liboracle.so")

SUM, COUNT, MIN, MAX = 0, 1, 2, 3
HLL_P = 14  # DESIGN.md reading R1


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no CUDA involved)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


_lib = None


def _load():
    global _lib
    if _lib is None:
        build()
        L = ctypes.CDLL(_LIB)
        L.oracle_groupby_run.restype = ctypes.c_void_p
        L.oracle_groupby_run.argtypes = [
            ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32,
            ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int32, ctypes.c_int32,
            ctypes.c_void_p, ctypes.c_int64]
        L.oracle_groupby_n_groups.restype = ctypes.c_int64
        L.oracle_groupby_n_groups.argtypes = [ctypes.c_void_p]
        L.oracle_groupby_status.restype = ctypes.c_int32
        L.oracle_groupby_status.argtypes = [ctypes.c_void_p]
        L.oracle_groupby_seconds.restype = ctypes.c_double
        L.oracle_groupby_seconds.argtypes = [ctypes.c_void_p]
        L.oracle_groupby_fetch.restype = None
        L.oracle_groupby_fetch.argtypes = [ctypes.c_void_p] * 3
        L.oracle_groupby_free.restype = None
        L.oracle_groupby_free.argtypes = [ctypes.c_void_p]
        L.oracle_exact_ndv.restype = ctypes.c_int64
        L.oracle_exact_ndv.argtypes = [ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64]
        L.oracle_minmax.restype = None
        L.oracle_minmax.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
        L.oracle_hash64.restype = ctypes.c_uint64
        L.oracle_hash64.argtypes = [ctypes.c_int64]
        L.oracle_hll_registers.restype = None
        L.oracle_hll_registers.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_void_p]
        L.oracle_hll_estimate.restype = ctypes.c_double
        L.oracle_hll_estimate.argtypes = [ctypes.c_void_p, ctypes.c_int32]
        L.oracle_dict_encode.restype = ctypes.c_int64
        L.oracle_dict_encode.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p]
        _lib = L
    return _lib


def _i64(a) -> np.ndarray:
    a = np.asarray(a)
    if a.dtype.kind not in "iu" or (a.dtype.kind == "u" and a.dtype.itemsize == 8):
        raise TypeError(f"integer keys expected, got {a.dtype}")
    return np.ascontiguousarray(a, dtype=np.int64)


def _ptr(a: np.ndarray | None):
    return None if a is None else a.ctypes.data_as(ctypes.c_void_p)


MAX_KEY_COLS = 4


def _ptrs(arrs):
    """array of pointers to the given numpy arrays, as a void*"""
    a = (ctypes.c_void_p * max(1, len(arrs)))(*[x.ctypes.data for x in arrs])
    return ctypes.cast(a, ctypes.c_void_p)


@dataclass
class GroupByResult:
    keys: list            # one int64 array per key column, sorted ascending
    aggs: list            # one array per aggregate (int64 or float64)
    n_groups: int
    seconds: float        # steady_clock around the aggregation loop only


def groupby(keys, vals, aggs, exact_f64_sum: bool = False, only=None) -> GroupByResult:
    """keys: one array or a list of 1-4 integer arrays; vals: list of int64/float64
    arrays; aggs: list of (op, val_col).  Result sorted by key."""
    L = _load()
    if isinstance(keys, np.ndarray):
        keys = [keys]
    if not 1 <= len(keys) <= MAX_KEY_COLS:
        raise ValueError("1 to 4 key columns")
    k = [_i64(x) for x in keys]
    n = int(k[0].shape[0])
    v, isf = [], []
    for col in vals:
        col = np.asarray(col)
        if col.dtype == np.float64:
            v.append(np.ascontiguousarray(col)); isf.append(1)
        elif col.dtype.kind == "i":
            v.append(np.ascontiguousarray(col, dtype=np.int64)); isf.append(0)
        else:
            raise TypeError(f"value dtype {col.dtype}")
        if v[-1].shape[0] != n:
            raise ValueError("column length mismatch")
    vp = (ctypes.c_void_p * max(1, len(v)))(*[x.ctypes.data for x in v])
    isf_a = np.asarray(isf + [0], dtype=np.int32)
    ops = np.asarray([a[0] for a in aggs], dtype=np.int32)
    cols = np.asarray([a[1] for a in aggs], dtype=np.int32)
    o = None
    if only is not None:
        if isinstance(only, np.ndarray):
            only = [only]
        o = [_i64(x) for x in only]
        if len(o) != len(k):
            raise ValueError("`only` needs one array per key column")
    h = L.oracle_groupby_run(_ptrs(k), len(k), n,
                             ctypes.cast(vp, ctypes.c_void_p), _ptr(isf_a), len(v),
                             _ptr(ops), _ptr(cols), len(aggs), 1 if exact_f64_sum else 0,
                             _ptrs(o) if o else None,
                             int(o[0].shape[0]) if o else 0)
    try:
        st = L.oracle_groupby_status(h)
        if st != 0:
            raise ValueError(f"oracle_groupby_run status {st}")
        g = L.oracle_groupby_n_groups(h)
        ok = [np.empty(g, dtype=np.int64) for _ in k]
        oa = [np.empty(g, dtype=np.int64) for _ in aggs]
        ap = (ctypes.c_void_p * max(1, len(oa)))(*[x.ctypes.data for x in oa])
        L.oracle_groupby_fetch(h, _ptrs(ok), ctypes.cast(ap, ctypes.c_void_p))
        secs = L.oracle_groupby_seconds(h)
    finally:
        L.oracle_groupby_free(h)
    out = []
    for (op, c), a in zip(aggs, oa):
        out.append(a.view(np.float64) if op != COUNT and isf[c] else a)
    return GroupByResult(ok, out, int(g), float(secs))


def exact_ndv(keys) -> int:
    L = _load()
    if isinstance(keys, np.ndarray):
        keys = [keys]
    k = [_i64(x) for x in keys]
    return int(L.oracle_exact_ndv(_ptrs(k), len(k), k[0].shape[0]))


def minmax(keys) -> tuple[int, int]:
    L = _load()
    k = _i64(keys)
    lo, hi = ctypes.c_int64(), ctypes.c_int64()
    L.oracle_minmax(_ptr(k), k.shape[0], ctypes.byref(lo), ctypes.byref(hi))
    return lo.value, hi.value


def hash64(key: int) -> int:
    return int(_load().oracle_hash64(ctypes.c_int64(int(key))))


def hll_registers(keys, p: int = HLL_P) -> np.ndarray:
    L = _load()
    k = _i64(keys)
    regs = np.empty(1 << p, dtype=np.uint8)
    L.oracle_hll_registers(_ptr(k), k.shape[0], p, _ptr(regs))
    return regs


def hll_estimate(regs: np.ndarray, p: int = HLL_P) -> float:
    L = _load()
    regs = np.ascontiguousarray(regs, dtype=np.uint8)
    assert regs.shape[0] == 1 << p
    return float(L.oracle_hll_estimate(_ptr(regs), p))


@dataclass
class Stats:
    min: int
    max: int
    ndv_est: float
    n: int


def profile(keys, p: int = HLL_P) -> Stats:
    """eiger_profile as the oracle computes it: exact min/max and the sketch estimate
    clamped to [0, min(n, max-min+1)] (reading R6)."""
    k = _i64(keys)
    n = int(k.shape[0])
    lo, hi = minmax(k)
    if n == 0:
        return Stats(lo, hi, 0.0, 0)
    est = hll_estimate(hll_registers(k, p), p)
    est = min(est, float(n), float(hi - lo + 1))
    return Stats(lo, hi, max(est, 0.0), n)


def dict_encode(keys):
    """Order-preserving dictionary encoding (Algorithm 1): returns (codes int64[n],
    dictionary int64[ndv] ascending, ndv) with dictionary[codes[i]] == keys[i]."""
    L = _load()
    k = _i64(keys)
    n = int(k.shape[0])
    codes = np.empty(n, dtype=np.int64)
    d = np.empty(max(n, 1), dtype=np.int64)
    ndv = int(L.oracle_dict_encode(_ptr(k), n, _ptr(codes), _ptr(d)))
    return codes, d[:ndv].copy(), ndv
