"""paper_2607_04489_b200 — thin Python binding of libeiger.so (include/eiger.h).

Argument marshalling only: every step of the path (profile, select, init, aggregate,
partition, compact) runs inside the C-ABI library's CUDA kernels.  PyTorch is used for
device memory and streams.  There is no CPU fallback: if the library is missing or
was not built for this GPU the import of the first symbol raises.

    import paper_2607_04489_b200 as eiger
    st  = eiger.profile(keys)                                   # eiger_profile
    res = eiger.groupby([keys], [vals], [(eiger.SUM, 0), (eiger.COUNT, 0)])
    res.keys[0], res.aggs[0], res.n_groups, res.variant
"""
from __future__ import annotations

import ctypes
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libeiger.so")

I8, I32, I64, F64 = 0, 1, 2, 3
SUM, COUNT, MIN, MAX = 0, 1, 2, 3
AUTO, DIRECT, SMEM, GLOBAL, PARTITION, SORT = 0, 1, 2, 3, 4, 5
VARIANT_NAMES = {AUTO: "auto", DIRECT: "direct", SMEM: "smem", GLOBAL: "global", PARTITION: "partition", SORT: "sort"}
OK, ERR_ARG, ERR_WORKSPACE, ERR_OUT_CAPACITY, ERR_INFEASIBLE, ERR_CUDA, ERR_TABLE_OVERFLOW, ERR_STATS, ERR_STATIC_LIMIT = 0, -1, -2, -3, -4, -5, -6, -7, -8
HLL_M = 1 << 14

# every symbol include/eiger.h declares (tests check the library exports each of them)
EXPORTS = [
    "eiger_profile", "eiger_profile_keys", "eiger_hll_registers", "eiger_hll_estimate_host", "eiger_groupby",
    "eiger_groupby_workspace_bytes", "eiger_select_variant", "eiger_groupby_host",
    "eiger_launch_count", "eiger_set_kernel_timing", "eiger_kernel_time_ms", "eiger_strerror",
    "eiger_last_cuda_error", "eiger_variant_name", "eiger_shutdown", "eiger_probe", "eiger_dict_encode", "eiger_dict_encode_workspace_bytes", "eiger_reload_tunables",
    "eiger_groupby_direct_static", "eiger_static_max_slots",
]

_DTYPES = {torch.int8: I8, torch.int32: I32, torch.int64: I64, torch.float64: F64}


class EigerError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"eiger error {code}: {msg}")
        self.code = code


class _Col(ctypes.Structure):
    _fields_ = [("data", ctypes.c_void_p), ("dtype", ctypes.c_int32), ("reserved", ctypes.c_int32)]


class _Agg(ctypes.Structure):
    _fields_ = [("op", ctypes.c_int32), ("val_col", ctypes.c_int32)]


class _Stats(ctypes.Structure):
    _fields_ = [("min", ctypes.c_int64), ("max", ctypes.c_int64), ("ndv_est", ctypes.c_double), ("n", ctypes.c_int64)]


class _CallInfo(ctypes.Structure):
    _fields_ = [("variant", ctypes.c_int32), ("attempts", ctypes.c_int32), ("partition_levels", ctypes.c_int32),
                ("partition_prehist", ctypes.c_int32), ("partition_key_bytes", ctypes.c_int32), ("sort_passes", ctypes.c_int32),
                ("ndv_est", ctypes.c_double), ("kernel_launches", ctypes.c_int64), ("spill_rows", ctypes.c_int64), ("dict_ids", ctypes.c_int32), ("reserved", ctypes.c_int32)]

    def as_dict(self) -> dict:
        return {name: getattr(self, name) for name, _ in self._fields_}


@dataclass
class Stats:
    min: int
    max: int
    ndv_est: float
    n: int


@dataclass
class GroupByResult:
    keys: list          # one tensor per key column (key dtype), n_groups long, order unspecified
    aggs: list          # one tensor per aggregate (int64 or float64)
    n_groups: int
    variant: int
    info: dict = None   # eiger_call_info of the call: attempts, partition_levels, ndv_est, kernel_launches, ...

    def sorted(self) -> "GroupByResult":
        """Groups ordered by key (for comparisons)."""
        if self.n_groups == 0:
            return self
        order = torch.arange(self.n_groups, device=self.keys[0].device)
        for k in reversed(self.keys):
            order = order[torch.sort(k[order], stable=True).indices]
        return GroupByResult([k[order] for k in self.keys], [a[order] for a in self.aggs], self.n_groups, self.variant, self.info)


_lib = None


def lib() -> ctypes.CDLL:
    """The loaded C-ABI library; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise ImportError(f"{_LIB_PATH} is missing: run `python -m paper_2607_04489_b200.build` "
                              "(or __graft_entry__.build()); there is no CPU fallback")
        L = ctypes.CDLL(_LIB_PATH)
        vp, i32, i64, sz = ctypes.c_void_p, ctypes.c_int32, ctypes.c_int64, ctypes.c_size_t
        L.eiger_profile.restype = ctypes.c_int
        L.eiger_profile.argtypes = [vp, i32, i64, ctypes.POINTER(_Stats), vp]
        L.eiger_profile_keys.restype = ctypes.c_int
        L.eiger_profile_keys.argtypes = [vp, i32, i64, vp, vp]
        L.eiger_hll_registers.restype = ctypes.c_int
        L.eiger_hll_registers.argtypes = [vp, i32, i64, vp, vp]
        L.eiger_hll_estimate_host.restype = ctypes.c_double
        L.eiger_hll_estimate_host.argtypes = [vp]
        L.eiger_groupby.restype = ctypes.c_int
        L.eiger_groupby.argtypes = [vp, i32, i64, vp, i32, vp, i32, vp, vp, vp, i64,
                                    ctypes.POINTER(i64), i32, ctypes.POINTER(i32), vp, sz, vp, ctypes.POINTER(_CallInfo)]
        L.eiger_groupby_workspace_bytes.restype = sz
        L.eiger_groupby_workspace_bytes.argtypes = [vp, i32, i64, vp, i32, vp, i32, vp, i32]
        L.eiger_select_variant.restype = i32
        L.eiger_select_variant.argtypes = [vp, i32, i64, vp, i32, vp, i32, vp]
        L.eiger_groupby_host.restype = ctypes.c_int
        L.eiger_groupby_host.argtypes = [vp, i32, i64, vp, i32, vp, i32, vp, vp, i64,
                                         ctypes.POINTER(i64), i32, ctypes.POINTER(i32),
                                         ctypes.POINTER(i64), ctypes.POINTER(i64), vp, ctypes.POINTER(_CallInfo)]
        L.eiger_launch_count.restype = i64
        L.eiger_set_kernel_timing.argtypes = [i32]
        L.eiger_kernel_time_ms.restype = ctypes.c_double
        L.eiger_kernel_time_ms.argtypes = [i32, i32, ctypes.POINTER(i64)]
        L.eiger_strerror.restype = ctypes.c_char_p
        L.eiger_strerror.argtypes = [ctypes.c_int]
        L.eiger_last_cuda_error.restype = ctypes.c_char_p
        L.eiger_variant_name.restype = ctypes.c_char_p
        L.eiger_variant_name.argtypes = [i32]
        L.eiger_shutdown.restype = None
        L.eiger_dict_encode.restype = ctypes.c_int
        L.eiger_dict_encode.argtypes = [vp, i32, i64, vp, vp, i64, ctypes.POINTER(i64), vp, sz, vp]
        L.eiger_dict_encode_workspace_bytes.restype = sz
        L.eiger_dict_encode_workspace_bytes.argtypes = [i32, i64, i64]
        L.eiger_groupby_direct_static.restype = ctypes.c_int
        L.eiger_groupby_direct_static.argtypes = [vp, i32, i64, i64, i64, vp, vp, vp, vp, i64, ctypes.POINTER(i64), vp]
        L.eiger_static_max_slots.restype = i64
        L.eiger_probe.restype = ctypes.c_int
        L.eiger_probe.argtypes = [ctypes.c_char_p, i64, i64, ctypes.POINTER(ctypes.c_double), vp]
        _lib = L
    return _lib


def _check(code: int):
    if code != OK:
        L = lib()
        msg = L.eiger_strerror(code).decode()
        if code == ERR_CUDA:
            msg += " — " + L.eiger_last_cuda_error().decode()
        raise EigerError(code, msg)


def _stream(device) -> int:
    return torch.cuda.current_stream(device).cuda_stream


def _cols(tensors, allowed) -> ctypes.Array:
    arr = (_Col * max(1, len(tensors)))()
    for i, t in enumerate(tensors):
        if t.dtype not in allowed:
            raise TypeError(f"unsupported column dtype {t.dtype}")
        if not t.is_contiguous():
            raise ValueError("columns must be contiguous")
        arr[i].data = t.data_ptr() if t.numel() else None
        arr[i].dtype = _DTYPES[t.dtype]
    return arr


def _aggs(aggs) -> ctypes.Array:
    arr = (_Agg * max(1, len(aggs)))()
    for i, (op, col) in enumerate(aggs):
        arr[i].op, arr[i].val_col = int(op), int(col)
    return arr


def _stats_arr(stats):
    if stats is None:
        return None
    arr = (_Stats * len(stats))()
    for i, s in enumerate(stats):
        arr[i].min, arr[i].max, arr[i].ndv_est, arr[i].n = s.min, s.max, s.ndv_est, s.n
    return arr


MAX_KEY_COLS = 4
_KEY_T = (torch.int8, torch.int32, torch.int64)
_VAL_T = (torch.int64, torch.float64, torch.int32)


def profile(keys: torch.Tensor) -> Stats:
    """eiger_profile: exact min/max and the HyperLogLog NDV estimate of a device key column."""
    if not keys.is_cuda:
        raise ValueError("keys must be a CUDA tensor")
    s = _Stats()
    with torch.cuda.device(keys.device):
        _check(lib().eiger_profile(_cols([keys], _KEY_T)[0].data, _DTYPES[keys.dtype], keys.numel(),
                                   ctypes.byref(s), _stream(keys.device)))
    return Stats(s.min, s.max, s.ndv_est, s.n)


def profile_keys(keys) -> list:
    """eiger_profile_keys: the statistics pass of the adaptive path (range first, sketch only
    where the range cannot decide), one read-back for all key columns."""
    if isinstance(keys, torch.Tensor):
        keys = [keys]
    arr = (_Stats * len(keys))()
    dev = keys[0].device
    with torch.cuda.device(dev):
        _check(lib().eiger_profile_keys(_cols(keys, _KEY_T), len(keys), keys[0].numel(), arr, _stream(dev)))
    return [Stats(s.min, s.max, s.ndv_est, s.n) for s in arr]


def hll_registers(keys: torch.Tensor) -> torch.Tensor:
    """eiger_hll_registers: the 16384 sketch registers (uint8, device)."""
    out = torch.empty(HLL_M, dtype=torch.uint8, device=keys.device)
    with torch.cuda.device(keys.device):
        _check(lib().eiger_hll_registers(_cols([keys], _KEY_T)[0].data, _DTYPES[keys.dtype], keys.numel(),
                                         out.data_ptr(), _stream(keys.device)))
    return out


def hll_estimate(regs) -> float:
    """eiger_hll_estimate_host on 16384 host registers."""
    r = torch.as_tensor(regs, dtype=torch.uint8).cpu().contiguous()
    assert r.numel() == HLL_M
    return float(lib().eiger_hll_estimate_host(r.data_ptr()))


def select_variant(keys, vals, aggs, stats) -> int:
    n = keys[0].numel()
    v = lib().eiger_select_variant(_cols(keys, _KEY_T), len(keys), n, _cols(vals, _VAL_T), len(vals),
                                   _aggs(aggs), len(aggs), _stats_arr(stats))
    if v < 0:
        _check(v)
    return v


def workspace_bytes(keys, vals, aggs, stats=None, force: int = AUTO) -> int:
    n = keys[0].numel()
    return int(lib().eiger_groupby_workspace_bytes(_cols(keys, _KEY_T), len(keys), n, _cols(vals, _VAL_T), len(vals),
                                                   _aggs(aggs), len(aggs), _stats_arr(stats), force))


class Workspace:
    """Reusable output columns (the scratch memory is the library's own arena)."""

    def __init__(self, device):
        self.device = device
        self.out = {}

    def column(self, name, n: int, dtype) -> torch.Tensor:
        t = self.out.get(name)
        if t is None or t.numel() < n or t.dtype != dtype:
            t = torch.empty(max(n, 1), dtype=dtype, device=self.device)
            self.out[name] = t
        return t


def groupby(keys, vals, aggs, force: int = AUTO, stats=None, out_capacity: int | None = None,
            workspace: Workspace | None = None, scratch: torch.Tensor | None = None) -> GroupByResult:
    """eiger_groupby on device columns.

    keys: 1-4 CUDA integer tensors; vals: CUDA int64 / float64 / int32 tensors; aggs: [(op, val_col)].
    With stats=None the statistics are gathered inside the call (that is what the adaptive path's
    time includes); pass stats from profile() to skip that.  Scratch memory is the library's own arena
    (workspace = NULL at the C ABI); `workspace` only keeps the output columns between calls.  The one
    decision taken here: when the caller fixed no out_capacity and the library reports more groups than
    the output columns hold (EIGER_ERR_OUT_CAPACITY carries the count), allocate that many and call again.
    `scratch`: a caller-owned uint8 CUDA tensor passed as the C ABI's workspace instead of the library arena
    (size it with workspace_bytes(); too small -> EIGER_ERR_WORKSPACE).
    """
    if isinstance(keys, torch.Tensor):
        keys = [keys]
    if not 1 <= len(keys) <= MAX_KEY_COLS:
        raise EigerError(ERR_ARG, f"1 to {MAX_KEY_COLS} key columns")
    dev = keys[0].device
    if not all(t.is_cuda for t in list(keys) + list(vals)):
        raise ValueError("all columns must be CUDA tensors")
    n = keys[0].numel()
    if any(t.numel() != n for t in list(keys) + list(vals)):
        raise ValueError("column length mismatch")
    L = lib()
    ws = workspace or Workspace(dev)
    kc, vc, ac, sc = _cols(keys, _KEY_T), _cols(vals, _VAL_T), _aggs(aggs), _stats_arr(stats)
    have = min([t.numel() for t in ws.out.values()], default=0)
    cap = out_capacity if out_capacity is not None else min(max(have, 1 << 20), max(n, 1))
    with torch.cuda.device(dev):
        for attempt in range(2):
            ok = [ws.column(("k", i), cap, k.dtype) for i, k in enumerate(keys)]
            oa = [ws.column(("a", j), cap, torch.float64 if (op != COUNT and vals[c].dtype == torch.float64) else torch.int64)
                  for j, (op, c) in enumerate(aggs)]
            okp = (ctypes.c_void_p * 4)(*[t.data_ptr() for t in ok])
            oap = (ctypes.c_void_p * 8)(*[t.data_ptr() for t in oa])
            ng, chosen, info = ctypes.c_int64(0), ctypes.c_int32(0), _CallInfo()
            rc = L.eiger_groupby(kc, len(keys), n, vc, len(vals), ac, len(aggs), sc, okp, oap, cap,
                                 ctypes.byref(ng), force, ctypes.byref(chosen),
                                 scratch.data_ptr() if scratch is not None else None, scratch.numel() if scratch is not None else 0,
                                 _stream(dev), ctypes.byref(info))
            if rc == ERR_OUT_CAPACITY and out_capacity is None and attempt == 0:
                cap = int(ng.value)
                continue
            _check(rc)
            g = int(ng.value)
            return GroupByResult([t[:g] for t in ok], [t[:g] for t in oa], g, int(chosen.value), info.as_dict())
    raise EigerError(ERR_OUT_CAPACITY, "more groups than the output columns hold")


def groupby_host(keys, vals, aggs, force: int = AUTO, out_capacity: int | None = None, out=None):
    """eiger_groupby_host: host tensors (ideally pinned) in, host tensors out; the H2D / D2H
    copies happen inside the library call.  Returns (GroupByResult on host, h2d_bytes, d2h_bytes)."""
    if isinstance(keys, torch.Tensor):
        keys = [keys]
    if any(t.is_cuda for t in list(keys) + list(vals)):
        raise ValueError("groupby_host takes host tensors")
    if not 1 <= len(keys) <= MAX_KEY_COLS:
        raise EigerError(ERR_ARG, f"1 to {MAX_KEY_COLS} key columns")
    n = keys[0].numel()
    L = lib()
    cap = n if out_capacity is None else out_capacity
    if out is None:
        ok = [torch.empty(max(cap, 1), dtype=k.dtype).pin_memory() for k in keys]
        oa = [torch.empty(max(cap, 1), dtype=torch.float64 if (op != COUNT and vals[c].dtype == torch.float64) else torch.int64).pin_memory()
              for (op, c) in aggs]
    else:
        ok, oa = out
    okp = (ctypes.c_void_p * 4)(*[t.data_ptr() for t in ok])
    oap = (ctypes.c_void_p * 8)(*[t.data_ptr() for t in oa])
    ng, chosen, h2d, d2h, info = ctypes.c_int64(0), ctypes.c_int32(0), ctypes.c_int64(0), ctypes.c_int64(0), _CallInfo()
    rc = L.eiger_groupby_host(_cols(keys, _KEY_T), len(keys), n, _cols(vals, _VAL_T), len(vals), _aggs(aggs), len(aggs),
                              okp, oap, cap, ctypes.byref(ng), force, ctypes.byref(chosen),
                              ctypes.byref(h2d), ctypes.byref(d2h), _stream(torch.device("cuda", torch.cuda.current_device())), ctypes.byref(info))
    _check(rc)
    g = int(ng.value)
    return GroupByResult([t[:g] for t in ok], [t[:g] for t in oa], g, int(chosen.value), info.as_dict()), int(h2d.value), int(d2h.value)


def launch_count() -> int:
    return int(lib().eiger_launch_count())


def set_kernel_timing(enabled: bool) -> None:
    lib().eiger_set_kernel_timing(1 if enabled else 0)


def kernel_time_ms(which: int = 0, reset: bool = True):
    n = ctypes.c_int64(0)
    ms = lib().eiger_kernel_time_ms(which, 1 if reset else 0, ctypes.byref(n))
    return float(ms), int(n.value)


def dict_encode(keys: torch.Tensor, dict_capacity: int | None = None):
    """eiger_dict_encode: order-preserving dictionary encoding (Algorithm 1).
    Returns (codes int32[n], dictionary[ndv] ascending, ndv) with dictionary[codes] == keys."""
    if not keys.is_cuda or keys.dtype not in _KEY_T or not keys.is_contiguous():
        raise ValueError("keys must be a contiguous CUDA int8 / int32 / int64 tensor")
    n = keys.numel()
    L = lib()
    cap = n if dict_capacity is None else int(dict_capacity)
    with torch.cuda.device(keys.device):
        codes = torch.empty(max(n, 1), dtype=torch.int32, device=keys.device)
        d = torch.empty(max(cap, 1), dtype=keys.dtype, device=keys.device)
        ws = torch.empty(max(256, int(L.eiger_dict_encode_workspace_bytes(_DTYPES[keys.dtype], n, cap))), dtype=torch.uint8, device=keys.device)
        ndv = ctypes.c_int64(0)
        _check(L.eiger_dict_encode(keys.data_ptr() if n else None, _DTYPES[keys.dtype], n, codes.data_ptr(), d.data_ptr(), cap,
                                   ctypes.byref(ndv), ws.data_ptr(), ws.numel(), _stream(keys.device)))
    g = int(ndv.value)
    return codes[:n], d[:g], g


def groupby_direct_static(keys: torch.Tensor, vals: torch.Tensor, key_min: int, key_max: int,
                          out_keys: torch.Tensor, out_sum: torch.Tensor, out_count: torch.Tensor) -> int:
    """eiger_groupby_direct_static: SUM + COUNT per key with the accumulator array in the library's static
    device scratch (no allocation anywhere in the call; key_max - key_min + 1 <= static_max_slots()).
    The caller owns the three output tensors (capacity = the shortest); returns the group count.
    Calls that overlap on the GPU race on the shared array (include/eiger.h)."""
    if not keys.is_cuda or keys.dtype not in _KEY_T or not keys.is_contiguous():
        raise ValueError("keys must be a contiguous CUDA int8 / int32 / int64 tensor")
    if vals.dtype != torch.int64 or vals.device != keys.device or not vals.is_contiguous() or vals.numel() != keys.numel():
        raise ValueError("vals must be a contiguous int64 tensor of the keys' length on the keys' device")
    for o, dt in ((out_keys, keys.dtype), (out_sum, torch.int64), (out_count, torch.int64)):
        if o.dtype != dt or o.device != keys.device or not o.is_contiguous():
            raise ValueError("outputs: contiguous tensors on the keys' device, out_keys of the keys' dtype, the others int64")
    cap = min(out_keys.numel(), out_sum.numel(), out_count.numel())
    n = keys.numel()
    g = ctypes.c_int64(0)
    with torch.cuda.device(keys.device):
        _check(lib().eiger_groupby_direct_static(keys.data_ptr() if n else None, _DTYPES[keys.dtype], n, int(key_min), int(key_max),
                                                 vals.data_ptr() if n else None, out_keys.data_ptr() if cap else None,
                                                 out_sum.data_ptr() if cap else None, out_count.data_ptr() if cap else None,
                                                 cap, ctypes.byref(g), _stream(keys.device)))
    return int(g.value)


def static_max_slots() -> int:
    """eiger_static_max_slots: the largest key range eiger_groupby_direct_static takes."""
    return int(lib().eiger_static_max_slots())


def probe(name: str, param: int = 0, param2: int = 0) -> float:
    """eiger_probe: one measured building-block rate of the current device (see include/eiger.h)."""
    r = ctypes.c_double(0.0)
    _check(lib().eiger_probe(name.encode(), int(param), int(param2), ctypes.byref(r),
                             _stream(torch.device("cuda", torch.cuda.current_device()))))
    return float(r.value)


def reload_tunables() -> None:
    """eiger_reload_tunables: re-read the EIGER_* environment variables."""
    lib().eiger_reload_tunables()


def shutdown() -> None:
    lib().eiger_shutdown()
