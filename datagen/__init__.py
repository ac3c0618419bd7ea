"""Seeded synthetic inputs for the five BASELINE.json configs.

This module serves both the oracle tests and the CUDA path and therefore holds
none of the method's arithmetic (no aggregation, no sketch hash, no selector): it
only draws inputs.  Everything is integer arithmetic on int64 torch tensors, so
the same call gives bit-identical data on ``cpu`` and on ``cuda`` (checked by
tests/test_datagen.py and tests/test_gpu_parity.py); the one floating-point
table (the Zipf CDF) is computed once on the host with numpy and turned into
integer thresholds before any device sees it.

Recipe:
  r(seed, col, i)   64-bit counter-based draw: two rounds of the murmur3 64-bit
                    finaliser over (i, col, seed) — NOT the sketch hash.
  integers in [lo, hi]: lo + ((r >> 32) * (hi - lo + 1) >> 32)  (range < 2^31)
  fp64 in [0, 1):   (r >> 11) * 2^-53   (so an exact fixed-point sum exists)
  known NDV:        pi(i) = (a*i + b) mod n with gcd(a, n) = 1; row i gets
                    id = pi(i) if pi(i) < D else a random id in [0, D)  =>  every
                    id in [0, D) appears, NDV = min(D, n) exactly.
  dense keys:       key = id;   scattered: key = bijection(id) (murmur3 fmix32 on
                    the id as uint32 for int32 keys; fmix64 of id + seed constant
                    for int64 keys).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np
import torch

_M64 = (1 << 64) - 1
_C1 = 0xFF51AFD7ED558CCD
_C2 = 0xC4CEB9FE1A85EC53
_GOLD = 0x9E3779B97F4A7C15
CHUNK = 1 << 25


def _s64(x: int) -> int:
    """Python int (mod 2^64) -> the int64 with the same bits."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical right shift of int64 (torch's >> is arithmetic)."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def fmix64(x: torch.Tensor) -> torch.Tensor:
    """murmur3 64-bit finaliser; a bijection of the 64-bit words."""
    x = x ^ _lsr(x, 33)
    x = x * _s64(_C1)
    x = x ^ _lsr(x, 33)
    x = x * _s64(_C2)
    x = x ^ _lsr(x, 33)
    return x


def fmix32(x: torch.Tensor) -> torch.Tensor:
    """murmur3 32-bit finaliser on values held in int64 (0 <= x < 2^32); bijection."""
    m = 0xFFFFFFFF
    x = x ^ (x >> 16)
    x = (x * 0x85EBCA6B) & m
    x = x ^ (x >> 13)
    x = (x * 0xC2B2AE35) & m
    x = x ^ (x >> 16)
    return x


def draw(seed: int, col: int, idx: torch.Tensor) -> torch.Tensor:
    """r(seed, col, i): one 64-bit draw per row index (int64 bit pattern)."""
    k = _s64((seed * 0xD1342543DE82EF95 + col * 0xAF251AF3B0F025B5 + 0x1234567) * _GOLD)
    return fmix64(fmix64(idx + k) ^ _s64(_GOLD * (col + 1) + seed))


def uniform_int(seed: int, col: int, idx: torch.Tensor, lo: int, hi: int) -> torch.Tensor:
    span = hi - lo + 1
    assert 0 < span < (1 << 31)
    return lo + ((_lsr(draw(seed, col, idx), 32) * span) >> 32)


def unit_f64(seed: int, col: int, idx: torch.Tensor) -> torch.Tensor:
    """k * 2^-53 with 0 <= k < 2^53."""
    return _lsr(draw(seed, col, idx), 11).to(torch.float64) * (2.0 ** -53)


def _affine(seed: int, n: int) -> tuple[int, int]:
    """(a, b) of a bijection i -> (a*i + b) mod n."""
    if n <= 1:
        return 1, 0
    h = (seed * 0x9E3779B97F4A7C15 + 0x7F4A7C15) & _M64
    a = ((h % n) | 1) + 2
    while math.gcd(a, n) != 1:
        a += 2
    b = (h >> 17) % n
    return a, b


def known_ndv_ids(seed: int, col: int, idx: torch.Tensor, n: int, D: int) -> torch.Tensor:
    """ids in [0, D) for rows idx of an n-row column such that every id < min(D, n) appears."""
    assert n < (1 << 31) and D >= 1
    a, b = _affine(seed, n)
    pi = (idx * a + b) % n
    if D >= n:
        return pi
    rnd = (_lsr(draw(seed, col, idx), 32) * D) >> 32
    return torch.where(pi < D, pi, rnd)


def scatter32(ids: torch.Tensor) -> torch.Tensor:
    """id (0 <= id < 2^32) -> int32-valued key spread over the whole int32 range."""
    x = fmix32(ids)
    return torch.where(x >= (1 << 31), x - (1 << 32), x)


def scatter64(seed: int, ids: torch.Tensor) -> torch.Tensor:
    return fmix64(ids + _s64(_GOLD * (seed + 1)))


def zipf_thresholds(s: float, N: int) -> np.ndarray:
    """Integer inverse-CDF table: rank k (0-based) is drawn when T[k-1] <= r63 < T[k]."""
    w = 1.0 / np.power(np.arange(1, N + 1, dtype=np.float64), s)
    cdf = np.cumsum(w)
    cdf /= cdf[-1]
    t = np.floor(cdf * float(1 << 62)).astype(np.int64) * 2
    t[-1] = np.iinfo(np.int64).max
    return t


@dataclass
class Dataset:
    name: str
    n: int
    keys: list                 # 1 to 4 tensors (int8 / int32 / int64)
    vals: list                 # int64 or float64 tensors
    aggs: list                 # [(op, val_col)], op codes: 0 SUM, 1 COUNT, 2 MIN, 3 MAX
    ndv: int | None = None     # exact NDV by construction, when known
    exact_f64_sum: bool = False
    meta: dict = field(default_factory=dict)

    @property
    def row_bytes(self) -> int:
        return sum(k.element_size() for k in self.keys) + sum(v.element_size() for v in self.vals)

    def cpu(self) -> "Dataset":
        return Dataset(self.name, self.n, [k.cpu() for k in self.keys], [v.cpu() for v in self.vals],
                       self.aggs, self.ndv, self.exact_f64_sum, dict(self.meta))


SUM, COUNT, MIN, MAX = 0, 1, 2, 3


def _fill(n: int, dtype, device, fn) -> torch.Tensor:
    out = torch.empty(n, dtype=dtype, device=device)
    for s in range(0, n, CHUNK):
        e = min(n, s + CHUNK)
        idx = torch.arange(s, e, dtype=torch.int64, device=device)
        out[s:e] = fn(idx).to(dtype)
    return out


def config1(device="cpu", n: int = 1_000_000, seed: int = 0) -> Dataset:
    """C1: int32 keys uniform over [0, 1000) (NDV = 1000 forced), int64 values in [-1000, 1000];
    SUM, COUNT, MIN, MAX."""
    D = 1000
    keys = _fill(n, torch.int32, device, lambda i: known_ndv_ids(seed, 0, i, n, D))
    vals = _fill(n, torch.int64, device, lambda i: uniform_int(seed, 1, i, -1000, 1000))
    return Dataset("C1", n, [keys], [vals], [(SUM, 0), (COUNT, 0), (MIN, 0), (MAX, 0)],
                   ndv=min(D, n), meta={"seed": seed})


def config2(device="cpu", n: int = 600_000_000, seed: int = 2, skewed: bool = False) -> Dataset:
    """C2: two int8 code columns (3 x 2 values), four int64 fixed-point value columns uniform in
    [1, 10^7]; SUM of each plus COUNT.  ``skewed`` = unequal weights with two combos absent."""
    if not skewed:
        def combo(i):
            return known_ndv_ids(seed, 0, i, n, 6)
        ndv = min(6, n)
    else:
        # weights 50 / 25 / 15 / 10 % over combos {0, 1, 3, 4}; combos 2 and 5 never appear
        def combo(i):
            u = uniform_int(seed, 0, i, 0, 99)
            c = torch.where(u < 50, 0, torch.where(u < 75, 1, torch.where(u < 90, 3, 4)))
            forced = torch.tensor([0, 1, 3, 4], dtype=torch.int64, device=i.device)
            return torch.where(i < 4, forced[torch.clamp(i, max=3)], c)
        ndv = min(4, n)
    k0 = _fill(n, torch.int8, device, lambda i: combo(i) // 2)
    k1 = _fill(n, torch.int8, device, lambda i: combo(i) % 2)
    vals = [_fill(n, torch.int64, device, lambda i, c=c: uniform_int(seed, 1 + c, i, 1, 10_000_000))
            for c in range(4)]
    return Dataset("C2", n, [k0, k1], vals, [(SUM, 0), (SUM, 1), (SUM, 2), (SUM, 3), (COUNT, 0)],
                   ndv=ndv, meta={"seed": seed, "skewed": skewed})


def config3(device="cpu", n: int = 200_000_000, seed: int = 3, D: int = 1_000_000,
            s: float = 1.1, dense: bool = False) -> Dataset:
    """C3: int64 keys, rank ~ Zipf(s) over D distinct values, randomly permuted and scattered
    over the int64 range; fp64 values k*2^-53; SUM, COUNT, MIN, MAX."""
    thr = torch.from_numpy(zipf_thresholds(s, D)).to(device)
    a2, b2 = _affine(seed + 77, D)

    def key(i):
        r63 = _lsr(draw(seed, 0, i), 1)
        rank = torch.clamp(torch.searchsorted(thr, r63, right=True), max=D - 1)
        a, b = _affine(seed, n)
        pi = (i * a + b) % n
        rank = torch.where(pi < D, pi, rank)          # coverage: every rank appears once at least
        ids = (rank * a2 + b2) % D                    # rank -> id by a seeded permutation
        return ids if dense else scatter64(seed, ids)
    keys = _fill(n, torch.int64, device, key)
    vals = _fill(n, torch.float64, device, lambda i: unit_f64(seed, 1, i))
    return Dataset("C3", n, [keys], [vals], [(SUM, 0), (COUNT, 0), (MIN, 0), (MAX, 0)],
                   ndv=min(D, n), exact_f64_sum=True, meta={"seed": seed, "zipf_s": s, "dense": dense})


def config4(device="cpu", n: int = 500_000_000, seed: int = 4, D: int = 100_000_000) -> Dataset:
    """C4: int64 keys uniform over D distinct scattered values (NDV exact), int64 values in
    [0, 2^31); SUM, COUNT."""
    keys = _fill(n, torch.int64, device, lambda i: scatter64(seed, known_ndv_ids(seed, 0, i, n, D)))
    vals = _fill(n, torch.int64, device, lambda i: uniform_int(seed, 1, i, 0, (1 << 31) - 2))
    return Dataset("C4", n, [keys], [vals], [(SUM, 0), (COUNT, 0)], ndv=min(D, n), meta={"seed": seed})


def config5(device="cpu", n: int = 1 << 28, seed: int = 5, ndv: int = 1 << 16,
            scattered: bool = False) -> Dataset:
    """C5: int32 keys with NDV exactly ``ndv``: dense range [0, ndv) or scattered over the whole
    int32 range; int64 values in [0, 2^31); SUM, COUNT."""
    def key(i):
        ids = known_ndv_ids(seed, 0, i, n, ndv)
        return scatter32(ids) if scattered else ids
    keys = _fill(n, torch.int32, device, key)
    vals = _fill(n, torch.int64, device, lambda i: uniform_int(seed, 1, i, 0, (1 << 31) - 2))
    return Dataset("C5", n, [keys], [vals], [(SUM, 0), (COUNT, 0)], ndv=min(ndv, n),
                   meta={"seed": seed, "ndv": ndv, "scattered": scattered})


MK_OFFSETS = (-7, 1000, 1 << 20, -(1 << 30))


def config_mk(device="cpu", n: int = 1 << 28, seed: int = 6, nk: int = 4, digit_bits: int = 4,
              dtypes=None) -> Dataset:
    """Multi-key group-by shaped like the paper's 4xI32 key tables (Table 4;
    §4.3): ``nk`` key columns, column c = digit c (``digit_bits`` bits) of an id
    with exactly min(n, 2^(nk * digit_bits)) distinct values, plus a per-column offset so that
    every column needs its own frame of reference; int64 values in [0, 2^31); SUM, COUNT."""
    D = 1 << (nk * digit_bits)
    dtypes = list(dtypes) if dtypes is not None else [torch.int32] * nk
    assert len(dtypes) == nk and 1 <= nk <= 4
    mask = (1 << digit_bits) - 1
    keys = []
    for c in range(nk):
        off = MK_OFFSETS[c] if dtypes[c] != torch.int8 else -3
        assert dtypes[c] != torch.int8 or mask + off <= 127
        keys.append(_fill(n, dtypes[c], device,
                          lambda i, c=c, off=off: ((known_ndv_ids(seed, 0, i, n, D) >> (c * digit_bits)) & mask) + off))
    vals = _fill(n, torch.int64, device, lambda i: uniform_int(seed, 1, i, 0, (1 << 31) - 2))
    return Dataset("MK", n, keys, [vals], [(SUM, 0), (COUNT, 0)], ndv=min(D, n),
                   meta={"seed": seed, "nk": nk, "digit_bits": digit_bits})
