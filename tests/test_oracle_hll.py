"""Pins for the oracle's sketch: hash, registers, estimate (no GPU).

Pinned to: published splitmix64 outputs and the survey's third-implementation
values (tests/golden/hll_hash_pins.txt, hll_sketch_pins.txt), a pure-Python
big-integer re-derivation, set invariants of the register array, the
linear-counting closed form, and the 1.04/sqrt(m) error bound on key sets whose
NDV is known by construction (BASELINE.json north_star; reading R6).
"""
import math

import numpy as np
import pytest
import torch

import datagen
import oracle

P = 14
M = 1 << P
SIGMA = 1.04 / math.sqrt(M)
MASK = (1 << 64) - 1


def py_hash(key: int) -> int:
    z = (key + 0x9E3779B97F4A7C15) & MASK
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & MASK
    return z ^ (z >> 31)


def py_idx_rho(key: int):
    z = py_hash(key)
    w = (z << P) & MASK
    lz = 64 - w.bit_length()
    return z >> (64 - P), min(lz, 64 - P) + 1


def test_hash_golden(golden):
    for key, h, idx, rho in golden("hll_hash_pins.txt"):
        key, h, idx, rho = int(key), int(h, 16), int(idx), int(rho)
        assert oracle.hash64(key) == h
        regs = oracle.hll_registers(np.array([key], dtype=np.int64))
        nz = np.flatnonzero(regs)
        assert nz.tolist() == [idx] and int(regs[idx]) == rho       # single key: one register
        assert py_idx_rho(key) == (idx, rho)


def test_registers_match_big_integer_rederivation():
    rng = np.random.default_rng(0)
    keys = np.concatenate([rng.integers(-(1 << 63), (1 << 63) - 1, size=3000),
                           np.arange(-500, 500)]).astype(np.int64)
    want = np.zeros(M, dtype=np.uint8)
    for k in keys.tolist():
        i, r = py_idx_rho(k)
        want[i] = max(want[i], r)
    assert np.array_equal(oracle.hll_registers(keys), want)


def test_rho_cap_when_remaining_bits_are_zero():
    # invert the mixer's last step is not needed: search a hash with w == 0 is infeasible, so
    # check the cap through p: with p = 4 the same code path caps at 64 - 4 + 1 = 61
    regs = oracle.hll_registers(np.arange(100000, dtype=np.int64), p=4)
    assert regs.max() <= 61 and regs.min() >= 1


def test_register_set_invariants():
    rng = np.random.default_rng(1)
    a = rng.integers(-10**12, 10**12, size=20000).astype(np.int64)
    b = rng.integers(-10**12, 10**12, size=20000).astype(np.int64)
    ra, rb = oracle.hll_registers(a), oracle.hll_registers(b)
    assert np.array_equal(oracle.hll_registers(np.concatenate([a, a])), ra)           # duplicates
    assert np.array_equal(oracle.hll_registers(a[rng.permutation(a.size)]), ra)       # order
    assert np.array_equal(oracle.hll_registers(np.concatenate([a, b])), np.maximum(ra, rb))  # merge
    assert not oracle.hll_registers(np.zeros(0, dtype=np.int64)).any()                # empty
    assert ra.max() <= 64 - P + 1


def test_int32_keys_are_sign_extended():
    k32 = np.array([-1, -(1 << 31), 5], dtype=np.int32)
    assert np.array_equal(oracle.hll_registers(k32), oracle.hll_registers(k32.astype(np.int64)))


def test_mixer_is_bijective_and_avalanches():
    x = np.arange(1 << 20, dtype=np.uint64)
    z = x + np.uint64(0x9E3779B97F4A7C15)
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    z = z ^ (z >> np.uint64(31))
    assert np.unique(z).size == x.size
    assert int(z[0]) == oracle.hash64(0) and int(z[12345]) == oracle.hash64(12345)
    flips = []
    for bit in range(0, 64, 7):
        for k in (0, 1, 999, 123456789):
            d = oracle.hash64(k) ^ oracle.hash64(k ^ (1 << bit) if k ^ (1 << bit) < (1 << 63) else k)
            flips.append(bin(d).count("1"))
    assert 28 < np.mean([f for f in flips if f]) < 36


def test_index_histogram_is_uniform():
    regs_idx = np.array([py_idx_rho(k)[0] for k in range(0, 1 << 18)])
    counts = np.bincount(regs_idx, minlength=M)
    expect = (1 << 18) / M
    chi2 = float(((counts - expect) ** 2 / expect).sum())
    assert abs(chi2 - M) < 6 * math.sqrt(2 * M)          # chi^2_(m-1): mean m, sd sqrt(2m)


def _keyset(layout, log2ndv):
    ids = torch.arange(1 << log2ndv, dtype=torch.int64)
    return (datagen.scatter32(ids) if layout == "scattered" else ids).numpy()


def test_whole_sketch_golden(golden):
    for row in golden("hll_sketch_pins.txt"):
        layout, lg, est = row[0], int(row[1]), float(row[5])
        regs = oracle.hll_registers(_keyset(layout, lg))
        assert oracle.hll_estimate(regs) == pytest.approx(est, abs=0.051)
        if row[2] != "-":
            assert int((regs == 0).sum()) == int(row[2])
            assert int(regs.sum()) == int(row[3]) and int(regs.max()) == int(row[4])
            hist = np.bincount(regs, minlength=64)
            assert hist[:len(row) - 6].tolist() == [int(x) for x in row[6:]]


def test_estimate_special_cases():
    assert oracle.hll_estimate(np.zeros(M, dtype=np.uint8)) == 0.0
    one = oracle.hll_registers(np.array([77], dtype=np.int64))
    assert oracle.hll_estimate(one) == pytest.approx(1.0, abs=0.01)
    # small-range closed form: with few keys the sketch carries (almost) only occupancy
    # information and the estimate must agree with linear counting m ln(m / V) (ref [14]'s
    # small-range rule) to well below sigma
    for n in (50, 500, 3000):
        regs = oracle.hll_registers(np.arange(1000, 1000 + n, dtype=np.int64) * 7919)
        lc = M * math.log(M / int((regs == 0).sum()))
        assert oracle.hll_estimate(regs) == pytest.approx(lc, rel=1e-4)
    # monotone: raising any register never lowers the estimate
    r = oracle.hll_registers(np.arange(5000, dtype=np.int64))
    e0 = oracle.hll_estimate(r)
    r2 = r.copy(); r2[np.argmin(r2)] += 3
    assert oracle.hll_estimate(r2) > e0


@pytest.mark.parametrize("lg", [0, 3, 6, 10, 13, 15, 17, 20, 22])
def test_error_bound_known_ndv(lg):
    errs = []
    for seed in range(4 if lg >= 20 else 16):
        ids = torch.arange(1 << lg, dtype=torch.int64)
        keys = datagen.scatter64(seed, ids).numpy()
        assert oracle.exact_ndv(keys) == 1 << lg if lg <= 17 else True
        est = oracle.hll_estimate(oracle.hll_registers(keys))
        errs.append((est - (1 << lg)) / (1 << lg))
    assert max(abs(e) for e in errs) <= 4 * SIGMA + 1e-9
    assert math.sqrt(np.mean(np.square(errs))) <= 1.3 * SIGMA + 1e-9


def test_profile_clamps():
    k = np.arange(100, 164, dtype=np.int64)
    s = oracle.profile(k)
    assert (s.min, s.max, s.n) == (100, 163, 64) and 60 <= s.ndv_est <= 64
    e = oracle.profile(np.zeros(0, dtype=np.int64))
    assert e.ndv_est == 0.0 and e.n == 0
