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


def _unxorshift(z: int, k: int) -> int:
    """inverse of z ^= z >> k on 64 bits"""
    x = z
    for _ in range(64 // k + 1):
        x = z ^ (x >> k)
    return x


INV1 = pow(0xBF58476D1CE4E5B9, -1, 1 << 64)
INV2 = pow(0x94D049BB133111EB, -1, 1 << 64)


def key_with_hash(h: int) -> int:
    """The int64 key whose sketch hash is exactly h: the splitmix64 output function is a bijection
    (two odd multipliers, three xor-shifts, one addition), inverted step by step."""
    z = _unxorshift(h & MASK, 31)
    z = (z * INV2) & MASK
    z = _unxorshift(z, 27)
    z = (z * INV1) & MASK
    z = _unxorshift(z, 30)
    x = (z - 0x9E3779B97F4A7C15) & MASK
    return x - (1 << 64) if x >= (1 << 63) else x


def deep_zero_keys():
    """Keys whose hash has a chosen register index and a chosen number of leading zeros in the
    remaining 50 bits: 0, 1, 17, 31, 32, 33, 48, 49 zeros, and all 50 zero (w = 0: rho = 51, the cap of
    reading R3).  By chance such hashes turn up once per 2^32 .. 2^50 keys."""
    rng = np.random.default_rng(7)
    out = []
    for j, lz in enumerate([0, 1, 17, 31, 32, 33, 48, 49, 50]):
        idx = 1000 + 37 * j
        if lz == 50:
            rest = 0
        else:
            low_bits = 49 - lz
            rest = (1 << low_bits) | (int(rng.integers(0, 1 << low_bits)) if low_bits else 0)
        h = (idx << 50) | rest
        out.append((key_with_hash(h), idx, lz + 1))
    return out


def test_rho_cap_and_deep_zero_runs():
    # (SURVEY.md C.3 step 4 / DESIGN.md R3: rho = min(clz64(w), 50) + 1, so w = 0 gives 51)
    cases = deep_zero_keys()
    for key, idx, rho in cases:
        assert oracle.hash64(key) >> 50 == idx
        assert py_idx_rho(key) == (idx, rho)
        regs = oracle.hll_registers(np.array([key], dtype=np.int64))
        assert np.flatnonzero(regs).tolist() == [idx] and int(regs[idx]) == rho
    keys = np.array([c[0] for c in cases], dtype=np.int64)
    regs = oracle.hll_registers(keys)
    want = np.zeros(M, dtype=np.uint8)
    for _, idx, rho in cases:
        want[idx] = rho
    assert np.array_equal(regs, want) and int(regs.max()) == 64 - P + 1
    # the cap again through another precision: p = 4 caps at 64 - 4 + 1 = 61
    k0 = key_with_hash(0x3 << 60)                      # idx 3, remaining 60 bits all zero
    r4 = oracle.hll_registers(np.array([k0], dtype=np.int64), p=4)
    assert int(r4[3]) == 61 and int(r4.sum()) == 61


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


# ---- estimator (reading R5) against an exact evaluation of the same formula --------------------
def _exact_estimate(hist, p=P):
    """z = m tau(1 - C[q+1]/m); for k = q..1: z = (z + C[k]) / 2; z += m sigma(C[0]/m);
    est = m^2 / (2 ln2 z), evaluated with 60 significant digits (mpmath), series summed to 1e-50."""
    import mpmath as mp
    mp.mp.dps = 60
    m, q = mp.mpf(1 << p), 64 - p

    def sigma(x):
        if x == 1:
            return mp.inf
        z, y = x, mp.mpf(1)
        for _ in range(400):
            x = x * x
            t = x * y
            z += t
            y += y
            if t < mp.mpf(10) ** -50:
                break
        return z

    def tau(x):
        if x == 0 or x == 1:
            return mp.mpf(0)
        z, y = 1 - x, mp.mpf(1)
        for _ in range(400):
            x = mp.sqrt(x)
            y *= mp.mpf(1) / 2
            t = (1 - x) ** 2 * y
            z -= t
            if t < mp.mpf(10) ** -50:
                break
        return z / 3

    z = m * tau(1 - mp.mpf(int(hist[q + 1])) / m)
    for k in range(q, 0, -1):
        z = (z + int(hist[k])) / 2
    z += m * sigma(mp.mpf(int(hist[0])) / m)
    if z == 0:
        return math.inf              # every register saturated
    return float(m * m / (2 * mp.log(2) * z))


def synthetic_register_arrays():
    """Register arrays no real key set of this size produces: many saturated registers (51), so that
    the tau term is far from its trivial value tau(1) = 0, next to zeros and mid values."""
    rng = np.random.default_rng(11)
    arrays = []
    for frac51, frac0 in [(0.0, 0.0), (0.01, 0.0), (0.25, 0.1), (0.5, 0.0), (0.9, 0.05), (0.999, 0.0), (1.0, 0.0), (0.0, 0.999), (0.3, 0.69)]:
        r = rng.integers(1, 51, size=M).astype(np.uint8)
        sel = rng.random(M)
        r[sel < frac51] = 51
        r[(sel >= frac51) & (sel < frac51 + frac0)] = 0
        if frac51 == 1.0:
            r[:] = 51
        arrays.append(r)
    arrays.append(rng.integers(0, 52, size=M).astype(np.uint8))         # uniform over 0 .. 51
    arrays.append(np.minimum(rng.geometric(0.5, size=M) + 40, 51).astype(np.uint8))   # piled up at the cap
    return arrays


def test_estimator_matches_exact_formula_including_tau():
    for regs in synthetic_register_arrays():
        hist = np.bincount(regs, minlength=64)
        want = _exact_estimate(hist)
        got = oracle.hll_estimate(regs)
        assert (got == want) if math.isinf(want) else got == pytest.approx(want, rel=1e-12), (hist[0], hist[51], got, want)
    # tau is really exercised: saturating registers moves the estimate
    base = np.full(M, 30, dtype=np.uint8)
    sat = base.copy(); sat[: M // 2] = 51
    assert oracle.hll_estimate(sat) > 1.5 * oracle.hll_estimate(base)
