"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle, element by element,
on the same seeded inputs.  Sizes span several tiles and a ragged tail."""
import numpy as np
import pytest
import torch

import datagen
import oracle
import paper_2607_04489_b200 as eiger
from parity import assert_matches, oracle_result

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
ALL_VARIANTS = [eiger.AUTO, eiger.DIRECT, eiger.SMEM, eiger.GLOBAL, eiger.PARTITION, eiger.SORT]


@pytest.fixture(autouse=True)
def _fresh_tunables():
    # the library reads its EIGER_* tunables once; tests that change them (monkeypatch.setenv + reload)
    # must not leak their values into the next test
    yield
    eiger.reload_tunables()


def set_tunable(monkeypatch, name, value):
    monkeypatch.setenv(name, str(value))
    eiger.reload_tunables()


@pytest.fixture(scope="module", autouse=True)
def _need_gpu():
    assert torch.cuda.is_available(), "these tests need the B200"
    eiger.lib()   # fails loudly if libeiger.so is missing: no fallback exists
    yield


def to_dev(ds):
    return datagen.Dataset(ds.name, ds.n, [k.to(DEV) for k in ds.keys], [v.to(DEV) for v in ds.vals],
                           ds.aggs, ds.ndv, ds.exact_f64_sum, ds.meta)


def run_all_variants(ds, variants=ALL_VARIANTS, expect_infeasible=()):
    want = oracle_result(ds)
    d = to_dev(ds)
    ran = []
    for v in variants:
        try:
            res = eiger.groupby(d.keys, d.vals, d.aggs, force=v)
        except eiger.EigerError as e:
            assert e.code == eiger.ERR_INFEASIBLE and v in expect_infeasible, (v, str(e))
            continue
        assert v == eiger.AUTO or res.variant == v
        assert_matches(res, want, d.aggs, d.vals)
        ran.append(res.variant)
    return ran


# ---- profile (A1-A3) ---------------------------------------------------------------------
@pytest.mark.parametrize("dtype", [torch.int8, torch.int32, torch.int64])
@pytest.mark.parametrize("n", [0, 1, 15, 17, 4097, 1_000_003])
def test_profile_parity(dtype, n):
    g = torch.Generator().manual_seed(n + 1)
    info = torch.iinfo(dtype)
    keys = torch.randint(max(info.min, -(1 << 62)), min(info.max, (1 << 62)), (n,), generator=g, dtype=torch.int64).to(dtype)
    if n > 4:
        keys[3] = info.min; keys[n - 2] = info.max
    want_regs = oracle.hll_registers(keys.numpy())
    got_regs = eiger.hll_registers(keys.to(DEV)).cpu().numpy()
    assert np.array_equal(got_regs, want_regs)                       # bit for bit
    st = eiger.profile(keys.to(DEV))
    ws = oracle.profile(keys.numpy())
    assert (st.min, st.max, st.n) == (ws.min, ws.max, ws.n)
    assert st.ndv_est == pytest.approx(ws.ndv_est, rel=1e-12, abs=1e-12)


def test_sketch_registers_deep_zero_runs_and_rho_cap():
    # keys constructed (by inverting the sketch hash, tests/test_oracle_hll.py) so that the remaining
    # 50 hash bits start with 31, 32, 33, 48, 49 zeros or are all zero: reaches the kernel's `wh == 0`
    # branch (profile.cu: hll_update), which random keys take once per 2^32
    from test_oracle_hll import deep_zero_keys
    cases = deep_zero_keys()
    filler = torch.arange(5000, dtype=torch.int64) * 7919 - 123456
    keys = torch.cat([torch.tensor([c[0] for c in cases], dtype=torch.int64), filler, torch.tensor([c[0] for c in cases], dtype=torch.int64)])
    want = oracle.hll_registers(keys.numpy())
    for _, idx, rho in cases:
        assert int(want[idx]) >= rho
    got = eiger.hll_registers(keys.to(DEV)).cpu().numpy()
    assert np.array_equal(got, want) and int(got.max()) == 51
    only = torch.tensor([c[0] for c in cases], dtype=torch.int64)
    got = eiger.hll_registers(only.to(DEV)).cpu().numpy()
    assert {int(i): int(got[i]) for i in np.flatnonzero(got)} == {idx: rho for _, idx, rho in cases}
    st, ws = eiger.profile(keys.to(DEV)), oracle.profile(keys.numpy())
    assert st.ndv_est == pytest.approx(ws.ndv_est, rel=1e-12)


@pytest.mark.parametrize("lg,scattered", [(4, False), (12, True), (16, False), (20, True)])
def test_profile_known_ndv(lg, scattered):
    ds = datagen.config5(n=1 << 22, ndv=1 << lg, scattered=scattered)
    st = eiger.profile(ds.keys[0].to(DEV))
    ndv = min(1 << lg, 1 << 22)
    assert abs(st.ndv_est - ndv) / ndv <= 4 * 1.04 / 128                 # 4 sigma, m = 2^14
    assert np.array_equal(eiger.hll_registers(ds.keys[0].to(DEV)).cpu().numpy(), oracle.hll_registers(ds.keys[0].numpy()))


def test_datagen_is_device_independent():
    a = datagen.config3(n=300_000, D=5000)
    b = datagen.config3(device=DEV, n=300_000, D=5000)
    assert torch.equal(a.keys[0], b.keys[0].cpu()) and torch.equal(a.vals[0], b.vals[0].cpu())
    a = datagen.config5(n=300_000, ndv=4096, scattered=True)
    b = datagen.config5(device=DEV, n=300_000, ndv=4096, scattered=True)
    assert torch.equal(a.keys[0], b.keys[0].cpu()) and torch.equal(a.vals[0], b.vals[0].cpu())


# ---- the five configs, every variant -------------------------------------------------------
def test_config1_all_variants():
    ran = run_all_variants(datagen.config1())
    assert ran[0] == eiger.DIRECT


@pytest.mark.parametrize("skewed", [False, True])
def test_config2_scaled(skewed):
    ds = datagen.config2(n=3_000_017, skewed=skewed)
    ran = run_all_variants(ds)
    assert ran[0] == eiger.DIRECT


@pytest.mark.parametrize("dense", [False, True])
def test_config3_scaled(dense):
    ds = datagen.config3(n=2_000_003, D=50_000, dense=dense)
    run_all_variants(ds, expect_infeasible=() if dense else (eiger.DIRECT,))


def test_config4_scaled():
    ds = datagen.config4(n=3_000_001, D=600_000)
    run_all_variants(ds, expect_infeasible=(eiger.DIRECT,))


@pytest.mark.parametrize("lg", [4, 8, 12, 16, 20])
@pytest.mark.parametrize("scattered", [False, True])
def test_config5_scaled(lg, scattered):
    ds = datagen.config5(n=(1 << 21) + 13, ndv=1 << lg, scattered=scattered)
    run_all_variants(ds)


# ---- edge cases ------------------------------------------------------------------------------
def test_empty_input():
    k = torch.zeros(0, dtype=torch.int64, device=DEV)
    v = torch.zeros(0, dtype=torch.int64, device=DEV)
    for f in ALL_VARIANTS:
        res = eiger.groupby([k], [v], [(eiger.SUM, 0), (eiger.COUNT, 0)], force=f)
        assert res.n_groups == 0
    st = eiger.profile(k)
    assert (st.min, st.max, st.ndv_est, st.n) == ((1 << 63) - 1, -(1 << 63), 0.0, 0)


@pytest.mark.parametrize("n", [1, 2, 31, 33, 511, 513, 2047, 2049, 100_001])
def test_ragged_sizes(n):
    i = torch.arange(n, dtype=torch.int64)
    ds = datagen.Dataset("rag", n, [(i % 7).to(torch.int32)], [i], [(eiger.COUNT, 0), (eiger.SUM, 0), (eiger.MIN, 0), (eiger.MAX, 0)])
    run_all_variants(ds)


def test_closed_form_without_oracle():
    # key_i = i mod D, value_i = i (SURVEY.md 8(c) C.5 iii): checks 64-bit sums at a size the
    # oracle is not needed for
    n, D = (1 << 24) + 5, 1000
    i = torch.arange(n, dtype=torch.int64, device=DEV)
    res = eiger.groupby([(i % D).to(torch.int32)], [i], [(eiger.COUNT, 0), (eiger.SUM, 0), (eiger.MIN, 0), (eiger.MAX, 0)]).sorted()
    k = torch.arange(D, dtype=torch.int64, device=DEV)
    c = (n - k + D - 1) // D
    assert torch.equal(res.keys[0].long(), k) and torch.equal(res.aggs[0], c)
    assert torch.equal(res.aggs[1], c * k + D * c * (c - 1) // 2)
    assert torch.equal(res.aggs[2], k) and torch.equal(res.aggs[3], k + D * (c - 1))


def test_int64_extremes_and_sentinel_key():
    k = torch.tensor([-(1 << 63), (1 << 63) - 1, -(1 << 63), 0, (1 << 63) - 1, 5, -1] * 300, dtype=torch.int64)
    v = torch.arange(k.numel(), dtype=torch.int64) - 1000
    ds = datagen.Dataset("ext", k.numel(), [k], [v], [(eiger.SUM, 0), (eiger.COUNT, 0), (eiger.MIN, 0), (eiger.MAX, 0)])
    run_all_variants(ds, expect_infeasible=(eiger.DIRECT,))
    k32 = torch.tensor([-(1 << 31), (1 << 31) - 1, 0, -1, (1 << 31) - 1] * 400, dtype=torch.int32)
    v = torch.arange(k32.numel(), dtype=torch.int64)
    ds = datagen.Dataset("ext32", k32.numel(), [k32], [v], [(eiger.SUM, 0), (eiger.COUNT, 0)])
    run_all_variants(ds)


def test_all_equal_and_all_distinct():
    n = 70_001
    v = torch.arange(n, dtype=torch.int64) * 3 - 7
    run_all_variants(datagen.Dataset("eq", n, [torch.full((n,), -42, dtype=torch.int64)], [v],
                                     [(eiger.SUM, 0), (eiger.COUNT, 0), (eiger.MIN, 0), (eiger.MAX, 0)]))
    perm = torch.randperm(n, generator=torch.Generator().manual_seed(1)).to(torch.int32)
    run_all_variants(datagen.Dataset("dist", n, [perm], [v], [(eiger.SUM, 0), (eiger.COUNT, 0)]))


def test_generic_signatures():
    g = torch.Generator().manual_seed(5)
    n = 200_003
    k0 = torch.randint(-3, 4, (n,), generator=g, dtype=torch.int64).to(torch.int8)
    k1 = torch.randint(100, 140, (n,), generator=g, dtype=torch.int64).to(torch.int32)
    vi = torch.randint(-10**9, 10**9, (n,), generator=g, dtype=torch.int64)
    vf = torch.randint(0, 1 << 53, (n,), generator=g, dtype=torch.int64).to(torch.float64) * 2.0 ** -53
    vneg = -vf - 1.0
    aggs = [(eiger.MIN, 1), (eiger.MAX, 0), (eiger.SUM, 1), (eiger.MAX, 2), (eiger.MIN, 2), (eiger.SUM, 0)]   # no COUNT
    # vf = k 2^-53: the oracle sums it exactly (128-bit integers, one rounding), tolerance 1e-12
    ds = datagen.Dataset("gen", n, [k0, k1], [vi, vf, vneg], aggs, exact_f64_sum=True)
    want = oracle_result(ds)
    d = to_dev(ds)
    for f in ALL_VARIANTS:
        res = eiger.groupby(d.keys, d.vals, d.aggs, force=f)
        assert_matches(res, want, d.aggs, d.vals)
    # single int8 key, COUNT only
    ds = datagen.Dataset("cnt", n, [k0], [], [(eiger.COUNT, 0)])
    run_all_variants(ds)


@pytest.mark.parametrize("g1", [1, 0])
def test_light_generic_signature_one_value_column(monkeypatch, g1):
    # plans of at most 4 accumulators over one value column: SIG_G1 (hashagg.cuh) or, switched off, the full generic
    # kernels - every hash variant, 32- and 64-bit keys, fp64 / int64 / int32 values, skewed and uniform keys
    set_tunable(monkeypatch, "EIGER_SIG_G1", g1)
    n = 700_003
    i = torch.arange(n, dtype=torch.int64)
    k32 = datagen.scatter64(3, datagen.uniform_int(31, 0, i, 0, 2999)).to(torch.int32)
    vf = datagen.unit_f64(31, 1, i)                     # k 2^-53: the oracle sums it exactly
    vneg = -vf - 1.0
    vi = datagen.uniform_int(31, 2, i, -(1 << 30), (1 << 30) - 2) * 4099
    v32 = datagen.uniform_int(31, 3, i, -(1 << 30), (1 << 30) - 2).to(torch.int32)
    hash_variants = (eiger.AUTO, eiger.SMEM, eiger.GLOBAL, eiger.PARTITION, eiger.SORT)
    for keys, vals, aggs in (
            ([k32], [vf], [(eiger.SUM, 0), (eiger.COUNT, 0)]),
            ([k32], [vneg], [(eiger.MAX, 0), (eiger.MIN, 0)]),
            ([k32], [vi], [(eiger.COUNT, 0), (eiger.MAX, 0), (eiger.SUM, 0), (eiger.SUM, 0)]),
            ([k32], [v32], [(eiger.MIN, 0), (eiger.SUM, 0)]),
            ([datagen.config3(n=n, D=40_000).keys[0]], [vf], [(eiger.SUM, 0)]),          # int64 keys, Zipf: heavy hitters
            ([datagen.config3(n=n, D=40_000).keys[0]], [vi], [(eiger.MIN, 0), (eiger.COUNT, 0), (eiger.SUM, 0)])):
        ds = datagen.Dataset("g1", n, keys, vals, aggs, exact_f64_sum=True)
        run_all_variants(ds, variants=hash_variants)


def test_table_overflow_retry_and_errors():
    ds = to_dev(datagen.config5(n=1 << 20, ndv=1 << 16, scattered=True))
    want = oracle_result(ds)
    st = eiger.profile(ds.keys[0])
    low = [eiger.Stats(st.min, st.max, 64.0, st.n)]                   # injected under-estimate (R10)
    for f in (eiger.SMEM, eiger.GLOBAL, eiger.PARTITION):
        res = eiger.groupby(ds.keys, ds.vals, ds.aggs, force=f, stats=low)
        assert_matches(res, want, ds.aggs, ds.vals)
    with pytest.raises(eiger.EigerError) as e:
        eiger.groupby(ds.keys, ds.vals, ds.aggs, out_capacity=10)
    assert e.value.code == eiger.ERR_OUT_CAPACITY
    with pytest.raises(eiger.EigerError) as e:                        # misaligned column
        eiger.groupby([ds.keys[0][1:]], [ds.vals[0][1:]], ds.aggs)
    assert e.value.code == eiger.ERR_ARG
    wide = to_dev(datagen.config4(n=10_000, D=5_000))
    with pytest.raises(eiger.EigerError) as e:
        eiger.groupby(wide.keys, wide.vals, wide.aggs, force=eiger.DIRECT)
    assert e.value.code == eiger.ERR_INFEASIBLE


def test_host_entry_point():
    ds = datagen.config1(n=300_007)
    want = oracle_result(ds)
    res, h2d, d2h = eiger.groupby_host([k.pin_memory() for k in ds.keys], [v.pin_memory() for v in ds.vals], ds.aggs)
    assert h2d == ds.n * ds.row_bytes and d2h == res.n_groups * (4 + 8 * 4)
    assert_matches(res, want, ds.aggs, ds.vals)


# ---- EIGER_AUTO's sample + speculative pass ------------------------------
SPEC_N = (1 << 22) + 4099          # >= the row count from which AUTO samples and speculates


def _auto_matches(ds, expect_variant=None):
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs)          # AUTO, statistics gathered inside the call
    assert_matches(res, want, d.aggs, d.vals)
    if expect_variant is not None:
        assert res.variant == expect_variant, eiger.VARIANT_NAMES[res.variant]
    return res


@pytest.mark.parametrize("lg,scattered,variant", [(4, False, eiger.DIRECT), (10, False, eiger.DIRECT),
                                                  (4, True, eiger.SMEM), (11, True, eiger.SMEM),
                                                  (18, False, eiger.DIRECT), (18, True, eiger.PARTITION)])
def test_auto_speculative_pass(lg, scattered, variant):
    _auto_matches(datagen.config5(n=SPEC_N, ndv=1 << lg, scattered=scattered), variant)


@pytest.mark.parametrize("ndv,passes", [(12000, 2), (1 << 14, 2)])
def test_auto_dictionary_passes(monkeypatch, ndv, passes):
    # more scattered keys than one large dictionary holds: two passes, each with the dictionary of one hash slice
    ds = datagen.config5(n=SPEC_N, ndv=ndv, scattered=True)
    res = _auto_matches(ds, eiger.SMEM)
    assert res.info["dict_ids"] * passes >= ndv and res.info["dict_ids"] <= 10112 and res.info["attempts"] == 1
    ds.keys[0][SPEC_N // 2 + 5] = 123456789                 # a key no dictionary holds: discarded, partition takes over
    res = _auto_matches(ds, eiger.PARTITION)
    assert res.n_groups == ndv + 1
    set_tunable(monkeypatch, "EIGER_DICT_MAX_PASS_LG", 0)
    res = _auto_matches(datagen.config5(n=SPEC_N, ndv=ndv, scattered=True), eiger.PARTITION)
    assert res.info["dict_ids"] == 0


@pytest.mark.parametrize("ndv", [5000, 7000, 8192])
def test_auto_large_dictionary_front(monkeypatch, ndv):
    # scattered keys beyond the small dictionary (4600) and up to 2^13: the compact dictionary layout (12 bytes per id,
    # 6 per entry, dictionary built from four times the sample); SUM + COUNT plans only
    ds = datagen.config5(n=SPEC_N, ndv=ndv, scattered=True)
    res = _auto_matches(ds, eiger.SMEM)
    assert res.info["dict_ids"] >= ndv and res.info["attempts"] == 1
    # a key that occurs once is not in the dictionary: the pass is discarded and the hash table takes over
    ds.keys[0][SPEC_N // 2 + 5] = 123456789
    res = _auto_matches(ds)
    assert res.n_groups == ndv + 1 and res.info["dict_ids"] == 0
    # other plans keep the hash table
    ds4 = datagen.Dataset("a4", ds.n, ds.keys, ds.vals, [(eiger.SUM, 0), (eiger.COUNT, 0), (eiger.MIN, 0), (eiger.MAX, 0)])
    res = _auto_matches(ds4)
    assert res.info["dict_ids"] == 0
    set_tunable(monkeypatch, "EIGER_DICT_BIG_MAX_KEYS", 0)
    res = _auto_matches(datagen.config5(n=SPEC_N, ndv=ndv, scattered=True))
    assert res.info["dict_ids"] == 0


def test_auto_speculation_gives_up_on_an_outlier():
    # 16 dense groups and ONE row far outside the range the sample sees: the speculative direct pass
    # must notice, discard its result and fall back to the full profile; the answer stays exact
    ds = datagen.config5(n=SPEC_N, ndv=16)
    ds.keys[0][SPEC_N // 3 + 7] = 1_000_000_007
    res = _auto_matches(ds)
    assert res.n_groups == 17
    ds = datagen.config2(n=SPEC_N)
    ds.keys[1][12345] = 100                      # an int8 code outside the sampled 0..1
    res = _auto_matches(ds)
    assert res.n_groups == 7


def test_auto_speculation_gives_up_when_tables_fill():
    # n = 2^22 makes the sample stride exactly 16: the sample only sees rows i = 0 mod 16, which
    # carry 8 scattered keys, while the other rows carry millions of distinct keys.  The plan from the
    # sample is a shared-memory hash pass; every CTA's table fills up -> give up, fall back, exact
    n = 1 << 22
    i = torch.arange(n, dtype=torch.int64)
    few = datagen.fmix32((i // 16) % 8 + 1000)
    many = datagen.fmix32(i + (1 << 24))
    k = torch.where(i % 16 == 0, few, many)
    keys = torch.where(k >= (1 << 31), k - (1 << 32), k).to(torch.int32)
    vals = datagen.uniform_int(9, 1, i, 0, 1000)
    res = _auto_matches(datagen.Dataset("adversarial", n, [keys], [vals], [(eiger.SUM, 0), (eiger.COUNT, 0)]))
    assert res.n_groups > 1_000_000


def test_auto_routes_hot_keys_to_the_global_table():
    ds = datagen.config3(n=SPEC_N, D=200_000)
    _auto_matches(ds, eiger.GLOBAL)


@pytest.mark.parametrize("frac", [0.5, 0.001])
def test_global_spill_buffer_partition_and_merge(monkeypatch, frac):
    # EIGER_GLOBAL: the rows the front cannot hold go through the spill buffer, are partitioned and merged into
    # the global table (frac 0.001: the buffer fills up and the rest of the misses take the global table)
    set_tunable(monkeypatch, "EIGER_GLOBAL_SPILL", 1)             # off by default (measured slower on C3)
    set_tunable(monkeypatch, "EIGER_SPILL_MIN_ROWS", 0)
    set_tunable(monkeypatch, "EIGER_SPILL_FRAC", frac)
    ds = datagen.config3(n=3_000_017, D=200_000)                 # fp64 SUM, COUNT, MIN, MAX; int64 keys
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.GLOBAL)
    assert res.info["spill_rows"] > 0 and res.info["partition_levels"] == 1
    if frac < 0.01:
        assert res.info["spill_rows"] <= 0.001 * ds.n + 2048
    assert_matches(res, want, d.aggs, d.vals)
    res = _auto_matches(datagen.config3(n=SPEC_N, D=200_000), eiger.GLOBAL)      # EIGER_AUTO takes the same path
    assert res.info["spill_rows"] > 0
    # SUM + COUNT on int64 values, keys uniform (almost every row misses the front), ragged size
    ds = datagen.config4(n=1_234_567, D=400_000)
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.GLOBAL)
    assert res.info["spill_rows"] > 0
    assert_matches(res, want, d.aggs, d.vals)
    # the spill buffer is off for 32-bit keys and gives the same groups when switched off
    set_tunable(monkeypatch, "EIGER_GLOBAL_SPILL", 0)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.GLOBAL)
    assert res.info["spill_rows"] == 0
    assert_matches(res, want, d.aggs, d.vals)


def test_global_spill_two_partition_levels_and_generic_signature(small_partition_tables, monkeypatch):
    set_tunable(monkeypatch, "EIGER_GLOBAL_SPILL", 1)
    set_tunable(monkeypatch, "EIGER_SPILL_MIN_ROWS", 0)
    ds = datagen.config4(n=6_000_011, D=5_000_000)
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.GLOBAL)
    assert res.info["spill_rows"] > 0 and res.info["partition_levels"] == 2
    assert_matches(res, want, d.aggs, d.vals)
    # two int64 key columns (fused 64-bit key), three aggregates over two value columns (generic signature)
    n = 2_000_003
    i = torch.arange(n, dtype=torch.int64)
    k0 = datagen.uniform_int(71, 0, i, -500, 499) * 1_000_003
    k1 = datagen.uniform_int(71, 1, i, 0, 299)
    v0 = datagen.uniform_int(71, 2, i, -1000, 1000)
    v1 = datagen.unit_f64(71, 3, i)
    ds = datagen.Dataset("two-key", n, [k0, k1], [v0, v1], [(eiger.MAX, 0), (eiger.SUM, 1), (eiger.MIN, 1)], exact_f64_sum=True)
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.GLOBAL)
    assert res.info["spill_rows"] > 0
    assert_matches(res, want, d.aggs, d.vals)


def test_partition_cuts_hot_partitions_into_items():
    # 2^24 rows over 2^7 partitions: the hot keys' partitions exceed twice the average and are cut
    # into several work items that merge through the global table
    ds = datagen.config3(n=1 << 24, D=300_000)
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.PARTITION)
    assert_matches(res, want, d.aggs, d.vals)


@pytest.mark.parametrize("part_kb,est_log2", [(None, 20), (48, 20), (None, 14), (48, 14)])
def test_partition_tables_close_without_duplicate_groups(monkeypatch, part_kb, est_log2):
    # Forced PARTITION with the NDV under-estimated (R10): 2^22 scattered keys, 16 rows each.
    # est = 2^20 sizes the fan-out so that every partition holds ~1.3x its table's slots in distinct keys:
    # the shared-memory tables CLOSE (0.85 x slots) and later rows go to the global table, whose capacity
    # (2 x est) still takes them - the configuration in which a key could end up in both tables and be
    # emitted twice (hashagg.cuh: s_spilled).  est = 2^14 additionally walks the overflow -> 4x re-run path.
    # Repeated, because the duplicate needs two lanes to race on one key.
    if part_kb is not None:
        set_tunable(monkeypatch, "EIGER_PART_KB", part_kb)
    ds = datagen.config5(n=1 << 26, ndv=1 << 22, scattered=True)
    want = oracle_result(ds)
    d = to_dev(ds)
    st = eiger.profile(d.keys[0])
    low = [eiger.Stats(st.min, st.max, float(1 << est_log2), st.n)]
    for rep in range(10 if est_log2 == 20 else 3):
        res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.PARTITION, stats=low)
        k = res.sorted().keys[0]
        assert bool((k[1:] > k[:-1]).all()), f"duplicate group keys in repetition {rep}"
        assert res.n_groups == 1 << 22
        assert_matches(res, want, d.aggs, d.vals)


@pytest.fixture
def small_partition_tables(monkeypatch):
    # 48 KB per-CTA tables (the tunables are re-read on every call): two partition levels are then
    # needed at sizes the oracle still handles in seconds
    set_tunable(monkeypatch, "EIGER_PART_KB", 48)
    set_tunable(monkeypatch, "EIGER_PART_THREADS", 256)


def test_two_level_partition(small_partition_tables):
    # enough distinct keys for two partition levels (more than 2^10 partitions)
    ds = datagen.config4(n=6_000_011, D=5_000_000)
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.PARTITION)
    assert res.info["partition_levels"] == 2
    assert_matches(res, want, d.aggs, d.vals)
    ds = datagen.config5(n=6_000_011, ndv=1 << 22, scattered=True)
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.PARTITION)
    assert res.info["partition_levels"] == 2
    assert_matches(res, want, d.aggs, d.vals)


# ---- EIGER_AUTO sizes PARTITION from a hash-space slice sketch ---------
@pytest.mark.parametrize("cfg,lg", [("c5", 15), ("c5", 18), ("c5", 22), ("c4", 21)])      # (2^14 int32 keys now take two dictionary passes)
def test_auto_slice_sketch(cfg, lg):
    # the sample settles PARTITION; one keys-only pass gives the level-1 histogram, exact min/max
    # and the NDV from the sketch of a slice of the partitions.  The estimate is checked against
    # the generator's exact NDV (head room 4 / sqrt(slice NDV) <= 9 % is added on purpose).
    D = 1 << lg
    ds = datagen.config5(n=SPEC_N + 12345, ndv=D, scattered=True) if cfg == "c5" else datagen.config4(n=SPEC_N + 777, D=D)
    res = _auto_matches(ds, eiger.PARTITION)
    assert res.n_groups == D
    est = res.info["ndv_est"]
    assert 0.93 * D <= est <= 1.20 * D, (est, D)


def test_auto_slice_sketch_two_levels(small_partition_tables):
    ds = datagen.config5(n=SPEC_N, ndv=1 << 22, scattered=True)
    res = _auto_matches(ds, eiger.PARTITION)
    assert res.info["partition_levels"] == 2 and res.n_groups == 1 << 22


def test_auto_slice_sketch_off_matches(monkeypatch):
    # same input through the full-column profile: same groups, and an estimate within the sketch's error
    set_tunable(monkeypatch, "EIGER_SLICE", 0)
    D = 1 << 18
    res = _auto_matches(datagen.config5(n=SPEC_N + 12345, ndv=D, scattered=True), eiger.PARTITION)
    assert res.n_groups == D and abs(res.info["ndv_est"] - D) <= 4 * 0.008125 * D


# ---- direct-index shared-memory array: the 1024-thread CTA at its size limits ---------------
@pytest.mark.parametrize("R", [4097, 8192, 10240, 10241])
def test_direct_wide_array_sizes(R):
    # SUM + COUNT: 16 bytes per slot, so 10240 slots fill the 160 KB limit of the shared-memory
    # array and 10241 fall to the global-atomics flavour; every key of the range is present
    n = 300_007
    i = torch.arange(n, dtype=torch.int64)
    keys = ((i * 7919) % R - R // 2).to(torch.int32)
    vals = (datagen.uniform_int(11, 1, i, 0, (1 << 31) - 2) - (1 << 30)) * 4099          # +-2^42: carries into the high word
    ds = datagen.Dataset("direct-wide", n, [keys], [vals], [(eiger.SUM, 0), (eiger.COUNT, 0)], ndv=R)
    want = oracle_result(ds)
    d = to_dev(ds)
    for force in (eiger.DIRECT, eiger.AUTO):
        res = eiger.groupby(d.keys, d.vals, d.aggs, force=force)
        assert res.variant == eiger.DIRECT and res.n_groups == R
        assert_matches(res, want, d.aggs, d.vals)


def test_direct_wide_array_all_aggregates():
    # SUM, COUNT, MIN, MAX of int64 and of fp64 on a 3000-slot array (the generic accumulate path
    # of the 1024-thread CTA)
    n = 200_003
    i = torch.arange(n, dtype=torch.int64)
    keys = ((i * 104729) % 3000).to(torch.int64)
    for fp in (False, True):
        vals = datagen.unit_f64(12, 1, i) if fp else datagen.uniform_int(12, 1, i, -1000, 1000)
        ds = datagen.Dataset("direct-wide-4", n, [keys], [vals], [(eiger.SUM, 0), (eiger.COUNT, 0), (eiger.MIN, 0), (eiger.MAX, 0)],
                             ndv=3000, exact_f64_sum=fp)
        want = oracle_result(ds)
        d = to_dev(ds)
        res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.DIRECT)
        assert_matches(res, want, d.aggs, d.vals)


def test_heavy_hitters_int32_keys():
    # Zipf keys as a dense int32 column: the sample flags them as skewed, the heavy hitters (top key
    # 12 % of the rows) take the warp-private cells of the whole-input hash kernel (32-bit key path)
    ds = datagen.config3(n=SPEC_N, D=200_000, dense=True)
    ds = datagen.Dataset("C3-int32", ds.n, [ds.keys[0].to(torch.int32) - 77_000], ds.vals, ds.aggs, ds.ndv, ds.exact_f64_sum, ds.meta)
    _auto_matches(ds, eiger.GLOBAL)


# ---- general multi-key group-by: smart key fusion without the dictionary step ----
@pytest.mark.parametrize("nk,digit_bits,n", [(3, 3, 300_007), (4, 2, 300_007), (4, 4, 1_500_001), (3, 6, 1_500_001)])
def test_multi_key_all_variants(nk, digit_bits, n):
    # fused domains 2^9, 2^8, 2^16 and 2^18: every variant (direct included) on 3 and 4 int32 columns
    ds = datagen.config_mk(n=n, nk=nk, digit_bits=digit_bits)
    ran = run_all_variants(ds)
    assert len(ran) == len(ALL_VARIANTS)


def test_multi_key_mixed_widths_and_four_aggregates():
    g = torch.Generator().manual_seed(11)
    n = 400_003
    k0 = torch.randint(-5, 6, (n,), generator=g, dtype=torch.int64).to(torch.int8)
    k1 = torch.randint(-(1 << 40), -(1 << 40) + 9, (n,), generator=g, dtype=torch.int64)
    k2 = torch.randint((1 << 31) - 20, (1 << 31), (n,), generator=g, dtype=torch.int64).to(torch.int32)   # up to INT32_MAX
    k3 = torch.randint(-128, -120, (n,), generator=g, dtype=torch.int64).to(torch.int8)                   # down to INT8_MIN
    vf = torch.randint(0, 1 << 53, (n,), generator=g, dtype=torch.int64).to(torch.float64) * 2.0 ** -53
    vi = torch.randint(-(1 << 62), 1 << 62, (n,), generator=g, dtype=torch.int64)
    aggs = [(eiger.SUM, 0), (eiger.COUNT, 0), (eiger.MIN, 0), (eiger.MAX, 0), (eiger.SUM, 1), (eiger.MIN, 1)]
    ds = datagen.Dataset("mk-mixed", n, [k0, k1, k2, k3], [vf, vi], aggs, exact_f64_sum=True)
    run_all_variants(ds)
    # three columns, the middle one constant
    ds = datagen.Dataset("mk-const", n, [k2, torch.full((n,), 77, dtype=torch.int64), k0], [vi], [(eiger.SUM, 0), (eiger.COUNT, 0)])
    run_all_variants(ds)


def test_multi_key_wide_ranges_and_infeasible():
    # three columns whose ranges multiply to ~2^61: the fused key needs the 64-bit path; DIRECT cannot run
    g = torch.Generator().manual_seed(12)
    n = 250_001
    ids = torch.randint(0, 5000, (n,), generator=g, dtype=torch.int64)          # 5000 distinct tuples
    k0 = (datagen.fmix64(ids) >> 44).to(torch.int32)                             # ~2^20 range
    k1 = datagen.fmix64(ids + 77) >> 34                                          # ~2^30 range, int64
    k2 = (datagen.fmix64(ids + 999) >> 53).to(torch.int32)                       # ~2^11 range
    v = torch.randint(0, 1 << 31, (n,), generator=g, dtype=torch.int64)
    ds = datagen.Dataset("mk-wide", n, [k0, k1, k2], [v], [(eiger.SUM, 0), (eiger.COUNT, 0)])
    ran = run_all_variants(ds, expect_infeasible=(eiger.DIRECT,))
    assert eiger.DIRECT not in ran[1:]
    # a fourth full-range int64 column: the product of the ranges no longer fits 64 bits.  Round 1 refused
    # (EIGER_ERR_INFEASIBLE); now the wide columns are dictionary-encoded (Algorithm 1), the
    # group-by runs on the codes and the dictionaries decode the group keys
    k3 = datagen.fmix64(ids + 5)
    over = datagen.Dataset("mk-over", n, [k0, k1, k2, k3], [v], [(eiger.SUM, 0), (eiger.COUNT, 0)])
    d = to_dev(over)
    want_over = oracle_result(over)
    for f in (eiger.AUTO, eiger.SMEM, eiger.PARTITION, eiger.SORT):
        res = eiger.groupby(d.keys, d.vals, d.aggs, force=f)
        assert_matches(res, want_over, d.aggs, d.vals)
    # two full-range columns of all-distinct values: no dictionary is small enough -> still refused
    i = torch.arange(n, dtype=torch.int64)
    wide2 = to_dev(datagen.Dataset("mk-hopeless", n, [datagen.fmix64(i), datagen.fmix64(i + n)], [v], [(eiger.COUNT, 0)]))
    res = eiger.groupby(wide2.keys, wide2.vals, wide2.aggs)         # n distinct pairs: codes of 18 + 18 bits fit
    assert res.n_groups == n
    with pytest.raises(eiger.EigerError) as e:                                   # five key columns
        eiger.groupby(d.keys + [d.keys[0]], d.vals, d.aggs)
    assert e.value.code == eiger.ERR_ARG


def test_multi_key_host_entry_point():
    ds = datagen.config_mk(n=200_003, nk=4, digit_bits=3)
    want = oracle_result(ds)
    res, h2d, d2h = eiger.groupby_host(ds.keys, ds.vals, ds.aggs)
    assert_matches(res, want, ds.aggs, ds.vals)
    assert h2d == ds.n * ds.row_bytes


def test_multi_key_fused_sketch():
    # 5000 distinct triples in a ~2^61 domain: the product of the ranges says nothing, the sketch of
    # the fused key does.  The oracle sketches the same fused values, restated here
    # with Python integers from the key columns' exact min/max.
    g = torch.Generator().manual_seed(12)
    n = 250_001
    ids = torch.randint(0, 5000, (n,), generator=g, dtype=torch.int64)
    k0 = (datagen.fmix64(ids) >> 44).to(torch.int32)
    k1 = datagen.fmix64(ids + 77) >> 34
    k2 = (datagen.fmix64(ids + 999) >> 53).to(torch.int32)
    cols = [k0, k1, k2]
    exact = oracle.exact_ndv([c.numpy() for c in cols])
    lo = [int(c.min()) for c in cols]
    rng = [int(c.max()) - int(c.min()) + 1 for c in cols]
    assert rng[0] * rng[1] * rng[2] > 1 << 50
    u = (((k0.to(torch.int64) - lo[0]) * rng[1]) + (k1 - lo[1])) * rng[2] + (k2.to(torch.int64) - lo[2])    # < 2^63: exact in int64
    want = oracle.hll_estimate(oracle.hll_registers(u.numpy()))
    st = eiger.profile_keys([c.to(DEV) for c in cols])
    assert [(s.min, s.max) for s in st] == [(lo[k], lo[k] + rng[k] - 1) for k in range(3)]
    assert st[0].ndv_est == pytest.approx(want, rel=1e-12) and st[1].ndv_est == 1.0 and st[2].ndv_est == 1.0
    assert abs(st[0].ndv_est - exact) <= 4 * 1.04 / 128 * exact          # 4 sigma of m = 2^14 registers
    v = torch.randint(0, 1 << 31, (n,), generator=g, dtype=torch.int64)
    ds = datagen.Dataset("mk-sketch", n, cols, [v], [(eiger.SUM, 0), (eiger.COUNT, 0)])
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs)
    assert_matches(res, oracle_result(ds), d.aggs, d.vals)
    assert res.info["ndv_est"] == pytest.approx(want, rel=1e-9)    # AUTO planned with it
    assert res.variant != eiger.DIRECT
    # small domains keep the range product: no sketch pass
    small = datagen.config_mk(n=100_001, nk=3, digit_bits=3)
    st = eiger.profile_keys([c.to(DEV) for c in small.keys])
    assert [s.ndv_est for s in st] == [8.0, 8.0, 8.0]


def test_multi_key_slice_sketch_single_profile_pass(monkeypatch):
    # EIGER_AUTO, several key columns, enough groups for PARTITION: one pass fuses the columns with the sample's
    # ranges, takes the level-1 histogram and sketches a slice of the fused keys
    def sparse_mk(**kw):
        ds = datagen.config_mk(n=SPEC_N, **kw)
        ds.keys[0] = ds.keys[0] * 1000                                   # a fused domain too wide for a direct array
        return ds
    ds = sparse_mk(nk=4, digit_bits=5)                                    # 2^20 groups, fused domain below 2^32
    res = _auto_matches(ds, eiger.PARTITION)
    assert res.info["partition_prehist"] == 1 and res.info["partition_key_bytes"] == 4
    assert abs(res.info["ndv_est"] / ds.ndv - 1.0) < 0.25                 # slice estimate incl. its head room
    ds = datagen.config_mk(n=SPEC_N, nk=3, digit_bits=7, dtypes=[torch.int64, torch.int32, torch.int64])
    ds.keys[0] = ds.keys[0] * 3_000_000_007                              # 64-bit fused keys
    res = _auto_matches(ds, eiger.PARTITION)
    assert res.info["partition_prehist"] == 1 and res.info["partition_key_bytes"] == 8
    # a row outside the sample's ranges flags the pass: the full profile runs after all, same groups
    ds = sparse_mk(nk=4, digit_bits=5)
    ds.keys[2][SPEC_N // 3 + 1] = (1 << 20) + 5000                        # the column's values are 2^20 .. 2^20 + 31
    res = _auto_matches(ds, eiger.PARTITION)
    assert res.info["partition_prehist"] == 0
    # few groups scattered over a large fused domain: the product of the columns' sample NDVs sends the sample's
    # plan to PARTITION, the slice sketch of the fused key says 2000 and the selector takes the shared-memory table
    g = torch.Generator().manual_seed(21)
    ids = torch.randint(0, 2000, (SPEC_N,), generator=g, dtype=torch.int64)
    cols = [(datagen.fmix64(ids) >> 44).to(torch.int32), datagen.fmix64(ids + 77) >> 34, (datagen.fmix64(ids + 999) >> 53).to(torch.int32)]
    v = torch.randint(0, 1 << 31, (SPEC_N,), generator=g, dtype=torch.int64)
    ds = datagen.Dataset("mk-sparse", SPEC_N, cols, [v], [(eiger.SUM, 0), (eiger.COUNT, 0)])
    res = _auto_matches(ds, eiger.SMEM)
    assert res.n_groups == 2000 and res.info["ndv_est"] < 6000
    # switched off: the round-1 sequence of passes, same groups
    set_tunable(monkeypatch, "EIGER_SLICE_FUSED", 0)
    res = _auto_matches(sparse_mk(nk=4, digit_bits=5), eiger.PARTITION)
    assert res.info["partition_prehist"] == 0


@pytest.mark.parametrize("n", [0, 1, 3, 1025, 4097])
def test_multi_key_tiny_and_ragged(n):
    g = torch.Generator().manual_seed(40 + n)
    k0 = torch.randint(-3, 4, (n,), generator=g, dtype=torch.int64).to(torch.int32)
    k1 = torch.randint(50, 53, (n,), generator=g, dtype=torch.int64).to(torch.int32)
    k2 = torch.randint(-2, 1, (n,), generator=g, dtype=torch.int64).to(torch.int8)
    v = torch.randint(-10**6, 10**6, (n,), generator=g, dtype=torch.int64)
    aggs = [(eiger.SUM, 0), (eiger.COUNT, 0), (eiger.MIN, 0), (eiger.MAX, 0)]
    run_all_variants(datagen.Dataset("mk-tiny", n, [k0, k1, k2], [v], aggs))          # mixed widths: generic loads
    run_all_variants(datagen.Dataset("mk-tiny32", n, [k0, k1], [v], [(eiger.SUM, 0), (eiger.COUNT, 0)]))   # all int32: 32-bit fusion
    if n:
        st = eiger.profile_keys([k0.to(DEV), k1.to(DEV), k2.to(DEV)])
        assert [(s.min, s.max) for s in st] == [(int(k.min()), int(k.max())) for k in (k0, k1, k2)]


# ---- statistics supplied by the caller, int64 margins, int32 payloads ---------------------------------
def test_auto_takes_direct_on_dense_nonnegative_int64_keys():
    # the slack added around the sampled range is clamped to the key type in unsigned arithmetic
    # (min - INT64_MIN overflowed int64 for every min >= 0 and sent such columns to PARTITION)
    ds = datagen.config5(n=SPEC_N, ndv=1 << 12)
    ds = datagen.Dataset("dense-i64", ds.n, [ds.keys[0].to(torch.int64) + 5], ds.vals, ds.aggs, ds.ndv)
    _auto_matches(ds, eiger.DIRECT)
    ds = datagen.Dataset("dense-i64-neg", ds.n, [ds.keys[0] - (1 << 40)], ds.vals, ds.aggs, ds.ndv)
    _auto_matches(ds, eiger.DIRECT)


def test_stale_statistics_are_detected_not_trusted():
    # statistics profiled on another batch: a direct-index array would be indexed out of bounds, a
    # fused multi-column key would alias onto another group -> EIGER_ERR_STATS, nothing is written
    n = 300_007
    i = torch.arange(n, dtype=torch.int64)
    keys = (i % 1000).to(torch.int32).to(DEV)
    vals = i.to(DEV)
    aggs = [(eiger.SUM, 0), (eiger.COUNT, 0)]
    good = eiger.profile(keys)
    stale = [eiger.Stats(0, 499, 500.0, n)]
    for stats, sig in ((stale, aggs), (stale, aggs + [(eiger.MIN, 0)])):
        with pytest.raises(eiger.EigerError) as e:
            eiger.groupby([keys], [vals], sig, force=eiger.DIRECT, stats=stats)
        assert e.value.code == eiger.ERR_STATS
    big = [eiger.Stats(0, 99_999, 1000.0, n)]                      # global-atomics flavour of DIRECT
    keys2 = keys.clone(); keys2[n // 2] = 100_000
    with pytest.raises(eiger.EigerError) as e:
        eiger.groupby([keys2], [vals], aggs, force=eiger.DIRECT, stats=big)
    assert e.value.code == eiger.ERR_STATS
    assert eiger.groupby([keys], [vals], aggs, force=eiger.DIRECT, stats=[good]).n_groups == 1000
    # single-column hash variants rebase modulo 2^32: stale bounds are harmless there
    for f in (eiger.SMEM, eiger.GLOBAL, eiger.PARTITION):
        assert eiger.groupby([keys], [vals], aggs, force=f, stats=[eiger.Stats(0, 499, 1000.0, n)]).n_groups == 1000
    # two key columns, the second one's statistics too narrow
    k1 = ((i // 1000) % 7).to(torch.int32).to(DEV)
    st2 = [eiger.Stats(0, 999, 1000.0, n), eiger.Stats(0, 3, 4.0, n)]
    for f in (eiger.DIRECT, eiger.SMEM, eiger.GLOBAL, eiger.PARTITION):      # (EIGER_SORT maps such rows to the marker key: one extra group)
        with pytest.raises(eiger.EigerError) as e:
            eiger.groupby([keys, k1], [vals], aggs, force=f, stats=st2)
        assert e.value.code == eiger.ERR_STATS, f
    ok = eiger.groupby([keys, k1], [vals], aggs, stats=eiger.profile_keys([keys, k1]))
    assert ok.n_groups == 7000


@pytest.mark.parametrize("kdtype", [torch.int32, torch.int64])
def test_int32_value_columns(kdtype):
    # 4-byte payloads ("both 4-byte data types (I32) and 8-byte"): widened on the fly,
    # results are int64 like the oracle's (which widens before it aggregates)
    n = (1 << 21) + 77
    for lg, scattered in ((6, False), (11, True), (17, True), (17, False)):
        ds = datagen.config5(n=n, ndv=1 << lg, scattered=scattered)
        v32 = (ds.vals[0] - (1 << 30)).to(torch.int32)                       # negative values too
        ds = datagen.Dataset(f"i32-{lg}", n, [ds.keys[0].to(kdtype)], [v32], [(eiger.SUM, 0), (eiger.COUNT, 0)], ds.ndv)
        run_all_variants(ds)
    v2 = datagen.uniform_int(21, 2, torch.arange(n, dtype=torch.int64), -(1 << 30), (1 << 30) - 2).to(torch.int32) * 2 + 1
    vf = datagen.unit_f64(21, 3, torch.arange(n, dtype=torch.int64))
    ds = datagen.config5(n=n, ndv=3000)                 # dense: the direct-index array of 7 aggregates stays small
    ds = datagen.Dataset("i32-mixed", n, [ds.keys[0].to(kdtype)], [v2, ds.vals[0], vf],
                         [(eiger.SUM, 0), (eiger.MIN, 0), (eiger.MAX, 0), (eiger.COUNT, 0), (eiger.SUM, 1), (eiger.SUM, 2), (eiger.MAX, 2)],
                         exact_f64_sum=True)
    run_all_variants(ds)


def test_int32_values_host_entry_point_and_two_keys():
    ds = datagen.config_mk(n=300_011, nk=2, digit_bits=5)
    v32 = (ds.vals[0] % 100_003 - 50_000).to(torch.int32)
    ds = datagen.Dataset("mk-i32", ds.n, ds.keys, [v32], [(eiger.SUM, 0), (eiger.COUNT, 0)], ds.ndv)
    run_all_variants(ds)
    want = oracle_result(ds)
    res, h2d, d2h = eiger.groupby_host(ds.keys, ds.vals, ds.aggs)
    assert_matches(res, want, ds.aggs, ds.vals)
    assert h2d == ds.n * (4 + 4 + 4)


# ---- order-preserving dictionary encoding (Algorithm 1) -----------------------------
@pytest.mark.parametrize("dtype", [torch.int8, torch.int32, torch.int64])
@pytest.mark.parametrize("n,ndv", [(0, 0), (1, 1), (1000, 7), (300_007, 5000), (1 << 21, 1 << 17)])
def test_dict_encode_matches_oracle(dtype, n, ndv):
    info = torch.iinfo(dtype)
    if n == 0:
        keys = torch.zeros(0, dtype=dtype)
    else:
        ids = datagen.known_ndv_ids(31, 0, torch.arange(n, dtype=torch.int64), n, min(ndv, info.max - info.min + 1))
        if dtype == torch.int8:
            keys = (ids % 256 - 128).to(dtype)
        elif dtype == torch.int32:
            keys = datagen.scatter32(ids).to(dtype)
        else:
            keys = datagen.scatter64(31, ids)
        if n > 4:
            keys[3] = info.min; keys[n - 2] = info.max            # the extremes (and the table's marker value -1 below)
            keys[1] = -1
    want_codes, want_dict, want_ndv = oracle.dict_encode(keys.numpy())
    codes, d, g = eiger.dict_encode(keys.to(DEV))
    assert g == want_ndv
    assert codes.dtype == torch.int32 and d.dtype == dtype
    assert np.array_equal(d.cpu().numpy().astype(np.int64), want_dict)
    assert np.array_equal(codes.cpu().numpy().astype(np.int64), want_codes)


def test_dict_encode_capacity_error_and_group_by_on_codes():
    ds = datagen.config5(n=400_003, ndv=3000, scattered=True)
    k = ds.keys[0].to(DEV)
    with pytest.raises(eiger.EigerError) as e:
        eiger.dict_encode(k, dict_capacity=100)
    assert e.value.code == eiger.ERR_OUT_CAPACITY
    # smart key fusion with the dictionary step: a sparse key column becomes a dense
    # code column; grouping by the codes and decoding gives the groups of the original column
    codes, d, g = eiger.dict_encode(k)
    assert g == 3000
    res = eiger.groupby([codes], [ds.vals[0].to(DEV)], ds.aggs).sorted()
    assert res.variant == eiger.DIRECT and res.n_groups == 3000
    want = oracle_result(ds)
    assert np.array_equal(d[res.keys[0].long()].cpu().numpy().astype(np.int64), want.keys[0])   # order-preserving: sorted codes = sorted keys
    for a, b in zip(res.aggs, want.aggs):
        assert np.array_equal(a.cpu().numpy(), b)


# ---- direct-index array split over co-operating CTAs (splitagg.cu) -------------------------------------
@pytest.mark.parametrize("R", [12_000, 1 << 16, (1 << 17) + 3, 180_000])
def test_split_direct_array(monkeypatch, R):
    set_tunable(monkeypatch, "EIGER_SPLIT_MAX", 16)          # groups of up to 16 CTAs (AUTO stops at 4: measured crossover)
    # ranges between one CTA's shared memory (10240 SUM + COUNT slots) and 16 CTAs' worth: every slot of
    # the range is present; ragged row count; values that carry into the high word
    n = (1 << 21) + 4099
    i = torch.arange(n, dtype=torch.int64)
    keys = ((i * 7919) % R - R // 3).to(torch.int32)
    vals = (datagen.uniform_int(13, 1, i, 0, (1 << 31) - 2) - (1 << 30)) * 4099
    ds = datagen.Dataset("split", n, [keys], [vals], [(eiger.SUM, 0), (eiger.COUNT, 0)], ndv=R)
    want = oracle_result(ds)
    d = to_dev(ds)
    for force in (eiger.DIRECT, eiger.AUTO):
        res = eiger.groupby(d.keys, d.vals, d.aggs, force=force)
        assert res.variant == eiger.DIRECT and res.n_groups == R
        assert_matches(res, want, d.aggs, d.vals)
    # four aggregates of fp64 and an int64 key column (generic signature, 64-bit rebased keys)
    vf = datagen.unit_f64(13, 2, i)
    ds = datagen.Dataset("split-f", n, [keys.to(torch.int64) * 1 + (1 << 40)], [vf], [(eiger.SUM, 0), (eiger.COUNT, 0), (eiger.MIN, 0), (eiger.MAX, 0)],
                         ndv=R, exact_f64_sum=True)
    want = oracle_result(ds)
    d = to_dev(ds)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.DIRECT)
    assert_matches(res, want, d.aggs, d.vals)


def test_split_direct_speculation_and_stale_statistics():
    ds = datagen.config5(n=SPEC_N, ndv=1 << 15)
    _auto_matches(ds, eiger.DIRECT)
    ds.keys[0][SPEC_N // 2 + 11] = 77_000_000                 # one row outside the sampled range: the pass is discarded
    res = _auto_matches(ds)
    assert res.n_groups == (1 << 15) + 1
    d = to_dev(datagen.config5(n=1 << 20, ndv=1 << 15))
    with pytest.raises(eiger.EigerError) as e:
        eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.DIRECT, stats=[eiger.Stats(0, (1 << 14) - 1, 1 << 14, d.n)])
    assert e.value.code == eiger.ERR_STATS


@pytest.mark.parametrize("lg", [13, 15, 16])
@pytest.mark.parametrize("kdtype", [torch.int32, torch.int64])
def test_split_hash_tables(monkeypatch, lg, kdtype):
    set_tunable(monkeypatch, "EIGER_SPLIT_HASH", 1)         # an experiment that lost: off by default, kept correct
    # scattered keys, more of them than one CTA's shared-memory table holds: EIGER_SMEM splits them over
    # 2 .. 16 co-operating CTAs (hash slices of the key space); AUTO speculates on it from the sample
    n = SPEC_N + 777
    ds = datagen.config5(n=n, ndv=1 << lg, scattered=True)
    ds = datagen.Dataset(ds.name, n, [ds.keys[0].to(kdtype)], ds.vals, ds.aggs, ds.ndv)
    want = oracle_result(ds)
    d = to_dev(ds)
    st = eiger.profile_keys(d.keys)
    res = eiger.groupby(d.keys, d.vals, d.aggs, force=eiger.SMEM, stats=st)
    assert_matches(res, want, d.aggs, d.vals)
    res = eiger.groupby(d.keys, d.vals, d.aggs)
    assert_matches(res, want, d.aggs, d.vals)
    # generic signature (no static plan), forced
    vf = datagen.unit_f64(17, 2, torch.arange(n, dtype=torch.int64))
    ds2 = datagen.Dataset("split-hash-gen", n, ds.keys, [ds.vals[0], vf], [(eiger.MAX, 0), (eiger.SUM, 1), (eiger.MIN, 1), (eiger.COUNT, 0)], ds.ndv, exact_f64_sum=True)
    d2 = to_dev(ds2)
    res = eiger.groupby(d2.keys, d2.vals, d2.aggs, force=eiger.SMEM, stats=st)
    assert_matches(res, oracle_result(ds2), d2.aggs, d2.vals)


def test_caller_owned_workspace():
    # the C ABI with the caller's scratch (sized by eiger_groupby_workspace_bytes) instead of the library arena
    ds = datagen.config5(n=(1 << 21) + 5, ndv=1 << 17, scattered=True)
    want = oracle_result(ds)
    d = to_dev(ds)
    st = eiger.profile_keys(d.keys)
    for f in (eiger.SMEM, eiger.GLOBAL, eiger.PARTITION, eiger.SORT):
        need = eiger.workspace_bytes(d.keys, d.vals, d.aggs, st, f)
        assert need > 0
        buf = torch.empty(need + 256, dtype=torch.uint8, device=DEV)
        off = (-buf.data_ptr()) % 256
        res = eiger.groupby(d.keys, d.vals, d.aggs, force=f, stats=st, scratch=buf[off:off + need])
        assert_matches(res, want, d.aggs, d.vals)
        with pytest.raises(eiger.EigerError) as e:
            eiger.groupby(d.keys, d.vals, d.aggs, force=f, stats=st, scratch=buf[off:off + 4096])
        assert e.value.code == eiger.ERR_WORKSPACE
    # no statistics: the worst case over the variants
    need = eiger.workspace_bytes(d.keys, d.vals, d.aggs)
    buf = torch.empty(need + 256, dtype=torch.uint8, device=DEV)
    off = (-buf.data_ptr()) % 256
    res = eiger.groupby(d.keys, d.vals, d.aggs, scratch=buf[off:off + need])
    assert_matches(res, want, d.aggs, d.vals)
