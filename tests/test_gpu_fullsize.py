"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(EIGER_AUTO, statistics gathered inside the call).

Where the oracle finishes a full config in tens of seconds (C3: 2x10^8 rows; C5 at 2^12 and 2^20
groups: 2^28 rows) the comparison is ELEMENT BY ELEMENT.  Elsewhere (C2 6x10^8 rows, C4 10^8 groups,
C5 2^24, the multi-key tables) the oracle computes SAMPLED output groups one by one - all rows of a
sampled key are gathered (torch indexing: plumbing) and handed to the oracle's group-by, whose single
group must equal the library's bit for bit (fp64 SUM: rel 1e-12) - next to properties that hold at
any size and need no oracle: n_groups = the generator's exact NDV; sum COUNT = n; the sum of the
SUMs = the column total (wrapping int64; fp64 rel 1e-9 against a pairwise device sum); min of MINs /
max of MAXes = the column's min / max; the output key set = the input's key set (strictly
increasing after sorting; sum and xor of the keys equal those of torch.unique of the input column)."""
import numpy as np
import pytest
import torch

import datagen
import oracle
import paper_2607_04489_b200 as eiger
from parity import assert_matches, oracle_result

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def _check_sampled_groups(ds, res, n_samples):
    g = res.n_groups
    picks = sorted({int(x) for x in np.linspace(0, g - 1, n_samples)})
    cnt_j = [j for j, (op, _) in enumerate(ds.aggs) if op == eiger.COUNT]
    for pos in picks:
        key = [k[pos] for k in res.keys]
        mask = ds.keys[0] == key[0]
        for kc, kv in zip(ds.keys[1:], key[1:]):
            mask &= kc == kv
        idx = mask.nonzero(as_tuple=True)[0]
        del mask
        want = oracle.groupby([k[idx].cpu().numpy() for k in ds.keys], [v[idx].cpu().numpy() for v in ds.vals], ds.aggs,
                              exact_f64_sum=ds.exact_f64_sum)
        assert want.n_groups == 1
        for (op, c), ag, aw in zip(ds.aggs, res.aggs, want.aggs):
            got = ag[pos].item()
            if op == eiger.SUM and ds.vals[c].dtype == torch.float64:
                assert abs(got - aw[0]) <= 1e-12 * abs(aw[0]), (pos, op, got, aw[0])
            else:
                assert got == aw[0].item(), (pos, op, got, aw[0])
        if cnt_j:
            assert res.aggs[cnt_j[0]][pos].item() == idx.numel()


def _xor_fold(t: torch.Tensor) -> int:
    """xor of all elements (halving on the device)."""
    t = t.clone()
    while t.numel() > 1:
        h = t.numel() // 2
        rest = t[2 * h:]
        t = t[:h] ^ t[h:2 * h]
        if rest.numel():
            t[0] ^= rest[0]
    return int(t.item()) if t.numel() else 0


def _check_whole_result_invariants(ds, res):
    """Properties of the whole result that hold at any size (no oracle involved)."""
    assert res.n_groups == ds.ndv
    for (op, c), ag in zip(ds.aggs, res.aggs):
        if op == eiger.COUNT:
            assert int(ag.sum().item()) == ds.n and int(ag.min().item()) >= 1
        elif op == eiger.SUM and ds.vals[c].dtype == torch.float64:
            tot = float(ds.vals[c].sum(dtype=torch.float64).item())
            assert abs(float(ag.sum(dtype=torch.float64).item()) - tot) <= 1e-9 * abs(tot)
        elif op == eiger.SUM:
            assert int(ag.sum().item()) == int(ds.vals[c].to(torch.int64).sum().item())        # both wrap modulo 2^64
        elif op == eiger.MIN:
            assert ag.min().item() == ds.vals[c].min().item()
        else:
            assert ag.max().item() == ds.vals[c].max().item()
    # the output key set is the input's key set
    if len(ds.keys) == 1:
        got = torch.sort(res.keys[0]).values
        assert bool((got[1:] > got[:-1]).all())                        # no key emitted twice
        want = torch.unique(ds.keys[0])
        assert want.numel() == got.numel()
        assert int(got.to(torch.int64).sum().item()) == int(want.to(torch.int64).sum().item())
        x = got.to(torch.int64); y = want.to(torch.int64)
        assert _xor_fold(x) == _xor_fold(y)
        del want, got, x, y
    else:
        r = res.sorted()
        lt = torch.zeros(r.n_groups - 1, dtype=torch.bool, device=r.keys[0].device)
        eq = torch.ones_like(lt)
        for k in r.keys:
            lt |= eq & (k[1:] > k[:-1])
            eq &= k[1:] == k[:-1]
        assert bool(lt.all())                                          # strictly increasing tuples: no duplicate group
    torch.cuda.empty_cache()


def _dataset(name):
    if name == "C2":
        return datagen.config2(DEV)
    if name == "C3":
        return datagen.config3(DEV)
    if name == "C4":
        return datagen.config4(DEV)
    parts = name.split(":")
    if name.startswith("MK"):                        # multi-key, 2^28 rows
        return datagen.config_mk(DEV, nk=int(parts[1]), digit_bits=int(parts[2]))
    return datagen.config5(DEV, ndv=1 << int(parts[1]), scattered=len(parts) > 2)


def _need_memory():
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < (90 << 30):
        pytest.skip("needs ~90 GB of free device memory")


@pytest.mark.parametrize("name,n_samples", [("C2", 2), ("C3", 6), ("C4", 8), ("C5:12", 4), ("C5:24:scattered", 8),
                                            ("MK:4:2", 4), ("MK:3:4", 4), ("MK:4:6", 6)])
def test_full_size_sampled_groups_and_invariants(name, n_samples):
    _need_memory()
    ds = _dataset(name)
    res = eiger.groupby(ds.keys, ds.vals, ds.aggs)          # EIGER_AUTO, as bench.py runs it
    _check_whole_result_invariants(ds, res)
    _check_sampled_groups(ds, res, n_samples)
    del ds, res
    torch.cuda.empty_cache()


@pytest.mark.parametrize("name", ["C3", "C5:12:scattered", "C5:20:scattered", "C5:16"])
def test_full_size_element_by_element(name):
    # every group of the full-size result against the oracle's (about 20-40 s of oracle time each)
    _need_memory()
    ds = _dataset(name)
    res = eiger.groupby(ds.keys, ds.vals, ds.aggs)
    want = oracle_result(ds)
    assert_matches(res, want, ds.aggs, ds.vals)
    del ds, res, want
    torch.cuda.empty_cache()
