"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times
(EIGER_AUTO, statistics gathered inside the call): the oracle cannot aggregate 6x10^8 rows in
seconds, so it computes SAMPLED output groups one by one - all rows of a sampled key are gathered
(torch indexing: plumbing) and handed to the oracle's group-by, whose single group must equal the
library's group bit for bit (fp64 SUM: rel 1e-12) - next to the properties that hold at any
size (n_groups = the generator's exact NDV, sum COUNT = n)."""
import numpy as np
import pytest
import torch

import datagen
import oracle
import paper_2607_04489_b200 as eiger

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


@pytest.mark.parametrize("name,n_samples", [("C2", 2), ("C3", 6), ("C4", 8), ("C5:12", 4), ("C5:24:scattered", 8),
                                            ("MK:4:2", 4), ("MK:3:4", 4), ("MK:4:6", 6)])
def test_full_size_sampled_groups(name, n_samples):
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < (90 << 30):
        pytest.skip("needs ~90 GB of free device memory")
    if name == "C2":
        ds = datagen.config2(DEV)
    elif name == "C3":
        ds = datagen.config3(DEV)
    elif name == "C4":
        ds = datagen.config4(DEV)
    elif name.startswith("MK"):
        parts = name.split(":")                      # multi-key, 2^28 rows
        ds = datagen.config_mk(DEV, nk=int(parts[1]), digit_bits=int(parts[2]))
    else:
        parts = name.split(":")
        ds = datagen.config5(DEV, ndv=1 << int(parts[1]), scattered=len(parts) > 2)
    res = eiger.groupby(ds.keys, ds.vals, ds.aggs)          # EIGER_AUTO, as bench.py runs it
    assert res.n_groups == ds.ndv
    cnt_j = [j for j, (op, _) in enumerate(ds.aggs) if op == eiger.COUNT][0]
    assert int(res.aggs[cnt_j].sum().item()) == ds.n
    _check_sampled_groups(ds, res, n_samples)
    del ds, res
    torch.cuda.empty_cache()
