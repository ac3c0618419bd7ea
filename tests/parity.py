"""Shared comparison helpers for the GPU parity tests (test infrastructure)."""
import numpy as np
import torch

import oracle
import paper_2607_04489_b200 as eiger


def oracle_result(ds, only=None):
    d = ds.cpu()
    return oracle.groupby([k.numpy() for k in d.keys], [v.numpy() for v in d.vals], d.aggs,
                          exact_f64_sum=d.exact_f64_sum, only=only)


def assert_matches(res: eiger.GroupByResult, want, aggs, vals, rel=1e-12):
    """Bit-exact group set and integer aggregates (after sorting by key); fp64 SUM within
    relative 1e-12 (BASELINE.json north_star); fp64 MIN/MAX bit-exact."""
    assert res.n_groups == want.n_groups, (res.n_groups, want.n_groups)
    r = res.sorted()
    for kg, kw in zip(r.keys, want.keys):
        assert np.array_equal(kg.cpu().numpy().astype(np.int64), kw)
    for (op, c), ag, aw in zip(aggs, r.aggs, want.aggs):
        got = ag.cpu().numpy()
        if op == eiger.SUM and vals[c].dtype == torch.float64:
            assert got.dtype == np.float64
            np.testing.assert_allclose(got, aw, rtol=rel, atol=0)
        else:
            assert got.dtype == aw.dtype, (got.dtype, aw.dtype)
            assert np.array_equal(got, aw), (op, c, np.flatnonzero(got != aw)[:5])
