"""The seeded input generators: determinism, ranges, exact-NDV construction (no GPU)."""
import numpy as np
import torch

import datagen
import oracle


def test_known_ndv_is_exact():
    for n, D in [(1000, 7), (5000, 5000), (4096, 1 << 20), (100_000, 65536), (12345, 1000)]:
        idx = torch.arange(n, dtype=torch.int64)
        ids = datagen.known_ndv_ids(5, 0, idx, n, D).numpy()
        assert ids.min() >= 0 and ids.max() < max(D, n)
        assert len(np.unique(ids)) == min(n, D)


def test_chunking_is_invisible_and_seeded():
    old = datagen.CHUNK
    a = datagen.config5(n=100_000, ndv=1 << 10, scattered=True)
    try:
        datagen.CHUNK = 4096
        b = datagen.config5(n=100_000, ndv=1 << 10, scattered=True)
    finally:
        datagen.CHUNK = old
    assert torch.equal(a.keys[0], b.keys[0]) and torch.equal(a.vals[0], b.vals[0])
    c = datagen.config5(n=100_000, ndv=1 << 10, scattered=True, seed=6)
    assert not torch.equal(a.keys[0], c.keys[0])


def test_config_shapes_and_ndv():
    c1 = datagen.config1()
    assert c1.n == 1_000_000 and c1.keys[0].dtype == torch.int32 and c1.vals[0].dtype == torch.int64
    assert int(c1.keys[0].min()) == 0 and int(c1.keys[0].max()) == 999
    assert int(c1.vals[0].min()) == -1000 and int(c1.vals[0].max()) == 1000
    assert oracle.exact_ndv(c1.keys[0].numpy()) == 1000 == c1.ndv
    c2 = datagen.config2(n=200_000)
    assert [k.dtype for k in c2.keys] == [torch.int8, torch.int8] and len(c2.vals) == 4
    assert oracle.exact_ndv([k.numpy() for k in c2.keys]) == 6
    assert int(c2.keys[0].max()) == 2 and int(c2.keys[1].max()) == 1
    assert all(int(v.min()) >= 1 and int(v.max()) <= 10_000_000 for v in c2.vals)
    c2s = datagen.config2(n=200_000, skewed=True)
    assert oracle.exact_ndv([k.numpy() for k in c2s.keys]) == 4
    c3 = datagen.config3(n=400_000, D=10_000)
    assert c3.keys[0].dtype == torch.int64 and c3.vals[0].dtype == torch.float64
    assert oracle.exact_ndv(c3.keys[0].numpy()) == 10_000
    v = c3.vals[0].numpy()
    assert v.min() >= 0 and v.max() < 1 and np.all(np.ldexp(v, 53) == np.floor(np.ldexp(v, 53)))
    top = np.unique(c3.keys[0].numpy(), return_counts=True)[1].max() / c3.n
    assert 0.05 < top < 0.25                                # Zipf(1.1): a heavy head
    c4 = datagen.config4(n=300_000, D=60_000)
    assert oracle.exact_ndv(c4.keys[0].numpy()) == 60_000
    assert int(c4.vals[0].min()) >= 0 and int(c4.vals[0].max()) < (1 << 31)
    for sc in (False, True):
        c5 = datagen.config5(n=1 << 18, ndv=1 << 12, scattered=sc)
        assert c5.keys[0].dtype == torch.int32
        assert oracle.exact_ndv(c5.keys[0].numpy()) == 1 << 12
        if not sc:
            assert int(c5.keys[0].max()) == (1 << 12) - 1
        else:
            assert int(c5.keys[0].max()) > (1 << 30) and int(c5.keys[0].min()) < -(1 << 30)


def test_scatter_bijections():
    ids = torch.arange(1 << 18, dtype=torch.int64)
    assert len(torch.unique(datagen.scatter32(ids))) == 1 << 18
    assert len(torch.unique(datagen.scatter64(3, ids))) == 1 << 18
    s = datagen.scatter32(ids)
    assert int(s.min()) >= -(1 << 31) and int(s.max()) < (1 << 31)


def test_config_mk_has_exact_ndv_and_per_column_frames():
    import oracle
    ds = datagen.config_mk(n=50_000, nk=3, digit_bits=3)
    assert len(ds.keys) == 3 and ds.ndv == 512
    assert oracle.exact_ndv([k.numpy() for k in ds.keys]) == 512
    for c, k in enumerate(ds.keys):
        assert int(k.min()) == datagen.MK_OFFSETS[c] and int(k.max()) == datagen.MK_OFFSETS[c] + 7
