"""The seeded synthetic-input generator (CPU).  Inputs only: no method arithmetic lives there."""
import numpy as np
import pytest
import torch

import workloads as W


def test_splitmix64_matches_bigint_reference():
    x = torch.tensor([0, 1, 2, -1, 123456789, 2**63 - 1, -2**63], dtype=torch.int64)
    got = W.splitmix64(x).tolist()
    want = [W._i64(W.splitmix64_py(v & W._M64)) for v in x.tolist()]
    assert got == want


def test_udivmod_is_unsigned():
    xs = torch.tensor([-1, -5, 10, 2**63 - 1, -2**63, -123456789012345], dtype=torch.int64)
    for m in [7, 1_800_000, 4, 29_000]:
        q, r = W.udivmod(xs, m)
        for xv, qv, rv in zip(xs.tolist(), q.tolist(), r.tolist()):
            assert (qv & W._M64, rv) == divmod(xv & W._M64, m)


def test_config1_shape_and_determinism():
    spec = W.CONFIGS[0]
    a = W.generate_tensor(spec)
    b = W.generate_tensor(spec)
    assert a.idx.dtype == torch.int32 and a.vals.dtype == torch.float32
    assert tuple(a.idx.shape) == (3, 100_000)
    assert torch.equal(a.idx, b.idx) and torch.equal(a.vals, b.vals)
    for m, d in enumerate(spec.dims):
        assert int(a.idx[m].min()) >= 0 and int(a.idx[m].max()) < d
    key = W._linear_key([a.idx[m].long() for m in range(3)], spec.dims)
    assert torch.unique(key).numel() == spec.nnz          # de-duplicated
    assert not bool((key[1:] >= key[:-1]).all())          # arrives unsorted
    assert 0.0 <= float(a.vals.min()) and float(a.vals.max()) < 1.0
    # uniform modes: every row of the smallest mode is hit about nnz / I times
    c = torch.bincount(a.idx[2].long(), minlength=600).double()
    assert abs(float(c.mean()) - 100_000 / 600) < 1e-9 and float(c.std()) < 0.2 * float(c.mean())


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_scaled_configs_keep_their_shape_class(cfg):
    spec = W.CONFIGS[cfg].scaled(60_000)
    t = W.generate_tensor(spec)
    N = len(spec.dims)
    assert tuple(t.idx.shape) == (N, 60_000)
    cols = [t.idx[m].long() for m in range(N)]
    for m, d in enumerate(spec.dims):
        assert int(cols[m].min()) >= 0 and int(cols[m].max()) < d
    # distinct tuples (two-column check avoids the 64-bit key wrap of config 3)
    tup = torch.stack(cols, dim=1)
    assert torch.unique(tup, dim=0).shape[0] == 60_000
    # Zipf modes are skewed (heaviest row far above the mean), uniform modes are not
    for m in range(N):
        c = torch.bincount(cols[m], minlength=spec.dims[m])
        mean_present = 60_000 / max(1, int((c > 0).sum()))
        if spec.zipf_s[m] > 0:
            assert int(c.max()) > 20 * mean_present
        elif spec.dims[m] < 6000:
            assert int(c.max()) < 3 * 60_000 / spec.dims[m] + 20
    if spec.values == "lognormal":
        assert float(t.vals.min()) > 0 and float(t.vals.max()) > 5.0


def test_factors_are_uniform_pm1_and_seeded():
    spec = W.CONFIGS[0]
    f = W.generate_factors(spec, 16)
    g = W.generate_factors(spec, 16)
    assert [tuple(x.shape) for x in f] == [(1000, 16), (800, 16), (600, 16)]
    for a, b in zip(f, g):
        assert a.dtype == torch.float32 and torch.equal(a, b)
        assert float(a.min()) >= -1.0 and float(a.max()) < 1.0
        assert abs(float(a.mean())) < 0.02
    assert not torch.equal(f[0][:600], f[2])


def test_zipf_cdf_is_the_truncated_power_law():
    c = W.zipf_cdf(1000, 1.1)
    w = np.arange(1, 1001, dtype=np.float64) ** -1.1
    np.testing.assert_allclose(np.diff(np.concatenate([[0.0], c])), w / w.sum(), rtol=1e-9, atol=1e-15)
    assert c[-1] == 1.0
    p = W.seeded_permutation(1000, 5)
    assert np.array_equal(np.sort(p), np.arange(1000))
