"""`mttkrp_get_perm_noalloc` against `mttkrp_get_perm`.

Why the entry point exists: `mttkrp_get_perm` needs a second nnz-word device buffer from its caller, and some
callers have no way to get one when they call - they run inside an application whose memory pool already holds
all of the GPU's memory (a direct cudaMalloc fails, or bypasses the pool), or on a multi-stream pipeline where
the device-wide stall of cudaMalloc / cudaFree is not acceptable.  The variant keeps that buffer in a fixed
16 MiB array inside the library (limit: MTTKRP_NOALLOC_MAX_NNZ = 2^22 nonzeros) and allocates nothing.

What is checked, through the C-ABI: the permutation is bit-identical to the existing path's (the bar every
permutation test in this suite uses: exact equality) on two calls in a row, including when the shared array
still holds another call's data; the second call takes no device memory; sizes over the limit are refused
with a clear error, the limit itself works.

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure in this side entry
point must not hide the parity tests.  It passes alone in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest
import torch

import workloads as W

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def P():
    import paper_2405_08470_b200 as pkg
    pkg.load_library()          # fails loudly if the CUDA library is missing
    assert torch.cuda.is_available()
    return pkg


def _random_coo(dims, nnz, seed, dev):
    """Seeded uniform indices, duplicates allowed (legal for the library); built on the device."""
    g = torch.Generator(device=dev)
    g.manual_seed(seed)
    idx = torch.stack([torch.randint(0, d, (nnz,), generator=g, device=dev, dtype=torch.int32) for d in dims])
    vals = torch.rand(nnz, generator=g, device=dev, dtype=torch.float32)
    return idx.contiguous(), vals


def test_two_calls_in_a_row_match_get_perm(P):
    dev = torch.device("cuda:0")
    spec = W.CONFIGS[0]                                       # 1000 x 800 x 600, 100k nonzeros
    t = W.generate_tensor(spec)
    h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev))
    N = len(spec.dims)
    want = [h.get_perm(d).clone() for d in range(N)]          # existing path: caller-allocated scratch
    out_a = torch.full((h.nnz,), -1, dtype=torch.int32, device=dev)
    out_b = torch.full((h.nnz,), -1, dtype=torch.int32, device=dev)
    for d in range(N):
        first = h.get_perm_noalloc(d, out=out_a)              # on a fresh process this is the set-up call
        torch.cuda.synchronize()
        free_before = torch.cuda.mem_get_info(dev)[0]
        second = h.get_perm_noalloc(d, out=out_b)             # second call in a row, same arguments
        torch.cuda.synchronize()
        free_after = torch.cuda.mem_get_info(dev)[0]
        assert torch.equal(first, want[d]), f"mode {d}: first call differs from mttkrp_get_perm"
        assert torch.equal(second, want[d]), f"mode {d}: second call differs from mttkrp_get_perm"
        assert free_after >= free_before, "the call took device memory"
    # the array now holds mode-(N-1) leftovers: calls for other modes, back to back, must not see them
    for d in (1, 0, N - 1, 1):
        got = h.get_perm_noalloc(d, out=out_a)
        assert torch.equal(got, want[d]), f"mode {d} after stale contents"
    # a permutation of [0, nnz) (Observation 1)
    assert np.array_equal(np.sort(out_a.cpu().numpy()), np.arange(h.nnz))
    h.destroy()


def test_four_modes_and_another_handle_share_the_array(P):
    dev = torch.device("cuda:0")
    dims = (300, 70, 900, 11)
    idx, vals = _random_coo(dims, 250_000, 7, dev)
    h1 = P.Mttkrp(dims, idx, vals)
    idx2, vals2 = _random_coo((50, 60, 70), 33_333, 8, dev)
    h2 = P.Mttkrp((50, 60, 70), idx2, vals2)
    for _ in range(2):
        for d in range(4):
            assert torch.equal(h1.get_perm_noalloc(d), h1.get_perm(d))
            if d < 3:                                         # same stream: ordered, so sharing is safe
                assert torch.equal(h2.get_perm_noalloc(d), h2.get_perm(d))
    h1.destroy()
    h2.destroy()


def test_limit_is_enforced_and_reachable(P):
    dev = torch.device("cuda:0")
    dims = (3000, 2000, 1000)
    limit = P.binding.NOALLOC_MAX_NNZ
    idx, vals = _random_coo(dims, limit + 1, 11, dev)
    h = P.Mttkrp(dims, idx[:, :limit].contiguous(), vals[:limit].contiguous())      # exactly the limit: whole array in use
    for d in (2, 1):
        assert torch.equal(h.get_perm_noalloc(d), h.get_perm(d))
    h.destroy()
    h = P.Mttkrp(dims, idx, vals)                             # one nonzero more
    out = torch.full((h.nnz,), -7, dtype=torch.int32, device=dev)
    with pytest.raises(P.MttkrpError) as e:
        h.get_perm_noalloc(1, out=out)
    assert e.value.status == P.binding.EUNSUPPORTED
    assert "MTTKRP_NOALLOC_MAX_NNZ" in str(e.value) and str(limit) in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == -7).all()), "a refused call must not launch anything"
    assert torch.equal(h.get_perm(1), h.get_perm(1))          # the handle is still usable through the normal path
    h.destroy()


def test_bad_arguments(P):
    dev = torch.device("cuda:0")
    idx, vals = _random_coo((5, 4, 3), 40, 3, dev)
    h = P.Mttkrp((5, 4, 3), idx, vals)
    lib = P.load_library()
    assert lib.mttkrp_get_perm_noalloc(None, 0, None, None) == P.binding.EINVAL
    assert lib.mttkrp_get_perm_noalloc(h._h, 3, None, None) == P.binding.EINVAL       # d out of range
    assert lib.mttkrp_get_perm_noalloc(h._h, 1, None, None) == P.binding.EINVAL       # NULL output
    h.destroy()
