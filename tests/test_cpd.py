"""CPD-ALS around the MTTKRP path: pins of the fp64 twin (CPU) and GPU parity."""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import cpd as ocpd


def _dense_rank_r(dims, R, seed):
    rng = np.random.default_rng(seed)
    fac = [rng.uniform(-1.0, 1.0, size=(d, R)) for d in dims]
    X = np.zeros(dims)
    for r in range(R):
        X += np.einsum("i,j,k->ijk", fac[0][:, r], fac[1][:, r], fac[2][:, r])
    grid = np.stack(np.meshgrid(*[np.arange(d) for d in dims], indexing="ij")).reshape(3, -1).astype(np.int32)
    return np.ascontiguousarray(grid), X.reshape(-1).astype(np.float32), X


def test_exact_low_rank_tensor_is_recovered_and_fit_is_monotone():
    dims, R = (6, 5, 4), 2
    idx, vals, X = _dense_rank_r(dims, R, 0)
    rng = np.random.default_rng(1)
    init = [rng.uniform(-1.0, 1.0, size=(d, R)).astype(np.float32) for d in dims]
    A, lam, fits = ocpd.cpd_als(dims, idx, vals, R, 100, init)
    assert fits[-1] > 0.9999                                   # a rank-2 tensor is fitted by rank-2 ALS
    assert all(b >= a - 1e-6 for a, b in zip(fits, fits[1:]))  # ALS never increases the residual
    # the fit formula equals the explicit dense residual (fp32-rounded values are the tensor being fitted)
    Xf = vals.astype(np.float64).reshape(dims)
    Xh = np.einsum("r,ir,jr,kr->ijk", lam, A[0], A[1], A[2])
    want = 1.0 - np.linalg.norm(Xf - Xh) / np.linalg.norm(Xf)
    assert abs(fits[-1] - want) < 1e-6


@pytest.mark.gpu
def test_gpu_cpd_matches_the_fp64_twin():
    import paper_2405_08470_b200 as P
    P.load_library()
    dims, R, iters = [60, 50, 40], 8, 4
    spec = W.TensorSpec("cpd", dims, 6_000, [1.1, 0.0, 0.0], "uniform", (R,), 93)
    t = W.generate_tensor(spec)
    rng = np.random.default_rng(2)
    init = [rng.uniform(0.1, 1.0, size=(d, R)).astype(np.float32) for d in dims]
    Ao, lamo, fo = ocpd.cpd_als(dims, t.idx.numpy(), t.vals.numpy(), R, iters, init)
    dev = torch.device("cuda:0")
    h = P.Mttkrp(dims, t.idx.to(dev), t.vals.to(dev))
    norm_x = float(np.sqrt(np.sum(t.vals.numpy().astype(np.float64) ** 2)))
    Ag, lamg, fg = P.cpd_als(h, dims, R, iters, [torch.from_numpy(a).to(dev) for a in init], norm_x)
    assert h.info()["remaps_done"] == 3 * iters - 1            # cyclic order: one remap per mode call after the first
    h.destroy()
    np.testing.assert_allclose(fg, fo, atol=2e-5)
    np.testing.assert_allclose(lamg.cpu().numpy(), lamo, rtol=2e-3)
    for m in range(3):
        np.testing.assert_allclose(Ag[m].cpu().numpy(), Ao[m], atol=2e-3)
    assert all(b >= a - 1e-5 for a, b in zip(fg, fg[1:]))
