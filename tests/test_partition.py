"""Alg. 1 of the paper: pins of the plain-Python twin (CPU) and GPU parity."""
import numpy as np
import pytest
import torch

import workloads as W
from oracle import partition as opart


def test_fig2_example():
    # PAPER.md:179 (Fig. 2, mode 0): vertex i_2 has two hyperedges and goes to B_{0,0}; i_0 and i_1 (one each) go
    # to B_{0,1}; both partitions hold two hyperedges.
    part, loads = opart.partition_rows([1, 1, 2], 2)
    assert loads == [2, 2]
    assert part[2] == 0 and part[0] == 1 and part[1] == 1


def test_four_thirds_bound_against_brute_force():
    # at most 4/3 of the optimum (Graham's bound for longest-first: 4/3 - 1/(3 kappa)).
    rng = np.random.default_rng(0)
    for _ in range(200):
        n, kappa = int(rng.integers(1, 8)), int(rng.integers(1, 4))
        deg = [int(x) for x in rng.integers(0, 12, size=n)]
        part, loads = opart.partition_rows(deg, kappa)
        assert sum(loads) == sum(deg)
        assert all(loads[z] == sum(d for v, d in enumerate(deg) if part[v] == z) for z in range(kappa))
        opt = opart.optimal_makespan(deg, kappa)
        assert max(loads) * 3 * kappa <= opt * (4 * kappa - 1)


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,nnz,kappa", [(1, 120_011, 148), (2, 90_007, 82), (3, 80_021, 148), (4, 60_013, 5)])
def test_gpu_partition_matches_the_twin(cfg, nnz, kappa):
    import paper_2405_08470_b200 as P
    P.load_library()
    base = W.CONFIGS[cfg]
    spec = base.scaled(nnz, dims=[max(2, d // 25) for d in base.dims])     # small modes keep the pure-Python twin fast
    t = W.generate_tensor(spec)
    dev = torch.device("cuda:0")
    h = P.Mttkrp(spec.dims, t.idx.to(dev), t.vals.to(dev))
    fac = [torch.zeros((d, 8), device=dev) for d in spec.dims]
    h.mttkrp_mode(1, fac)                                        # degrees must not depend on the resident layout
    for d in range(len(spec.dims)):
        deg = np.bincount(t.idx[d].numpy(), minlength=spec.dims[d])
        part, loads = h.partition_rows(d, kappa)
        want_part, want_loads = opart.partition_rows([int(x) for x in deg], kappa)
        np.testing.assert_array_equal(loads, np.array(want_loads))
        np.testing.assert_array_equal(part, np.array(want_part, dtype=np.int32))
        assert loads.sum() == nnz                               # every nonzero in exactly one partition (Observation 2)
    h.destroy()


def _alg1_perm(dims, idx_np, order, kappa):
    """Expected layout of mode d = order[0] under the Alg. 1 policy: stable sort by (partition of the output row,
    then the layout's key tuple), the partition from the plain-Python twin (hyperedges ordered by
    partition id)."""
    d = order[0]
    deg = np.bincount(idx_np[d], minlength=dims[d])
    part, loads = opart.partition_rows([int(x) for x in deg], kappa)
    part = np.asarray(part, dtype=np.int64)
    keys = tuple(idx_np[m] for m in reversed(list(order))) + (part[idx_np[d]],)      # lexsort: last key is primary
    return np.lexsort(keys).astype(np.int64), loads


@pytest.mark.gpu
@pytest.mark.parametrize("case", [("tiny3", (7, 5, 6), 60, 3, 8), ("tiny5", (3, 4, 5, 3, 2), 120, 4, 16),
                                  ("cfg1", 1, 150_011, 5, 32), ("cfg2", 2, 120_007, 148, 32), ("cfg3", 3, 90_013, 37, 32),
                                  ("cfg4", 4, 60_017, 148, 16), ("more-bins-than-rows", (6, 40, 9), 900, 16, 8)])
def test_alg1_shard_policy_is_executable(monkeypatch, case):
    # the paper's Alg. 1 as a shard policy.  MTTKRP_SHARD_POLICY=alg1 orders every layout by
    # (partition of the output row, key tuple), one thread block walks one partition, rows never span blocks
    # (Observation 2): the permutation equals the twin's, the remapped copy is that order, every
    # entry of every Y_d matches the oracle, and no row goes through the carry / fix-up path.
    import oracle
    import paper_2405_08470_b200 as P
    P.load_library()
    name, shape, nnz, kappa, R = case
    if isinstance(shape, int):
        base = W.CONFIGS[shape]
        spec = base.scaled(nnz, dims=[max(2, dd // 25) for dd in base.dims])
        t = W.generate_tensor(spec)
        dims = list(spec.dims)
    else:
        dims = list(shape)
        t = W.tiny_tensor(dims, nnz, seed=nnz, duplicates=True)
    monkeypatch.setenv("MTTKRP_SHARD_POLICY", "alg1")
    monkeypatch.setenv("MTTKRP_KAPPA", str(kappa))
    dev = torch.device("cuda:0")
    N = len(dims)
    h = P.Mttkrp(dims, t.idx.to(dev), t.vals.to(dev))
    info = h.info()
    assert info["shard_policy"] == "alg1" and info["kappa"] == kappa and info["num_split_rows"] == [0] * N
    idx_np, vals_np = t.idx.numpy(), t.vals.numpy()
    rng = np.random.default_rng(7)
    fac_np = [rng.uniform(-1, 1, size=(dd, R)).astype(np.float32) for dd in dims]
    fac = [torch.from_numpy(f).to(dev) for f in fac_np]
    for d in list(range(N)) + [0]:
        perm, loads = _alg1_perm(dims, idx_np, info["key_order"][d], kappa)
        assert info["max_partition_nnz"][d] == max(loads) and info["min_partition_nnz"][d] == min(loads)
        np.testing.assert_array_equal(h.get_perm(d).cpu().numpy().astype(np.int64), perm)
        out = torch.full((dims[d], R), float("nan"), dtype=torch.float32, device=dev)
        Y = h.mttkrp_mode(d, fac, out=out).cpu().numpy()
        gi, gv = h.export_coo()
        np.testing.assert_array_equal(gi.cpu().numpy(), idx_np[:, perm])
        np.testing.assert_array_equal(gv.cpu().numpy(), vals_np[perm])
        Yo, So = oracle.mttkrp_mode(dims, idx_np, vals_np, fac_np, d, perm=perm)
        err, zeros_ok = oracle.normalised_error(Y, Yo, So)
        assert zeros_ok and err <= 1e-5, f"{name} mode {d}: normalised error {err:.3e}"
    h.destroy()
