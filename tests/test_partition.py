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
