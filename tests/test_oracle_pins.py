"""Pins for the fp64 oracle (CPU only).  Each test checks oracle/ against something other
than itself: the mathematics (brute force on the dense unfolding, closed forms, invariants)
or a library routine (scipy.sparse, np.bincount, np.lexsort)."""
import itertools

import numpy as np
import pytest
import scipy.sparse as sp

import oracle
import workloads as W

TINY_SHAPES = [((4, 3, 5), 30), ((3, 4, 2, 3), 40), ((2, 3, 2, 2, 3), 50), ((5, 4), 12)]


def _np(t):
    return t.idx.numpy(), t.vals.numpy()


def _factors(dims, R, seed, ones=False):
    rng = np.random.default_rng(seed)
    if ones:
        return [np.ones((d, R), dtype=np.float32) for d in dims]
    return [rng.uniform(-1, 1, size=(d, R)).astype(np.float32) for d in dims]


def brute_force(dims, idx, vals, factors, d):
    """Eq. 1 literally: densify X, unfold along d, form the Khatri-Rao
    product of the other factors explicitly, multiply.  numpy C order: the remaining modes in
    increasing order, last fastest (reading 1)."""
    X = np.zeros(dims, dtype=np.float64)
    np.add.at(X, tuple(idx[m] for m in range(len(dims))), vals.astype(np.float64))
    Xd = np.moveaxis(X, d, 0).reshape(dims[d], -1)
    R = factors[0].shape[1]
    kr = None
    for m in range(len(dims)):
        if m == d:
            continue
        A = factors[m].astype(np.float64)
        kr = A if kr is None else (kr[:, None, :] * A[None, :, :]).reshape(-1, R)
    return Xd @ kr


def test_hand_worked_example():
    # tests/golden/hand_worked_3mode.txt: PAPER.md:121 worked by hand for three nonzeros (exact in fp64).
    from conftest import load_golden
    dims, idx, vals, factors, want = load_golden("hand_worked_3mode.txt")
    for d in range(3):
        Y, S = oracle.mttkrp_mode(dims, idx, vals, factors, d)
        np.testing.assert_array_equal(Y, want[d])
        assert np.all(S >= np.abs(Y))
        Yn, _ = oracle.mttkrp_numpy(dims, idx, vals, factors, d)
        np.testing.assert_array_equal(Yn, want[d])


@pytest.mark.parametrize("dims,nnz", TINY_SHAPES)
@pytest.mark.parametrize("dup", [False, True])
def test_brute_force_dense_unfold_khatri_rao(dims, nnz, dup):
    t = W.tiny_tensor(dims, nnz, seed=len(dims) * 10 + int(dup), duplicates=dup)
    idx, vals = _np(t)
    fac = _factors(dims, 3, seed=7)
    for d in range(len(dims)):
        want = brute_force(dims, idx, vals, fac, d)
        Y, S = oracle.mttkrp_mode(dims, idx, vals, fac, d)
        np.testing.assert_allclose(Y, want, rtol=1e-12, atol=1e-13)
        Yn, Sn = oracle.mttkrp_numpy(dims, idx, vals, fac, d)
        np.testing.assert_allclose(Yn, want, rtol=1e-12, atol=1e-13)
        np.testing.assert_allclose(S, Sn, rtol=1e-12)
        # the normaliser is the same sum with absolute values: brute force on |.|
        Sw = brute_force(dims, idx, np.abs(vals), [np.abs(f) for f in fac], d)
        np.testing.assert_allclose(S, Sw, rtol=1e-12, atol=1e-13)
        assert np.all(S + 1e-15 >= np.abs(Y))


@pytest.mark.parametrize("dims", [(4, 3, 5), (3, 2, 4, 2), (2, 3, 2, 2, 3)])
def test_all_ones_closed_form(dims):
    # north_star: all-ones dense tensor, all-ones factors => Y_d[i,r] = prod of the other dims (exact).
    grid = np.array(list(itertools.product(*[range(d) for d in dims])), dtype=np.int32).T
    vals = np.ones(grid.shape[1], dtype=np.float32)
    fac = _factors(dims, 4, 0, ones=True)
    for d in range(len(dims)):
        Y, S = oracle.mttkrp_mode(dims, grid, vals, fac, d)
        want = float(np.prod(dims)) / dims[d]
        assert np.all(Y == want)
        assert np.all(S == want)


@pytest.mark.parametrize("dims,nnz", TINY_SHAPES + [((40, 30, 20), 2000)])
def test_cross_mode_invariant(dims, nnz):
    # sum_i sum_r Y_d[i,r] A_d[i,r] = sum_k val_k sum_r prod_m A_m[i_m(k), r], the same for every d.
    t = W.tiny_tensor(dims, nnz, seed=3)
    idx, vals = _np(t)
    fac = _factors(dims, 5, seed=11)
    direct = 0.0
    for k in range(idx.shape[1]):
        term = np.full(5, float(vals[k]))
        for m in range(len(dims)):
            term = term * fac[m][idx[m, k]].astype(np.float64)
        direct += term.sum()
    for d in range(len(dims)):
        Y, _ = oracle.mttkrp_mode(dims, idx, vals, fac, d)
        inner = float((Y * fac[d].astype(np.float64)).sum())
        assert abs(inner - direct) <= 1e-10 * max(1.0, abs(direct))


def test_two_modes_is_spmm():
    # N = 2: Y_0 = X A_1 and Y_1 = X^T A_0 (library special case, scipy.sparse in fp64).
    dims = (50, 40)
    t = W.tiny_tensor(dims, 600, seed=5)
    idx, vals = _np(t)
    fac = _factors(dims, 6, seed=2)
    X = sp.coo_matrix((vals.astype(np.float64), (idx[0], idx[1])), shape=dims).tocsr()
    Y0, _ = oracle.mttkrp_mode(dims, idx, vals, fac, 0)
    Y1, _ = oracle.mttkrp_mode(dims, idx, vals, fac, 1)
    np.testing.assert_allclose(Y0, X @ fac[1].astype(np.float64), rtol=1e-12, atol=1e-13)
    np.testing.assert_allclose(Y1, X.T @ fac[0].astype(np.float64), rtol=1e-12, atol=1e-13)


def test_rank_one_ones_is_bincount():
    # R = 1 with all-ones factors: Y_d[i] = sum of the values in slice i (np.bincount).
    dims = (30, 20, 10)
    t = W.tiny_tensor(dims, 900, seed=9)
    idx, vals = _np(t)
    fac = _factors(dims, 1, 0, ones=True)
    for d in range(3):
        Y, _ = oracle.mttkrp_mode(dims, idx, vals, fac, d)
        want = np.bincount(idx[d], weights=vals.astype(np.float64), minlength=dims[d])
        np.testing.assert_allclose(Y[:, 0], want, rtol=1e-13, atol=1e-14)


def test_linearity_permutation_and_duplicate_splitting():
    dims = (12, 9, 7, 5)
    t = W.tiny_tensor(dims, 500, seed=4)
    idx, vals = _np(t)
    fac = _factors(dims, 4, seed=1)
    fac2 = _factors(dims, 4, seed=2)
    rng = np.random.default_rng(0)
    for d in range(4):
        Y, S = oracle.mttkrp_mode(dims, idx, vals, fac, d)
        # linear in val (2.5 * v is exact in fp32 only sometimes, so scale by a power of two)
        Y2, _ = oracle.mttkrp_mode(dims, idx, vals * np.float32(4.0), fac, d)
        np.testing.assert_allclose(Y2, 4.0 * Y, rtol=1e-14)
        # linear in one factor: A_m -> A_m + B_m, for m != d
        m = (d + 1) % 4
        mix = list(fac)
        mix[m] = fac2[m]
        Yb, _ = oracle.mttkrp_mode(dims, idx, vals, mix, d)
        both = list(fac)
        both[m] = (fac[m].astype(np.float64) + fac2[m].astype(np.float64))
        # the sum is not fp32-exact in general; feed it through the numpy twin in fp64 instead
        l = vals.astype(np.float64)[:, None] * np.ones((1, 4))
        for w in range(4):
            if w != d:
                l = l * (both[w] if w == m else fac[w].astype(np.float64))[idx[w]]
        want = np.zeros_like(Y)
        np.add.at(want, idx[d], l)
        np.testing.assert_allclose(Y + Yb, want, rtol=1e-11, atol=1e-12)
        # invariant under a permutation of the COO order (to fp64 rounding)
        p = rng.permutation(idx.shape[1])
        Yp, Sp = oracle.mttkrp_mode(dims, idx[:, p], vals[p], fac, d)
        np.testing.assert_allclose(Yp, Y, rtol=1e-11, atol=1e-13)
        np.testing.assert_allclose(Sp, S, rtol=1e-12)
        # A_d is not read
        junk = list(fac)
        junk[d] = np.full_like(fac[d], np.nan)
        Yj, _ = oracle.mttkrp_mode(dims, idx, vals, junk, d)
        np.testing.assert_array_equal(Yj, Y)
        # splitting a nonzero into two duplicates with halved values changes nothing (halving is exact)
        idx_s = np.concatenate([idx, idx[:, :50]], axis=1)
        vals_s = np.concatenate([vals, vals[:50] * np.float32(0.5)])
        vals_s[:50] = vals[:50] * np.float32(0.5)
        Ys, _ = oracle.mttkrp_mode(dims, idx_s, vals_s, fac, d)
        np.testing.assert_allclose(Ys, Y, rtol=1e-11, atol=1e-13)


def test_visit_order_and_row_variant_agree():
    dims = (64, 48, 32)
    t = W.tiny_tensor(dims, 5000, seed=6)
    idx, vals = _np(t)
    fac = _factors(dims, 8, seed=3)
    for d in range(3):
        order = [d] + [m for m in range(3) if m != d]
        perm = oracle.sort_perm(dims, idx, order)
        Y1, S1 = oracle.mttkrp_mode(dims, idx, vals, fac, d, perm=perm)
        Yr, Sr = oracle.mttkrp_mode(dims, idx, vals, fac, d, perm=perm, threads=4)
        np.testing.assert_array_equal(Y1, Yr)      # bit-identical for any thread count
        np.testing.assert_array_equal(S1, Sr)
        Y0, _ = oracle.mttkrp_mode(dims, idx, vals, fac, d)
        np.testing.assert_allclose(Y1, Y0, rtol=1e-11, atol=1e-13)
        rows = np.array([0, 5, dims[d] - 1, 17], dtype=np.int64)
        Ys, Ss = oracle.mttkrp_rows(dims, idx, vals, fac, d, rows, perm=perm)
        np.testing.assert_array_equal(Ys, Y1[rows])
        np.testing.assert_array_equal(Ss, S1[rows])


@pytest.mark.parametrize("dup", [False, True])
def test_sort_perm_is_stable_lexsort(dup):
    dims = (9, 7, 5, 3)
    t = W.tiny_tensor(dims, 800, seed=8, duplicates=dup) if dup else W.tiny_tensor(dims, 800, seed=8)
    idx, _ = _np(t)
    if dup:
        idx = np.concatenate([idx, idx[:, ::3]], axis=1)    # plenty of equal tuples
    nnz = idx.shape[1]
    for order in [(0,), (2,), (1, 0, 2, 3), (3, 2, 1, 0), (2, 0, 1, 3)]:
        perm = oracle.sort_perm(dims, idx, order)
        # bijection (Observation 1)
        assert np.array_equal(np.sort(perm), np.arange(nnz))
        # library routine: np.lexsort is stable, so ties keep the COO order
        assert np.array_equal(perm, oracle.sort_perm_numpy(idx, order))
        # keys non-decreasing, ties in original order
        keys = np.stack([idx[m][perm] for m in order], axis=1)
        for a, b, pa, pb in zip(keys[:-1], keys[1:], perm[:-1], perm[1:]):
            ta, tb = tuple(a), tuple(b)
            assert ta < tb or (ta == tb and pa < pb)
    # single key == np.argsort(kind="stable")
    assert np.array_equal(oracle.sort_perm(dims, idx, (1,)), np.argsort(idx[1], kind="stable"))


def test_empty_and_bad_inputs():
    dims = (4, 3, 2)
    idx = np.zeros((3, 0), dtype=np.int32)
    vals = np.zeros(0, dtype=np.float32)
    fac = _factors(dims, 2, 0)
    Y, S = oracle.mttkrp_mode(dims, idx, vals, fac, 1)
    assert Y.shape == (3, 2) and not Y.any() and not S.any()
    assert oracle.sort_perm(dims, idx, (0, 1, 2)).shape == (0,)
    bad = np.array([[0], [3], [0]], dtype=np.int32)
    with pytest.raises(RuntimeError):
        oracle.sort_perm(dims, bad, (1,))


def test_normalised_error_helper():
    Yref = np.array([[1.0, 0.0], [2.0, -4.0]])
    S = np.array([[2.0, 0.0], [2.0, 8.0]])
    err, zeros_ok = oracle.normalised_error(Yref + np.array([[2e-6, 0], [0, 8e-6]]), Yref, S)
    assert abs(err - 1e-6) < 1e-12 and zeros_ok
    err, zeros_ok = oracle.normalised_error(Yref + np.array([[0, 1e-30], [0, 0]]), Yref, S)
    assert not zeros_ok
