"""fp64 CPU twin of paper_2405_08470_b200/cpd.py.  TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Textbook CPD-ALS (the paper names it, and gives no further detail) on top of the oracle's
MTTKRP: for d = 0..N-1: M = MTTKRP_d; G = Hadamard_{m != d} A_m^T A_m; A_d = M G^{-1}; normalise columns.
fit = 1 - ||X - X^|| / ||X|| with <X, X^> = sum_r lam_r sum_i M[i,r] A_d[i,r], ||X^||^2 = lam^T (Hadamard_m
A_m^T A_m) lam.  Pinned in tests/test_cpd.py: an exactly rank-R tensor is recovered (fit -> 1), the fit
never decreases, and the fit formula equals the explicit dense residual.
"""
from __future__ import annotations

import numpy as np

from . import mttkrp_mode


def cpd_als(dims, idx, vals, R, iters, init):
    N = len(dims)
    A = [np.array(a, dtype=np.float64) for a in init]
    norm_x = float(np.sqrt(np.sum(vals.astype(np.float64) ** 2)))      # distinct coordinates assumed
    lam = np.ones(R)
    fits = []
    for _ in range(iters):
        M = None
        for d in range(N):
            M, _ = mttkrp_mode(dims, idx, vals, [a.astype(np.float32) for a in A], d)
            G = np.ones((R, R))
            for m in range(N):
                if m != d:
                    G = G * (A[m].T @ A[m])
            Ad = np.linalg.solve(G + 1e-12 * np.eye(R), M.T).T
            lam = np.linalg.norm(Ad, axis=0)
            lam = np.where(lam > 0, lam, 1.0)
            A[d] = (Ad / lam).astype(np.float32).astype(np.float64)     # factors are handed on in fp32, as on the GPU
        d = N - 1
        inner = float(np.sum(lam * np.sum(M * A[d], axis=0)))
        G = np.ones((R, R))
        for m in range(N):
            G = G * (A[m].T @ A[m])
        resid2 = max(norm_x ** 2 - 2.0 * inner + float(lam @ G @ lam), 0.0)
        fits.append(1.0 - np.sqrt(resid2) / norm_x)
    return A, lam, fits
