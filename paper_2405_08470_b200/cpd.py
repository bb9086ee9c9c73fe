"""CPD-ALS driver around the MTTKRP path.

The paper motivates spMTTKRP as the bottleneck of CP decomposition by alternating least squares
(Sec. 2.1.4: "ALS iterates Eq. 1 over the modes") and gives no detail beyond the
name; this is the textbook iteration.  Per sweep, for d = 0..N-1 (the cyclic order of Alg. 5,
PAPER.md:305-330, so every call costs exactly one remap):

    M   = MTTKRP_d(X; A_0..A_{N-1})            library: remap into layout d + k_mttkrp  (the hot path)
    G   = Hadamard_{m != d} (A_m^T A_m)        R x R, torch
    A_d = M G^+                                R x R solve, torch
    lam = column norms of A_d;  A_d /= lam     torch

and after the last mode  fit = 1 - ||X - X^|| / ||X||  from  <X, X^> = sum_r lam_r sum_i M[i,r] A_d[i,r]
and ||X^||^2 = lam^T (Hadamard_m A_m^T A_m) lam.  Everything of size nnz or I_d x R on the MTTKRP side runs
in the library's kernels; torch is used for the R x R algebra and the I_d x R Gram products (cuBLAS GEMMs).
"""
from __future__ import annotations

from typing import List, Optional, Sequence, Tuple

import torch

from .binding import Mttkrp


def cpd_als(h: Mttkrp, dims: Sequence[int], R: int, iters: int, init: Sequence[torch.Tensor],
            norm_x: float) -> Tuple[List[torch.Tensor], torch.Tensor, List[float]]:
    """Run `iters` ALS sweeps from the factor matrices `init` (fp32 CUDA, I_m x R).  `norm_x` = ||X||_F.
    Returns (unit-column factors, lam, fit after every sweep)."""
    N = len(dims)
    A = [a.clone().contiguous() for a in init]
    dev = A[0].device
    grams = [a.double().T @ a.double() for a in A]
    lam = torch.ones(R, dtype=torch.float64, device=dev)
    outs = [torch.empty((int(d), R), dtype=torch.float32, device=dev) for d in dims]
    fits: List[float] = []
    for _ in range(iters):
        M = None
        for d in range(N):
            M = h.mttkrp_mode(d, A, out=outs[d])
            G = torch.ones((R, R), dtype=torch.float64, device=dev)
            for m in range(N):
                if m != d:
                    G = G * grams[m]
            Ad = torch.linalg.solve(G + 1e-12 * torch.eye(R, dtype=torch.float64, device=dev), M.double().T).T
            lam = torch.linalg.norm(Ad, dim=0)
            lam = torch.where(lam > 0, lam, torch.ones_like(lam))
            Ad = Ad / lam
            A[d] = Ad.float().contiguous()
            grams[d] = A[d].double().T @ A[d].double()
        # fit from the last mode's MTTKRP (computed with the other factors already updated)
        d = N - 1
        inner = float((lam * (M.double() * A[d].double()).sum(dim=0)).sum().item())
        G = torch.ones((R, R), dtype=torch.float64, device=dev)
        for m in range(N):
            G = G * grams[m]
        norm_hat2 = float((lam @ G @ lam).item())
        resid2 = max(norm_x * norm_x - 2.0 * inner + norm_hat2, 0.0)
        fits.append(1.0 - (resid2 ** 0.5) / norm_x)
    return A, lam, fits
