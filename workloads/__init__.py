"""Seeded synthetic sparse-tensor workloads (inputs only; none of the method's arithmetic).

This module serves both the CPU oracle (`oracle/`) and the CUDA path
(`paper_2405_08470_b200/`); it imports neither.  It stands in for the paper's public
tensors (Table 3), which are not available offline: BASELINE.json's five
configs keep their shape class (3-5 modes, Zipf-skewed and uniform modes, tiny and huge
modes side by side).

Everything random is drawn from a counter-based generator (splitmix64 over
`(stream seed, element counter)`), written with wrapping int64 torch ops, so the same call
yields bit-identical tensors on CPU and on CUDA.  The large configs are generated on the
GPU in seconds; the small ones on the CPU in the `-m "not gpu"` tests.

Recipe:
 1. Zipf(s) on a mode of size I is the truncated law P(rank j) ~ j^-s, j = 1..I (float64
    CDF built on the host with numpy, inverted with `searchsorted`), and the drawn rank is
    mapped through a seeded random permutation of [0, I).  s = 0 means uniform integers.
 2. Index tuples are linearised to a 64-bit mixed-radix key (wrapping arithmetic; the key
    space of every config is < 2^64 so the map is injective), de-duplicated with `unique`,
    topped up until at least `nnz` distinct cells exist.
 3. The distinct cells are ordered by a bijective 64-bit hash of their key and the first
    `nnz` are kept: a seeded random subset in a seeded random (unsorted) order.
 4. Values: fp32 uniform[0,1) (24 random bits) or lognormal(0,1); factors fp32
    uniform(-1,1), I_m x R row-major.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence

import numpy as np
import torch

BASE_SEED = 24050847  # arXiv id 2405.08470 with the dot dropped

_M64 = (1 << 64) - 1


def _i64(x: int) -> int:
    """Two's-complement int64 view of an unsigned 64-bit constant."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLDEN = _i64(0x9E3779B97F4A7C15)
_MUL1 = _i64(0xBF58476D1CE4E5B9)
_MUL2 = _i64(0x94D049BB133111EB)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right on int64 (torch's >> is arithmetic)."""
    return (x >> s) & ((1 << (64 - s)) - 1)


def splitmix64(x: torch.Tensor) -> torch.Tensor:
    """Bijective 64-bit mix (the splitmix64 finaliser) on wrapping int64."""
    z = x + _GOLDEN
    z = (z ^ _lsr(z, 30)) * _MUL1
    z = (z ^ _lsr(z, 27)) * _MUL2
    return z ^ _lsr(z, 31)


def splitmix64_py(x: int) -> int:
    """Pure-Python big-int twin of `splitmix64`, used by the tests to pin the torch version."""
    z = (x + 0x9E3779B97F4A7C15) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def stream_seed(*words: int) -> int:
    """Derive a 64-bit stream seed from integer words (config id, tag, ...)."""
    s = BASE_SEED
    for w in words:
        s = splitmix64_py((s ^ (w & _M64)) & _M64)
    return _i64(s)


def random_bits(seed: int, start: int, n: int, device) -> torch.Tensor:
    """n pseudo-random int64 words: splitmix64(seed + GOLDEN*(start + i))."""
    ctr = torch.arange(start, start + n, dtype=torch.int64, device=device)
    return splitmix64(ctr * _GOLDEN + seed)


def uniform01_f64(seed: int, start: int, n: int, device) -> torch.Tensor:
    """float64 uniform on [0,1) with 53 random bits (exact on any device)."""
    return _lsr(random_bits(seed, start, n, device), 11).to(torch.float64) * (2.0 ** -53)


def uniform01_f32(seed: int, start: int, n: int, device) -> torch.Tensor:
    """float32 uniform on [0,1) with 24 random bits (exact on any device)."""
    return (_lsr(random_bits(seed, start, n, device), 40).to(torch.float32)) * (2.0 ** -24)


def udivmod(x: torch.Tensor, m: int):
    """Unsigned 64-bit divmod of a two's-complement int64 tensor by a positive int m < 2^62."""
    q1 = torch.div(x, m, rounding_mode="floor")
    r1 = x - q1 * m  # in [0, m)
    if m < 4:        # 2^64 // m would not fit int64; only needed when the key space is >= 2^63
        if bool((x < 0).any()):
            raise ValueError("udivmod: wrapped key with a modulus < 4")
        return q1, r1
    q2, r2 = divmod(1 << 64, m)
    neg = (x < 0).to(torch.int64)
    r = r1 + neg * r2
    carry = (r >= m).to(torch.int64)
    r = r - carry * m
    q = q1 + neg * q2 + carry
    return q, r


def zipf_cdf(size: int, s: float) -> np.ndarray:
    """float64 CDF of the truncated Zipf law P(j) ~ j^-s, j = 1..size (host, numpy)."""
    w = np.arange(1, size + 1, dtype=np.float64) ** (-float(s))
    c = np.cumsum(w)
    c /= c[-1]
    c[-1] = 1.0
    return c


def seeded_permutation(size: int, seed: int) -> np.ndarray:
    """Random permutation of [0,size): stable argsort of hashed counters (host, numpy)."""
    h = random_bits(seed, 0, size, "cpu").numpy()
    return np.argsort(h, kind="stable").astype(np.int64)


@dataclass
class TensorSpec:
    name: str
    dims: Sequence[int]
    nnz: int
    zipf_s: Sequence[float]          # per mode; 0.0 = uniform
    values: str = "uniform"          # "uniform" | "lognormal"
    ranks: Sequence[int] = (32,)
    config_id: int = 0

    def scaled(self, nnz: int, dims: Optional[Sequence[int]] = None, name: Optional[str] = None) -> "TensorSpec":
        """Same shape class at a smaller size (for tests)."""
        return TensorSpec(name or f"{self.name}-scaled", list(dims or self.dims), int(nnz), list(self.zipf_s),
                          self.values, tuple(self.ranks), self.config_id)


# BASELINE.json "configs" (0-based here; SURVEY.md numbers them 1..5).
CONFIGS: List[TensorSpec] = [
    TensorSpec("cfg1-3mode-uniform-100k", [1000, 800, 600], 100_000, [0.0, 0.0, 0.0], "uniform", (16,), 1),
    TensorSpec("cfg2-3mode-zipf1.1-77M", [12_000, 9_000, 29_000], 77_000_000, [1.1, 1.1, 1.1], "uniform", (32,), 2),
    TensorSpec("cfg3-3mode-skewed-200M", [4_800_000, 1_800_000, 1_800_000], 200_000_000, [1.3, 1.05, 1.05],
               "uniform", (32,), 3),
    TensorSpec("cfg4-4mode-zipf1.1-100M", [200_000, 50_000, 200_000, 1_000], 100_000_000, [1.1, 1.1, 1.1, 1.1],
               "lognormal", (32,), 4),
    TensorSpec("cfg5-5mode-60M", [2_000, 3_000, 1_000_000, 5_000, 24], 60_000_000, [0.0, 0.0, 1.2, 0.0, 0.0],
               "uniform", (8, 16, 32, 64), 5),
]


@dataclass
class SparseTensor:
    spec: TensorSpec
    idx: torch.Tensor     # int32 [N, nnz] (SoA), 0-based, distinct tuples, unsorted
    vals: torch.Tensor    # float32 [nnz]
    draws: int = 0        # tuples drawn before de-duplication
    checksums: dict = field(default_factory=dict)

    @property
    def nnz(self) -> int:
        return int(self.vals.numel())

    @property
    def dims(self) -> List[int]:
        return list(self.spec.dims)


def _draw_mode(spec: TensorSpec, m: int, start: int, n: int, device, cache: dict) -> torch.Tensor:
    size = int(spec.dims[m])
    s = float(spec.zipf_s[m])
    u = uniform01_f64(stream_seed(spec.config_id, 100 + m), start, n, device)
    if s == 0.0:
        return torch.clamp((u * size).to(torch.int64), max=size - 1)
    if m not in cache:
        cdf = torch.from_numpy(zipf_cdf(size, s)).to(device)
        perm = torch.from_numpy(seeded_permutation(size, stream_seed(spec.config_id, 200 + m))).to(device)
        cache[m] = (cdf, perm)
    cdf, perm = cache[m]
    j = torch.searchsorted(cdf, u, right=True).clamp_(max=size - 1)
    return perm[j]


def _linear_key(cols: Sequence[torch.Tensor], dims: Sequence[int]) -> torch.Tensor:
    key = cols[0].clone()
    for m in range(1, len(dims)):
        key = key * int(dims[m]) + cols[m]
    return key


def generate_tensor(spec: TensorSpec, device="cpu", batch: Optional[int] = None) -> SparseTensor:
    """Build the de-duplicated, shuffled COO tensor for `spec` on `device`."""
    N = len(spec.dims)
    cells = 1
    for d in spec.dims:
        cells *= int(d)
    if cells >= (1 << 64):
        raise ValueError("key space must fit 64 bits")
    if spec.nnz > cells:
        raise ValueError("more nonzeros than cells")
    device = torch.device(device)
    cache: dict = {}
    target = int(spec.nnz)
    batch = int(batch or max(1024, target // 2))
    uniq = torch.empty(0, dtype=torch.int64, device=device)
    drawn = 0
    while uniq.numel() < target:
        cols = [_draw_mode(spec, m, drawn, batch, device, cache) for m in range(N)]
        key = _linear_key(cols, spec.dims)
        del cols
        uniq = torch.unique(torch.cat([uniq, key]))
        del key
        drawn += batch
    # Seeded random subset in seeded random order: sort by a bijective hash of the key.
    h = splitmix64(uniq ^ stream_seed(spec.config_id, 300))
    order = torch.argsort(h)[:target]
    del h
    key = uniq[order]
    del uniq, order
    idx = torch.empty((N, target), dtype=torch.int32, device=device)
    rest = key
    for m in range(N - 1, 0, -1):
        rest, r = udivmod(rest, int(spec.dims[m]))
        idx[m] = r.to(torch.int32)
    idx[0] = rest.to(torch.int32)
    del rest, key
    if spec.values == "uniform":
        vals = uniform01_f32(stream_seed(spec.config_id, 400), 0, target, device)
    elif spec.values == "lognormal":
        u1 = uniform01_f64(stream_seed(spec.config_id, 401), 0, target, device)
        u2 = uniform01_f64(stream_seed(spec.config_id, 402), 0, target, device)
        z = torch.sqrt(-2.0 * torch.log1p(-u1)) * torch.cos(2.0 * np.pi * u2)
        vals = torch.exp(z).to(torch.float32)
    else:
        raise ValueError(spec.values)
    t = SparseTensor(spec, idx, vals, drawn)
    t.checksums = {
        "idx_sum": [int(idx[m].to(torch.int64).sum().item()) for m in range(N)],
        "vals_sum_f64": float(vals.to(torch.float64).sum().item()),
    }
    return t


def generate_factors(spec: TensorSpec, R: int, device="cpu") -> List[torch.Tensor]:
    """Factor matrices A_m: float32 [I_m, R] row-major, uniform(-1,1) (23-bit grid)."""
    out = []
    for m, size in enumerate(spec.dims):
        n = int(size) * int(R)
        u = uniform01_f32(stream_seed(spec.config_id, 500 + m, R), 0, n, device)
        out.append((u * 2.0 - 1.0).reshape(int(size), int(R)).contiguous())
    return out


def tiny_tensor(dims: Sequence[int], nnz: int, seed: int, duplicates: bool = False, device="cpu") -> SparseTensor:
    """Small uniform tensor for brute-force tests; with `duplicates` some coordinates repeat."""
    spec = TensorSpec(f"tiny-{seed}", list(dims), int(nnz), [0.0] * len(dims), "uniform", (4,), 1000 + seed)
    if not duplicates:
        return generate_tensor(spec, device)
    N = len(dims)
    cols = [_draw_mode(spec, m, 0, nnz, device, {}) for m in range(N)]
    idx = torch.stack(cols).to(torch.int32)
    # force at least one repeated coordinate
    if nnz >= 2:
        idx[:, -1] = idx[:, 0]
    vals = uniform01_f32(stream_seed(spec.config_id, 400), 0, nnz, device)
    return SparseTensor(spec, idx, vals, nnz)


def distinct_per_mode(t: SparseTensor) -> List[int]:
    """U_m = number of distinct indices present in mode m (for the compulsory-byte model)."""
    return [int(torch.unique(t.idx[m]).numel()) for m in range(len(t.spec.dims))]
