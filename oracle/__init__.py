"""fp64 CPU oracle for all-mode sparse MTTKRP.  TEST INFRASTRUCTURE ONLY.

Only `tests/`, `__graft_entry__.smoke()` and `bench.py`'s `cpu_baseline` / `--impl reference`
legs may import this package.  It shares no code with `paper_2405_08470_b200/` and never
imports it; the product path never imports this package and has no CPU fallback.

Two implementations of the same definition (PAPER.md:121 elementwise form; Eq. 1,
PAPER.md:100; Alg. 2):

* `mttkrp_oracle.c` - plain C, one nonzero at a time in the mode-d order, double
  accumulation.  Used at every size (built on demand with gcc into `oracle/_build/`).
* `mttkrp_numpy` / `sort_perm_numpy` - a numpy twin for small cases (np.add.at + np.lexsort),
  used to cross-check the C code in the pins.

What is returned for mode d:
  Y_d[i,r] = sum_k val_k * prod_{m != d} A_m[i_m(k), r]                (fp64)
  S_d[i,r] = sum_k |val_k| * prod_{m != d} |A_m[i_m(k), r]|            (fp64, error normaliser)
  perm_d   = stable sort of the COO list by the key tuple the handle documents
             (reading 4), ties keeping the original COO order.

Parity status: every function here is pinned by tests/test_oracle_pins.py (brute force by
densify + unfold + explicit Khatri-Rao, all-ones closed form, cross-mode invariant, scipy
SpMM for N=2, bincount for R=1, algebraic properties, np.lexsort).  Nothing is unpinned.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from typing import List, Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mttkrp_oracle.c")
_BUILD = os.path.join(_HERE, "_build")
_LIBPATH = os.path.join(_BUILD, "liboracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle with gcc (-O2 -fopenmp).  Building the checker is not using it."""
    os.makedirs(_BUILD, exist_ok=True)
    if force or not os.path.exists(_LIBPATH) or os.path.getmtime(_LIBPATH) < os.path.getmtime(_SRC):
        tmp = _LIBPATH + f".{os.getpid()}.tmp"
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"])
        os.replace(tmp, _LIBPATH)
    return _LIBPATH


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        i64p = ctypes.POINTER(ctypes.c_int64)
        i32p = ctypes.POINTER(ctypes.c_int32)
        f32p = ctypes.POINTER(ctypes.c_float)
        f64p = ctypes.POINTER(ctypes.c_double)
        fpp = ctypes.POINTER(f32p)
        lib.oracle_sort_perm.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, i32p, ctypes.c_int, i32p, i64p]
        lib.oracle_sort_perm.restype = ctypes.c_int
        lib.oracle_mttkrp_mode.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, i32p, f32p, fpp, ctypes.c_int,
                                           ctypes.c_int, i64p, f64p, f64p]
        lib.oracle_mttkrp_mode.restype = ctypes.c_int
        lib.oracle_mttkrp_mode_rows.argtypes = lib.oracle_mttkrp_mode.argtypes + [ctypes.c_int]
        lib.oracle_mttkrp_mode_rows.restype = ctypes.c_int
        lib.oracle_mttkrp_rows_subset.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, i32p, f32p, fpp, ctypes.c_int,
                                                  ctypes.c_int, i64p, ctypes.c_int64, i64p, f64p, f64p]
        lib.oracle_mttkrp_rows_subset.restype = ctypes.c_int
        lib.oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _ptr(a: Optional[np.ndarray], ctype):
    if a is None:
        return ctypes.cast(None, ctypes.POINTER(ctype))
    return a.ctypes.data_as(ctypes.POINTER(ctype))


def _prep(dims, idx, vals, factors):
    dims = np.ascontiguousarray(np.asarray(dims, dtype=np.int64))
    idx = np.ascontiguousarray(np.asarray(idx, dtype=np.int32))
    vals = np.ascontiguousarray(np.asarray(vals, dtype=np.float32))
    assert idx.ndim == 2 and idx.shape[0] == dims.shape[0] and idx.shape[1] == vals.shape[0]
    fac = None
    if factors is not None:
        fac = [np.ascontiguousarray(np.asarray(f, dtype=np.float32)) for f in factors]
        for m, f in enumerate(fac):
            assert f.ndim == 2 and f.shape[0] == dims[m]
    return dims, idx, vals, fac


def _facptrs(fac: List[np.ndarray]):
    f32p = ctypes.POINTER(ctypes.c_float)
    arr = (f32p * len(fac))()
    for m, f in enumerate(fac):
        arr[m] = f.ctypes.data_as(f32p)
    return arr


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def sort_perm(dims: Sequence[int], idx: np.ndarray, order: Sequence[int]) -> np.ndarray:
    """perm (int64[nnz]): stable sort of COO positions by (i_order[0], i_order[1], ...)."""
    dims_a = np.ascontiguousarray(np.asarray(dims, dtype=np.int64))
    idx = np.ascontiguousarray(np.asarray(idx, dtype=np.int32))
    order_a = np.ascontiguousarray(np.asarray(order, dtype=np.int32))
    nnz = idx.shape[1]
    perm = np.empty(nnz, dtype=np.int64)
    rc = _load().oracle_sort_perm(len(dims_a), _ptr(dims_a, ctypes.c_int64), nnz, _ptr(idx, ctypes.c_int32),
                                  len(order_a), _ptr(order_a, ctypes.c_int32), _ptr(perm, ctypes.c_int64))
    if rc != 0:
        raise RuntimeError("oracle_sort_perm failed (bad index or allocation)")
    return perm


def mttkrp_mode(dims, idx, vals, factors, d: int, perm: Optional[np.ndarray] = None,
                threads: int = 1) -> Tuple[np.ndarray, np.ndarray]:
    """(Y_d, S_d) in fp64.  threads > 1 uses the row-partitioned variant (needs a mode-d perm)."""
    dims, idx, vals, fac = _prep(dims, idx, vals, factors)
    R = fac[(d + 1) % len(fac)].shape[1]
    nnz = idx.shape[1]
    Y = np.empty((int(dims[d]), R), dtype=np.float64)
    S = np.empty_like(Y)
    p = None if perm is None else np.ascontiguousarray(perm, dtype=np.int64)
    lib = _load()
    if threads == 1:
        rc = lib.oracle_mttkrp_mode(len(dims), _ptr(dims, ctypes.c_int64), nnz, _ptr(idx, ctypes.c_int32),
                                    _ptr(vals, ctypes.c_float), _facptrs(fac), R, d, _ptr(p, ctypes.c_int64),
                                    _ptr(Y, ctypes.c_double), _ptr(S, ctypes.c_double))
    else:
        rc = lib.oracle_mttkrp_mode_rows(len(dims), _ptr(dims, ctypes.c_int64), nnz, _ptr(idx, ctypes.c_int32),
                                         _ptr(vals, ctypes.c_float), _facptrs(fac), R, d, _ptr(p, ctypes.c_int64),
                                         _ptr(Y, ctypes.c_double), _ptr(S, ctypes.c_double), int(threads))
        rc = 0 if rc > 0 else -1
    if rc != 0:
        raise RuntimeError("oracle_mttkrp_mode failed")
    return Y, S


def mttkrp_rows(dims, idx, vals, factors, d: int, rows: np.ndarray,
                perm: Optional[np.ndarray] = None) -> Tuple[np.ndarray, np.ndarray]:
    """(Y_d[rows,:], S_d[rows,:]) in fp64 for a sample of output rows (full-size parity)."""
    dims, idx, vals, fac = _prep(dims, idx, vals, factors)
    R = fac[(d + 1) % len(fac)].shape[1]
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    Y = np.empty((rows.shape[0], R), dtype=np.float64)
    S = np.empty_like(Y)
    p = None if perm is None else np.ascontiguousarray(perm, dtype=np.int64)
    rc = _load().oracle_mttkrp_rows_subset(len(dims), _ptr(dims, ctypes.c_int64), idx.shape[1],
                                           _ptr(idx, ctypes.c_int32), _ptr(vals, ctypes.c_float), _facptrs(fac), R, d,
                                           _ptr(p, ctypes.c_int64), rows.shape[0], _ptr(rows, ctypes.c_int64),
                                           _ptr(Y, ctypes.c_double), _ptr(S, ctypes.c_double))
    if rc != 0:
        raise RuntimeError("oracle_mttkrp_rows_subset failed")
    return Y, S


# ----------------------------------------------------------------------------- numpy twin

def sort_perm_numpy(idx: np.ndarray, order: Sequence[int]) -> np.ndarray:
    """np.lexsort twin of `sort_perm` (lexsort is stable; its LAST key is the primary one)."""
    keys = tuple(np.asarray(idx[m]) for m in reversed(list(order)))
    return np.lexsort(keys).astype(np.int64)


def mttkrp_numpy(dims, idx, vals, factors, d: int) -> Tuple[np.ndarray, np.ndarray]:
    """Vectorised numpy twin of the definition, fp64, for small cases."""
    dims, idx, vals, fac = _prep(dims, idx, vals, factors)
    R = fac[(d + 1) % len(fac)].shape[1]
    l = np.repeat(vals.astype(np.float64)[:, None], R, axis=1)
    labs = np.abs(l)
    for w in range(len(dims)):
        if w == d:
            continue
        rows = fac[w].astype(np.float64)[idx[w]]
        l = l * rows
        labs = labs * np.abs(rows)
    Y = np.zeros((int(dims[d]), R), dtype=np.float64)
    S = np.zeros_like(Y)
    np.add.at(Y, idx[d], l)
    np.add.at(S, idx[d], labs)
    return Y, S


# ----------------------------------------------------------------------------- acceptance

def normalised_error(Y_test: np.ndarray, Y_ref: np.ndarray, S_ref: np.ndarray) -> Tuple[float, bool]:
    """north_star acceptance: max |Y_test - Y_ref| / S_ref over entries with S_ref > 0, and whether
    every entry with S_ref == 0 is exactly 0 in Y_test."""
    Yt = np.asarray(Y_test, dtype=np.float64)
    diff = np.abs(Yt - Y_ref)
    pos = S_ref > 0
    err = float((diff[pos] / S_ref[pos]).max()) if pos.any() else 0.0
    zeros_ok = bool(np.all(Yt[~pos] == 0.0)) and bool(np.all(np.isfinite(Yt)))
    return err, zeros_ok
