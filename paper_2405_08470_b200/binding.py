"""ctypes binding of libmttkrp_b200 (include/mttkrp.h).  Argument marshalling only.

Every step of the path (format build, remap, MTTKRP, fix-up) runs in the library's CUDA kernels;
PyTorch is used for device memory and the current stream.  There is no CPU fallback: if the shared
library is missing, or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes
import os
from typing import List, Optional, Sequence

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libmttkrp_b200.so")
MAX_MODES = 8
NOALLOC_MAX_NNZ = 1 << 22          # MTTKRP_NOALLOC_MAX_NNZ in include/mttkrp.h

OK, EINVAL, EINDEX, EUNSUPPORTED, EWORKSPACE, ECUDA = range(6)
_STATUS_NAMES = {0: "MTTKRP_OK", 1: "MTTKRP_EINVAL", 2: "MTTKRP_EINDEX", 3: "MTTKRP_EUNSUPPORTED",
                 4: "MTTKRP_EWORKSPACE", 5: "MTTKRP_ECUDA"}

EXPORTS = ["mttkrp_workspace_bytes", "mttkrp_create", "mttkrp_mode", "mttkrp_sweep", "mttkrp_remap_to",
           "mttkrp_sweep_host", "mttkrp_destroy", "mttkrp_last_error", "mttkrp_get_info", "mttkrp_get_perm",
           "mttkrp_get_perm_noalloc", "mttkrp_export_coo", "mttkrp_timing_begin", "mttkrp_timing_end", "mttkrp_partition_rows", "mttkrp_version"]


class MttkrpError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"{_STATUS_NAMES.get(status, status)}: {message}")
        self.status = status


class Info(ctypes.Structure):
    _fields_ = [("nmodes", ctypes.c_int32), ("cur_layout", ctypes.c_int32), ("nnz", ctypes.c_int64),
                ("dims", ctypes.c_int64 * MAX_MODES), ("record_bytes", ctypes.c_int32),
                ("shard_nnz", ctypes.c_int32), ("num_shards", ctypes.c_int64),
                ("num_split_rows", ctypes.c_int64 * MAX_MODES), ("num_empty_rows", ctypes.c_int64 * MAX_MODES),
                ("bytes_held", ctypes.c_int64), ("bytes_paper_format", ctypes.c_int64),
                ("remaps_done", ctypes.c_int64), ("key_order", (ctypes.c_int32 * MAX_MODES) * MAX_MODES),
                ("remap_blocked", ctypes.c_int32 * MAX_MODES), ("remap_avg_run", ctypes.c_double * MAX_MODES),
                ("shard_policy", ctypes.c_int32), ("kappa", ctypes.c_int32),
                ("max_partition_nnz", ctypes.c_int64 * MAX_MODES), ("min_partition_nnz", ctypes.c_int64 * MAX_MODES),
                ("remap_plain_ms", ctypes.c_double * MAX_MODES), ("remap_twopass_ms", ctypes.c_double * MAX_MODES),
                ("fused_remap", ctypes.c_int32), ("reserved_", ctypes.c_int32),
                ("cold_rows", ctypes.c_int64 * MAX_MODES), ("cold_degree", ctypes.c_int64 * MAX_MODES)]


class Timing(ctypes.Structure):
    _fields_ = [("remap_ms", ctypes.c_double), ("zero_ms", ctypes.c_double), ("mttkrp_ms", ctypes.c_double),
                ("fixup_ms", ctypes.c_double), ("remap_launches", ctypes.c_int64), ("zero_launches", ctypes.c_int64),
                ("mttkrp_launches", ctypes.c_int64), ("fixup_launches", ctypes.c_int64)]


_lib = None


def load_library(path: Optional[str] = None) -> ctypes.CDLL:
    """dlopen the in-tree shared library (built by `python -m paper_2405_08470_b200.build`)."""
    global _lib
    if _lib is not None and path is None:
        return _lib
    p = path or LIB_PATH
    if not os.path.exists(p):
        raise ImportError(f"{p} not found: build it with `python -m paper_2405_08470_b200.build` "
                          "(there is no CPU fallback)")
    lib = ctypes.CDLL(p)
    vp, i64p, szp = ctypes.c_void_p, ctypes.POINTER(ctypes.c_int64), ctypes.POINTER(ctypes.c_size_t)
    vpp = ctypes.POINTER(ctypes.c_void_p)
    lib.mttkrp_workspace_bytes.argtypes = [ctypes.c_int, i64p, ctypes.c_int64, ctypes.c_int, szp]
    lib.mttkrp_create.argtypes = [vpp, ctypes.c_int, i64p, ctypes.c_int64, vp, vp, ctypes.c_int, vp, ctypes.c_size_t, vp]
    lib.mttkrp_mode.argtypes = [vp, ctypes.c_int, vpp, ctypes.c_int, vp, vp]
    lib.mttkrp_sweep.argtypes = [vp, vpp, ctypes.c_int, vpp, vp]
    lib.mttkrp_remap_to.argtypes = [vp, ctypes.c_int, vp]
    lib.mttkrp_sweep_host.argtypes = [vp, vpp, ctypes.c_int, vpp, vp]
    lib.mttkrp_destroy.argtypes = [vp]
    lib.mttkrp_get_info.argtypes = [vp, ctypes.POINTER(Info)]
    lib.mttkrp_get_perm.argtypes = [vp, ctypes.c_int, vp, vp, vp]
    lib.mttkrp_get_perm_noalloc.argtypes = [vp, ctypes.c_int, vp, vp]
    lib.mttkrp_export_coo.argtypes = [vp, vp, vp, vp]
    lib.mttkrp_partition_rows.argtypes = [vp, ctypes.c_int, ctypes.c_int, vp, vp, vp, vp]
    lib.mttkrp_timing_begin.argtypes = [vp]
    lib.mttkrp_timing_end.argtypes = [vp, ctypes.POINTER(Timing), vp]
    for name in EXPORTS:
        getattr(lib, name).restype = ctypes.c_int
    lib.mttkrp_last_error.restype = ctypes.c_char_p
    lib.mttkrp_last_error.argtypes = []
    lib.mttkrp_version.restype = ctypes.c_char_p
    lib.mttkrp_version.argtypes = []
    if path is None:
        _lib = lib
    return lib


def _check(status: int):
    if status != OK:
        raise MttkrpError(status, load_library().mttkrp_last_error().decode())


def _dims_array(dims: Sequence[int]):
    return (ctypes.c_int64 * len(dims))(*[int(d) for d in dims])


def _stream() -> int:
    return int(torch.cuda.current_stream().cuda_stream)


def _ptr_array(tensors: Sequence[Optional[torch.Tensor]]):
    arr = (ctypes.c_void_p * len(tensors))()
    for i, t in enumerate(tensors):
        arr[i] = None if t is None else t.data_ptr()
    return arr


def version() -> str:
    return load_library().mttkrp_version().decode()


def mttkrp_workspace_bytes(dims: Sequence[int], nnz: int, max_rank: int = 0) -> int:
    out = ctypes.c_size_t(0)
    _check(load_library().mttkrp_workspace_bytes(len(dims), _dims_array(dims), int(nnz), int(max_rank), ctypes.byref(out)))
    return int(out.value)


class Mttkrp:
    """Handle over `mttkrp_create` / `mttkrp_mode` / `mttkrp_destroy`.

    idx: int32 [nmodes, nnz] CUDA tensor (SoA COO), vals: float32 [nnz] CUDA tensor.
    """

    def __init__(self, dims: Sequence[int], idx: torch.Tensor, vals: torch.Tensor, max_rank: int = 0):
        lib = load_library()
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2405_08470_b200 needs a CUDA device (no CPU fallback)")
        if not (idx.is_cuda and vals.is_cuda):
            raise ValueError("idx and vals must be CUDA tensors")
        if idx.dtype != torch.int32 or vals.dtype != torch.float32:
            raise ValueError("idx must be int32 and vals float32")
        idx = idx.contiguous()
        vals = vals.contiguous()
        self.dims = [int(d) for d in dims]
        self.nmodes = len(self.dims)
        self.nnz = int(vals.numel())
        if idx.dim() != 2 or idx.shape[0] != self.nmodes or idx.shape[1] != self.nnz:
            raise ValueError("idx must be [nmodes, nnz]")
        self.device = vals.device
        nbytes = mttkrp_workspace_bytes(self.dims, self.nnz, max_rank)
        self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
        base = self.workspace.data_ptr()
        self._ws_ptr = (base + 255) // 256 * 256
        self._h = ctypes.c_void_p(None)
        with torch.cuda.device(self.device):
            st = lib.mttkrp_create(ctypes.byref(self._h), self.nmodes, _dims_array(self.dims), self.nnz,
                                   idx.data_ptr() if self.nnz else None, vals.data_ptr() if self.nnz else None,
                                   int(max_rank), self._ws_ptr, nbytes, _stream())
        if st != OK:
            self._h = ctypes.c_void_p(None)
            _check(st)

    # -- compute ---------------------------------------------------------------------------------
    def _check_factors(self, factors: Sequence[Optional[torch.Tensor]], skip: Optional[int]) -> int:
        if len(factors) != self.nmodes:
            raise ValueError("need one factor per mode")
        R = None
        for m, f in enumerate(factors):
            if m == skip and f is None:
                continue
            if f is None or not f.is_cuda or f.dtype != torch.float32 or not f.is_contiguous():
                raise ValueError(f"factors[{m}] must be a contiguous float32 CUDA tensor")
            if f.dim() != 2 or f.shape[0] != self.dims[m]:
                raise ValueError(f"factors[{m}] must be [{self.dims[m]}, R]")
            R = f.shape[1] if R is None else R
            if f.shape[1] != R:
                raise ValueError("all factors must have the same rank")
        return int(R)

    def mttkrp_mode(self, d: int, factors: Sequence[Optional[torch.Tensor]], out: Optional[torch.Tensor] = None) -> torch.Tensor:
        R = self._check_factors(factors, d)
        if out is None:
            out = torch.empty((self.dims[d], R), dtype=torch.float32, device=self.device)
        elif out.shape != (self.dims[d], R) or out.dtype != torch.float32 or not out.is_contiguous() or not out.is_cuda:
            raise ValueError("out must be a contiguous float32 CUDA tensor [dims[d], R]")
        fac = [None if m == d else f for m, f in enumerate(factors)]
        with torch.cuda.device(self.device):
            _check(load_library().mttkrp_mode(self._h, int(d), _ptr_array(fac), R, out.data_ptr(), _stream()))
        return out

    def mttkrp_sweep(self, factors: Sequence[torch.Tensor], outs: Optional[List[torch.Tensor]] = None) -> List[torch.Tensor]:
        R = self._check_factors(factors, None)
        if outs is None:
            outs = [torch.empty((self.dims[d], R), dtype=torch.float32, device=self.device) for d in range(self.nmodes)]
        with torch.cuda.device(self.device):
            _check(load_library().mttkrp_sweep(self._h, _ptr_array(factors), R, _ptr_array(outs), _stream()))
        return outs

    def mttkrp_sweep_host(self, factors: Sequence[torch.Tensor], outs: Sequence[torch.Tensor]) -> Sequence[torch.Tensor]:
        """HOST tensors in, HOST tensors out (pinned memory recommended); synchronous."""
        R = int(factors[0].shape[1])
        for m, (f, o) in enumerate(zip(factors, outs)):
            if f.is_cuda or o.is_cuda or f.dtype != torch.float32 or o.dtype != torch.float32:
                raise ValueError("host entry point takes float32 CPU tensors")
            if tuple(f.shape) != (self.dims[m], R) or tuple(o.shape) != (self.dims[m], R) or not f.is_contiguous() or not o.is_contiguous():
                raise ValueError(f"factors[{m}] / outs[{m}] must be contiguous [{self.dims[m]}, {R}]")
        with torch.cuda.device(self.device):
            _check(load_library().mttkrp_sweep_host(self._h, _ptr_array(factors), R, _ptr_array(outs), _stream()))
        return outs

    def remap_to(self, d: int) -> None:
        with torch.cuda.device(self.device):
            _check(load_library().mttkrp_remap_to(self._h, int(d), _stream()))

    # -- introspection ---------------------------------------------------------------------------
    def info(self) -> dict:
        raw = Info()
        _check(load_library().mttkrp_get_info(self._h, ctypes.byref(raw)))
        n = raw.nmodes
        return {
            "nmodes": n, "cur_layout": raw.cur_layout, "nnz": raw.nnz, "dims": list(raw.dims)[:n],
            "record_bytes": raw.record_bytes, "shard_nnz": raw.shard_nnz, "num_shards": raw.num_shards,
            "num_split_rows": list(raw.num_split_rows)[:n], "num_empty_rows": list(raw.num_empty_rows)[:n],
            "bytes_held": raw.bytes_held, "bytes_paper_format": raw.bytes_paper_format,
            "remaps_done": raw.remaps_done,
            "key_order": [list(raw.key_order[d])[:n] for d in range(n)],
            "remap_blocked": list(raw.remap_blocked)[:n], "remap_avg_run": list(raw.remap_avg_run)[:n],
            "shard_policy": "alg1" if raw.shard_policy else "equal", "kappa": raw.kappa, "fused_remap": bool(raw.fused_remap),
            "remap_plain_ms": list(raw.remap_plain_ms)[:n], "remap_twopass_ms": list(raw.remap_twopass_ms)[:n],
            "max_partition_nnz": list(raw.max_partition_nnz)[:n], "min_partition_nnz": list(raw.min_partition_nnz)[:n],
            "cold_rows": list(raw.cold_rows)[:n], "cold_degree": list(raw.cold_degree)[:n],
        }

    def partition_rows(self, d: int, kappa: int):
        """Alg. 1 of the paper for mode d: (partition of every row [int32, host], nonzeros per partition [int64])."""
        import numpy as np
        deg = torch.empty(int(self.dims[d]), dtype=torch.int32, device=self.device)
        part = np.empty(int(self.dims[d]), dtype=np.int32)
        loads = np.empty(int(kappa), dtype=np.int64)
        with torch.cuda.device(self.device):
            _check(load_library().mttkrp_partition_rows(self._h, int(d), int(kappa), deg.data_ptr(),
                                                        part.ctypes.data, loads.ctypes.data, _stream()))
        return part, loads

    def get_perm(self, d: int) -> torch.Tensor:
        perm = torch.empty(max(self.nnz, 1), dtype=torch.int32, device=self.device)
        scratch = torch.empty_like(perm)
        with torch.cuda.device(self.device):
            _check(load_library().mttkrp_get_perm(self._h, int(d), perm.data_ptr(), scratch.data_ptr(), _stream()))
        return perm[: self.nnz]

    def get_perm_noalloc(self, d: int, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        """`get_perm` for callers that cannot allocate device memory at call time (all of the GPU's memory already
        belongs to the host application's pool, or cudaMalloc's device-wide stall is not acceptable): the second
        buffer `get_perm` allocates is a fixed 16 MiB array inside the library instead.  Pass a preallocated int32
        `out` of nnz elements and this method allocates nothing on the device either.  Handles with more than
        NOALLOC_MAX_NNZ nonzeros raise MTTKRP_EUNSUPPORTED.  All calls on a device share the array: do not let two
        of them overlap on the GPU."""
        if out is None:
            out = torch.empty(max(self.nnz, 1), dtype=torch.int32, device=self.device)
        elif not out.is_cuda or out.dtype != torch.int32 or not out.is_contiguous() or out.numel() < self.nnz:
            raise ValueError("out must be a contiguous int32 CUDA tensor with at least nnz elements")
        with torch.cuda.device(self.device):
            _check(load_library().mttkrp_get_perm_noalloc(self._h, int(d), out.data_ptr(), _stream()))
        return out[: self.nnz]

    def export_coo(self):
        idx = torch.empty((self.nmodes, max(self.nnz, 1)), dtype=torch.int32, device=self.device)[:, : self.nnz].contiguous()
        vals = torch.empty(max(self.nnz, 1), dtype=torch.float32, device=self.device)[: self.nnz]
        if self.nnz:
            with torch.cuda.device(self.device):
                _check(load_library().mttkrp_export_coo(self._h, idx.data_ptr(), vals.data_ptr(), _stream()))
        return idx, vals

    def timing_begin(self) -> None:
        _check(load_library().mttkrp_timing_begin(self._h))

    def timing_end(self) -> dict:
        raw = Timing()
        with torch.cuda.device(self.device):
            _check(load_library().mttkrp_timing_end(self._h, ctypes.byref(raw), _stream()))
        return {name: getattr(raw, name) for name, _ in Timing._fields_}

    def destroy(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            load_library().mttkrp_destroy(self._h)
            self._h = ctypes.c_void_p(None)
            self.workspace = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
