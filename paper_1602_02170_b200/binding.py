"""ctypes binding of ``librpy_matvec.so`` (C ABI: ``include/rpy_matvec.h``).

Argument marshalling only: every function here checks tensor dtype / shape / device /
contiguity, takes raw pointers and the current CUDA stream from PyTorch, and calls the C
entry point of the same name.  All arithmetic of the method runs in the
CUDA kernels behind that ABI.  PyTorch is used for device memory and streams, nothing else.

There is no fallback: if the shared library is missing it is built with nvcc
(``paper_1602_02170_b200.build``); if that fails, or no CUDA device is present when a
matvec is called, an exception is raised.
"""
from __future__ import annotations

import ctypes
from typing import Optional

import torch

from . import build as _build

RPY_OK = 0
RPY_PREC_F64 = 0
RPY_PREC_F32_ACC64 = 1

_STATUS_NAMES = {0: "RPY_OK", 1: "RPY_ERR_NULL", 2: "RPY_ERR_ARG", 3: "RPY_ERR_ALIAS",
                 4: "RPY_ERR_WORKSPACE", 5: "RPY_ERR_CUDA"}


class RpyError(RuntimeError):
    """A C-ABI call returned a status other than RPY_OK."""

    def __init__(self, status: int, message: str):
        super().__init__(message)
        self.status = int(status)
        self.name = _STATUS_NAMES.get(int(status), "?")


_lib = None

_vp, _i64, _int, _dbl, _sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_size_t

# name -> (restype, argtypes); also the list of symbols the header declares (tests check it)
SIGNATURES = {
    "rpy_matvec_workspace_bytes": (_sz, [_int, _i64, _int]),
    "rpy_wall_matvec": (_int, [_int, _i64, _int, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_free_matvec": (_int, [_int, _i64, _int, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_wall_matvec_rows": (_int, [_int, _i64, _int, _i64, _i64, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_free_matvec_rows": (_int, [_int, _i64, _int, _i64, _i64, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_wall_matvec_shard": (_int, [_int, _i64, _int, _int, _int, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_free_matvec_shard": (_int, [_int, _i64, _int, _int, _int, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_matvec_rect_workspace_bytes": (_sz, [_int, _i64, _i64, _int]),
    "rpy_wall_matvec_rect": (_int, [_int, _i64, _i64, _int, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_free_matvec_rect": (_int, [_int, _i64, _i64, _int, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_flow_subdivide": (_int, [_int, _i64, _int, _int, _vp, _vp, _vp, _vp, _vp, _vp]),
    "rpy_matvec_host_scratch_bytes": (_sz, [_int, _i64, _int]),
    "rpy_wall_matvec_host": (_int, [_int, _i64, _int, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_free_matvec_host": (_int, [_int, _i64, _int, _vp, _vp, _vp, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_wall_count_below": (_int, [_int, _i64, _vp, _dbl, _vp, _vp]),
    "rpy_matvec_launch_plan": (_int, [_int, _i64, _int, _i64, ctypes.POINTER(_int), ctypes.POINTER(_int),
                                      ctypes.POINTER(_int), ctypes.POINTER(_i64), ctypes.POINTER(_int)]),
    "rpy_status_string": (ctypes.c_char_p, [_int]),
    "rpy_last_cuda_error": (_int, []),
    "rpy_abi_version": (_int, []),
}


def library_path() -> str:
    return str(_build.LIB)


def load_library(rebuild: bool = False):
    """Load (building first if needed) the native library; raises if it cannot be had."""
    global _lib
    if _lib is None or rebuild:
        path = _build.build(force=rebuild)
        lib = ctypes.CDLL(str(path))
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)       # AttributeError if the library does not export it
            fn.restype = res
            fn.argtypes = args
        _lib = lib
    return _lib


def rpy_status_string(status: int) -> str:
    return load_library().rpy_status_string(int(status)).decode()


def _check(status: int):
    if status != RPY_OK:
        lib = load_library()
        msg = lib.rpy_status_string(int(status)).decode()
        if status == 5:
            msg += f" [cudaError {lib.rpy_last_cuda_error()}]"
        raise RpyError(status, msg)


def _prec_of(dtype) -> int:
    if dtype == torch.float64:
        return RPY_PREC_F64
    if dtype == torch.float32:
        return RPY_PREC_F32_ACC64
    raise TypeError(f"positions must be float64 (fp64 path) or float32 (fp32 path with fp64 "
                    f"accumulation), got {dtype}")


def _prec_code(prec) -> int:
    if prec in (RPY_PREC_F64, "f64", torch.float64):
        return RPY_PREC_F64
    if prec in (RPY_PREC_F32_ACC64, "f32", torch.float32):
        return RPY_PREC_F32_ACC64
    raise ValueError(f"unknown precision {prec!r}")


def rpy_matvec_workspace_bytes(prec, n_blobs: int, n_rhs: int = 1) -> int:
    return int(load_library().rpy_matvec_workspace_bytes(_prec_code(prec), int(n_blobs), int(n_rhs)))


def rpy_matvec_host_scratch_bytes(prec, n_blobs: int, n_rhs: int = 1) -> int:
    return int(load_library().rpy_matvec_host_scratch_bytes(_prec_code(prec), int(n_blobs), int(n_rhs)))


def rpy_matvec_launch_plan(prec, n_blobs: int, n_rhs: int = 1, row_count: Optional[int] = None) -> dict:
    """Launch geometry of the all-pairs kernel (pure host arithmetic, works without a GPU)."""
    lib = load_library()
    tpc, nch, ts, nct, sym = _int(), _int(), _int(), _i64(), _int()
    rc = n_blobs if row_count is None else row_count
    _check(lib.rpy_matvec_launch_plan(_prec_code(prec), int(n_blobs), int(n_rhs), int(rc),
                                      ctypes.byref(tpc), ctypes.byref(nch), ctypes.byref(ts), ctypes.byref(nct),
                                      ctypes.byref(sym)))
    return {"targets_per_cta": tpc.value, "n_source_chunks": nch.value, "tile_sources": ts.value,
            "n_ctas": nct.value, "symmetric": bool(sym.value)}


def _require_cuda(t: torch.Tensor, what: str):
    if not torch.cuda.is_available():
        raise RuntimeError("rpy matvec needs a CUDA device (sm_100a); there is no CPU fallback")
    if not t.is_cuda:
        raise ValueError(f"{what} must be a CUDA tensor (use the *_host call for host buffers)")


def _shape_inputs(pos: torch.Tensor, force: torch.Tensor):
    if pos.dim() != 2 or pos.shape[1] != 3:
        raise ValueError("pos must have shape [n_blobs, 3]")
    n = pos.shape[0]
    if force.dim() == 2:
        single = True
        if tuple(force.shape) != (n, 3):
            raise ValueError("force must have shape [n_blobs, 3] or [n_rhs, n_blobs, 3]")
        k = 1
    elif force.dim() == 3 and force.shape[1] == n and force.shape[2] == 3 and force.shape[0] >= 1:
        single = False
        k = force.shape[0]
    else:
        raise ValueError("force must have shape [n_blobs, 3] or [n_rhs, n_blobs, 3]")
    if force.dtype != pos.dtype:
        raise TypeError("pos and force must have the same dtype")
    if not pos.is_contiguous() or not force.is_contiguous():
        raise ValueError("pos and force must be contiguous")
    return n, k, single


def _workspace(prec: int, n: int, k: int, device, workspace: Optional[torch.Tensor]):
    need = rpy_matvec_workspace_bytes(prec, n, k)
    if workspace is None:
        workspace = torch.empty(max(need, 1), dtype=torch.uint8, device=device)
    else:
        if workspace.dtype != torch.uint8 or not workspace.is_contiguous() or workspace.device != device:
            raise ValueError("workspace must be a contiguous uint8 tensor on the same device")
    return workspace, int(workspace.numel())


def _matvec(fn_name: str, pos, force, a, eta, out, workspace, rows):
    lib = load_library()
    _require_cuda(pos, "pos")
    _require_cuda(force, "force")
    n, k, single = _shape_inputs(pos, force)
    prec = _prec_of(pos.dtype)
    if rows is None:
        row_begin, row_count = 0, n
    else:
        row_begin, row_count = int(rows[0]), int(rows[1])
    oshape = (row_count, 3) if single else (k, row_count, 3)
    if out is None:
        out = torch.empty(oshape, dtype=pos.dtype, device=pos.device)
    else:
        if tuple(out.shape) != oshape or out.dtype != pos.dtype or out.device != pos.device or not out.is_contiguous():
            raise ValueError(f"out must be a contiguous {pos.dtype} tensor of shape {oshape} on {pos.device}")
    ws, ws_bytes = _workspace(prec, n, k, pos.device, workspace)
    with torch.cuda.device(pos.device):
        stream = torch.cuda.current_stream(pos.device).cuda_stream
        fn = getattr(lib, fn_name + ("_rows" if rows is not None else ""))
        args = [prec, n, k]
        if rows is not None:
            args += [row_begin, row_count]
        args += [pos.data_ptr() or None, force.data_ptr() or None, out.data_ptr() or None,
                 float(a), float(eta), ws.data_ptr(), ws_bytes, stream]
        _check(fn(*args))
    return out


def rpy_wall_matvec(pos: torch.Tensor, force: torch.Tensor, a: float = 1.0, eta: float = 1.0, *,
                    out: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
                    rows: Optional[tuple] = None) -> torch.Tensor:
    """u = M lambda with the wall-corrected RPY tensor, on the current stream.

    pos [n,3], force [n,3] or [k,n,3] CUDA tensors, float64 (fp64 path) or float32 (fp32
    path with fp64 accumulation).  ``rows=(row_begin, row_count)`` computes only those
    target rows (against all sources).  Returns velocities shaped like ``force``.
    """
    return _matvec("rpy_wall_matvec", pos, force, a, eta, out, workspace, rows)


def rpy_free_matvec(pos: torch.Tensor, force: torch.Tensor, a: float = 1.0, eta: float = 1.0, *,
                    out: Optional[torch.Tensor] = None, workspace: Optional[torch.Tensor] = None,
                    rows: Optional[tuple] = None) -> torch.Tensor:
    """u = M lambda with the free-space RPY tensor, Eq. (9)."""
    return _matvec("rpy_free_matvec", pos, force, a, eta, out, workspace, rows)


def _matvec_shard(fn_name: str, pos, force, shard, n_shards, a, eta, out, workspace):
    lib = load_library()
    _require_cuda(pos, "pos")
    _require_cuda(force, "force")
    n, k, single = _shape_inputs(pos, force)
    prec = _prec_of(pos.dtype)
    oshape = (n, 3) if single else (k, n, 3)
    # partial velocities are float64 on both paths (the cross-shard sum keeps the fp64 accumulation)
    if out is None:
        out = torch.empty(oshape, dtype=torch.float64, device=pos.device)
    elif tuple(out.shape) != oshape or out.dtype != torch.float64 or out.device != pos.device or not out.is_contiguous():
        raise ValueError(f"out must be a contiguous float64 tensor of shape {oshape} on {pos.device}")
    ws, ws_bytes = _workspace(prec, n, k, pos.device, workspace)
    with torch.cuda.device(pos.device):
        stream = torch.cuda.current_stream(pos.device).cuda_stream
        _check(getattr(lib, fn_name)(prec, n, k, int(shard), int(n_shards), pos.data_ptr() or None,
                                     force.data_ptr() or None, out.data_ptr() or None, float(a), float(eta),
                                     ws.data_ptr(), ws_bytes, stream))
    return out


def rpy_wall_matvec_shard(pos: torch.Tensor, force: torch.Tensor, shard: int, n_shards: int, a: float = 1.0,
                          eta: float = 1.0, *, out=None, workspace=None) -> torch.Tensor:
    """Shard `shard` of `n_shards` of u = M lambda (wall tensor): a partial result for ALL rows, always
    float64; the sum over the shards is the product (multi-GPU: one all-reduce).  Uses the symmetric kernel."""
    return _matvec_shard("rpy_wall_matvec_shard", pos, force, shard, n_shards, a, eta, out, workspace)


def rpy_free_matvec_shard(pos: torch.Tensor, force: torch.Tensor, shard: int, n_shards: int, a: float = 1.0,
                          eta: float = 1.0, *, out=None, workspace=None) -> torch.Tensor:
    return _matvec_shard("rpy_free_matvec_shard", pos, force, shard, n_shards, a, eta, out, workspace)


def rpy_matvec_rect_workspace_bytes(prec, n_targets: int, n_sources: int, n_rhs: int = 1) -> int:
    return int(load_library().rpy_matvec_rect_workspace_bytes(_prec_code(prec), int(n_targets), int(n_sources), int(n_rhs)))


def _matvec_rect(fn_name: str, targets, pos, force, a, eta, out, workspace):
    lib = load_library()
    _require_cuda(pos, "pos")
    _require_cuda(force, "force")
    _require_cuda(targets, "targets")
    n, k, single = _shape_inputs(pos, force)
    if targets.dim() != 2 or targets.shape[1] != 3 or targets.dtype != pos.dtype or not targets.is_contiguous():
        raise ValueError("targets must be a contiguous [n_targets, 3] tensor of the positions' dtype")
    nt = targets.shape[0]
    prec = _prec_of(pos.dtype)
    oshape = (nt, 3) if single else (k, nt, 3)
    if out is None:
        out = torch.empty(oshape, dtype=pos.dtype, device=pos.device)
    elif tuple(out.shape) != oshape or out.dtype != pos.dtype or out.device != pos.device or not out.is_contiguous():
        raise ValueError(f"out must be a contiguous {pos.dtype} tensor of shape {oshape} on {pos.device}")
    need = rpy_matvec_rect_workspace_bytes(prec, nt, n, k)
    if workspace is None:
        workspace = torch.empty(max(need, 1), dtype=torch.uint8, device=pos.device)
    with torch.cuda.device(pos.device):
        stream = torch.cuda.current_stream(pos.device).cuda_stream
        _check(getattr(lib, fn_name)(prec, nt, n, k, targets.data_ptr() or None, pos.data_ptr() or None,
                                     force.data_ptr() or None, out.data_ptr() or None, float(a), float(eta),
                                     workspace.data_ptr(), int(workspace.numel()), stream))
    return out


def rpy_wall_matvec_rect(targets: torch.Tensor, pos: torch.Tensor, force: torch.Tensor, a: float = 1.0,
                         eta: float = 1.0, *, out=None, workspace=None) -> torch.Tensor:
    """Velocities at `targets` [n_targets,3] induced by forces on the blobs at `pos` (wall tensor):
    the flow-field evaluation of Appendix B with tracer radius a."""
    return _matvec_rect("rpy_wall_matvec_rect", targets, pos, force, a, eta, out, workspace)


def rpy_free_matvec_rect(targets: torch.Tensor, pos: torch.Tensor, force: torch.Tensor, a: float = 1.0,
                         eta: float = 1.0, *, out=None, workspace=None) -> torch.Tensor:
    return _matvec_rect("rpy_free_matvec_rect", targets, pos, force, a, eta, out, workspace)


def rpy_flow_subdivide(pos: torch.Tensor, force: torch.Tensor, template: torch.Tensor):
    """Appendix B's refinement: every blob -> len(template) small blobs at r_i + template[s], force
    divided uniformly.  Returns (sub_pos [n*n_sub,3], sub_force shaped like force with n*n_sub blobs)."""
    lib = load_library()
    _require_cuda(pos, "pos")
    n, k, single = _shape_inputs(pos, force)
    if template.dim() != 2 or template.shape[1] != 3 or template.dtype != pos.dtype or not template.is_cuda \
            or not template.is_contiguous():
        raise ValueError("template must be a contiguous CUDA [n_sub, 3] tensor of the positions' dtype")
    ns = template.shape[0]
    sub_pos = torch.empty((n * ns, 3), dtype=pos.dtype, device=pos.device)
    sub_force = torch.empty((n * ns, 3) if single else (k, n * ns, 3), dtype=pos.dtype, device=pos.device)
    with torch.cuda.device(pos.device):
        stream = torch.cuda.current_stream(pos.device).cuda_stream
        _check(lib.rpy_flow_subdivide(_prec_of(pos.dtype), n, k, ns, pos.data_ptr() or None, force.data_ptr() or None,
                                      template.data_ptr(), sub_pos.data_ptr() or None, sub_force.data_ptr() or None, stream))
    return sub_pos, sub_force


def _matvec_host(fn_name: str, pos, force, a, eta, out, scratch, device):
    lib = load_library()
    if not torch.cuda.is_available():
        raise RuntimeError("rpy matvec needs a CUDA device (sm_100a); there is no CPU fallback")
    if pos.is_cuda or force.is_cuda:
        raise ValueError("the *_host calls take host (CPU) tensors")
    n, k, single = _shape_inputs(pos, force)
    prec = _prec_of(pos.dtype)
    oshape = (n, 3) if single else (k, n, 3)
    if out is None:
        out = torch.empty(oshape, dtype=pos.dtype, pin_memory=True)
    elif tuple(out.shape) != oshape or out.dtype != pos.dtype or out.is_cuda or not out.is_contiguous():
        raise ValueError(f"out must be a contiguous host {pos.dtype} tensor of shape {oshape}")
    device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    need = rpy_matvec_host_scratch_bytes(prec, n, k)
    if scratch is None:
        scratch = torch.empty(max(need, 1), dtype=torch.uint8, device=device)
    elif scratch.dtype != torch.uint8 or not scratch.is_cuda or not scratch.is_contiguous():
        raise ValueError("scratch must be a contiguous CUDA uint8 tensor")
    with torch.cuda.device(scratch.device):
        stream = torch.cuda.current_stream(scratch.device).cuda_stream
        _check(getattr(lib, fn_name)(prec, n, k, pos.data_ptr() or None, force.data_ptr() or None,
                                     out.data_ptr() or None, float(a), float(eta),
                                     scratch.data_ptr(), int(scratch.numel()), stream))
    return out


def rpy_wall_matvec_host(pos, force, a: float = 1.0, eta: float = 1.0, *, out=None, scratch=None, device=None):
    """Host-buffer form: copies pos/force up, runs the wall matvec, copies u back, synchronises."""
    return _matvec_host("rpy_wall_matvec_host", pos, force, a, eta, out, scratch, device)


def rpy_free_matvec_host(pos, force, a: float = 1.0, eta: float = 1.0, *, out=None, scratch=None, device=None):
    return _matvec_host("rpy_free_matvec_host", pos, force, a, eta, out, scratch, device)


def rpy_wall_count_below(pos: torch.Tensor, zmin: float) -> int:
    """Number of blobs with z < zmin (blobs overlapping the wall for zmin = a)."""
    lib = load_library()
    _require_cuda(pos, "pos")
    if pos.dim() != 2 or pos.shape[1] != 3 or not pos.is_contiguous():
        raise ValueError("pos must be a contiguous [n_blobs, 3] tensor")
    prec = _prec_of(pos.dtype)
    cnt = torch.empty(1, dtype=torch.int64, device=pos.device)
    with torch.cuda.device(pos.device):
        stream = torch.cuda.current_stream(pos.device).cuda_stream
        _check(lib.rpy_wall_count_below(prec, pos.shape[0], pos.data_ptr() or None, float(zmin),
                                        cnt.data_ptr(), stream))
    return int(cnt.item())
