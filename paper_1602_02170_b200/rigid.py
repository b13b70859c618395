"""ctypes binding of the rigid-multiblob entry points (C ABI: ``include/rpy_rigid.h``).

Argument marshalling only: tensor checks, raw pointers, the current CUDA stream.  K, K^T
(PAPER.md:79-84, 156-161), the block-diagonal preconditioner and the GMRES solve
of Eq. (11) all run in the CUDA kernels of ``csrc/rpy_rigid.cu``.  No CPU
fallback: without the built library or a CUDA device every call raises.
"""
from __future__ import annotations

import ctypes
from dataclasses import dataclass
from typing import Optional

import torch

from . import binding
from .binding import RPY_PREC_F64, RPY_PREC_F32_ACC64, RpyError, _prec_code  # noqa: F401

RPY_ERR_NOT_SPD = 6
RPY_PREC_MIXED = 2       # solve only: fp32 products inside a cycle, fp64 residual per cycle
RPY_RIGID_MAX_BODY_BLOBS = 1024
RPY_RIGID_MAX_RESTART = 128
RPY_RIGID_MAX_BATCH = 8

_vp, _i64, _int, _dbl, _sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
_i64p, _dblp, _intp = ctypes.POINTER(_i64), ctypes.POINTER(_dbl), ctypes.POINTER(_int)

# int reduce(void* ctx, double* d_buf, int64_t count, void* cuda_stream): sums d_buf over the ranks in place
REDUCE_FN = ctypes.CFUNCTYPE(_int, _vp, _vp, _i64, _vp)


class SolveExt(ctypes.Structure):
    """rpy_rigid_solve_ext: the caller's side stream and event, and the multi-GPU share of the product."""
    _fields_ = [("side_stream", _vp), ("side_event", _vp), ("shard", _int), ("n_shards", _int),
                ("reduce", REDUCE_FN), ("reduce_ctx", _vp)]


_extp = ctypes.POINTER(SolveExt)

SIGNATURES = {
    "rpy_rigid_K_apply": (_int, [_i64, _i64, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp, _vp]),
    "rpy_rigid_KT_apply": (_int, [_i64, _i64, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp, _vp]),
    "rpy_rigid_blob_positions": (_int, [_int, _i64, _int, _vp, _vp, _vp, _vp, _vp]),
    "rpy_rigid_precond_bytes": (_sz, [_i64, _i64p]),
    "rpy_rigid_precond_build": (_int, [_int, _i64, _i64, _vp, _vp, _i64p, _dbl, _dbl, _vp, _sz, _vp]),
    "rpy_rigid_precond_info": (_int, [_i64, _vp, _i64p, _vp]),
    "rpy_rigid_precond_apply": (_int, [_i64, _i64, _vp, _vp, _vp, _vp]),
    "rpy_rigid_precond_get": (_int, [_i64, _i64p, _vp, _i64, _vp, _vp, _vp]),
    "rpy_rigid_solve_workspace_bytes": (_sz, [_int, _i64, _i64, _int]),
    "rpy_rigid_mobility_solve": (_int, [_int, _int, _i64, _i64, _vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp, _dbl,
                                        _int, _int, _vp, _vp, _dblp, _intp, _dblp, _vp, _sz, _vp, _extp]),
    "rpy_rigid_solve_batch_workspace_bytes": (_sz, [_int, _i64, _i64, _int, _int]),
    "rpy_rigid_mobility_solve_batch": (_int, [_int, _int, _i64, _i64, _int, _vp, _vp, _vp, _vp, _vp, _dbl, _dbl, _vp, _dbl,
                                              _int, _int, _vp, _vp, _dblp, _intp, _dblp, _vp, _sz, _vp, _extp]),
    "rpy_rigid_saddle_apply": (_int, [_int, _int, _i64, _i64, _vp, _vp, _vp, _dbl, _dbl, _vp, _vp, _vp, _sz, _vp]),
}

_ready = False


def _lib():
    global _ready
    lib = binding.load_library()
    if not _ready:
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(lib, name)
            fn.restype = res
            fn.argtypes = args
        _ready = True
    return lib


def _check(status: int):
    if status == RPY_ERR_NOT_SPD:
        raise RpyError(status, "RPY_ERR_NOT_SPD: a body's blob mobility M^(pp) (or its K^T M^-1 K) is not positive "
                               "(semi-)definite (a blob overlapping the wall, or coincident blobs)")
    binding._check(status)


def _f64(t: torch.Tensor, shape, what: str):
    if not torch.cuda.is_available():
        raise RuntimeError("the rigid layer needs a CUDA device (sm_100a); there is no CPU fallback")
    if not t.is_cuda or t.dtype != torch.float64 or not t.is_contiguous() or tuple(t.shape) != tuple(shape):
        raise ValueError(f"{what} must be a contiguous float64 CUDA tensor of shape {tuple(shape)}")
    return t


def _stream(t: torch.Tensor):
    return torch.cuda.current_stream(t.device).cuda_stream


@dataclass
class Bodies:
    """Device view of the rigid bodies: positions of all blobs, tracking points, contiguous runs."""
    pos: torch.Tensor            # [n_blobs, 3] float64 CUDA
    q: torch.Tensor              # [n_bodies, 3] float64 CUDA
    offsets: torch.Tensor        # [n_bodies + 1] int64 CUDA
    h_offsets: torch.Tensor      # the same on the host (sizes the preconditioner)

    @property
    def n_blobs(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_bodies(self) -> int:
        return int(self.q.shape[0])

    @property
    def n(self) -> int:
        return 3 * self.n_blobs + 6 * self.n_bodies


def bodies(pos: torch.Tensor, q: torch.Tensor, offsets) -> Bodies:
    """Bundles the inputs every rigid call needs; `offsets` is any int sequence / tensor [n_bodies+1]."""
    h = torch.as_tensor(offsets, dtype=torch.int64).cpu().contiguous()
    nb = h.numel() - 1
    _f64(pos, (pos.shape[0], 3), "pos")
    _f64(q, (nb, 3), "q")
    if nb < 1 or int(h[0]) != 0 or int(h[-1]) != pos.shape[0] or bool((h[1:] <= h[:-1]).any()):
        raise ValueError("offsets must start at 0, increase strictly and end at n_blobs")
    return Bodies(pos, q, h.to(pos.device), h)


def rpy_rigid_K_apply(b: Bodies, U: torch.Tensor, alpha: float = 1.0, beta: float = 0.0,
                      out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """out = beta out + alpha K U: blob velocities of the rigid motions U [n_bodies, 6] (Eq. (2))."""
    _f64(U, (b.n_bodies, 6), "U")
    if out is None:
        if beta != 0.0:
            raise ValueError("beta != 0 needs out")
        out = torch.empty_like(b.pos)
    _f64(out, (b.n_blobs, 3), "out")
    with torch.cuda.device(b.pos.device):
        _check(_lib().rpy_rigid_K_apply(b.n_blobs, b.n_bodies, b.pos.data_ptr(), b.q.data_ptr(), b.offsets.data_ptr(),
                                        U.data_ptr(), float(alpha), float(beta), out.data_ptr(), _stream(b.pos)))
    return out


def rpy_rigid_KT_apply(b: Bodies, lam: torch.Tensor, alpha: float = 1.0, beta: float = 0.0,
                       out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """out = beta out + alpha K^T lambda: force and torque per body [n_bodies, 6] (Eq. (10))."""
    _f64(lam, (b.n_blobs, 3), "lam")
    if out is None:
        if beta != 0.0:
            raise ValueError("beta != 0 needs out")
        out = torch.empty((b.n_bodies, 6), dtype=torch.float64, device=b.pos.device)
    _f64(out, (b.n_bodies, 6), "out")
    with torch.cuda.device(b.pos.device):
        _check(_lib().rpy_rigid_KT_apply(b.n_blobs, b.n_bodies, b.pos.data_ptr(), b.q.data_ptr(), b.offsets.data_ptr(),
                                         lam.data_ptr(), float(alpha), float(beta), out.data_ptr(), _stream(b.pos)))
    return out


def rpy_rigid_blob_positions(template: torch.Tensor, centres: torch.Tensor, quats: torch.Tensor) -> torch.Tensor:
    """Blob positions [n_bodies * blobs_per_body, 3] of identical bodies from their poses:
    r = c_p + R(theta_p) template_t, quaternions (s, p1, p2, p3).  float64 or float32 CUDA tensors."""
    if not torch.cuda.is_available():
        raise RuntimeError("the rigid layer needs a CUDA device (sm_100a); there is no CPU fallback")
    nb, bpb = centres.shape[0], template.shape[0]
    for t, shape, what in ((template, (bpb, 3), "template"), (centres, (nb, 3), "centres"), (quats, (nb, 4), "quats")):
        if not t.is_cuda or t.dtype != template.dtype or not t.is_contiguous() or tuple(t.shape) != shape:
            raise ValueError(f"{what} must be a contiguous CUDA tensor of shape {shape} and the template's dtype")
    pos = torch.empty((nb * bpb, 3), dtype=template.dtype, device=template.device)
    with torch.cuda.device(template.device):
        _check(_lib().rpy_rigid_blob_positions(binding._prec_of(template.dtype), nb, bpb, template.data_ptr(),
                                               centres.data_ptr() or None, quats.data_ptr() or None,
                                               pos.data_ptr() or None, _stream(template)))
    return pos


def _hptr(h: torch.Tensor):
    return ctypes.cast(h.data_ptr(), _i64p)


def rpy_rigid_precond_bytes(offsets) -> int:
    h = torch.as_tensor(offsets, dtype=torch.int64).cpu().contiguous()
    return int(_lib().rpy_rigid_precond_bytes(h.numel() - 1, _hptr(h)))


@dataclass
class Precond:
    """A built block-diagonal preconditioner (device buffer + the bodies it belongs to)."""
    buf: torch.Tensor
    bodies: Bodies
    variant: str


def rpy_rigid_precond_build(b: Bodies, variant: str = "wall", a: float = 1.0, eta: float = 1.0,
                            check: bool = True, buf: Optional[torch.Tensor] = None) -> Precond:
    """Dense M^(pp), its explicit inverse, Y, N~ for every body (Eqs. (17)-(19)); `variant` 'wall' or 'free'.
    `buf`: a CUDA uint8 tensor of at least rpy_rigid_precond_bytes(offsets) bytes to build into (a time-stepping
    caller rebuilds the preconditioner every step); allocated when None."""
    lib = _lib()
    need = int(lib.rpy_rigid_precond_bytes(b.n_bodies, _hptr(b.h_offsets)))
    if need == 0:
        raise ValueError("invalid body offsets (or a body above RPY_RIGID_MAX_BODY_BLOBS)")
    if buf is None:
        buf = torch.empty(need, dtype=torch.uint8, device=b.pos.device)
    elif buf.dtype != torch.uint8 or not buf.is_cuda or not buf.is_contiguous() or buf.numel() < need:
        raise ValueError(f"buf must be a contiguous CUDA uint8 tensor of at least {need} bytes")
    with torch.cuda.device(b.pos.device):
        _check(lib.rpy_rigid_precond_build(1 if variant == "wall" else 0, b.n_blobs, b.n_bodies, b.pos.data_ptr(),
                                           b.q.data_ptr(), _hptr(b.h_offsets), float(a), float(eta),
                                           buf.data_ptr(), need, _stream(b.pos)))
        pc = Precond(buf, b, variant)
        if check:
            rpy_rigid_precond_info(pc)
    return pc


def rpy_rigid_precond_info(pc: Precond) -> int:
    """-1 if every factorisation succeeded; raises RpyError(RPY_ERR_NOT_SPD) naming the first bad body."""
    bad = _i64(-1)
    with torch.cuda.device(pc.buf.device):
        st = _lib().rpy_rigid_precond_info(pc.bodies.n_bodies, pc.buf.data_ptr(), ctypes.byref(bad), _stream(pc.buf))
    if st == RPY_ERR_NOT_SPD:
        raise RpyError(st, f"RPY_ERR_NOT_SPD: M^(pp) of body {bad.value} is not positive definite")
    _check(st)
    return int(bad.value)


def rpy_rigid_precond_apply(pc: Precond, x: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
    """[lambda; U] = P^-1 x for a solver vector x of 3 n_blobs + 6 n_bodies doubles (Eq. (19))."""
    b = pc.bodies
    _f64(x, (b.n,), "x")
    if out is None:
        out = torch.empty_like(x)
    _f64(out, (b.n,), "out")
    with torch.cuda.device(x.device):
        _check(_lib().rpy_rigid_precond_apply(b.n_blobs, b.n_bodies, pc.buf.data_ptr(), x.data_ptr(), out.data_ptr(),
                                              _stream(x)))
    return out


def rpy_rigid_precond_get(pc: Precond, body: int):
    """((M^(pp))^-1 [m, m], N~_pp [6, 6]) of one body."""
    b = pc.bodies
    m = 3 * int(b.h_offsets[body + 1] - b.h_offsets[body])
    fac = torch.empty((m, m), dtype=torch.float64, device=pc.buf.device)
    nt = torch.empty((6, 6), dtype=torch.float64, device=pc.buf.device)
    with torch.cuda.device(pc.buf.device):
        _check(_lib().rpy_rigid_precond_get(b.n_bodies, _hptr(b.h_offsets), pc.buf.data_ptr(), int(body),
                                            fac.data_ptr(), nt.data_ptr(), _stream(pc.buf)))
    return fac, nt


def rpy_rigid_solve_workspace_bytes(matvec_prec, n_blobs: int, n_bodies: int, restart: int) -> int:
    prec = RPY_PREC_MIXED if matvec_prec in ("mixed", RPY_PREC_MIXED) else _prec_code(matvec_prec)
    return int(_lib().rpy_rigid_solve_workspace_bytes(prec, int(n_blobs), int(n_bodies), int(restart)))


def rpy_rigid_saddle_apply(b: Bodies, x: torch.Tensor, variant: str = "wall", a: float = 1.0, eta: float = 1.0,
                           matvec_prec="f64") -> torch.Tensor:
    """[M lambda - K U; -K^T lambda] for a solver vector x (the operator of Eq. (11))."""
    _f64(x, (b.n,), "x")
    prec = _prec_code(matvec_prec)
    need = rpy_rigid_solve_workspace_bytes(prec, b.n_blobs, b.n_bodies, 1)
    ws = torch.empty(need, dtype=torch.uint8, device=x.device)
    out = torch.empty_like(x)
    with torch.cuda.device(x.device):
        _check(_lib().rpy_rigid_saddle_apply(1 if variant == "wall" else 0, prec, b.n_blobs, b.n_bodies,
                                             b.pos.data_ptr(), b.q.data_ptr(), b.offsets.data_ptr(), float(a),
                                             float(eta), x.data_ptr(), out.data_ptr(), ws.data_ptr(), need, _stream(x)))
    return out


_side = {}          # (device index, thread) -> (side stream, event): created once, handed to every solve


def _solve_ext(device, shard: int = 0, n_shards: int = 1, reduce=None, side: bool = True):
    """(SolveExt, keep-alive objects): the side stream and event the solve reads its status on, and -- for a
    multi-GPU solve -- this rank's share and the hook that sums the partial products over the ranks."""
    ext = SolveExt()
    keep = []
    if side:
        import threading
        idx = torch.device(device).index
        idx = torch.cuda.current_device() if idx is None else idx
        key = (idx, threading.get_ident())                   # concurrent solves must not share an event
        if key not in _side:
            with torch.cuda.device(idx):
                st, ev = torch.cuda.Stream(), torch.cuda.Event()
                ev.record(torch.cuda.current_stream())       # torch creates the cudaEvent_t lazily
                _side[key] = (st, ev)
        st, ev = _side[key]
        ext.side_stream, ext.side_event = st.cuda_stream, ev.cuda_event
    ext.shard, ext.n_shards = int(shard), int(n_shards)
    if n_shards > 1:
        if reduce is None:
            raise ValueError("a sharded solve needs a reduce hook")

        def hook(_ctx, ptr, count, _stream):
            try:
                reduce(int(ptr), int(count))
                return 0
            except Exception:      # pragma: no cover
                import traceback
                traceback.print_exc()
                return 1
        cb = REDUCE_FN(hook)
        keep.append(cb)
        ext.reduce = cb
    return ext, keep


def rpy_rigid_mobility_solve(b: Bodies, pc: Precond, F: torch.Tensor, slip: Optional[torch.Tensor] = None,
                             variant: str = "wall", a: float = 1.0, eta: float = 1.0, tol: float = 1e-8,
                             restart: int = 60, max_iter: int = 200, matvec_prec="f64",
                             workspace: Optional[torch.Tensor] = None, shard: int = 0, n_shards: int = 1,
                             reduce=None, side_stream: bool = True) -> dict:
    """Solves Eq. (11) by preconditioned GMRES.  Returns {'lambda', 'U', 'history', 'n_iter', 'rel_resid'}.

    Multi-GPU: every rank calls with the same arguments and its own ``shard`` of ``n_shards``;
    ``reduce(ptr, count)`` must sum ``count`` doubles at device address ``ptr`` over the ranks in place, in
    stream order on the current stream (``sharding.solve_reduce_hook`` binds it to torch.distributed)."""
    _f64(F, (b.n_bodies, 6), "F")
    if slip is not None:
        _f64(slip, (b.n_blobs, 3), "slip")
    prec = RPY_PREC_MIXED if matvec_prec in ("mixed", RPY_PREC_MIXED) else _prec_code(matvec_prec)
    need = rpy_rigid_solve_workspace_bytes(prec, b.n_blobs, b.n_bodies, restart)
    if need == 0:
        raise ValueError("invalid sizes or restart length")
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=b.pos.device)
    lam = torch.empty_like(b.pos)
    U = torch.empty((b.n_bodies, 6), dtype=torch.float64, device=b.pos.device)
    hist = (_dbl * (max_iter + 1))()
    n_iter, rel = _int(0), _dbl(0.0)
    with torch.cuda.device(b.pos.device):
        ext, keep = _solve_ext(b.pos.device, shard, n_shards, reduce, side_stream)
        _check(_lib().rpy_rigid_mobility_solve(
            1 if variant == "wall" else 0, prec, b.n_blobs, b.n_bodies, b.pos.data_ptr(), b.q.data_ptr(),
            b.offsets.data_ptr(), F.data_ptr(), slip.data_ptr() if slip is not None else None, float(a), float(eta),
            pc.buf.data_ptr(), float(tol), int(restart), int(max_iter), lam.data_ptr(), U.data_ptr(),
            hist, ctypes.byref(n_iter), ctypes.byref(rel), workspace.data_ptr(), int(workspace.numel()),
            _stream(b.pos), ctypes.byref(ext)))
    del keep
    return {"lambda": lam, "U": U, "history": list(hist[:n_iter.value + 1]), "n_iter": n_iter.value,
            "rel_resid": rel.value}


def rpy_rigid_solve_batch_workspace_bytes(matvec_prec, n_blobs: int, n_bodies: int, restart: int, n_rhs: int) -> int:
    prec = RPY_PREC_MIXED if matvec_prec in ("mixed", RPY_PREC_MIXED) else _prec_code(matvec_prec)
    return int(_lib().rpy_rigid_solve_batch_workspace_bytes(prec, int(n_blobs), int(n_bodies), int(restart), int(n_rhs)))


def rpy_rigid_mobility_solve_batch(b: Bodies, pc: Precond, F: torch.Tensor, slip: Optional[torch.Tensor] = None,
                                   variant: str = "wall", a: float = 1.0, eta: float = 1.0, tol: float = 1e-8,
                                   restart: int = 60, max_iter: int = 200, matvec_prec="f64",
                                   workspace: Optional[torch.Tensor] = None) -> dict:
    """Eq. (11) for k = F.shape[0] <= 8 right-hand sides at once (lockstep GMRES sharing one k-right-hand-side
    product per iteration).  F [k, n_bodies, 6], slip [k, n_blobs, 3] or None.
    Returns {'lambda' [k,N,3], 'U' [k,nb,6], 'history' [k][n_iter+1], 'n_iter', 'rel_resid' [k]}."""
    if F.dim() != 3:
        raise ValueError("F must have shape [k, n_bodies, 6]")
    k = int(F.shape[0])
    _f64(F, (k, b.n_bodies, 6), "F")
    if slip is not None:
        _f64(slip, (k, b.n_blobs, 3), "slip")
    prec = RPY_PREC_MIXED if matvec_prec in ("mixed", RPY_PREC_MIXED) else _prec_code(matvec_prec)
    need = rpy_rigid_solve_batch_workspace_bytes(prec, b.n_blobs, b.n_bodies, restart, k)
    if need == 0:
        raise ValueError("invalid sizes, restart length or batch size (1..8)")
    if workspace is None:
        workspace = torch.empty(need, dtype=torch.uint8, device=b.pos.device)
    lam = torch.empty((k, b.n_blobs, 3), dtype=torch.float64, device=b.pos.device)
    U = torch.empty((k, b.n_bodies, 6), dtype=torch.float64, device=b.pos.device)
    hist = (_dbl * (k * (max_iter + 1)))()
    n_iter, rel = _int(0), (_dbl * k)()
    with torch.cuda.device(b.pos.device):
        ext, _keep = _solve_ext(b.pos.device)
        _check(_lib().rpy_rigid_mobility_solve_batch(
            1 if variant == "wall" else 0, prec, b.n_blobs, b.n_bodies, k, b.pos.data_ptr(), b.q.data_ptr(),
            b.offsets.data_ptr(), F.data_ptr(), slip.data_ptr() if slip is not None else None, float(a), float(eta),
            pc.buf.data_ptr(), float(tol), int(restart), int(max_iter), lam.data_ptr(), U.data_ptr(),
            hist, ctypes.byref(n_iter), rel, workspace.data_ptr(), int(workspace.numel()), _stream(b.pos),
            ctypes.byref(ext)))
    it = n_iter.value
    return {"lambda": lam, "U": U, "n_iter": it, "rel_resid": list(rel),
            "history": [list(hist[r * (max_iter + 1): r * (max_iter + 1) + it + 1]) for r in range(k)]}
