"""CPU oracle for the RPY / wall-RPY mobility matvec -- TEST INFRASTRUCTURE.

ctypes front end of ``oracle/rpy_oracle.c`` (plain float64 double loop, long-double
row sums; what it computes and which passages of arXiv:1602.02170 it follows are
stated in that file's header).  Only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package;
the product (``paper_1602_02170_b200``) never does, and this package never imports
the product.

``build()`` compiles the C file with gcc (``-O2 -fopenmp``, no fast-math) into
``oracle/librpy_oracle.so``; the loader builds on demand when the library is missing
or older than its source.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
from pathlib import Path

import numpy as np

FREE = 0
WALL = 1

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "rpy_oracle.c"
_LIB = _HERE / "librpy_oracle.so"
_lib = None


def build(force: bool = False) -> Path:
    """Compile oracle/rpy_oracle.c -> oracle/librpy_oracle.so (gcc -O2 -fopenmp)."""
    if force or not _LIB.exists() or _LIB.stat().st_mtime < _SRC.stat().st_mtime:
        tmp = _LIB.with_suffix(f".so.tmp{os.getpid()}")
        cmd = ["gcc", "-O2", "-std=gnu99", "-fopenmp", "-fPIC", "-shared",
               "-Wall", "-Wextra", "-o", str(tmp), str(_SRC), "-lm"]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(str(build()))
        dp = ctypes.POINTER(ctypes.c_double)
        ip = ctypes.POINTER(ctypes.c_int64)
        lib.rpy_oracle_pair.argtypes = [ctypes.c_int, dp, dp, ctypes.c_double, ctypes.c_double, dp]
        lib.rpy_oracle_pair.restype = None
        lib.rpy_oracle_wall_block.argtypes = [dp, dp, ctypes.c_double, dp]
        lib.rpy_oracle_wall_block.restype = None
        lib.rpy_oracle_dense.argtypes = [ctypes.c_int, ctypes.c_int64, dp, ctypes.c_double,
                                         ctypes.c_double, dp]
        lib.rpy_oracle_dense.restype = None
        lib.rpy_oracle_matvec.argtypes = [ctypes.c_int, ctypes.c_int64, ctypes.c_int, dp, dp,
                                          ctypes.c_double, ctypes.c_double, ctypes.c_int64, ip, dp]
        lib.rpy_oracle_matvec.restype = None
        lib.rpy_oracle_flow.argtypes = [ctypes.c_int, ctypes.c_int64, dp, ctypes.c_int64, dp, ctypes.c_int, dp,
                                        ctypes.c_double, ctypes.c_double, dp]
        lib.rpy_oracle_flow.restype = None
        lib.rpy_oracle_num_threads.argtypes = []
        lib.rpy_oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def _dptr(x: np.ndarray):
    return x.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def _f64(x, shape=None) -> np.ndarray:
    x = np.ascontiguousarray(x, dtype=np.float64)
    if shape is not None:
        x = x.reshape(shape)
    return x


def pair(variant: int, ri, rj, a: float = 1.0, eta: float = 1.0) -> np.ndarray:
    """3x3 block M_ij (row = velocity component at i, column = force component at j)."""
    ri = _f64(ri, (3,)); rj = _f64(rj, (3,))
    out = np.empty(9)
    _load().rpy_oracle_pair(int(variant), _dptr(ri), _dptr(rj), float(a), float(eta), _dptr(out))
    return out.reshape(3, 3)


def wall_block(ri, rj, a: float = 1.0) -> np.ndarray:
    """Dimensionless wall block (3a/4) W(r_i, r_j) = 6 pi eta a (M_wall - M_free)."""
    ri = _f64(ri, (3,)); rj = _f64(rj, (3,))
    out = np.empty(9)
    _load().rpy_oracle_wall_block(_dptr(ri), _dptr(rj), float(a), _dptr(out))
    return out.reshape(3, 3)


def dense(variant: int, pos, a: float = 1.0, eta: float = 1.0) -> np.ndarray:
    """Dense (3n)x(3n) mobility matrix in the block layout of PAPER.md:120."""
    pos = _f64(pos); n = pos.shape[0]
    assert pos.shape == (n, 3)
    out = np.empty((3 * n, 3 * n))
    _load().rpy_oracle_dense(int(variant), n, _dptr(pos), float(a), float(eta), _dptr(out))
    return out


def matvec(variant: int, pos, force, a: float = 1.0, eta: float = 1.0, rows=None) -> np.ndarray:
    """u = M lambda by the plain double loop.

    pos [n,3]; force [n,3] or [k,n,3]; rows: optional int array of target rows.
    Returns [nrows,3] or [k,nrows,3] to match ``force``.
    """
    pos = _f64(pos); n = pos.shape[0]
    assert pos.shape == (n, 3)
    force = _f64(force)
    single = force.ndim == 2
    k = 1 if single else force.shape[0]
    f3 = force.reshape(k, n, 3)
    if rows is None:
        nrows = n; rptr = None
    else:
        rows = np.ascontiguousarray(rows, dtype=np.int64)
        assert rows.ndim == 1 and (rows.size == 0 or (rows.min() >= 0 and rows.max() < n))
        nrows = rows.size
        rptr = rows.ctypes.data_as(ctypes.POINTER(ctypes.c_int64))
    out = np.zeros((k, nrows, 3))
    if n > 0 and nrows > 0:
        _load().rpy_oracle_matvec(int(variant), n, k, _dptr(pos), _dptr(f3), float(a), float(eta),
                                  nrows, rptr, _dptr(out))
    return out[0] if single else out


def flow(variant: int, targets, pos, force, a: float = 1.0, eta: float = 1.0) -> np.ndarray:
    """Flow field of Appendix B: v(r_t) = sum_j M'(r_t, r_j) lambda_j, tracer radius a.

    targets [nt,3]; pos [ns,3]; force [ns,3] or [k,ns,3].  Returns [nt,3] or [k,nt,3]."""
    targets = _f64(targets); pos = _f64(pos); force = _f64(force)
    nt, ns = targets.shape[0], pos.shape[0]
    assert targets.shape == (nt, 3) and pos.shape == (ns, 3)
    single = force.ndim == 2
    k = 1 if single else force.shape[0]
    f3 = np.ascontiguousarray(force.reshape(k, ns, 3))
    out = np.zeros((k, nt, 3))
    if nt > 0 and ns > 0:
        _load().rpy_oracle_flow(int(variant), nt, _dptr(targets), ns, _dptr(pos), k, _dptr(f3), float(a), float(eta),
                                _dptr(out))
    return out[0] if single else out


def subdivide(pos, force, template):
    """Appendix B: blob i -> small blobs at r_i + template[s], lambda' = lambda_i / n_sub."""
    pos = _f64(pos); force = _f64(force); template = _f64(template)
    ns = template.shape[0]
    sub_pos = (pos[:, None, :] + template[None, :, :]).reshape(-1, 3)
    sub_force = np.repeat(force, ns, axis=-2) / ns
    return sub_pos, sub_force


def num_threads() -> int:
    """Threads the oracle's row loop uses (OpenMP max threads)."""
    return int(_load().rpy_oracle_num_threads())
