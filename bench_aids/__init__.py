"""Measurement aids of ``bench.py`` (C ABI: ``bench_aids/rpy_bench_aids.h``) -- not part of the product.

    python -m bench_aids [--force]      builds bench_aids/librpy_bench_aids.so with nvcc for sm_100a

* ``pipe_probe``      FMA-chain rates of the FP32 / FP64 / MUFU pipes (the ALU roofline's denominator)
* ``operand_probe``   what an FFMA2 / DFMA costs by the form of its operands (register pairs, reuse, scalar, immediate)
* ``coissue_probe``   DFMA chains beside FFMA2 chains on every SM
* ``matvec_phases``   the product (``librpy_matvec.so``) with CUDA events around each of its kernels

Argument marshalling only.  The library links against the product library for ``matvec_phases`` (an
internal, non-ABI entry: ``csrc/rpy_internal.h``); the product never loads this one.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import sys
from pathlib import Path
from typing import Optional

HERE = Path(__file__).resolve().parent
LIB = HERE / "librpy_bench_aids.so"
SOURCES = [HERE / "rpy_bench_aids.cu"]
DEPS = SOURCES + [HERE / "rpy_bench_aids.h"]

_lib = None


def _product_build():
    from paper_1602_02170_b200 import build as product_build
    return product_build


def needs_build() -> bool:
    if not LIB.exists():
        return True
    t = LIB.stat().st_mtime
    pb = _product_build()
    return any(d.stat().st_mtime > t for d in DEPS) or (pb.LIB.exists() and pb.LIB.stat().st_mtime > t)


def build(force: bool = False) -> Path:
    pb = _product_build()
    product = pb.build(force=False)
    if not force and not needs_build():
        return LIB
    tmp = LIB.with_suffix(f".so.tmp{os.getpid()}")
    cmd = [pb.nvcc(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
           "-Xcompiler", "-fPIC", "-shared", "-I", str(pb.INCLUDE), "-o", str(tmp), *map(str, SOURCES),
           "-L", str(product.parent), f"-l:{product.name}",
           "-Xlinker", "-rpath", "-Xlinker", "$ORIGIN/../" + product.parent.name]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building librpy_bench_aids.so")
    os.replace(tmp, LIB)
    return LIB


def load_library(rebuild: bool = False):
    global _lib
    if _lib is None or rebuild:
        from paper_1602_02170_b200 import binding
        binding.load_library()                          # the product first: its symbols resolve ours
        ctypes.CDLL(binding.library_path(), mode=ctypes.RTLD_GLOBAL)
        lib = ctypes.CDLL(str(build(force=rebuild)))
        vp, i64, cint, dbl, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        fp, dp = ctypes.POINTER(ctypes.c_float), ctypes.POINTER(ctypes.c_double)
        lib.rpy_bench_pipe_probe.restype = cint
        lib.rpy_bench_pipe_probe.argtypes = [cint, cint, vp, fp, dp, vp]
        lib.rpy_bench_operand_probe.restype = cint
        lib.rpy_bench_operand_probe.argtypes = [cint, cint, cint, vp, fp, dp, vp]
        lib.rpy_bench_coissue_probe.restype = cint
        lib.rpy_bench_coissue_probe.argtypes = [cint, cint, cint, cint, vp, fp, dp, dp, vp]
        lib.rpy_bench_matvec_phases.restype = cint
        lib.rpy_bench_matvec_phases.argtypes = [cint, cint, i64, cint, vp, vp, vp, dbl, dbl, vp, sz, vp, ctypes.POINTER(vp)]
        _lib = lib
    return _lib


def pipe_probe(kind: int, iters: int = 4096, device=None) -> dict:
    """{'ms', 'fma', 'gfma_per_s'} for kind 0 FFMA, 1 FFMA2, 2 DFMA, 3 MUFU.RSQ, 4/5 three-register forms."""
    import torch
    lib = load_library()
    device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    sink = torch.zeros(8, dtype=torch.float64, device=device)
    ms, cnt = ctypes.c_float(), ctypes.c_double()
    with torch.cuda.device(device):
        stream = torch.cuda.current_stream(device).cuda_stream
        rc = lib.rpy_bench_pipe_probe(int(kind), int(iters), sink.data_ptr(), ctypes.byref(ms), ctypes.byref(cnt), stream)
    if rc != 0:
        raise RuntimeError(f"rpy_bench_pipe_probe failed with status {rc}")
    return {"ms": ms.value, "fma": cnt.value, "gfma_per_s": cnt.value / (ms.value * 1e-3) / 1e9}


OPERAND_FORMS = {0: "ffma2_two_pairs", 1: "ffma2_two_pairs_imm", 2: "ffma2_three_pairs", 3: "ffma2_three_pairs_one_reused",
                 4: "ffma2_two_pairs_one_scalar", 5: "dfma_two_regs", 6: "dfma_three_regs", 7: "dfma_three_regs_one_reused"}


def operand_probe(kind: int, ctas_per_sm: int = 4, iters: int = 8192, device=None) -> dict:
    """Lane operations per second of an FFMA2 (kind 0-4) or DFMA (5-7) stream by operand form (OPERAND_FORMS)."""
    import torch
    lib = load_library()
    device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    scratch = torch.zeros(8 + 8 * 128 * 4 * 12, dtype=torch.uint8, device=device)
    ms, cnt = ctypes.c_float(), ctypes.c_double()
    with torch.cuda.device(device):
        stream = torch.cuda.current_stream(device).cuda_stream
        rc = lib.rpy_bench_operand_probe(int(kind), int(ctas_per_sm), int(iters), scratch.data_ptr(), ctypes.byref(ms),
                                         ctypes.byref(cnt), stream)
    if rc != 0:
        raise RuntimeError(f"rpy_bench_operand_probe failed with status {rc}")
    return {"form": OPERAND_FORMS[int(kind)], "ms": ms.value, "tlaneops_per_s": cnt.value / (ms.value * 1e-3) / 1e12}


def coissue_probe(n64_per_sm: int, iters32: int, iters64: int, three_reg: bool = False, device=None) -> dict:
    """Lane operations per second of FFMA2 chains and of DFMA chains running side by side on every SM."""
    import torch
    lib = load_library()
    device = torch.device("cuda", torch.cuda.current_device()) if device is None else torch.device(device)
    scratch = torch.zeros(2048, dtype=torch.uint8, device=device)
    ms, o32, o64 = ctypes.c_float(), ctypes.c_double(), ctypes.c_double()
    with torch.cuda.device(device):
        stream = torch.cuda.current_stream(device).cuda_stream
        rc = lib.rpy_bench_coissue_probe(int(n64_per_sm), int(iters32), int(iters64), int(bool(three_reg)),
                                         scratch.data_ptr(), ctypes.byref(ms), ctypes.byref(o32), ctypes.byref(o64), stream)
    if rc != 0:
        raise RuntimeError(f"rpy_bench_coissue_probe failed with status {rc}")
    t = ms.value * 1e-3
    return {"ms": ms.value, "f32_tlaneops_per_s": o32.value / t / 1e12, "f64_tlaneops_per_s": o64.value / t / 1e12}


def matvec_phases(variant: str, pos, force, a: float = 1.0, eta: float = 1.0, *, out=None,
                  workspace: Optional["torch.Tensor"] = None, events=None):
    """Whole-matrix product with four CUDA events recorded around its phases.

    Returns (u, events); after synchronising, ``events[1].elapsed_time(events[2])`` is the duration of
    the all-pairs kernel in ms."""
    import torch
    from paper_1602_02170_b200 import binding
    lib = load_library()
    if not (pos.is_cuda and force.is_cuda and pos.is_contiguous() and force.is_contiguous() and pos.dtype == force.dtype):
        raise ValueError("pos and force must be contiguous CUDA tensors of one dtype")
    n = pos.shape[0]
    single = force.dim() == 2
    k = 1 if single else force.shape[0]
    prec = 0 if pos.dtype == torch.float64 else 1
    if out is None:
        out = torch.empty((n, 3) if single else (k, n, 3), dtype=pos.dtype, device=pos.device)
    need = binding.rpy_matvec_workspace_bytes(prec, n, k)
    if workspace is None:
        workspace = torch.empty(max(need, 1), dtype=torch.uint8, device=pos.device)
    with torch.cuda.device(pos.device):
        stream0 = torch.cuda.current_stream(pos.device)
        if events is None:
            events = [torch.cuda.Event(enable_timing=True) for _ in range(4)]
            for e in events:
                e.record(stream0)         # torch creates the cudaEvent_t lazily, on first record
        handles = (ctypes.c_void_p * 4)(*[e.cuda_event for e in events])
        rc = lib.rpy_bench_matvec_phases(1 if variant == "wall" else 0, prec, n, k, pos.data_ptr(), force.data_ptr(),
                                         out.data_ptr(), float(a), float(eta), workspace.data_ptr(), int(workspace.numel()),
                                         stream0.cuda_stream, handles)
    if rc != 0:
        raise RuntimeError(f"rpy_bench_matvec_phases: {binding.rpy_status_string(rc)}")
    return out, events

