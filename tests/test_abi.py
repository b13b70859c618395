"""Host-side checks of the C ABI that need no GPU: the library builds and loads, exports every
symbol include/rpy_matvec.h declares, validates arguments before touching CUDA, and its launch
planning / workspace arithmetic is consistent."""
import ctypes
import os
import re

import pytest

from paper_1602_02170_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "rpy_matvec.h")

F64, F32 = binding.RPY_PREC_F64, binding.RPY_PREC_F32_ACC64


def _declared_symbols():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(rpy_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    lib = binding.load_library()
    names = _declared_symbols()
    assert "rpy_wall_matvec" in names and "rpy_free_matvec" in names and len(names) >= 14
    for n in names:
        assert hasattr(lib, n), f"{n} declared in the header but not exported"
    assert set(names) == set(binding.SIGNATURES), "binding and header disagree on the symbol list"
    assert lib.rpy_abi_version() == 5


def test_no_torch_or_oracle_in_native_symbols():
    # the boundary is plain C: no C++-mangled torch symbols are needed to load it
    out = os.popen(f"nm -D --undefined-only {binding.library_path()}").read()
    assert "c10" not in out and "at::" not in out and "torch" not in out
    assert "rpy_oracle" not in out


def test_status_strings():
    for code, name in [(0, "RPY_OK"), (1, "RPY_ERR_NULL"), (2, "RPY_ERR_ARG"), (3, "RPY_ERR_ALIAS"),
                       (4, "RPY_ERR_WORKSPACE"), (5, "RPY_ERR_CUDA")]:
        assert binding.rpy_status_string(code).startswith(name)
    assert "unknown" in binding.rpy_status_string(99)


def test_workspace_bytes_monotone_and_zero_cases():
    w = binding.rpy_matvec_workspace_bytes
    assert w(F64, 0, 1) == 0 and w(F32, -5, 1) == 0 and w(F64, 100, 0) == 0
    for prec in (F64, F32):
        prev = 0
        for n in (1, 127, 128, 129, 2000, 15000, 172032, 1 << 20):
            b = w(prec, n, 1)
            assert b >= prev and b % 256 == 0 and b > 0
            prev = b
        assert w(prec, 2000, 8) > w(prec, 2000, 1)
        # n_rhs = 11 is processed as groups 8 + 2 + 1: the largest group sizes the workspace
        assert w(prec, 2000, 11) == w(prec, 2000, 8)
    # fp32 records are half the size of fp64 ones
    assert w(F32, 1 << 20, 1) < w(F64, 1 << 20, 1)
    # host scratch = inputs + output + workspace
    h = binding.rpy_matvec_host_scratch_bytes
    assert h(F64, 1000, 2) >= w(F64, 1000, 2) + 3 * 1000 * 3 * 8
    assert h(F32, 0, 1) == 0


@pytest.mark.parametrize("prec", [F64, F32])
@pytest.mark.parametrize("n,k", [(2000, 1), (15000, 1), (172032, 1), (1 << 20, 1), (172032, 8), (1, 1), (129, 3)])
def test_launch_plan_covers_all_sources_and_fits_workspace(prec, n, k):
    for rows in sorted({n, max(1, n // 2), 1}):
        p = binding.rpy_matvec_launch_plan(prec, n, k, rows)
        ts, tpc, nch = p["tile_sources"], p["targets_per_cta"], p["n_source_chunks"]
        kg = 8 if k >= 8 else 4 if k >= 4 else 2 if k >= 2 else 1
        w = 2 if prec == F32 else 1
        es = 4 if prec == F32 else 8
        rec = -(-((3 + 3 * kg) * w * es) // 16) * 16
        if p["symmetric"]:
            # symmetric kernel: one RHS, all rows, tiles of 128 (n < 50,000) or 256 blobs, chunks of the
            # tile distances 0..nt/2
            assert k == 1 and rows == n and n >= 1152 and ts == tpc == (128 if n < 50000 else 256)
            nt = -(-n // ts)
            count = nt // 2 + 1
            assert 1 <= nch <= count
            d_per_chunk = -(-count // nch)
            assert d_per_chunk * nch >= count and d_per_chunk * (nch - 1) < count
            assert p["n_ctas"] in (nt * nch, 2 * nt * nch, 4 * nt * nch)       # small problems: tile pairs cut in 2 or 4
            # records padded to whole tiles + the ONE double accumulator that receives both halves of every CTA's
            # work through fp64 atomics
            need = (nt * ts // w) * rec + n * 3 * 8
        else:
            n_tiles = -(-n // ts)
            assert 1 <= nch <= max(1, n_tiles)
            tiles_per_chunk = -(-n_tiles // nch)
            assert tiles_per_chunk * nch >= n_tiles                 # every tile is in some chunk
            assert tiles_per_chunk * (nch - 1) < n_tiles            # no empty chunk
            assert p["n_ctas"] == -(-rows // tpc) * nch
            # partial sums [chunk][k][rows][3] doubles + packed records fit the advertised workspace
            need = (-(-n // ts) * ts // w) * rec + nch * kg * rows * 3 * 8
        assert need <= binding.rpy_matvec_workspace_bytes(prec, n, k)
    if n >= 172032 and k == 1:
        full = binding.rpy_matvec_launch_plan(prec, n, k, n)
        assert full["symmetric"]
        assert full["n_ctas"] >= 148 * 4      # enough CTAs for several waves on 148 SMs
        assert not binding.rpy_matvec_launch_plan(prec, n, k, n - 1)["symmetric"]   # row ranges: plain kernel


def test_argument_errors_are_returned_before_any_cuda_work():
    lib = binding.load_library()
    one = ctypes.create_string_buffer(4096)
    p = ctypes.addressof(one)

    def call(prec=F64, n=4, k=1, pos=p, force=p + 1024, vel=p + 2048, a=1.0, eta=1.0, ws=p, wsb=0, fn="rpy_wall_matvec"):
        return getattr(lib, fn)(prec, n, k, pos, force, vel, a, eta, ws, wsb, None)

    for fn in ("rpy_wall_matvec", "rpy_free_matvec", "rpy_wall_matvec_host", "rpy_free_matvec_host"):
        assert call(n=-1, fn=fn) == 2
        assert call(k=0, fn=fn) == 2
        assert call(prec=7, fn=fn) == 2
        assert call(a=0.0, fn=fn) == 2 and call(a=-1.0, fn=fn) == 2 and call(a=float("nan"), fn=fn) == 2
        assert call(eta=0.0, fn=fn) == 2 and call(eta=float("inf"), fn=fn) == 2
        assert call(n=0, fn=fn) == 0                              # empty problem: OK, no-op
        assert call(pos=None, fn=fn) == 1 and call(force=None, fn=fn) == 1 and call(vel=None, fn=fn) == 1
        assert call(ws=None, fn=fn) == 1
        assert call(wsb=16, fn=fn) == 4                           # workspace too small
    assert call(n=(1 << 26) + 1) == 2
    big = binding.rpy_matvec_workspace_bytes(F64, 4, 1)
    aligned = (p + 255) // 256 * 256
    # misaligned workspace, then aliasing output
    assert call(ws=aligned + 8, wsb=big) == 4
    assert call(ws=aligned, wsb=big, vel=p, pos=p) == 3
    assert call(ws=aligned, wsb=big, vel=p + 1024 + 8, force=p + 1024) == 3
    # row ranges
    rows = lib.rpy_wall_matvec_rows
    assert rows(F64, 4, 1, -1, 2, p, p, p, 1.0, 1.0, p, 0, None) == 2
    assert rows(F64, 4, 1, 3, 2, p, p, p, 1.0, 1.0, p, 0, None) == 2
    assert rows(F64, 4, 1, 2, 0, p, p, p, 1.0, 1.0, p, 0, None) == 0
    assert lib.rpy_free_matvec_rows(F64, -4, 1, 0, 0, p, p, p, 1.0, 1.0, p, 0, None) == 2
    # count_below / plan argument checks
    assert lib.rpy_wall_count_below(F64, -1, p, 1.0, p, None) == 2
    assert lib.rpy_wall_count_below(F64, 4, p, 1.0, None, None) == 1
    assert lib.rpy_matvec_launch_plan(F64, 10, 1, 11, None, None, None, None, None) == 2
    assert lib.rpy_last_cuda_error() == 0


def test_python_binding_refuses_cpu_tensors_and_bad_shapes():
    import torch
    pos = torch.zeros(4, 3, dtype=torch.float64)
    lam = torch.zeros(4, 3, dtype=torch.float64)
    with pytest.raises((RuntimeError, ValueError)):
        binding.rpy_wall_matvec(pos, lam)            # no CUDA / CPU tensor: no fallback
    with pytest.raises((RuntimeError, ValueError)):
        binding.rpy_free_matvec(pos, lam)
    with pytest.raises(TypeError):
        binding._prec_of(torch.float16)
    with pytest.raises(ValueError):
        binding._shape_inputs(torch.zeros(4, 2), lam)
    with pytest.raises(ValueError):
        binding._shape_inputs(pos, torch.zeros(2, 5, 3, dtype=torch.float64))
    with pytest.raises(TypeError):
        binding._shape_inputs(pos, torch.zeros(4, 3, dtype=torch.float32))
    assert binding._shape_inputs(pos, torch.zeros(2, 4, 3, dtype=torch.float64)) == (4, 2, False)


def test_product_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_1602_02170_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "rpy_oracle" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_1602_02170_b200 import" not in txt and "import paper_1602_02170_b200" not in txt


def test_bench_aids_are_a_library_of_their_own():
    """The measurement aids (FMA-chain probes, per-kernel events) are not part of the product ABI: they
    live in bench_aids/ with their own header, build against the product and export what that header declares."""
    import bench_aids
    lib = bench_aids.load_library()
    hdr = re.sub(r"/\*.*?\*/", "", open(os.path.join(ROOT, "bench_aids", "rpy_bench_aids.h")).read(), flags=re.S)
    names = sorted(set(re.findall(r"\b(rpy_bench_[a-z0-9_]+)\s*\(", hdr)))
    assert names == ["rpy_bench_coissue_probe", "rpy_bench_matvec_phases", "rpy_bench_operand_probe", "rpy_bench_pipe_probe"]
    for n in names:
        assert hasattr(lib, n)
    product = binding.load_library()
    for n in ("rpy_pipe_peak_probe", "rpy_matvec_phases", "rpy_bench_pipe_probe"):
        assert not hasattr(product, n), f"{n} is a measurement aid and must not be exported by the product"
    assert "probe" not in open(HEADER).read()
    # argument checks reach no CUDA call
    one = ctypes.c_void_p(256)
    assert lib.rpy_bench_pipe_probe(9, 10, one, None, None, None) == 2
    assert lib.rpy_bench_pipe_probe(0, 10, None, None, None, None) == 1
    assert lib.rpy_bench_coissue_probe(9, 10, 10, 0, one, None, None, None, None) == 2
    assert lib.rpy_bench_operand_probe(8, 4, 10, one, None, None, None) == 2
    assert lib.rpy_bench_operand_probe(0, 5, 10, one, None, None, None) == 2
    assert lib.rpy_bench_operand_probe(0, 4, 10, None, None, None, None) == 1
    assert lib.rpy_bench_matvec_phases(1, 0, 10, 1, one, one, one, 1.0, 1.0, one, 1 << 20, None, None) == 1


# ------------------------------------------------------------------ include/rpy_rigid.h
RIGID_HEADER = os.path.join(ROOT, "include", "rpy_rigid.h")


def test_rigid_header_symbols_are_exported_and_bound():
    from paper_1602_02170_b200 import rigid
    src = re.sub(r"/\*.*?\*/", "", open(RIGID_HEADER).read(), flags=re.S)
    names = sorted(set(re.findall(r"\b(rpy_rigid_[a-z0-9_A-Z]+)\s*\(", src)))
    lib = rigid._lib()
    assert len(names) == 13
    for n in names:
        assert hasattr(lib, n), f"{n} declared in rpy_rigid.h but not exported"
    assert set(names) == set(rigid.SIGNATURES)


def test_rigid_host_arithmetic_and_argument_checks():
    import numpy as np
    from paper_1602_02170_b200 import rigid
    lib = rigid._lib()
    pb = rigid.rpy_rigid_precond_bytes
    assert pb([0, 15, 30]) > 2 * 45 * 45 * 8 and pb([0, 15, 30]) % 256 == 0
    assert pb([0, 15, 57, 117]) > pb([0, 15, 57])
    assert pb([1, 15]) == 0 and pb([0, 5, 5]) == 0 and pb([0, 1200]) == 0     # bad start, empty body, body too large
    w = rigid.rpy_rigid_solve_workspace_bytes
    n, nb = 15000, 1000
    assert w("f64", n, nb, 60) >= 65 * (3 * n + 6 * nb) * 8
    assert w("f32", n, nb, 60) > 0 and w("f64", n, nb, 0) == 0 and w("f64", n, nb, 129) == 0 and w("f64", n, 0, 10) == 0
    assert w("f64", n, nb, 30) < w("f64", n, nb, 60)
    # argument errors are detected before any CUDA call (works without a GPU)
    one = ctypes.c_void_p(256)
    assert lib.rpy_rigid_K_apply(10, 2, None, one, one, one, 1.0, 0.0, one, None) == 1
    assert lib.rpy_rigid_K_apply(-1, 2, one, one, one, one, 1.0, 0.0, one, None) == 2
    assert lib.rpy_rigid_KT_apply(10, 11, one, one, one, one, 1.0, 0.0, one, None) == 2
    assert lib.rpy_rigid_KT_apply(10, 2, one, one, one, one, float("nan"), 0.0, one, None) == 2
    off = (ctypes.c_int64 * 3)(0, 4, 10)
    assert lib.rpy_rigid_precond_build(1, 10, 2, one, one, off, -1.0, 1.0, one, 1 << 20, None) == 2
    assert lib.rpy_rigid_precond_build(1, 11, 2, one, one, off, 1.0, 1.0, one, 1 << 20, None) == 2
    assert lib.rpy_rigid_precond_build(1, 10, 2, one, one, off, 1.0, 1.0, one, 16, None) == 4
    assert lib.rpy_rigid_precond_apply(10, 2, one, one, one, None) == 3            # in aliases out
    n_it, rr = ctypes.c_int(), ctypes.c_double()
    args = lambda tol, restart, ws, ext=None: (1, 0, 10, 2, one, one, one, one, None, 1.0, 1.0, one, tol, restart, 50, one, one,
                                               None, ctypes.byref(n_it), ctypes.byref(rr), one, ws, None, ext)
    assert lib.rpy_rigid_mobility_solve(*args(-1.0, 10, 1 << 30)) == 2
    assert lib.rpy_rigid_mobility_solve(*args(1e-8, 500, 1 << 30)) == 2
    assert lib.rpy_rigid_mobility_solve(*args(1e-8, 10, 64)) == 4
    # the optional extras: a share of the product needs a reduction hook, one right-hand side and the symmetric kernel
    big = 1 << 30
    ext = rigid.SolveExt(); ext.shard, ext.n_shards = 2, 2
    assert lib.rpy_rigid_mobility_solve(*args(1e-8, 10, big, ctypes.byref(ext))) == 2      # shard >= n_shards
    ext.shard = 0
    assert lib.rpy_rigid_mobility_solve(*args(1e-8, 10, big, ctypes.byref(ext))) == 1      # no hook
    ext.reduce = rigid.REDUCE_FN(lambda c, p, n, s: 0)
    assert lib.rpy_rigid_mobility_solve(*args(1e-8, 10, big, ctypes.byref(ext))) == 2      # 10 blobs: no symmetric kernel


def test_rigid_and_sharded_bindings_refuse_cpu_tensors():
    """No CPU fallback anywhere: the rigid layer, the work shards and the rectangular product raise on
    host tensors (and on a box without CUDA) instead of computing something else."""
    import torch
    from paper_1602_02170_b200 import rigid
    pos = torch.zeros(6, 3, dtype=torch.float64); q = torch.zeros(2, 3, dtype=torch.float64)
    with pytest.raises((RuntimeError, ValueError)):
        rigid.bodies(pos, q, [0, 3, 6])
    with pytest.raises((RuntimeError, ValueError)):
        rigid.rpy_rigid_blob_positions(pos, q, torch.zeros(2, 4, dtype=torch.float64))
    lam = torch.zeros(6, 3, dtype=torch.float64)
    with pytest.raises((RuntimeError, ValueError)):
        binding.rpy_wall_matvec_shard(pos, lam, 0, 2)
    with pytest.raises((RuntimeError, ValueError)):
        binding.rpy_free_matvec_rect(pos, pos, lam)
    with pytest.raises((RuntimeError, ValueError)):
        binding.rpy_flow_subdivide(pos, lam, torch.zeros(3, 3, dtype=torch.float64))
    # host-side argument checks of the sharded / rectangular entry points (no CUDA call is reached)
    lib = rigid._lib()                      # the same CDLL, with the rigid signatures set
    one = ctypes.c_void_p(256)
    assert lib.rpy_wall_matvec_shard(F64, 10, 1, 2, 2, one, one, one, 1.0, 1.0, one, 1 << 20, None) == 2    # shard >= n_shards
    assert lib.rpy_wall_matvec_shard(F64, 10, 1, 0, 0, one, one, one, 1.0, 1.0, one, 1 << 20, None) == 2
    assert lib.rpy_free_matvec_shard(F64, 10, 1, 0, 2, one, one, None, 1.0, 1.0, one, 1 << 20, None) == 1
    assert lib.rpy_wall_matvec_rect(F64, 5, 10, 1, one, one, one, one, 1.0, 1.0, one, 16, None) == 4
    assert lib.rpy_wall_matvec_rect(F64, -1, 10, 1, one, one, one, one, 1.0, 1.0, one, 16, None) == 2
    assert binding.rpy_matvec_rect_workspace_bytes(F64, 100, 200, 1) > binding.rpy_matvec_workspace_bytes(F64, 200, 1)
    assert lib.rpy_flow_subdivide(F64, 10, 1, 0, one, one, one, one, one, None) == 2
    assert lib.rpy_rigid_solve_batch_workspace_bytes(F64, 1000, 10, 30, 9) == 0
    assert lib.rpy_rigid_solve_batch_workspace_bytes(F64, 1000, 10, 30, 8) > 8 * 31 * (3000 + 60) * 8
