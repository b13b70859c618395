"""Host-side pieces of bench.py that need no GPU: the parity figures, the per-pair work model, the DRAM-traffic
table read from profiles/, and that the kernel-coverage cases import cleanly."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402


def test_parity_of_reports_rel_l2_and_per_blob_max_and_gates_on_the_tolerance():
    rng = np.random.default_rng(0)
    ref = rng.standard_normal((2, 50, 3))
    full = rng.standard_normal((2, 400, 3))
    rows = np.sort(rng.choice(400, 50, replace=False))
    full[:, rows, :] = ref
    p = bench.parity_of(torch.from_numpy(full), ref, rows, "f64")
    assert p["rel_l2"] == 0.0 and p["per_blob_max"] == 0.0 and p["ok"] and p["rows"] == 50 and p["tol"] == 1e-12
    bad = full.copy()
    bad[1, rows[7], :] += 1e-3 * np.linalg.norm(ref[1, 7])          # one wrong blob among 100
    p = bench.parity_of(torch.from_numpy(bad), ref, rows, "f32")
    assert p["per_blob_max"] == pytest_approx(1e-3 * np.sqrt(3)) and 1e-5 < p["rel_l2"] < 1e-3 and not p["ok"]
    nan = full.copy(); nan[0, rows[0], 0] = np.nan
    assert not bench.parity_of(torch.from_numpy(nan), ref, rows, "f32")["ok"]
    # a single right-hand side given as [N, 3]
    p1 = bench.parity_of(torch.from_numpy(full[0]), ref[0], rows, "f64")
    assert p1["ok"] and p1["rows"] == 50


def pytest_approx(x):
    import pytest
    return pytest.approx(x, rel=1e-6)


def test_work_model_matches_the_expression_tree_counts():
    # wall 44 + 10k lane-ops per ordered pair (plain), (44 + 20k) / 2 symmetric; fp64 adds the roots
    assert bench.work_per_pair("f32", "wall", 1) == (54, 88)
    assert bench.work_per_pair("f32", "wall", 8) == (124, 214)
    assert bench.work_per_pair("f32", "wall", 1, symmetric=True) == (32.0, 53.0)
    assert bench.work_per_pair("f64", "wall", 1, symmetric=True) == (36.0, 59.0)
    assert bench.work_per_pair("f32", "free", 1, symmetric=True) == (16.0, 27.5)
    assert abs(bench.peak_tflops("f32") - 74.45) < 0.01 and abs(bench.peak_tflops("f64") - 37.22) < 0.01


def test_dram_traffic_table_is_read_from_the_committed_profile_summary():
    b, src = bench.ncu_traffic(3, "f32", "wall")
    assert b is not None and 1e6 < b < 1e9 and os.path.exists(os.path.join(ROOT, src))
    assert bench.ncu_traffic(1, "f32", "free") == (None, None)
    txt = open(os.path.join(ROOT, src)).read()               # the figure is the one in that summary
    rd = float(txt.split("`dram__bytes_read.sum` | ")[1].split(" |")[0]) * 1e6
    wr = float(txt.split("`dram__bytes_write.sum` | ")[1].split(" |")[0]) * 1e6
    assert abs(b - (rd + wr)) < 1.0


def test_kernel_cases_cover_the_documented_paths():
    sys.path.insert(0, os.path.join(ROOT, "tests"))
    import kernel_cases
    assert set(kernel_cases.CASES) == {"products_small", "symmetric_128", "symmetric_256", "rect_and_flow",
                                       "precond_all_paths", "solves"}
