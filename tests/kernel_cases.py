"""Cases that launch every kernel of the product at least once, on inputs that reach each code path; not a pytest file.

    python tests/kernel_cases.py [--only NAME,...]

Written for compute-sanitizer (memcheck, racecheck, synccheck on the double-buffered staging
and the rigid layer).  The tool is CLOSED on this GPU pool ("compute-sanitizer is closed on this pool and stays
closed", profiles/r2_sanitizer_closed.md), so the same cases run instead under the instrumentation of
tests/test_memory_safety_gpu.py: guard bands around every buffer the bindings allocate (a write outside a
buffer is seen), NaN-poisoned workspaces and outputs (a read of memory the call should have written first is
seen), and repeated runs compared bit for bit where the result is promised to be reproducible.

The cases: the plain all-pairs kernel (k = 1, 2, 8; both precisions; wall and free; a ragged last tile), the
symmetric kernel with 128-blob tiles (config 2) and with 256-blob tiles (N = 50,177: an odd tile count with a
one-blob last tile), row ranges, work shards, the rectangular product, the preconditioner build on its three
paths (register-resident sweep, shared-memory Cholesky, global-memory Cholesky), its application with one and
with four warps per body, K / K^T, and the fp64, fp32 and mixed GMRES solves incl. the batched one.  Results
are only checked to be finite here (parity is tests/test_*_gpu.py's job).
"""
from __future__ import annotations

import argparse
import os
import sys
import time

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1602_02170_b200 import binding, rigid, workloads  # noqa: E402


def dev(x, dt=torch.float64):
    return torch.from_numpy(np.ascontiguousarray(x)).to(dt).cuda()


def finite(t, what):
    assert bool(torch.isfinite(t).all()), what


def case_products_small():
    w = workloads.make(1)
    for dt in (torch.float64, torch.float32):
        pos, lam = dev(w.pos, dt), dev(w.force, dt)
        for fn in (binding.rpy_wall_matvec, binding.rpy_free_matvec):
            finite(fn(pos, lam), "cfg1")
            finite(fn(pos, lam, rows=(517, 300)), "cfg1 rows")
    rng = np.random.default_rng(0)
    n = 1000 + 77                                             # ragged last tile, k = 2 and 8
    pos = np.column_stack([rng.uniform(0, 30, n), rng.uniform(0, 30, n), rng.uniform(1.1, 8, n)])
    for k in (2, 8):
        lam = rng.standard_normal((k, n, 3))
        for dt in (torch.float64, torch.float32):
            finite(binding.rpy_wall_matvec(dev(pos, dt), dev(lam, dt)), f"k={k}")
            finite(binding.rpy_free_matvec(dev(pos, dt), dev(lam, dt)), f"k={k} free")


def case_symmetric_128():
    w = workloads.make(2)                                     # 15,000 blobs: symmetric kernel, 128-blob tiles
    for dt in (torch.float64, torch.float32):
        pos, lam = dev(w.pos, dt), dev(w.force, dt)
        for fn, sh in ((binding.rpy_wall_matvec, binding.rpy_wall_matvec_shard),
                       (binding.rpy_free_matvec, binding.rpy_free_matvec_shard)):
            finite(fn(pos, lam), "cfg2")
            finite(sh(pos, lam, 1, 3), "cfg2 shard")


def case_symmetric_256():
    n = 50177                                                 # 197 tiles of 256, the last one holds one blob
    rng = np.random.default_rng(1)
    pos = np.column_stack([rng.uniform(0, 110, n), rng.uniform(0, 110, n), rng.uniform(1.1, 9, n)])
    lam = rng.standard_normal((1, n, 3))
    for dt in (torch.float64, torch.float32):
        assert binding.rpy_matvec_launch_plan("f64" if dt == torch.float64 else "f32", n, 1, n)["tile_sources"] == 256
        finite(binding.rpy_wall_matvec(dev(pos, dt), dev(lam, dt)), "sym256")


def case_rect_and_flow():
    w = workloads.config2(n_bodies=40)
    rng = np.random.default_rng(2)
    targets = np.column_stack([rng.uniform(0, 100, 333), rng.uniform(0, 100, 333), rng.uniform(0.5, 9, 333)])
    for dt in (torch.float64, torch.float32):
        pos, lam = dev(w.pos, dt), dev(w.force, dt)
        finite(binding.rpy_wall_matvec_rect(dev(targets, dt), pos, lam), "rect")
        tmpl = dev(0.3 * workloads.shell_template(12), dt)
        sp, sf = binding.rpy_flow_subdivide(pos, lam, tmpl)
        finite(sp, "subdivide")
    assert binding.rpy_wall_count_below(dev(w.pos), 1.5) >= 0


def _mixed_bodies():
    pos, b, lam = workloads.mixed_suspension(1, 2)            # 15-, 42- and 60-blob bodies
    cyl = workloads.cylinder_template(n_rings=50, per_ring=6, radius=1.2, spacing=2.0) + np.array([300.0, 0.0, 4.0])
    pos = np.concatenate([pos, cyl])                          # + one 300-blob body: the global-memory path
    off = np.concatenate([b.offsets, [b.offsets[-1] + 300]])
    q = np.concatenate([b.q, cyl.mean(axis=0)[None, :]])
    return pos, q, off


def case_precond_all_paths():
    pos, q, off = _mixed_bodies()
    db = rigid.bodies(dev(pos), dev(q), off)
    for variant in ("wall", "free"):
        pc = rigid.rpy_rigid_precond_build(db, variant)
        x = torch.randn(db.n, dtype=torch.float64, device="cuda")
        finite(rigid.rpy_rigid_precond_apply(pc, x), "precond apply (4 warps per body)")
    U = torch.randn(db.n_bodies, 6, dtype=torch.float64, device="cuda")
    finite(rigid.rpy_rigid_K_apply(db, U), "K")
    finite(rigid.rpy_rigid_KT_apply(db, torch.randn(db.n_blobs, 3, dtype=torch.float64, device="cuda")), "KT")
    # one warp per body needs >= 2,048 bodies: single blobs
    n = 2100
    rng = np.random.default_rng(3)
    p1 = np.column_stack([rng.uniform(0, 900, n), rng.uniform(0, 900, n), rng.uniform(1.5, 4, n)])
    d1 = rigid.bodies(dev(p1), dev(p1), np.arange(n + 1))
    pc1 = rigid.rpy_rigid_precond_build(d1, "wall")
    finite(rigid.rpy_rigid_precond_apply(pc1, torch.randn(d1.n, dtype=torch.float64, device="cuda")), "precond apply (1 warp)")
    t = dev(workloads.boomerang_template())
    c = torch.rand(5, 3, dtype=torch.float64, device="cuda") * 50 + 20
    qt = torch.randn(5, 4, dtype=torch.float64, device="cuda")
    finite(rigid.rpy_rigid_blob_positions(t, c, qt), "blob positions")


def case_solves():
    w = workloads.config2(seed=2, n_bodies=300)               # 4,500 blobs: symmetric kernel inside the solve
    hb = workloads.bodies_of(w)
    db = rigid.bodies(dev(w.pos), dev(hb.q), hb.offsets)
    pc = rigid.rpy_rigid_precond_build(db, "wall")
    F = dev(hb.F)
    slip = dev(0.1 * np.random.default_rng(4).standard_normal(w.pos.shape))
    for prec, tol in (("f64", 1e-8), ("mixed", 1e-8), ("f32", 1e-5)):
        r = rigid.rpy_rigid_mobility_solve(db, pc, F, slip, "wall", tol=tol, matvec_prec=prec, restart=12)
        assert r["rel_resid"] <= 10 * tol, (prec, r["rel_resid"], r["n_iter"])
        finite(r["U"], "solve")
    r = rigid.rpy_rigid_mobility_solve(db, pc, F, slip, "wall", tol=1e-8, side_stream=False)
    assert r["rel_resid"] <= 1e-8
    small = workloads.config2(seed=3, n_bodies=30)            # plain kernel, batched solves with 3 and 8 right-hand sides
    sb = workloads.bodies_of(small)
    d2 = rigid.bodies(dev(small.pos), dev(sb.q), sb.offsets)
    pc2 = rigid.rpy_rigid_precond_build(d2, "wall")
    for k in (3, 8):
        Fk = torch.randn(k, d2.n_bodies, 6, dtype=torch.float64, device="cuda")
        for prec in ("f64", "mixed"):
            r = rigid.rpy_rigid_mobility_solve_batch(d2, pc2, Fk, None, "wall", tol=1e-8, matvec_prec=prec)
            assert max(r["rel_resid"]) <= 1e-7, (k, prec, r["rel_resid"])
    x = torch.randn(d2.n, dtype=torch.float64, device="cuda")
    for prec in ("f64", "f32"):
        finite(rigid.rpy_rigid_saddle_apply(d2, x, "wall", matvec_prec=prec), "saddle")


CASES = {
    "products_small": case_products_small,
    "symmetric_128": case_symmetric_128,
    "symmetric_256": case_symmetric_256,
    "rect_and_flow": case_rect_and_flow,
    "precond_all_paths": case_precond_all_paths,
    "solves": case_solves,
}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", default="", help="comma-separated case names (default: all)")
    args = ap.parse_args()
    names = [n for n in args.only.split(",") if n] or list(CASES)
    torch.cuda.set_device(0)
    binding.load_library()
    for n in names:
        t0 = time.perf_counter()
        CASES[n]()
        torch.cuda.synchronize()
        print(f"[kernel_cases] {n}: ok ({time.perf_counter() - t0:.1f} s)", flush=True)
    print("[kernel_cases] all cases ran", flush=True)


if __name__ == "__main__":
    main()
