"""CUDA path vs the CPU oracle, element by element, through the C ABI (-m gpu).

Tolerances are north_star's: relative L2 error <= 1e-12 for the fp64 path and <= 1e-5 for the
fp32 path with fp64 accumulation, over all 3 N k output components (sampled rows at the full
sizes: the oracle computes each sampled row against ALL sources).  For the fp32 path the oracle
consumes exactly the values that cross the boundary: the fp32-rounded positions and forces
promoted to double (reading A8).  The per-blob maximum max_i |du_i| / |u_i| is gated too,
loosely (PB_TOL): a blob whose velocity nearly cancels may lose digits relative to ITS OWN magnitude
without the method being wrong, but a single wrong row among 10^5 must not hide inside the norm.
"""
import numpy as np
import pytest
import torch

import oracle
from paper_1602_02170_b200 import binding, workloads

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
PB_TOL = {"f64": 1e-11, "f32": 2e-4}         # per-blob gate (A11); measured maxima: 4e-14 and 3e-5
DT = {"f64": torch.float64, "f32": torch.float32}
NP = {"f64": np.float64, "f32": np.float32}
ORACLE_VARIANT = {"wall": oracle.WALL, "free": oracle.FREE}
GPU_FN = {"wall": binding.rpy_wall_matvec, "free": binding.rpy_free_matvec}


def rel_l2(u, ref):
    return float(np.linalg.norm((u - ref).ravel()) / np.linalg.norm(ref.ravel()))


def per_blob_max(u, ref):
    num = np.linalg.norm(u - ref, axis=-1)
    den = np.linalg.norm(ref, axis=-1)
    return float((num / np.maximum(den, 1e-300)).max())


def run_case(pos64, force64, prec, variant, a=1.0, eta=1.0, rows=None, gpu_rows=None):
    """Returns (gpu result as float64 numpy [k,nrows,3], oracle result) on the same inputs."""
    pos_b = pos64.astype(NP[prec])        # the values that cross the boundary
    force_b = force64.astype(NP[prec])
    d_pos = torch.from_numpy(pos_b).cuda()
    d_force = torch.from_numpy(force_b).cuda()
    u = GPU_FN[variant](d_pos, d_force, a, eta, rows=gpu_rows)
    torch.cuda.synchronize()
    u = u.cpu().numpy().astype(np.float64)
    if gpu_rows is not None:
        orows = np.arange(gpu_rows[0], gpu_rows[0] + gpu_rows[1], dtype=np.int64)
        ref = oracle.matvec(ORACLE_VARIANT[variant], pos_b.astype(np.float64), force_b.astype(np.float64), a, eta, rows=orows)
    else:
        ref = oracle.matvec(ORACLE_VARIANT[variant], pos_b.astype(np.float64), force_b.astype(np.float64), a, eta, rows=rows)
        if rows is not None:
            u = u[..., rows, :]
    return u, ref


def check(u, ref, prec, what):
    e = rel_l2(u, ref)
    pb = per_blob_max(u, ref)
    print(f"{what}: prec={prec} rel-L2={e:.3e} per-blob-max={pb:.3e}")
    assert np.isfinite(u).all()
    assert e <= TOL[prec], f"{what}: rel-L2 {e:.3e} > {TOL[prec]}"
    assert pb <= PB_TOL[prec], f"{what}: per-blob max {pb:.3e} > {PB_TOL[prec]}"


# ------------------------------------------------------------------ small cases, every row
@pytest.mark.parametrize("variant", ["wall", "free"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config1_all_rows(prec, variant):
    w = workloads.make(1)
    u, ref = run_case(w.pos, w.force, prec, variant)
    check(u, ref, prec, f"cfg1 {variant}")


@pytest.mark.parametrize("variant", ["wall", "free"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [1, 2, 3, 63, 64, 65, 127, 128, 129, 257, 1000])
def test_ragged_sizes(prec, variant, n):
    """Sizes around the tile (64 / 128 sources) and CTA (128 targets) edges; a != 1, eta != 1."""
    rng = np.random.default_rng(100 + n)
    pos = np.column_stack([rng.uniform(0, 12, n), rng.uniform(0, 12, n), rng.uniform(0.7 * 1.1, 6, n)])
    lam = rng.standard_normal((1, n, 3))
    u, ref = run_case(pos, lam, prec, variant, a=0.7, eta=1.3)
    check(u, ref, prec, f"ragged n={n} {variant}")


@pytest.mark.parametrize("variant", ["wall", "free"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("k", [2, 3, 4, 8, 11])
def test_multi_rhs(prec, variant, k):
    rng = np.random.default_rng(200 + k)
    n = 777
    pos = np.column_stack([rng.uniform(0, 30, n), rng.uniform(0, 30, n), rng.uniform(1.1, 8, n)])
    lam = rng.standard_normal((k, n, 3))
    u, ref = run_case(pos, lam, prec, variant)
    assert u.shape == (k, n, 3)
    check(u, ref, prec, f"k={k} {variant}")
    for s in range(k):                       # every right-hand side on its own
        assert rel_l2(u[s], ref[s]) <= TOL[prec]


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_config2_boomerangs_all_rows(prec):
    w = workloads.make(2)
    u, ref = run_case(w.pos, w.force, prec, "wall")
    check(u, ref, prec, "cfg2 wall")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_small_shell_lattice_all_rows(prec):
    """Config-3 recipe with 8x8 shells (2,688 blobs): intra-body overlapping pairs."""
    w = workloads.config3(side=8)
    u, ref = run_case(w.pos, w.force, prec, "wall")
    check(u, ref, prec, "cfg3-small wall")
    w5 = workloads.config5(side=8)
    for variant in ("wall", "free"):
        u, ref = run_case(w5.pos, w5.force, "f32", variant)
        check(u, ref, "f32", f"cfg5-small {variant}")


# ------------------------------------------------------------------ symmetric kernel (n >= 1,152, k = 1, all rows)
@pytest.mark.parametrize("variant", ["wall", "free"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [1152, 1153, 1999, 2048, 3584, 3585, 6144, 6145, 6400 + 77, 7 * 1024 + 1])
def test_symmetric_kernel_tile_edges(prec, variant, n):
    """The path that uses M_ij = M_ji^T, 128-blob tiles (n < 50,000): even tile count (16, 28, 48: the
    half-distance case), odd (9, 29, 49), ragged last tile, tile pairs cut into two (fp32) or four (fp64)
    parts of the source tile where one CTA per tile pair would not fill the chip (n < ~4,000); dense enough
    that overlapping pairs (r < 2a) occur across tiles."""
    plan = binding.rpy_matvec_launch_plan(prec, n, 1, n)
    assert plan["symmetric"] and plan["tile_sources"] == 128
    assert not binding.rpy_matvec_launch_plan(prec, 1151, 1, 1151)["symmetric"]
    rng = np.random.default_rng(300 + n)
    side = 40.0
    pos = np.column_stack([rng.uniform(0, side, n), rng.uniform(0, side, n), rng.uniform(1.1, 9, n)])
    lam = rng.standard_normal((1, n, 3))
    u, ref = run_case(pos, lam, prec, variant, a=0.9, eta=1.7)
    check(u, ref, prec, f"symmetric n={n} {variant}")


@pytest.mark.parametrize("variant", ["wall", "free"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [50176, 50177, 50000 + 3 * 256 + 19])
def test_symmetric_kernel_256_blob_tiles_sampled_rows(prec, variant, n):
    """n >= 50,000: 256-blob tiles -- even tile count (196), odd with a one-blob last tile (197), ragged
    (199); the oracle computes a seeded sample of rows against all sources."""
    plan = binding.rpy_matvec_launch_plan(prec, n, 1, n)
    assert plan["symmetric"] and plan["tile_sources"] == 256
    rng = np.random.default_rng(500 + n)
    side = 110.0
    pos = np.column_stack([rng.uniform(0, side, n), rng.uniform(0, side, n), rng.uniform(1.1, 9, n)])
    lam = rng.standard_normal((1, n, 3))
    rows = np.unique(np.concatenate([workloads.sample_rows(n, 700, seed=n), np.arange(n - 300, n), np.arange(0, 40)]))
    u, ref = run_case(pos, lam, prec, variant, rows=rows)
    check(u, ref, prec, f"symmetric-256 n={n} {variant}")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_symmetric_and_plain_kernels_agree(prec):
    """Same inputs through the symmetric kernel (all rows) and the plain kernel (two row ranges)."""
    w = workloads.config2(n_bodies=600)          # 9,000 blobs
    n = w.n_blobs
    pos = torch.from_numpy(w.pos.astype(NP[prec])).cuda(); lam = torch.from_numpy(w.force.astype(NP[prec])).cuda()
    assert binding.rpy_matvec_launch_plan(prec, n, 1, n)["symmetric"]
    assert not binding.rpy_matvec_launch_plan(prec, n, 1, n // 2)["symmetric"]
    for fn in (binding.rpy_wall_matvec, binding.rpy_free_matvec):
        full = fn(pos, lam)
        halves = torch.cat([fn(pos, lam, rows=(0, n // 2)), fn(pos, lam, rows=(n // 2, n - n // 2))], dim=1)
        e = rel_l2(full.cpu().numpy().astype(np.float64), halves.cpu().numpy().astype(np.float64))
        print(f"symmetric vs plain kernel, {prec}: rel-L2 {e:.3e}")
        assert e <= (1e-13 if prec == "f64" else 2e-6)
        # the symmetric path is reproducible to rounding of the fp64 atomics, not bit for bit
        again = fn(pos, lam)
        assert rel_l2(again.cpu().numpy().astype(np.float64), full.cpu().numpy().astype(np.float64)) <= 1e-14


# ------------------------------------------------------------------ degenerate cases
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_single_blob_and_coincident_blobs(prec):
    # one blob: u = M_ii lambda (PAPER.md:146 + wall self term)
    u, ref = run_case(np.array([[3.0, 4.0, 2.0]]), np.array([[[1.0, 2.0, 3.0]]]), prec, "wall")
    check(u, ref, prec, "single blob")
    # two coincident distinct blobs (r = 0 between different blobs) and a pair exactly at r = 2a
    pos = np.array([[0.0, 0.0, 2.0], [0.0, 0.0, 2.0], [2.0, 0.0, 2.0], [7.0, 1.0, 1.5]])
    lam = np.array([[[1.0, -2.0, 0.5], [0.3, 0.1, -1.0], [2.0, 1.0, 1.0], [-1.0, 0.0, 1.0]]])
    for variant in ("wall", "free"):
        u, ref = run_case(pos, lam, prec, variant)
        check(u, ref, prec, f"coincident/r=2a {variant}")


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("n", [700, 4000])
def test_dense_cluster_where_most_pairs_overlap(prec, n):
    """The r <= 2a branch of Eq. (9) is rare in the configured workloads (it sits behind a warp vote); here it is the rule:
    blobs packed into a box 3a wide (every pair overlaps) or 12a wide (most warp steps take the vote), plain kernel (n = 700)
    and symmetric kernel (n = 4,000); two blobs coincide."""
    rng = np.random.default_rng(31)
    side = 3.0 if n == 700 else 12.0
    pos = np.column_stack([rng.uniform(0, side, n), rng.uniform(0, side, n), rng.uniform(1.1, 1.1 + side, n)])
    pos[n // 2] = pos[n // 3]
    lam = rng.standard_normal((1, n, 3))
    for variant in ("wall", "free"):
        u, ref = run_case(pos, lam, prec, variant)
        check(u, ref, prec, f"dense cluster n={n} {variant}")


@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_blobs_overlapping_the_wall_formula_as_is(prec):
    """Reading A6: for z < a the tensor is not meaningful but it is evaluated as written, with no
    clamping inside the library: blobs at heights 0.3a .. a (and some below 0.05a) give the oracle's numbers."""
    rng = np.random.default_rng(32)
    n = 900
    pos = np.column_stack([rng.uniform(0, 40, n), rng.uniform(0, 40, n), rng.uniform(0.3, 1.0, n)])
    pos[:20, 2] = rng.uniform(0.01, 0.05, 20)
    lam = rng.standard_normal((2, n, 3))
    u, ref = run_case(pos, lam, prec, "wall")
    check(u, ref, prec, "blobs overlapping the wall")


def test_empty_and_zero_force():
    e = torch.zeros(0, 3, dtype=torch.float64, device="cuda")
    assert binding.rpy_wall_matvec(e, e).shape == (0, 3)
    assert binding.rpy_free_matvec(e, torch.zeros(2, 0, 3, dtype=torch.float64, device="cuda")).shape == (2, 0, 3)
    w = workloads.make(1)
    pos = torch.from_numpy(w.pos).cuda()
    u = binding.rpy_wall_matvec(pos, torch.zeros_like(pos))
    assert torch.count_nonzero(u).item() == 0


def test_fp64_result_is_deterministic_and_workspace_reuse():
    w = workloads.config1(n=1000)                   # below 1,152 blobs: the plain kernel
    pos = torch.from_numpy(w.pos).cuda(); lam = torch.from_numpy(w.force).cuda()
    ws = torch.empty(binding.rpy_matvec_workspace_bytes("f64", w.n_blobs, 1), dtype=torch.uint8, device="cuda")
    out = torch.empty_like(lam)
    u1 = binding.rpy_wall_matvec(pos, lam, workspace=ws).clone()
    u2 = binding.rpy_wall_matvec(pos, lam, workspace=ws, out=out)
    assert u2.data_ptr() == out.data_ptr()
    assert torch.equal(u1, u2)                      # chunk partials are added in a fixed order
    # a workspace that is one byte short is refused
    with pytest.raises(binding.RpyError) as ei:
        binding.rpy_wall_matvec(pos, lam, workspace=ws[:-256])
    assert ei.value.status == 4
    with pytest.raises(binding.RpyError) as ei:
        binding.rpy_wall_matvec(pos, lam[0], out=pos)     # output aliases an input
    assert ei.value.status == 3


def test_symmetry_and_positivity_of_the_gpu_operator():
    """Properties that hold at any size: l2.(M l1) = l1.(M l2), l.(M l) > 0."""
    w = workloads.config2(n_bodies=200)
    pos = torch.from_numpy(w.pos).cuda()
    rng = np.random.default_rng(5)
    l = torch.from_numpy(rng.standard_normal((2, w.n_blobs, 3))).cuda()
    for fn in (binding.rpy_wall_matvec, binding.rpy_free_matvec):
        u = fn(pos, l)
        a = torch.sum(l[1] * u[0]).item(); b = torch.sum(l[0] * u[1]).item()
        assert a == pytest.approx(b, rel=1e-11)
        assert torch.sum(l[0] * u[0]).item() > 0 and torch.sum(l[1] * u[1]).item() > 0


# ------------------------------------------------------------------ row-sharded and host forms
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_row_range_calls_match_full_result(prec):
    w = workloads.config2(n_bodies=150)          # 2,250 blobs
    n = w.n_blobs
    pos = torch.from_numpy(w.pos.astype(NP[prec])).cuda(); lam = torch.from_numpy(w.force.astype(NP[prec])).cuda()
    full = binding.rpy_wall_matvec(pos, lam)
    for rb, rc in [(0, 1), (0, 1000), (1000, 1250), (n - 1, 1), (517, 3)]:
        part = binding.rpy_wall_matvec(pos, lam, rows=(rb, rc))
        assert part.shape == (1, rc, 3)
        ref = full[:, rb:rb + rc]
        # the full product comes from the symmetric kernel, the row range from the plain one
        d = float((part.double() - ref.double()).norm() / ref.double().norm())
        assert d <= (1e-13 if prec == "f64" else 2e-6), d
    u, ref = run_case(w.pos, w.force, prec, "wall", gpu_rows=(700, 900))
    check(u, ref, prec, "row range vs oracle")


@pytest.mark.parametrize("variant", ["wall", "free"])
@pytest.mark.parametrize("prec", ["f64", "f32"])
def test_host_buffer_call(prec, variant):
    w = workloads.config1(n=1500, k=2)
    pos = torch.from_numpy(w.pos.astype(NP[prec])); lam = torch.from_numpy(w.force.astype(NP[prec]))
    fn = binding.rpy_wall_matvec_host if variant == "wall" else binding.rpy_free_matvec_host
    u = fn(pos, lam, 1.0, 1.0)
    assert not u.is_cuda and u.shape == (2, 1500, 3)
    ref = oracle.matvec(ORACLE_VARIANT[variant], pos.numpy().astype(np.float64), lam.numpy().astype(np.float64))
    check(u.numpy().astype(np.float64), ref, prec, f"host call {variant}")


def test_count_below():
    w = workloads.make(2)
    for dt in (torch.float64, torch.float32):
        pos = torch.from_numpy(w.pos).to(dt).cuda()
        assert binding.rpy_wall_count_below(pos, 1.0) == 0
        expect = int((w.pos[:, 2].astype(np.float32 if dt == torch.float32 else np.float64) < 1.5).sum())
        assert binding.rpy_wall_count_below(pos, 1.5) == expect


# ------------------------------------------------------------------ full sizes, sampled rows
def _full_size(cfg, prec, variant, n_rows):
    w = workloads.make(cfg)
    rows = workloads.sample_rows(w.n_blobs, n_rows)
    u, ref = run_case(w.pos, w.force, prec, variant, rows=rows)
    check(u, ref, prec, f"cfg{cfg} full size {variant} ({len(rows)} sampled rows x {w.n_blobs} sources)")


@pytest.mark.parametrize("prec", ["f32", "f64"])
def test_config3_full_size_sampled_rows(prec):
    _full_size(3, prec, "wall", 2048)


def test_config4_full_size_sampled_rows():
    _full_size(4, "f32", "wall", 2048)


@pytest.mark.parametrize("variant", ["wall", "free"])
def test_config5_full_size_sampled_rows(variant):
    _full_size(5, "f32", variant, 2048)


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("variant", ["wall", "free"])
@pytest.mark.parametrize("n_bodies,n_shards,k", [(600, 2, 1), (600, 3, 1), (600, 8, 1), (430, 40, 1), (40, 3, 1), (600, 2, 3)])
def test_work_shards_sum_to_the_full_product(prec, variant, n_bodies, n_shards, k):
    """rpy_*_matvec_shard: the partial results of all shards (computed one after the other on this
    GPU -- on a multi-GPU job each rank computes one and an all-reduce adds them) sum to u.
    9,000 blobs: symmetric kernel, shards = ranges of tile distances (18 distances: 40 shards leaves
    some empty); 600 blobs or k = 3: plain kernel, shards = ranges of rows."""
    w = workloads.config2(seed=4, n_bodies=n_bodies, k=k)
    pos_b = w.pos.astype(NP[prec]); lam_b = w.force.astype(NP[prec])
    pos = torch.from_numpy(pos_b).cuda(); lam = torch.from_numpy(lam_b).cuda()
    fn = binding.rpy_wall_matvec_shard if variant == "wall" else binding.rpy_free_matvec_shard
    total = torch.zeros((k, w.n_blobs, 3), dtype=torch.float64, device="cuda")
    for s in range(n_shards):
        part = fn(pos, lam, s, n_shards)
        assert part.shape == (k, w.n_blobs, 3)
        total += part.double()
    ref = oracle.matvec(ORACLE_VARIANT[variant], pos_b.astype(np.float64), lam_b.astype(np.float64))
    check(total.cpu().numpy(), ref, prec, f"shards n={w.n_blobs} G={n_shards} {variant}")
    one = fn(pos, lam, 0, 1)                          # a single shard is the whole product
    check(one.cpu().numpy().astype(np.float64), ref, prec, "single shard")


@pytest.mark.parametrize("n", [2000, 6000])
def test_product_is_capturable_in_a_cuda_graph(n):
    """The device forms allocate nothing, create no CUDA object and never synchronise (include/rpy_matvec.h), so a
    caller can capture the whole product -- three kernels chained by programmatic dependent launch -- in a CUDA
    graph and replay it; plain (n = 2,000) and symmetric (n = 6,000) kernel.  The replay on new inputs equals the
    eager call."""
    w = workloads.config1(seed=3, n=n)
    pos = torch.from_numpy(w.pos).cuda(); lam = torch.from_numpy(w.force).cuda()
    ws = torch.empty(binding.rpy_matvec_workspace_bytes("f64", n, 1), dtype=torch.uint8, device="cuda")
    out = torch.empty_like(lam)
    binding.rpy_wall_matvec(pos, lam, out=out, workspace=ws)            # loads the module before capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        with torch.cuda.graph(g, stream=side):
            binding.rpy_wall_matvec(pos, lam, out=out, workspace=ws)
    lam2 = torch.from_numpy(np.random.default_rng(9).standard_normal(w.force.shape)).cuda()
    lam.copy_(lam2)                                                     # new forces in the captured buffers
    out.zero_()
    g.replay()
    torch.cuda.synchronize()
    eager = binding.rpy_wall_matvec(pos, lam2)
    assert float((out - eager).norm() / eager.norm()) <= 1e-14
    ref = oracle.matvec(oracle.WALL, w.pos, lam2.cpu().numpy())
    check(out.cpu().numpy(), ref, "f64", f"graph replay n={n}")
