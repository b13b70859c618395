"""Rectangular product / flow fields (Appendix B) on the GPU vs the oracle."""
import numpy as np
import pytest
import torch

import oracle
from paper_1602_02170_b200 import binding, workloads

pytestmark = pytest.mark.gpu

TOL = {"f64": 1e-12, "f32": 1e-5}
NP = {"f64": np.float64, "f32": np.float32}
OV = {"wall": oracle.WALL, "free": oracle.FREE}
FN = {"wall": binding.rpy_wall_matvec_rect, "free": binding.rpy_free_matvec_rect}


def rel(u, ref):
    return float(np.linalg.norm((u - ref).ravel()) / np.linalg.norm(ref.ravel()))


def cloud(seed, nt, ns, k):
    rng = np.random.default_rng(seed)
    src = rng.uniform([0, 0, 1.1], [40, 40, 8], size=(ns, 3))
    tgt = rng.uniform([-5, -5, 1.0], [45, 45, 12], size=(nt, 3))
    lam = rng.standard_normal((k, ns, 3))
    return tgt, src, lam


def run(tgt, src, lam, prec, variant, a=1.0, eta=1.0):
    tb, sb, lb = tgt.astype(NP[prec]), src.astype(NP[prec]), lam.astype(NP[prec])
    u = FN[variant](torch.from_numpy(tb).cuda(), torch.from_numpy(sb).cuda(), torch.from_numpy(lb).cuda(), a, eta)
    torch.cuda.synchronize()
    ref = oracle.flow(OV[variant], tb.astype(np.float64), sb.astype(np.float64), lb.astype(np.float64), a, eta)
    return u.cpu().numpy().astype(np.float64), ref


@pytest.mark.parametrize("prec", ["f64", "f32"])
@pytest.mark.parametrize("variant", ["wall", "free"])
@pytest.mark.parametrize("nt,ns,k", [(777, 1000, 1), (1, 1, 1), (5000, 300, 3), (130, 4100, 8), (257, 129, 2)])
def test_rect_matches_oracle(prec, variant, nt, ns, k):
    tgt, src, lam = cloud(nt + ns, nt, ns, k)
    u, ref = run(tgt, src, lam, prec, variant, a=0.7, eta=1.3)
    assert np.isfinite(u).all() and rel(u, ref) <= TOL[prec]


def test_targets_on_sources_inside_blobs_and_empty_inputs():
    tgt, src, lam = cloud(1, 64, 200, 1)
    tgt[:10] = src[:10]                       # coincident: self block
    tgt[10:20] = src[10:20] + 0.3             # inside a blob: overlap branch of Eq. (9)
    for prec in ("f64", "f32"):
        u, ref = run(tgt, src, lam, prec, "wall")
        assert rel(u, ref) <= TOL[prec]
    dt = torch.float64
    z = binding.rpy_wall_matvec_rect(torch.from_numpy(tgt).cuda(), torch.empty((0, 3), dtype=dt).cuda(),
                                     torch.empty((0, 3), dtype=dt).cuda())
    assert z.shape == (64, 3) and not z.any()
    e = binding.rpy_wall_matvec_rect(torch.empty((0, 3), dtype=dt).cuda(), torch.from_numpy(src).cuda(),
                                     torch.from_numpy(lam[0]).cuda())
    assert e.shape == (0, 3)


def test_rect_with_targets_equal_sources_is_the_plain_matvec_bit_for_bit():
    w = workloads.config2(n_bodies=200, k=2)                        # two right-hand sides: the plain (non-symmetric) kernel
    pos = torch.from_numpy(w.pos).cuda(); lam = torch.from_numpy(w.force).cuda()
    a = binding.rpy_wall_matvec_rect(pos, pos, lam)
    b = binding.rpy_wall_matvec(pos, lam)
    assert torch.equal(a, b)


def test_subdivide_matches_oracle_exactly_and_flow_through_refined_sources():
    """Appendix B end to end: blobs -> 12 small blobs each (icosahedron of radius a - a'), tracer
    radius a', flow on a plane of targets."""
    w = workloads.config2(n_bodies=30, k=2)
    a_t = 0.25
    tmpl = (1.0 - a_t) * workloads.shell_template(12)
    for prec in ("f64", "f32"):
        pb, fb, tb = w.pos.astype(NP[prec]), w.force.astype(NP[prec]), tmpl.astype(NP[prec])
        sp, sf = binding.rpy_flow_subdivide(torch.from_numpy(pb).cuda(), torch.from_numpy(fb).cuda(), torch.from_numpy(tb).cuda())
        osp, osf = oracle.subdivide(pb, fb, tb) if prec == "f64" else (None, None)
        if prec == "f64":
            assert np.array_equal(sp.cpu().numpy(), osp) and np.array_equal(sf.cpu().numpy(), osf)
        xs = np.linspace(w.pos[:, 0].min(), w.pos[:, 0].max(), 40)
        tg = np.stack(np.meshgrid(xs, xs, [3.0], indexing="ij"), -1).reshape(-1, 3).astype(NP[prec])
        v = binding.rpy_wall_matvec_rect(torch.from_numpy(tg).cuda(), sp, sf, a_t, 1.0)
        ref = oracle.flow(oracle.WALL, tg.astype(np.float64), sp.cpu().numpy().astype(np.float64),
                          sf.cpu().numpy().astype(np.float64), a_t, 1.0)
        assert rel(v.cpu().numpy().astype(np.float64), ref) <= TOL[prec]


def test_full_size_flow_field_sampled_rows():
    """Config-3 sources (172,032 blobs) and a 256 x 256 plane of tracers, fp32 path: sampled targets."""
    w = workloads.make(3)
    xs = np.linspace(0.0, 512.0, 256)
    tg = np.stack(np.meshgrid(xs, xs, [12.0], indexing="ij"), -1).reshape(-1, 3).astype(np.float32)
    pb, fb = w.pos.astype(np.float32), w.force.astype(np.float32)
    v = binding.rpy_wall_matvec_rect(torch.from_numpy(tg).cuda(), torch.from_numpy(pb).cuda(), torch.from_numpy(fb).cuda())
    rows = workloads.sample_rows(tg.shape[0], 256, seed=3)
    ref = oracle.flow(oracle.WALL, tg[rows].astype(np.float64), pb.astype(np.float64), fb.astype(np.float64))
    assert rel(v.cpu().numpy()[:, rows].astype(np.float64), ref) <= 1e-5
