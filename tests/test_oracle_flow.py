"""Pins for the flow-field oracle (Appendix B): oracle.flow, oracle.subdivide.

None calls oracle.flow to check oracle.flow: a brute-force sum over the separately pinned pair
blocks, the Oseen far field (Eq. (8)), incompressibility by finite differences, no-slip at the wall
for a vanishing tracer, force conservation of the subdivision."""
import numpy as np
import pytest

import oracle

EIGHTPI = 8.0 * np.pi


def _cloud(seed=0, ns=7, nt=5):
    rng = np.random.default_rng(seed)
    src = rng.uniform([0, 0, 1.5], [6, 6, 5], size=(ns, 3))
    tgt = rng.uniform([-2, -2, 1.2], [8, 8, 7], size=(nt, 3))
    lam = rng.standard_normal((2, ns, 3))
    return src, tgt, lam


@pytest.mark.parametrize("variant", [oracle.FREE, oracle.WALL])
def test_flow_is_the_block_by_block_sum(variant):
    src, tgt, lam = _cloud()
    a, eta = 0.3, 1.7
    v = oracle.flow(variant, tgt, src, lam, a, eta)
    ref = np.zeros_like(v)
    for t in range(tgt.shape[0]):
        for j in range(src.shape[0]):
            B = oracle.pair(variant, tgt[t], src[j], a, eta)         # pinned by P1-P11
            for s in range(2):
                ref[s, t] += B @ lam[s, j]
    assert np.allclose(v, ref, rtol=1e-13, atol=1e-15)
    assert np.allclose(oracle.flow(variant, tgt, src, lam[0], a, eta), v[0])
    # a target on a source sees that source's self block
    v0 = oracle.flow(oracle.FREE, src[:1], src[:1], lam[0, :1], a, eta)
    assert np.allclose(v0[0], lam[0, 0] / (6 * np.pi * eta * a))


def test_far_field_is_the_oseen_tensor():
    """Eq. (8): v -> (1/(8 pi eta r)) (I + rhat rhat) F far from a force, any tracer size."""
    F = np.array([[0.3, -1.0, 0.5]])
    r = np.array([[300.0, -200.0, 150.0]])
    d = np.linalg.norm(r); rh = r[0] / d
    oseen = (F[0] + rh * np.dot(rh, F[0])) / (EIGHTPI * 1.3 * d)
    v = oracle.flow(oracle.FREE, r, np.zeros((1, 3)), F, 0.05, 1.3)
    assert np.allclose(v[0], oseen, rtol=1e-6)


@pytest.mark.parametrize("variant", [oracle.FREE, oracle.WALL])
def test_flow_field_is_divergence_free(variant):
    """The regularised Green's function of Eq. (7) inherits incompressibility from G."""
    src, tgt, lam = _cloud(seed=3)
    a, h = 0.2, 1e-4
    for t in tgt:
        if np.min(np.linalg.norm(src - t, axis=1)) < 2.5 * a:
            continue
        div = 0.0
        for c in range(3):
            e = np.zeros(3); e[c] = h
            vp = oracle.flow(variant, (t + e)[None], src, lam[0], a)
            vm = oracle.flow(variant, (t - e)[None], src, lam[0], a)
            div += (vp[0, c] - vm[0, c]) / (2 * h)
        scale = np.linalg.norm(oracle.flow(variant, t[None], src, lam[0], a)) / np.min(np.linalg.norm(src - t, axis=1))
        assert abs(div) < 1e-6 * scale


def test_no_slip_at_the_wall_for_a_vanishing_tracer():
    """Blake's tensor vanishes on the wall (PAPER.md:148 [72]); the tracer's Faxen terms are O(a'^2)."""
    src, _, lam = _cloud(seed=5)
    tgt = np.array([[1.0, 2.0, 0.0], [4.0, 0.5, 0.0]])
    v_small = oracle.flow(oracle.WALL, tgt, src, lam[0], 1e-4)
    v_bulk = oracle.flow(oracle.WALL, tgt + [0, 0, 2.0], src, lam[0], 1e-4)
    assert np.linalg.norm(v_small) < 1e-6 * np.linalg.norm(v_bulk)


def test_subdivision_conserves_force_and_first_moment():
    rng = np.random.default_rng(1)
    pos = rng.standard_normal((4, 3)); lam = rng.standard_normal((2, 4, 3))
    tmpl = rng.standard_normal((6, 3)); tmpl -= tmpl.mean(axis=0)
    sp, sf = oracle.subdivide(pos, lam, tmpl)
    assert sp.shape == (24, 3) and sf.shape == (2, 24, 3)
    assert np.allclose(sp[6:12], pos[1] + tmpl)                       # sub-blob s of blob i at i*n_sub + s
    assert np.allclose(sf[:, 6:12].sum(axis=1), lam[:, 1])            # uniform split, total force kept
    assert np.allclose(sf[0, 7], lam[0, 1] / 6)
    # far away the refined sources give the same flow as the original blobs (same total force and centroid)
    far = np.array([[400.0, 300.0, 500.0]])
    assert np.allclose(oracle.flow(oracle.FREE, far, sp, sf, 0.1), oracle.flow(oracle.FREE, far, pos, lam, 0.1), rtol=1e-4)
