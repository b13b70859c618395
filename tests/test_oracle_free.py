"""Pins for the free-space part of the oracle (Eq. (9)).

Each test checks the oracle against something the paper or the mathematics fixes:
hand-computed entries of both branches (P1), continuity at r = 2a (P2), the self block
(P3), the Oseen far field Eq. (8), symmetry, invariances (P8) and the effective radii
the paper prints in Table I (P9).  Nothing here calls the CUDA path.
"""
import os

import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
SIXPI = 6.0 * np.pi


def fg_from_block(B, rhat):
    """Split B = f I + g rhat rhat^T using a direction orthogonal to rhat."""
    t = np.cross(rhat, [0.3, -0.5, 0.8]); t /= np.linalg.norm(t)
    f = t @ B @ t
    g = rhat @ B @ rhat - f
    return f, g


@pytest.mark.parametrize("a,eta", [(1.0, 1.0), (0.37, 2.5)])
def test_p1_closed_form_entries_both_branches(a, eta):
    # r = 4a: C1 = 3/16 + 1/128, C2 = 3/16 - 3/128 ; r = a: C3 = 23/32, C4 = 3/32 (Eq. (9))
    rhat = np.array([2.0, -1.0, 2.0]) / 3.0
    ri = np.array([0.2, 0.1, -0.4])
    for r_over_a, f_exp, g_exp in [(4.0, 3 / 16 + 1 / 128, 3 / 16 - 3 / 128), (1.0, 23 / 32, 3 / 32)]:
        rj = ri - r_over_a * a * rhat
        B = oracle.pair(oracle.FREE, ri, rj, a, eta) * SIXPI * eta * a
        f, g = fg_from_block(B, rhat)
        assert f == pytest.approx(f_exp, rel=1e-14)
        assert g == pytest.approx(g_exp, rel=1e-13)
        # the full block is f I + g rhat rhat^T, nothing else
        assert np.allclose(B, f_exp * np.eye(3) + g_exp * np.outer(rhat, rhat), rtol=0, atol=1e-15)


def test_p1_dimensional_prefactor():
    # M scales as 1/(6 pi eta a) at fixed r/a (prefactor of Eq. (9))
    ri = np.array([0.0, 0.0, 0.0]); d = np.array([1.0, 2.0, 2.0])   # |d| = 3
    B1 = oracle.pair(oracle.FREE, ri, d, 1.0, 1.0)
    B2 = oracle.pair(oracle.FREE, ri, 2.0 * d, 2.0, 3.0)
    assert np.allclose(B2, B1 / 6.0, rtol=1e-15)
    # explicit far entry along the line of centres: (1/(6 pi eta a)) (C1 + C2) = (1/(6 pi))(3/2r - 1/r^3), a=1
    rh = d / 3.0
    assert rh @ B1 @ rh == pytest.approx((1.5 / 3.0 - 1.0 / 27.0) / SIXPI, rel=1e-14)


def test_p2_continuity_at_2a():
    a = 0.8
    rhat = np.array([0.0, 0.6, 0.8])
    z = np.zeros(3)
    for eps in (0.0, 1e-9, -1e-9):
        B = oracle.pair(oracle.FREE, (2 * a + eps) * rhat, z, a, 1.0) * SIXPI * a
        f, g = fg_from_block(B, rhat)
        assert f == pytest.approx(7 / 16, abs=2e-9)
        assert g == pytest.approx(3 / 16, abs=2e-9)
    # exactly at r = 2a both branch formulas give 7/16, 3/16
    B = oracle.pair(oracle.FREE, 2 * a * rhat, z, a, 1.0) * SIXPI * a
    f, g = fg_from_block(B, rhat)
    assert f == pytest.approx(7 / 16, rel=1e-14) and g == pytest.approx(3 / 16, rel=1e-13)
    # |M(2a+e) - M(2a-e)| = O(e)
    for e in (1e-3, 1e-5):
        Bp = oracle.pair(oracle.FREE, (2 * a + e) * rhat, z, a, 1.0)
        Bm = oracle.pair(oracle.FREE, (2 * a - e) * rhat, z, a, 1.0)
        assert np.abs(Bp - Bm).max() * SIXPI * a < 2.0 * e / a


def test_p3_self_block_and_r_to_zero():
    a, eta = 1.3, 0.7
    p = np.array([0.4, -2.0, 5.0])
    B = oracle.pair(oracle.FREE, p, p, a, eta)
    assert np.array_equal(B, np.eye(3) / (SIXPI * eta * a))
    for r in (1e-3, 1e-8, 1e-300):
        Br = oracle.pair(oracle.FREE, p + np.array([r, 0, 0]), p, a, eta) * SIXPI * eta * a
        assert np.abs(Br - np.eye(3)).max() <= 0.3 * r / a + 1e-16


def test_far_field_is_oseen():
    # Eq. (8): M -> (1/(8 pi eta r)) (I + rhat rhat^T); the RPY correction is O(a^2/r^2)
    a, eta = 1.0, 1.0
    rhat = np.array([1.0, 2.0, -2.0]) / 3.0
    for r in (1e2, 1e4):
        B = oracle.pair(oracle.FREE, r * rhat, np.zeros(3), a, eta)
        oseen = (np.eye(3) + np.outer(rhat, rhat)) / (8 * np.pi * eta * r)
        assert np.abs(B - oseen).max() / np.abs(oseen).max() < 1.1 * (a / r) ** 2


def test_symmetry_and_isotropy_free():
    rng = np.random.default_rng(3)
    for _ in range(50):
        ri, rj = rng.uniform(-3, 3, (2, 3))
        Bij = oracle.pair(oracle.FREE, ri, rj, 1.0, 1.0)
        Bji = oracle.pair(oracle.FREE, rj, ri, 1.0, 1.0)
        assert np.allclose(Bij, Bij.T, rtol=0, atol=1e-17)
        assert np.allclose(Bij, Bji.T, rtol=0, atol=1e-17)
        # P8: a rigid rotation Q conjugates the block; a translation leaves it unchanged
        Q, _ = np.linalg.qr(rng.standard_normal((3, 3)))
        t = rng.uniform(-10, 10, 3)
        Brot = oracle.pair(oracle.FREE, Q @ ri + t, Q @ rj + t, 1.0, 1.0)
        assert np.allclose(Brot, Q @ Bij @ Q.T, rtol=0, atol=1e-15)


def _body_mobility(pos, a, eta=1.0):
    """N = (K^T M^-1 K)^-1, Eqs. (2),(3),(12), tracking point = origin."""
    n = pos.shape[0]
    M = oracle.dense(oracle.FREE, pos, a, eta)
    K = np.zeros((3 * n, 6))
    for i, r in enumerate(pos):
        K[3 * i:3 * i + 3, 0:3] = np.eye(3)
        # omega x r = -[r]x omega
        K[3 * i:3 * i + 3, 3:6] = -np.array([[0, -r[2], r[1]], [r[2], 0, -r[0]], [-r[1], r[0], 0]])
    return np.linalg.inv(K.T @ np.linalg.solve(M, K))


def test_p9_table1_effective_radii():
    """Table I (left): R_h/R_g and R_tau/R_g of 12-, 42-, 162- and 642-blob shells.
    Pins the far branch, the r = 2a boundary (a/s = 1/2 puts neighbours exactly at 2a),
    the r<2a branch is not reached here; also pins the 1/(6 pi eta a) prefactor."""
    from paper_1602_02170_b200.workloads import shell_template
    rows = [l.split() for l in open(os.path.join(GOLDEN, "table1_radii.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 8
    for nb, a_over_s, rh_exp, rt_exp in rows:
        pos = shell_template(int(nb))                          # R_g = 1
        d = np.linalg.norm(pos[:, None] - pos[None], axis=2)
        s = d[d > 1e-9].min()
        a = float(a_over_s) * s
        N = _body_mobility(pos, a)
        mu_tt = np.trace(N[:3, :3]) / 3.0
        mu_rr = np.trace(N[3:, 3:]) / 3.0
        Rh = 1.0 / (SIXPI * mu_tt)
        Rt = (1.0 / (8 * np.pi * mu_rr)) ** (1.0 / 3.0)
        assert Rh == pytest.approx(float(rh_exp), abs=1.5e-4), (nb, a_over_s, Rh)
        assert Rt == pytest.approx(float(rt_exp), abs=1.5e-4), (nb, a_over_s, Rt)
