"""Pins for the wall (Rotne-Prager-Blake) part of the oracle.

The paper defines the wall block by Eq. (7) on the half-space Green's function and cites
[13] for the closed form without printing it.  The oracle codes a closed form; these
tests pin it to things that do not depend on that closed form:

 P5  Blake's tensor written out separately here (itself pinned by exact no-slip at z = 0,
     reciprocity and the Oseen limit), with both Faxen operators of Eq. (7) applied by
     4th-order central differences in 60-digit arithmetic (mpmath);
 P11 the survey's worked examples (tests/golden/wall_pairs.txt), also re-derived by P5;
 P6  the wall-corrected self mobility polynomial in a/h and Table VI's -9/16;
 P7  the wall term vanishing like (9/8)(a/H);
 P4  symmetry M_ij = M_ji^T and positive definiteness of the dense matrix, eigenvalues by
     a Jacobi sweep written here;
 P8  invariance under x-y translation, rotation about z and x<->y swap.
Nothing here calls the CUDA path.
"""
import os

import mpmath as mp
import numpy as np
import pytest

import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
SIXPI = 6.0 * np.pi


# ----------------------------------------------------------------------------------------
# Blake's half-space Green's function [72], unit viscosity, wall z = 0, written out on its
# own: target x, source y at height h = y3, r = x - y, R = x - (y1, y2, -h),
#   8 pi G_ij = S_ij(r) - S_ij(R) + 2 h D_jj d/dR_j [ h R_i/|R|^3 - S_i3(R) ]   (no sum on j)
# with S_ij(v) = delta_ij/|v| + v_i v_j/|v|^3 and D = diag(1, 1, -1).
# ----------------------------------------------------------------------------------------
def _S(v):
    n = mp.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    return [[(1 if i == j else 0) / n + v[i] * v[j] / n ** 3 for j in range(3)] for i in range(3)]


def blake_image_8pi(x, y):
    """8 pi (G_Blake - Oseen)(x, y) as a 3x3 list; row = velocity comp. at x, col = force comp. at y."""
    h = y[2]
    R = [x[0] - y[0], x[1] - y[1], x[2] + y[2]]
    n = mp.sqrt(R[0] ** 2 + R[1] ** 2 + R[2] ** 2)
    SR = _S(R)
    D = [1, 1, -1]
    out = [[None] * 3 for _ in range(3)]
    for i in range(3):
        for j in range(3):
            dij = 1 if i == j else 0
            di3 = 1 if i == 2 else 0
            dj3 = 1 if j == 2 else 0
            d_dipole = h * (dij / n ** 3 - 3 * R[i] * R[j] / n ** 5)
            d_S_i3 = (-di3 * R[j] / n ** 3
                      + (dij * R[2] + R[i] * dj3) / n ** 3
                      - 3 * R[i] * R[2] * R[j] / n ** 5)
            out[i][j] = -SR[i][j] + 2 * h * D[j] * (d_dipole - d_S_i3)
    return out


def blake_full_8pi(x, y):
    r = [x[0] - y[0], x[1] - y[1], x[2] - y[2]]
    Sr = _S(r)
    img = blake_image_8pi(x, y)
    return [[Sr[i][j] + img[i][j] for j in range(3)] for i in range(3)]


def _mat(fn, x, y):
    return mp.matrix(fn([mp.mpf(c) for c in x], [mp.mpf(c) for c in y]))


def _lap(fn, x, y, which, d):
    """4th-order central-difference Laplacian of the matrix function fn in x (which=0) or y (1)."""
    c = [mp.mpf(-1) / 12, mp.mpf(4) / 3, mp.mpf(-5) / 2, mp.mpf(4) / 3, mp.mpf(-1) / 12]
    acc = mp.zeros(3, 3)
    for ax in range(3):
        for s, w in zip((-2, -1, 0, 1, 2), c):
            xx = list(x); yy = list(y)
            if which == 0:
                xx[ax] = xx[ax] + s * d
            else:
                yy[ax] = yy[ax] + s * d
            acc += w * fn(xx, yy)
    return acc / d ** 2


def wall_block_fd(xi, xj, a):
    """(3a/4) * 8 pi (1 + a^2/6 lap_x)(1 + a^2/6 lap_y)[G_Blake - Oseen](x_i, x_j): Eq. (7)."""
    mp.mp.dps = 60
    d = mp.mpf("1e-6")
    x = [mp.mpf(repr(float(c))) if not isinstance(c, str) else mp.mpf(c) for c in xi]
    y = [mp.mpf(repr(float(c))) if not isinstance(c, str) else mp.mpf(c) for c in xj]
    a = mp.mpf(repr(float(a)))
    F = lambda xx, yy: mp.matrix(blake_image_8pi(xx, yy))
    LyF = lambda xx, yy: _lap(F, xx, yy, 1, d)
    W = F(x, y) + a ** 2 / 6 * (_lap(F, x, y, 0, d) + LyF(x, y)) + a ** 4 / 36 * _lap(LyF, x, y, 0, d)
    W = W * (3 * a / 4)
    return np.array([[float(W[i, j]) for j in range(3)] for i in range(3)])


# ------------------------------ pins on Blake's tensor itself ---------------------------
def test_blake_tensor_no_slip_reciprocity_oseen():
    mp.mp.dps = 40
    rng = np.random.default_rng(0)
    for _ in range(10):
        x = list(rng.uniform(-2, 2, 3)); y = list(rng.uniform(-2, 2, 3))
        x[2] = abs(x[2]) + 0.1; y[2] = abs(y[2]) + 0.1
        # velocity vanishes on the wall for any source
        G0 = _mat(blake_full_8pi, [x[0], x[1], 0.0], y)
        assert max(abs(v) for v in G0) < mp.mpf("1e-35")
        # reciprocity G_ij(x,y) = G_ji(y,x)
        Gxy = _mat(blake_full_8pi, x, y); Gyx = _mat(blake_full_8pi, y, x)
        assert max(abs(v) for v in (Gxy - Gyx.T)) < mp.mpf("1e-35")
    # far from the wall the image part is O(1/H) and G -> Oseen, Eq. (8)
    x = [0.3, -0.2, 1e6 + 0.5]; y = [-0.4, 0.1, 1e6]
    img = _mat(blake_image_8pi, x, y)
    assert max(abs(v) for v in img) < 2e-6


# ------------------------------ P5: Eq. (7) on Blake vs the oracle ----------------------
@pytest.mark.parametrize("seed", range(8))
def test_p5_wall_block_equals_faxen_of_blake(seed):
    rng = np.random.default_rng(100 + seed)
    a = float(rng.uniform(0.4, 1.6))
    xi = rng.uniform(-3, 3, 3); xj = rng.uniform(-3, 3, 3)
    xi[2] = rng.uniform(1.0, 5.0) * a; xj[2] = rng.uniform(1.0, 5.0) * a
    if seed == 0:
        xj = xi.copy()                                  # self term i = j
    if seed == 1:
        xj = xi + np.array([0.5, -0.3, 0.2]) * a        # overlapping pair, r < 2a
    ref = wall_block_fd(xi, xj, a)
    got = oracle.wall_block(xi, xj, a)
    assert np.abs(got - ref).max() <= 2e-14 * np.abs(ref).max()


def test_p11_golden_worked_examples():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "wall_pairs.txt")) if l.strip() and l[0] != "#"]
    assert len(rows) == 4
    for row in rows:
        tag = row[0]
        v = np.array([float(t) for t in row[1:]])
        xi, xj, exp = v[0:3], v[3:6], v[6:15].reshape(3, 3)
        if tag.endswith("_wall"):
            got = oracle.wall_block(xi, xj, 1.0)
            # the stored numbers are themselves Eq. (7) on Blake: re-derive them here
            assert np.abs(wall_block_fd(xi, xj, 1.0) - exp).max() < 5e-16
        else:
            got = oracle.pair(oracle.WALL, xi, xj, 1.0, 1.0) * SIXPI
        assert np.abs(got - exp).max() < 5e-16, tag
    # in one block the xz and zx entries differ: the symmetry is M_ij = M_ji^T, not per block
    B = oracle.pair(oracle.WALL, [0.3, -1.1, 1.7], [1.9, 0.4, 1.3])
    assert abs(B[0, 2] - B[2, 0]) > 1e-3


def test_small_radius_limit_is_blake_green_function():
    # a -> 0: 6 pi eta a M_ij -> (3a/4) 8 pi G_Blake(r_i, r_j) (Faxen terms are O(a^2)); Eq. (7)
    mp.mp.dps = 30
    xi = [0.3, -1.1, 1.7]; xj = [1.9, 0.4, 1.3]
    G = np.array(_mat(blake_full_8pi, xi, xj).tolist(), dtype=float)
    for a in (1e-3, 1e-4):
        B = oracle.pair(oracle.WALL, xi, xj, a, 1.0) * SIXPI * a
        assert np.abs(B - 0.75 * a * G).max() / (0.75 * a * np.abs(G).max()) < 3.0 * a * a
    # a target on the wall does not move in that limit
    a = 1e-5
    B = oracle.pair(oracle.WALL, [0.3, -1.1, 0.0], xj, a, 1.0) * SIXPI * a
    assert np.abs(B).max() < 10 * a ** 3


# ------------------------------ P6: self mobility above the wall ------------------------
@pytest.mark.parametrize("a,eta", [(1.0, 1.0), (0.6, 1.7)])
def test_p6_self_mobility_polynomial(a, eta):
    mu0 = 1.0 / (SIXPI * eta * a)
    for h_over_a in (1.0, 1.1, 1.5, 2.0, 3.7, 10.0, 123.0):
        h = h_over_a * a
        t = a / h
        p = np.array([0.7, -0.2, h])
        B = oracle.pair(oracle.WALL, p, p, a, eta) / mu0
        par = 1 - 9 * t / 16 + t ** 3 / 8 - t ** 5 / 16
        perp = 1 - 9 * t / 8 + t ** 3 / 2 - t ** 5 / 8
        assert np.allclose(B, np.diag([par, par, perp]), rtol=0, atol=4e-16)
    # h = 1.5a: diag(1271/1944, 1271/1944, 371/972)
    B = oracle.pair(oracle.WALL, [0, 0, 1.5 * a], [0, 0, 1.5 * a], a, eta) / mu0
    assert np.allclose(np.diag(B), [1271 / 1944, 1271 / 1944, 371 / 972], rtol=2e-16 * 4)


def test_p6_leading_wall_coefficient_is_table6():
    # Table VI: mu_par/mu0 = 1 - (9/16)(R_h/H) + ...  (f_{n,2} = -9/16)
    for H in (1e3, 1e4, 1e5):
        B = oracle.pair(oracle.WALL, [0, 0, H], [0, 0, H], 1.0, 1.0) * SIXPI
        assert (B[0, 0] - 1.0) * H == pytest.approx(-9 / 16, rel=0, abs=2e-7 + 1e-11 * H)
        assert (B[2, 2] - 1.0) * H == pytest.approx(-9 / 8, rel=0, abs=6e-7 + 1e-11 * H)


# ------------------------------ P7: wall term vanishes as h grows -----------------------
def test_p7_wall_term_vanishes_with_height():
    d = np.array([2.5, 0.5, 0.3])
    for H, expect in ((10.0, 0.112), (1e2, 0.01125), (1e3, 1.125e-3), (1e4, 1.125e-4)):
        ri = np.array([0.0, 0.0, H]); rj = ri + d
        diff = (oracle.pair(oracle.WALL, ri, rj) - oracle.pair(oracle.FREE, ri, rj)) * SIXPI
        # for H >> |d| the block tends to the self term of P6: -(a/H) diag(9/16, 9/16, 9/8),
        # whose 2-norm is (9/8)(a/H)  (0.112, 0.01125, ... in SURVEY.md 8(c) P7)
        nrm = np.linalg.norm(diff, 2)
        assert nrm == pytest.approx(1.125 / H, rel=0.06)
        assert nrm == pytest.approx(expect, rel=0.06)
    # ratio wall/free -> 0 linearly in 1/H
    r1 = np.linalg.norm((oracle.pair(oracle.WALL, [0, 0, 1e3], [1, 1, 1e3 + 1])
                         - oracle.pair(oracle.FREE, [0, 0, 1e3], [1, 1, 1e3 + 1])))
    r2 = np.linalg.norm((oracle.pair(oracle.WALL, [0, 0, 1e5], [1, 1, 1e5 + 1])
                         - oracle.pair(oracle.FREE, [0, 0, 1e5], [1, 1, 1e5 + 1])))
    assert r1 / r2 == pytest.approx(100.0, rel=1e-2)


# ------------------------------ P4: symmetry and positive definiteness ------------------
def jacobi_eigenvalues(A, sweeps=30, tol=1e-14):
    """Eigenvalues of a symmetric matrix by cyclic Jacobi rotations (brute force, no LAPACK)."""
    A = np.array(A, dtype=float)
    n = A.shape[0]
    for _ in range(sweeps):
        off = np.sqrt(np.sum(np.tril(A, -1) ** 2))
        if off < tol * np.sqrt(np.sum(np.diag(A) ** 2)):
            break
        for p in range(n - 1):
            for q in range(p + 1, n):
                if abs(A[p, q]) < 1e-300:
                    continue
                theta = (A[q, q] - A[p, p]) / (2.0 * A[p, q])
                t = np.sign(theta) / (abs(theta) + np.sqrt(theta * theta + 1.0)) if theta != 0 else 1.0
                c = 1.0 / np.sqrt(t * t + 1.0); s = t * c
                rp = A[p, :].copy(); rq = A[q, :].copy()
                A[p, :] = c * rp - s * rq; A[q, :] = s * rp + c * rq
                cp = A[:, p].copy(); cq = A[:, q].copy()
                A[:, p] = c * cp - s * cq; A[:, q] = s * cp + c * cq
    return np.sort(np.diag(A))


def test_jacobi_solver_on_known_spectrum():
    rng = np.random.default_rng(5)
    Q, _ = np.linalg.qr(rng.standard_normal((12, 12)))
    lam = np.linspace(0.1, 3.0, 12)
    assert np.allclose(jacobi_eigenvalues(Q @ np.diag(lam) @ Q.T), lam, atol=1e-13)


@pytest.mark.parametrize("variant", [oracle.FREE, oracle.WALL])
def test_p4_dense_symmetric_positive_definite(variant):
    rng = np.random.default_rng(11)
    n = 30
    pos = np.column_stack([rng.uniform(0, 8, n), rng.uniform(0, 8, n), rng.uniform(1.1, 8, n)])
    d = np.linalg.norm(pos[:, None] - pos[None], axis=2)
    assert ((d < 2.0) & (d > 0)).sum() >= 4                  # overlapping pairs are present
    M = oracle.dense(variant, pos, 1.0, 1.0)
    assert np.abs(M - M.T).max() <= 1e-15 * np.abs(M).max()  # M_ij = M_ji^T
    ev = jacobi_eigenvalues(0.5 * (M + M.T))
    assert ev[0] > 1e-3 / SIXPI                               # strictly positive
    assert np.allclose(ev, np.linalg.eigvalsh(0.5 * (M + M.T)), rtol=0, atol=1e-13)
    lam = rng.standard_normal(3 * n)
    assert lam @ M @ lam > 0


def test_wall_overlap_loses_definiteness():
    # not guaranteed SPD when blobs overlap the wall (z < a)
    rng = np.random.default_rng(2)
    n = 30
    pos = np.column_stack([rng.uniform(0, 5, n), rng.uniform(0, 5, n), rng.uniform(0.3, 1.0, n)])
    M = oracle.dense(oracle.WALL, pos, 1.0, 1.0)
    assert np.linalg.eigvalsh(0.5 * (M + M.T))[0] < 0


def test_pair_symmetry_wall_blockwise():
    rng = np.random.default_rng(4)
    for _ in range(100):
        ri = rng.uniform(-3, 3, 3); rj = rng.uniform(-3, 3, 3)
        ri[2] = rng.uniform(1, 6); rj[2] = rng.uniform(1, 6)
        Bij = oracle.pair(oracle.WALL, ri, rj, 0.9, 1.3)
        Bji = oracle.pair(oracle.WALL, rj, ri, 0.9, 1.3)
        assert np.abs(Bij - Bji.T).max() <= 1e-15 * np.abs(Bij).max()


# ------------------------------ P8: invariances with the wall ---------------------------
def test_p8_wall_invariances():
    rng = np.random.default_rng(9)
    for _ in range(30):
        ri = rng.uniform(-3, 3, 3); rj = rng.uniform(-3, 3, 3)
        ri[2] = rng.uniform(1, 6); rj[2] = rng.uniform(1, 6)
        B = oracle.pair(oracle.WALL, ri, rj)
        t = np.array([rng.uniform(-50, 50), rng.uniform(-50, 50), 0.0])
        assert np.allclose(oracle.pair(oracle.WALL, ri + t, rj + t), B, rtol=0, atol=1e-14 * np.abs(B).max() * 50)
        th = rng.uniform(0, 2 * np.pi)
        Q = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1]])
        assert np.allclose(oracle.pair(oracle.WALL, Q @ ri, Q @ rj), Q @ B @ Q.T, rtol=0, atol=1e-15)
        P = np.array([[0, 1, 0], [1, 0, 0], [0, 0, 1.0]])
        assert np.allclose(oracle.pair(oracle.WALL, P @ ri, P @ rj), P @ B @ P.T, rtol=0, atol=1e-16)
        # a shift in z is NOT a symmetry
        assert not np.allclose(oracle.pair(oracle.WALL, ri + [0, 0, 1], rj + [0, 0, 1]), B, rtol=1e-6, atol=0)
