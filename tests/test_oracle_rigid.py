"""Pins for oracle/rigid.py (the rigid-multiblob layer: K, Eq. (11), Eq. (12), Eq. (19)).

None of these calls the oracle to check the oracle: printed values of the paper (Table I),
hand-computed entries, identities re-evaluated term by term, and a textbook special case.
"""
import os

import numpy as np
import pytest

import oracle
from oracle import rigid
from paper_1602_02170_b200 import workloads

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
SIXPI = 6.0 * np.pi


def _small_suspension(n_bodies=4, seed=3):
    w = workloads.config2(seed=seed, n_bodies=n_bodies)
    return w, workloads.bodies_of(w)


def test_k_entries_by_hand():
    """Eq. (2): r' = u + omega x (r - q)."""
    pos = np.array([[2.0, 1.0, 5.0], [1.0, 3.0, 5.0]])
    q = np.array([[1.0, 1.0, 5.0]])
    off = np.array([0, 2])
    # rotation about z with unit rate: the blob at q + (1,0,0) moves in +y, the one at q + (0,2,0) in -x
    v = rigid.K_apply(pos, q, off, np.array([[0, 0, 0, 0, 0, 1.0]]))
    assert np.allclose(v, [[0, 1, 0], [-2, 0, 0]])
    v = rigid.K_apply(pos, q, off, np.array([[0.5, -1, 2, 0, 0, 0.0]]))
    assert np.allclose(v, [[0.5, -1, 2], [0.5, -1, 2]])
    # Eq. (10): a force (0, 1, 0) on the first blob gives torque (1,0,0) x (0,1,0) = +z about q
    FT = rigid.KT_apply(pos, q, off, np.array([[0, 1.0, 0], [0, 0, 0]]))
    assert np.allclose(FT, [[0, 1, 0, 0, 0, 1]])


def test_kt_is_the_adjoint_of_k_and_rigid_motion_preserves_distances():
    w, b = _small_suspension()
    rng = np.random.default_rng(0)
    U = rng.standard_normal((b.n_bodies, 6)); lam = rng.standard_normal(w.pos.shape)
    lhs = np.sum(rigid.K_apply(w.pos, b.q, b.offsets, U) * lam)
    rhs = np.sum(U * rigid.KT_apply(w.pos, b.q, b.offsets, lam))
    assert lhs == pytest.approx(rhs, rel=1e-13)
    K = rigid.K_matrix(w.pos, b.q, b.offsets)
    assert np.allclose(K.T @ lam.reshape(-1), rigid.KT_apply(w.pos, b.q, b.offsets, lam).reshape(-1), atol=1e-12)
    # rigid: relative velocity of two blobs of one body is perpendicular to their separation
    v = rigid.K_apply(w.pos, b.q, b.offsets, U)
    i, j = b.offsets[1], b.offsets[1] + 9
    assert abs(np.dot(v[i] - v[j], w.pos[i] - w.pos[j])) < 1e-12


def test_table1_effective_radii_through_body_mobility():
    """Table I (left), through rigid.body_mobility and through the saddle-point
    solve (11): an isolated shell pulled with force f moves with u = f / (6 pi eta R_h)."""
    rows = [l.split() for l in open(os.path.join(GOLDEN, "table1_radii.txt")) if l.strip() and l[0] != "#"]
    for nb, a_over_s, rh_exp, rt_exp in rows:
        pos = workloads.shell_template(int(nb))
        d = np.linalg.norm(pos[:, None] - pos[None], axis=2)
        a = float(a_over_s) * d[d > 1e-9].min()
        off = np.array([0, pos.shape[0]]); q = np.zeros((1, 3))
        N = rigid.body_mobility(oracle.FREE, pos, q, off, a, 1.0)
        assert 1.0 / (SIXPI * np.trace(N[:3, :3]) / 3) == pytest.approx(float(rh_exp), abs=1.5e-4)
        assert (1.0 / (8 * np.pi * np.trace(N[3:, 3:]) / 3)) ** (1 / 3) == pytest.approx(float(rt_exp), abs=1.5e-4)
        lam, U = rigid.mobility_solve(oracle.FREE, pos, q, off, np.array([[1.0, 0, 0, 0, 0, 0]]), None, a, 1.0)
        assert U[0, 0] == pytest.approx(1.0 / (SIXPI * float(rh_exp)), rel=2e-4)
        assert np.allclose(U[0, 1:], 0, atol=1e-9)          # icosahedral symmetry: no coupling
        assert np.allclose(lam.sum(axis=0), [1, 0, 0], atol=1e-12)


@pytest.mark.parametrize("variant", [oracle.FREE, oracle.WALL])
def test_mobility_solve_satisfies_eq10_term_by_term(variant):
    """The three equations of (10), re-evaluated with the matvec oracle (row
    loop, not the dense assembly) and explicit cross products."""
    w, b = _small_suspension(n_bodies=5)
    rng = np.random.default_rng(1)
    slip = 0.1 * rng.standard_normal(w.pos.shape)
    lam, U = rigid.mobility_solve(variant, w.pos, b.q, b.offsets, b.F, slip, 1.0, 1.0)
    Ml = oracle.matvec(variant, w.pos, lam)
    for p in range(b.n_bodies):
        f = np.zeros(3); t = np.zeros(3)
        for i in range(b.offsets[p], b.offsets[p + 1]):
            rhs = U[p, :3] + np.cross(U[p, 3:], w.pos[i] - b.q[p]) + slip[i]
            assert np.allclose(Ml[i], rhs, atol=1e-10)
            f += lam[i]; t += np.cross(w.pos[i] - b.q[p], lam[i])
        assert np.allclose(f, b.F[p, :3], atol=1e-10) and np.allclose(t, b.F[p, 3:], atol=1e-10)


def test_body_mobility_is_spd_and_wall_slows_the_body():
    w, b = _small_suspension(n_bodies=3)
    for variant in (oracle.FREE, oracle.WALL):
        N = rigid.body_mobility(variant, w.pos, b.q, b.offsets)
        assert np.allclose(N, N.T, atol=1e-12)
        assert np.linalg.eigvalsh(N).min() > 0          # PAPER.md:177 "evidently SPD since M is"
    # one shell: the wall reduces the translational mobility (Fig. 5)
    pos = 3.0 * workloads.shell_template(42) + np.array([0, 0, 4.5])
    off = np.array([0, 42]); q = np.array([[0, 0, 4.5]])
    Nf = rigid.body_mobility(oracle.FREE, pos, q, off); Nw = rigid.body_mobility(oracle.WALL, pos, q, off)
    assert 0.3 * Nf[0, 0] < Nw[0, 0] < 0.9 * Nf[0, 0] and Nw[2, 2] < Nw[0, 0]


def test_preconditioner_is_exact_for_one_body_and_block_diagonal_otherwise():
    """Eq. (17)-(19)."""
    w, b = _small_suspension(n_bodies=1)
    rng = np.random.default_rng(2)
    x = rng.standard_normal(w.pos.shape)
    lam, U = rigid.precond_solve(oracle.WALL, w.pos, b.q, b.offsets, x, -b.F)
    lam2, U2 = rigid.mobility_solve(oracle.WALL, w.pos, b.q, b.offsets, b.F, x)
    assert np.allclose(lam, lam2, atol=1e-10) and np.allclose(U, U2, atol=1e-10)
    # several bodies: the solve of body p ignores every other body's blobs
    w, b = _small_suspension(n_bodies=3)
    x = rng.standard_normal(w.pos.shape)
    lam, U = rigid.precond_solve(oracle.WALL, w.pos, b.q, b.offsets, x, -b.F)
    s = slice(b.offsets[1], b.offsets[2])
    lam1, U1 = rigid.mobility_solve(oracle.WALL, w.pos[s], b.q[1:2], np.array([0, 15]), b.F[1:2], x[s])
    assert np.allclose(lam[s], lam1, atol=1e-10) and np.allclose(U[1], U1[0], atol=1e-10)
    # residual of (19) with the block-diagonal M~ assembled from body_blocks
    blocks = rigid.body_blocks(oracle.WALL, w.pos, b.offsets)
    for p, Mpp in enumerate(blocks):
        sp = slice(b.offsets[p], b.offsets[p + 1])
        r = Mpp @ lam[sp].reshape(-1) - rigid.K_apply(w.pos[sp], b.q[p:p + 1], np.array([0, 15]), U[p:p + 1]).reshape(-1)
        assert np.allclose(r, x[sp].reshape(-1), atol=1e-10)


def test_blob_positions_from_poses_by_hand_and_by_group_properties():
    """Footnote 4.  Quarter turns computed by hand; rotations preserve lengths; the
    quaternion product composes rotations; the seeded generator's own matrix form agrees."""
    tmpl = np.array([[1.0, 0, 0], [0, 2.0, 0], [0, 0, 3.0]])
    c = np.array([[10.0, 20.0, 30.0]])
    h = np.sqrt(0.5)
    # quarter turn about z: x -> y, y -> -x
    out = rigid.blob_positions(tmpl, c, np.array([[h, 0, 0, h]]))
    assert np.allclose(out, c + np.array([[0, 1.0, 0], [-2.0, 0, 0], [0, 0, 3.0]]), atol=1e-15)
    # quarter turn about x: y -> z, z -> -y ; an unnormalised quaternion gives the same rotation
    out = rigid.blob_positions(tmpl, c, np.array([[3.0, 3.0, 0, 0]]))
    assert np.allclose(out, c + np.array([[1.0, 0, 0], [0, 0, 2.0], [0, -3.0, 0]]), atol=1e-14)
    rng = np.random.default_rng(0)
    q1, q2 = rng.standard_normal(4), rng.standard_normal(4)
    q1 /= np.linalg.norm(q1); q2 /= np.linalg.norm(q2)
    q12 = np.concatenate([[q1[0] * q2[0] - q1[1:] @ q2[1:]], q1[0] * q2[1:] + q2[0] * q1[1:] + np.cross(q1[1:], q2[1:])])
    t = rng.standard_normal((5, 3)); z = np.zeros((1, 3))
    two = rigid.blob_positions(rigid.blob_positions(t, z, q2[None]), z, q1[None])
    assert np.allclose(two, rigid.blob_positions(t, z, q12[None]), atol=1e-14)
    assert np.allclose(np.linalg.norm(two, axis=1), np.linalg.norm(t, axis=1))
    assert np.allclose(rigid.blob_positions(t, c, q1[None]), t @ workloads.quat_to_rot(q1[None])[0].T + c, atol=1e-14)


def test_table6_sphere_near_a_wall_through_the_wall_corrected_body_mobility():
    """Appendix D / Table VI (Fig. 5): the paper's fits of the
    mobility of its 642-blob sphere at height H above the wall.  The 42-blob shell (a/s = 1/2, R_h and
    R_tau from Table I) run through the oracle's WALL pair tensor, K and Eq. (12) must reproduce them:
    a body-level check of the whole wall correction (translation, rotation and their coupling) that
    no pair-level pin sees.  Tolerances: the fit's own error plus the 42- vs 642-blob resolution."""
    fits = {}
    for l in open(os.path.join(GOLDEN, "table6_fits.txt")):
        if l.strip() and l[0] != "#":
            t = l.split(); fits[t[0]] = [float(v) for v in t[1:8]]

    def fit(name, x):
        de, al, f2, f1, f0, d1, d0 = fits[name]
        return de + (1.0 / x) ** al * (f2 * x * x + f1 * x + f0) / (x * x + d1 * x + d0)

    pos0 = workloads.shell_template(42)
    d = np.linalg.norm(pos0[:, None] - pos0[None], axis=2)
    a = 0.5 * d[d > 1e-9].min()
    off = np.array([0, 42])
    Nf = rigid.body_mobility(oracle.FREE, pos0, np.zeros((1, 3)), off, a, 1.0)
    Rh = 1.0 / (SIXPI * np.trace(Nf[:3, :3]) / 3); Rt = (1.0 / (8 * np.pi * np.trace(Nf[3:, 3:]) / 3)) ** (1 / 3)
    assert Rh == pytest.approx(1.1220, abs=2e-4) and Rt == pytest.approx(1.1019, abs=2e-4)       # Table I
    for x in (1.5, 2.0, 3.0, 5.0, 8.0):
        H = x * Rh
        N = rigid.body_mobility(oracle.WALL, pos0 + [0, 0, H], np.array([[0, 0, H]]), off, a, 1.0)
        tt = 0.5 * (N[0, 0] + N[1, 1]) * SIXPI * Rh
        rr_par = 0.5 * (N[3, 3] + N[4, 4]) * 8 * np.pi * Rt ** 3
        rr_perp = N[5, 5] * 8 * np.pi * Rt ** 3
        rt = 0.5 * (N[0, 4] - N[1, 3]) * SIXPI * Rh ** 2          # u_x from tau_y = -(u_y from tau_x)
        assert tt == pytest.approx(fit("tt_par", x), rel=8e-3)
        assert rr_par == pytest.approx(fit("rr_par", x), rel=8e-3)
        assert rr_perp == pytest.approx(fit("rr_perp", x), rel=3e-3)
        assert N[0, 4] == pytest.approx(-N[1, 3], rel=2e-2)        # isotropy in the wall plane, up to the shell's own
                                                                   # anisotropy (the paper averages over orientations)
        if x <= 5.0:
            assert rt == pytest.approx(fit("rt_par", x), rel=5e-2)
        assert N[2, 2] < 0.5 * (N[0, 0] + N[1, 1])                # perpendicular motion is hindered more (Fig. 5)


def test_straight_rods_minimum_norm_solution():
    """the paper's minimally resolved rods are blobs on a line segment; K^T M^-1 K is
    singular (no torque about the axis) and pseudo-inverses are meant.  The minimum-norm solution of
    (11) satisfies Eq. (10) term by term, does not spin about the axis, equals pinv(K^T M^-1 K) F, turns
    with the rod in free space, and shows the slender-body anisotropy."""
    rng = np.random.default_rng(4)
    nblob = 7
    axis = np.array([np.cos(0.3), np.sin(0.3), 0.0])
    rods, q, off = [], [], [0]
    for c in ([0.0, 0.0, 3.0], [3.0, 9.0, 4.0]):
        r = np.array(c) + np.outer(2.0 * (np.arange(nblob) - 3), axis)
        rods.append(r); q.append(r[3]); off.append(off[-1] + nblob)
    pos = np.concatenate(rods); q = np.array(q); off = np.array(off)
    F = rng.standard_normal((2, 6))
    F[:, 3:] -= np.outer(F[:, 3:] @ axis, axis)                      # no torque about the axis: consistent
    lam, U = rigid.mobility_solve(oracle.WALL, pos, q, off, F, None, rank_deficient=True)
    assert np.allclose(U[:, 3:] @ axis, 0.0, atol=1e-10)
    Ml = oracle.matvec(oracle.WALL, pos, lam)
    assert np.allclose(Ml, rigid.K_apply(pos, q, off, U), atol=1e-9)
    assert np.allclose(rigid.KT_apply(pos, q, off, lam), F, atol=1e-9)
    # the same through the Schur complement with a pseudo-inverse (Eq. (12) as PAPER.md:192 reads it)
    M = oracle.dense(oracle.WALL, pos)
    K = rigid.K_matrix(pos, q, off)
    Npinv = np.linalg.pinv(K.T @ np.linalg.solve(M, K), rcond=1e-10)
    assert np.allclose(U.reshape(-1), Npinv @ F.reshape(-1), rtol=1e-8, atol=1e-12)
    # free space: turning rod and load together turns the motion (one rod, quarter turn about z)
    rod = rods[0] - rods[0][3]
    Rz = np.array([[0.0, -1.0, 0.0], [1.0, 0.0, 0.0], [0.0, 0.0, 1.0]])
    f = F[:1].copy()
    _, U0 = rigid.mobility_solve(oracle.FREE, rod, np.zeros((1, 3)), np.array([0, nblob]), f, None, rank_deficient=True)
    fr = np.concatenate([f[0, :3] @ Rz.T, f[0, 3:] @ Rz.T])[None]
    _, U1 = rigid.mobility_solve(oracle.FREE, rod @ Rz.T, np.zeros((1, 3)), np.array([0, nblob]), fr, None, rank_deficient=True)
    assert np.allclose(U1[0, :3], U0[0, :3] @ Rz.T, atol=1e-12) and np.allclose(U1[0, 3:], U0[0, 3:] @ Rz.T, atol=1e-12)
    # a rod moves more easily along its axis than across it (slender-body ratio between 1 and 2)
    Nf = np.linalg.pinv(rigid.K_matrix(rod, np.zeros((1, 3)), np.array([0, nblob])).T @ np.linalg.solve(
        oracle.dense(oracle.FREE, rod), rigid.K_matrix(rod, np.zeros((1, 3)), np.array([0, nblob]))), rcond=1e-10)
    mu_par = axis @ Nf[:3, :3] @ axis; mu_perp = Nf[2, 2]
    assert 1.2 < mu_par / mu_perp < 2.0
