"""CPU oracle for the rigid-multiblob layer around the matvec -- TEST INFRASTRUCTURE.

Plain numpy float64 restatement of arXiv:1602.02170 Section II (line numbers: PAPER.md):

  K, K^T            the kinematic matrix of Eqs. (2), (3) and the force / torque
                    sums of Eq. (10), written as explicit loops;
  mobility_solve    the saddle-point system (11) assembled densely from the
                    oracle's own pair tensor and handed to numpy.linalg.solve: the definition;
  body_mobility     N = (K^T M^-1 K)^-1, Eq. (12);
  precond_solve     the block-diagonal preconditioner system (19) with M~ of Eq. (17)
                    (PAPER.md:228-244), one small dense saddle-point solve per body.

Bodies are contiguous runs of blobs: body p owns blobs offsets[p] .. offsets[p+1]-1 and has the
tracking point q[p].  U = [u_p, omega_p] and F = [f_p, tau_p] are stored [n_bodies, 6].

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it
shares no code with paper_1602_02170_b200 (the CUDA side never forms (11), it runs GMRES).

Pins (tests/test_oracle_rigid.py): Table I effective radii (printed values), the adjoint identity,
hand-computed K entries, the three equations of (10) re-evaluated term by term, SPD of N.
"""
from __future__ import annotations

import numpy as np

from . import dense as _dense_mobility


def _check(pos, q, offsets):
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    q = np.ascontiguousarray(q, dtype=np.float64)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    nb = q.shape[0]
    assert pos.ndim == 2 and pos.shape[1] == 3 and q.shape == (nb, 3)
    assert offsets.shape == (nb + 1,) and offsets[0] == 0 and offsets[-1] == pos.shape[0]
    assert np.all(np.diff(offsets) >= 1)
    return pos, q, offsets, nb


def K_apply(pos, q, offsets, U) -> np.ndarray:
    """Blob velocities of rigid motion, Eq. (2): r_i' = u_p + omega_p x (r_i - q_p)."""
    pos, q, offsets, nb = _check(pos, q, offsets)
    U = np.asarray(U, dtype=np.float64).reshape(nb, 6)
    out = np.zeros_like(pos)
    for p in range(nb):
        for i in range(offsets[p], offsets[p + 1]):
            out[i] = U[p, :3] + np.cross(U[p, 3:], pos[i] - q[p])
    return out


def KT_apply(pos, q, offsets, lam) -> np.ndarray:
    """Total force and torque per body, Eq. (10): f_p = sum lambda_i, tau_p = sum (r_i - q_p) x lambda_i."""
    pos, q, offsets, nb = _check(pos, q, offsets)
    lam = np.asarray(lam, dtype=np.float64).reshape(pos.shape)
    out = np.zeros((nb, 6))
    for p in range(nb):
        for i in range(offsets[p], offsets[p + 1]):
            out[p, :3] += lam[i]
            out[p, 3:] += np.cross(pos[i] - q[p], lam[i])
    return out


def blob_positions(template, centres, quats) -> np.ndarray:
    """Blob positions of identical bodies from their poses (footnote 4; Eq. (1)'s
    r_i = q + R (r_i^ref)): rotation by the unit quaternion theta = (s, p) applied as
    v' = v + 2 s (p x v) + 2 p x (p x v)  (no rotation matrix is formed)."""
    template = np.asarray(template, dtype=np.float64); centres = np.asarray(centres, dtype=np.float64)
    quats = np.asarray(quats, dtype=np.float64)
    out = np.zeros((centres.shape[0], template.shape[0], 3))
    for b in range(centres.shape[0]):
        th = quats[b] / np.linalg.norm(quats[b])
        s, p = th[0], th[1:]
        for t in range(template.shape[0]):
            v = template[t]
            pv = np.cross(p, v)
            out[b, t] = centres[b] + v + 2.0 * s * pv + 2.0 * np.cross(p, pv)
    return out.reshape(-1, 3)


def K_matrix(pos, q, offsets) -> np.ndarray:
    """Dense K, (3 N_b) x (6 N_bodies): column c is K applied to the c-th unit motion."""
    pos, q, offsets, nb = _check(pos, q, offsets)
    K = np.zeros((3 * pos.shape[0], 6 * nb))
    for c in range(6 * nb):
        e = np.zeros(6 * nb); e[c] = 1.0
        K[:, c] = K_apply(pos, q, offsets, e.reshape(nb, 6)).reshape(-1)
    return K


def mobility_solve(variant, pos, q, offsets, F, slip=None, a=1.0, eta=1.0, rank_deficient=False):
    """Solves Eq. (11):  [M -K; -K^T 0] [lambda; U] = [slip; -F].  Returns (lambda [N,3], U [nb,6]).

    rank_deficient=True: bodies whose blobs lie on a straight line cannot resist a torque about that
    line, K has a zero column and (11) is singular; "in practice all inverses should be replaced by
    pseudo-inverses ... no problem ... if the applied force is in the appropriate range"
    (PAPER.md:192): the minimum-norm least-squares solution (numpy.linalg.lstsq), whose rotation
    rate about the line is zero."""
    pos, q, offsets, nb = _check(pos, q, offsets)
    n = pos.shape[0]
    M = _dense_mobility(variant, pos, a, eta)
    K = K_matrix(pos, q, offsets)
    A = np.zeros((3 * n + 6 * nb, 3 * n + 6 * nb))
    A[:3 * n, :3 * n] = M
    A[:3 * n, 3 * n:] = -K
    A[3 * n:, :3 * n] = -K.T
    b = np.zeros(3 * n + 6 * nb)
    if slip is not None:
        b[:3 * n] = np.asarray(slip, dtype=np.float64).reshape(-1)
    b[3 * n:] = -np.asarray(F, dtype=np.float64).reshape(-1)
    x = np.linalg.lstsq(A, b, rcond=1e-12)[0] if rank_deficient else np.linalg.solve(A, b)
    return x[:3 * n].reshape(n, 3), x[3 * n:].reshape(nb, 6)


def body_mobility(variant, pos, q, offsets, a=1.0, eta=1.0) -> np.ndarray:
    """N = (K^T M^-1 K)^-1, Eq. (12), for all bodies together: (6 nb) x (6 nb)."""
    pos, q, offsets, nb = _check(pos, q, offsets)
    M = _dense_mobility(variant, pos, a, eta)
    K = K_matrix(pos, q, offsets)
    return np.linalg.inv(K.T @ np.linalg.solve(M, K))


def body_blocks(variant, pos, offsets, a=1.0, eta=1.0):
    """The diagonal blocks M^(pp) of Eq. (17): each body alone (with the wall when variant = WALL)."""
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    return [_dense_mobility(variant, pos[offsets[p]:offsets[p + 1]], a, eta) for p in range(len(offsets) - 1)]


def precond_solve(variant, pos, q, offsets, x, y, a=1.0, eta=1.0, rank_deficient=False):
    """Solves Eq. (19) body by body:  [M~ -K; -K^T 0] [lambda; U] = [x; y]  with M~ of Eq. (17)
    (rank_deficient=True: minimum-norm least squares per body, see mobility_solve)."""
    pos, q, offsets, nb = _check(pos, q, offsets)
    x = np.asarray(x, dtype=np.float64).reshape(pos.shape)
    y = np.asarray(y, dtype=np.float64).reshape(nb, 6)
    lam = np.zeros_like(pos); U = np.zeros((nb, 6))
    for p in range(nb):
        s = slice(offsets[p], offsets[p + 1])
        m = 3 * (offsets[p + 1] - offsets[p])
        Mpp = _dense_mobility(variant, pos[s], a, eta)
        Kp = K_matrix(pos[s], q[p:p + 1], np.array([0, m // 3]))
        A = np.zeros((m + 6, m + 6))
        A[:m, :m] = Mpp; A[:m, m:] = -Kp; A[m:, :m] = -Kp.T
        rhs = np.concatenate([x[s].reshape(-1), y[p]])
        sol = np.linalg.lstsq(A, rhs, rcond=1e-12)[0] if rank_deficient else np.linalg.solve(A, rhs)
        lam[s] = sol[:m].reshape(-1, 3); U[p] = sol[m:]
    return lam, U
