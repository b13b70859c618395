"""CPU oracle for the iterative mobility solver -- TEST INFRASTRUCTURE.

arXiv:1602.02170 Section II.B: the saddle-point system (11) is solved "directly
using a preconditioned iterative Krylov method" -- GMRES with the indefinite
block-diagonal preconditioner P of Eq. (18), applied by solving Eq. (19).  The paper takes GMRES
from PETSc and prints no algorithm, so this file follows the textbook statement (Saad & Schultz
1986: Arnoldi with modified Gram-Schmidt, Givens rotations on the Hessenberg matrix), step by step,
in numpy float64.  Readings (A16-A18): RIGHT preconditioning (the monitored residual is
the true residual of (11)), zero initial guess, convergence when ||r_k|| <= tol ||b||
("reduce the residual by a factor of 10^8", Table III), restart length `restart`.

  gmres            the algorithm on abstract operators
  mobility_gmres   operators of (11) and (19) built from the matvec oracle and oracle/rigid.py

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline leg may import this module; it
shares no code with paper_1602_02170_b200.

Pins (tests/test_oracle_gmres.py): the k-th iterate is the brute-force least-squares minimiser
over the explicitly built Krylov space; exact solve in <= n steps; one step when P = A; residual
history monotone; mobility_gmres reproduces the dense solve of (11) and Table I.
"""
from __future__ import annotations

import numpy as np


def gmres(apply_A, apply_Pinv, b, tol=1e-8, restart=60, max_iter=200):
    """Right-preconditioned restarted GMRES for A x = b, x0 = 0.

    Solves (A P^-1) y = b, x = P^-1 y.  Returns (x, history, n_iter): history[k] is the residual
    norm ||b - A x_k|| / ||b|| estimated by the rotated right-hand side after k iterations
    (history[0] = 1); n_iter counts applications of A inside Arnoldi.
    """
    b = np.asarray(b, dtype=np.float64).reshape(-1)
    n = b.size
    bnorm = np.linalg.norm(b)
    x = np.zeros(n)
    history = [1.0]
    if bnorm == 0.0:
        return x, history, 0
    n_iter = 0
    r = b.copy()
    while n_iter < max_iter:
        beta = np.linalg.norm(r)
        m = min(restart, max_iter - n_iter)
        V = np.zeros((m + 1, n))
        H = np.zeros((m + 1, m))
        cs = np.zeros(m); sn = np.zeros(m)
        g = np.zeros(m + 1); g[0] = beta
        V[0] = r / beta
        j_done = 0
        converged = False
        for j in range(m):
            w = apply_A(apply_Pinv(V[j]))
            n_iter += 1
            for i in range(j + 1):                     # modified Gram-Schmidt
                H[i, j] = np.dot(V[i], w)
                w = w - H[i, j] * V[i]
            H[j + 1, j] = np.linalg.norm(w)
            if H[j + 1, j] > 0.0:
                V[j + 1] = w / H[j + 1, j]
            for i in range(j):                         # earlier rotations on the new column
                t = cs[i] * H[i, j] + sn[i] * H[i + 1, j]
                H[i + 1, j] = -sn[i] * H[i, j] + cs[i] * H[i + 1, j]
                H[i, j] = t
            d = np.hypot(H[j, j], H[j + 1, j])         # new rotation annihilates H[j+1, j]
            cs[j] = H[j, j] / d; sn[j] = H[j + 1, j] / d
            H[j, j] = d; H[j + 1, j] = 0.0
            g[j + 1] = -sn[j] * g[j]
            g[j] = cs[j] * g[j]
            j_done = j + 1
            history.append(abs(g[j + 1]) / bnorm)
            if abs(g[j + 1]) <= tol * bnorm:
                converged = True
                break
        y = np.zeros(j_done)
        for i in range(j_done - 1, -1, -1):            # back substitution R y = g
            y[i] = (g[i] - np.dot(H[i, i + 1:j_done], y[i + 1:])) / H[i, i]
        x = x + apply_Pinv(V[:j_done].T @ y)
        if converged:
            break
        r = b - apply_A(x)
    return x, history, n_iter


def mobility_gmres(variant, pos, q, offsets, F, slip=None, a=1.0, eta=1.0, tol=1e-8, restart=60,
                   max_iter=200, precond_variant=None):
    """GMRES on Eq. (11) with the preconditioner of Eq. (18)-(19).

    Unknown x = [lambda (3 N_b); U (6 N_bodies)], right-hand side [slip; -F].  `precond_variant`
    chooses the tensor of the diagonal blocks M^(pp) (default: the same as `variant`; FREE with a
    WALL matvec is the "unbounded" preconditioner of Table III).
    Returns (lambda [N,3], U [nb,6], history, n_iter).
    """
    from . import matvec as _matvec
    from . import dense as _dense
    from . import rigid

    pos = np.ascontiguousarray(pos, dtype=np.float64)
    q = np.ascontiguousarray(q, dtype=np.float64)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    n = pos.shape[0]; nb = q.shape[0]
    pv = variant if precond_variant is None else precond_variant
    b = np.zeros(3 * n + 6 * nb)
    if slip is not None:
        b[:3 * n] = np.asarray(slip, dtype=np.float64).reshape(-1)
    b[3 * n:] = -np.asarray(F, dtype=np.float64).reshape(-1)

    def apply_A(x):
        lam = x[:3 * n].reshape(n, 3); U = x[3 * n:].reshape(nb, 6)
        top = _matvec(variant, pos, lam, a, eta) - rigid.K_apply(pos, q, offsets, U)
        bot = -rigid.KT_apply(pos, q, offsets, lam)
        return np.concatenate([top.reshape(-1), bot.reshape(-1)])

    # Eq. (19), body by body; the per-body saddle matrices do not change between applications
    blocks = []
    for p in range(nb):
        s = slice(offsets[p], offsets[p + 1]); m = 3 * (offsets[p + 1] - offsets[p])
        Ap = np.zeros((m + 6, m + 6))
        Kp = rigid.K_matrix(pos[s], q[p:p + 1], np.array([0, m // 3]))
        Ap[:m, :m] = _dense(pv, pos[s], a, eta); Ap[:m, m:] = -Kp; Ap[m:, :m] = -Kp.T
        blocks.append(Ap)

    def apply_Pinv(x):
        out = np.empty_like(x)
        for p in range(nb):
            lo, hi = 3 * offsets[p], 3 * offsets[p + 1]
            sol = np.linalg.solve(blocks[p], np.concatenate([x[lo:hi], x[3 * n + 6 * p:3 * n + 6 * p + 6]]))
            out[lo:hi] = sol[:hi - lo]; out[3 * n + 6 * p:3 * n + 6 * p + 6] = sol[hi - lo:]
        return out

    x, history, n_iter = gmres(apply_A, apply_Pinv, b, tol, restart, max_iter)
    return x[:3 * n].reshape(n, 3), x[3 * n:].reshape(nb, 6), history, n_iter
