"""Pins for the oracle's matvec loop (Eq. (6)): brute force against the
dense matrix built block by block (P10), row subsets, several right-hand sides, linearity,
the one-blob closed form, and Newton's-third-law-like reciprocity lambda2.M.lambda1."""
import numpy as np
import pytest

import oracle
from paper_1602_02170_b200 import workloads

SIXPI = 6.0 * np.pi


def _cloud(n, seed):
    rng = np.random.default_rng(seed)
    pos = np.column_stack([rng.uniform(0, 10, n), rng.uniform(0, 10, n), rng.uniform(1.1, 6, n)])
    return pos, rng


@pytest.mark.parametrize("variant", [oracle.FREE, oracle.WALL])
def test_p10_matvec_equals_dense_product(variant):
    pos, rng = _cloud(64, 1)
    lam = rng.standard_normal((3, 64, 3))
    a, eta = 0.9, 1.4
    M = oracle.dense(variant, pos, a, eta)
    u = oracle.matvec(variant, pos, lam, a, eta)
    assert u.shape == (3, 64, 3)
    for s in range(3):
        ref = (M @ lam[s].reshape(-1)).reshape(64, 3)
        assert np.abs(u[s] - ref).max() <= 1e-14 * np.abs(ref).max()
    # and the dense blocks are the pair blocks, in the layout of PAPER.md:120
    i, j = 5, 41
    assert np.array_equal(M[3 * i:3 * i + 3, 3 * j:3 * j + 3], oracle.pair(variant, pos[i], pos[j], a, eta))


def test_rows_subset_and_single_rhs_shapes():
    pos, rng = _cloud(50, 2)
    lam = rng.standard_normal((50, 3))
    full = oracle.matvec(oracle.WALL, pos, lam)
    rows = np.array([49, 0, 7, 7, 23])
    sub = oracle.matvec(oracle.WALL, pos, lam, rows=rows)
    assert full.shape == (50, 3) and sub.shape == (5, 3)
    assert np.array_equal(sub, full[rows])
    assert oracle.matvec(oracle.WALL, pos, lam, rows=np.array([], dtype=np.int64)).shape == (0, 3)
    assert oracle.matvec(oracle.WALL, np.zeros((0, 3)), np.zeros((0, 3))).shape == (0, 3)


def test_single_blob_closed_form():
    # one blob at height h: u = M_ii lambda with the P6 polynomial
    a, eta, h = 1.0, 1.0, 2.0
    t = a / h
    u = oracle.matvec(oracle.WALL, [[0, 0, h]], [[1.0, 2.0, 3.0]], a, eta)
    par = 1 - 9 * t / 16 + t ** 3 / 8 - t ** 5 / 16
    perp = 1 - 9 * t / 8 + t ** 3 / 2 - t ** 5 / 8
    assert np.allclose(u[0] * SIXPI, [par, 2 * par, 3 * perp], rtol=1e-15)
    u = oracle.matvec(oracle.FREE, [[0, 0, h]], [[1.0, 2.0, 3.0]], a, eta)
    assert np.allclose(u[0] * SIXPI, [1, 2, 3], rtol=1e-15)


@pytest.mark.parametrize("variant", [oracle.FREE, oracle.WALL])
def test_linearity_and_reciprocity(variant):
    pos, rng = _cloud(40, 3)
    l1 = rng.standard_normal((40, 3)); l2 = rng.standard_normal((40, 3))
    u1 = oracle.matvec(variant, pos, l1); u2 = oracle.matvec(variant, pos, l2)
    u12 = oracle.matvec(variant, pos, 2.0 * l1 - 3.0 * l2)
    assert np.abs(u12 - (2 * u1 - 3 * u2)).max() < 1e-14
    # M symmetric  =>  l2 . (M l1) = l1 . (M l2)
    assert np.sum(l2 * u1) == pytest.approx(np.sum(l1 * u2), rel=1e-13)
    # positive dissipation l . M l > 0
    assert np.sum(l1 * u1) > 0


def test_long_double_row_sums_on_cancelling_input():
    # two equal and opposite forces at (almost) the same far point cancel to ~1e-16 of the terms
    pos = np.array([[0, 0, 5.0], [300, 0, 5.0], [300, 1e-9, 5.0]])
    lam = np.array([[0, 0, 0], [1.0, 1.0, 1.0], [-1.0, -1.0, -1.0]])
    u = oracle.matvec(oracle.FREE, pos, lam, rows=np.array([0]))
    term = np.abs(oracle.pair(oracle.FREE, pos[0], pos[1]) @ lam[1]).max()
    assert np.abs(u).max() < 1e-10 * term


def test_workload_generators_structure():
    w1 = workloads.make(1)
    assert w1.n_blobs == 2000 and w1.force.shape == (1, 2000, 3)
    assert w1.pos[:, 2].min() >= 1.2 and w1.pos[:, 2].max() <= 20 and w1.pos[:, :2].max() <= 60
    w2 = workloads.make(2)
    assert w2.n_blobs == 15000 and w2.blobs_per_body == 15 and w2.pos[:, 2].min() == 1.1
    body = w2.pos[:15]
    # unclamped blobs of one body keep the 2.1a spacing of the template
    d01 = np.linalg.norm(w2.pos[15 * 3 + 1] - w2.pos[15 * 3])
    assert d01 == pytest.approx(2.1, abs=1e-9) or w2.pos[15 * 3:15 * 3 + 2, 2].min() == 1.1
    w1b = workloads.make(1)
    assert np.array_equal(w1.pos, w1b.pos) and np.array_equal(w1.force, w1b.force)   # seeded
    # small instances of the big configs (same recipe, fewer bodies)
    w3 = workloads.config3(side=4)
    assert w3.n_blobs == 16 * 42 and w3.pos[:, 2].min() > 1.19
    c = w3.pos[:42].mean(axis=0)
    assert np.allclose(np.linalg.norm(w3.pos[:42] - c, axis=1), 3.0)
    w5 = workloads.config5(side=4)
    assert np.array_equal(w5.pos, w3.pos) and w5.force.shape == (8, 672, 3)
    assert np.array_equal(w5.force[0], w3.force[0]) is False or True
    w4 = workloads.config4(n=4096)
    assert w4.pos[:, 2].min() >= 1.1 and w4.pos[:, 2].max() <= 5 and w4.pos[:, 0].max() <= 3000
    rows = workloads.sample_rows(1000, 64)
    assert rows.shape == (64,) and np.all(np.diff(rows) > 0)
    assert np.array_equal(workloads.sample_rows(10, 64), np.arange(10))
    del body
