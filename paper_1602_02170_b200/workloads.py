"""Seeded synthetic inputs for the mobility matvec (shared by tests, bench and oracle legs).

This module holds geometry and random draws only -- none of the method's arithmetic
(no RPY or wall formula appears here) -- so that the CUDA path and the CPU oracle can
be fed the same inputs without sharing any code of the method itself.

The five workloads are the ones ``BASELINE.json:configs`` names, made concrete in
SURVEY.md 8(d) / DESIGN.md "Input recipe".  They stand in for the paper's own timing
workload (rigid rods sedimented above a no-slip wall, a random force on every blob,
PAPER.md:643), whose hard-rectangle packings are not available.

Generator: ``numpy.random.default_rng(seed)`` (PCG64), float64, draws in the order
written in each function; lengths in units of the blob radius a = 1, eta = 1; blob
order is body-major.  The wall is z = 0 and the fluid occupies z > 0.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np


@dataclass
class Workload:
    name: str
    pos: np.ndarray            # [N,3] float64 blob positions
    force: np.ndarray          # [k,N,3] float64 blob forces lambda
    a: float = 1.0
    eta: float = 1.0
    blobs_per_body: int = 1
    precisions: tuple = ("f64",)
    variants: tuple = ("wall",)
    meta: dict = field(default_factory=dict)

    @property
    def n_blobs(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_rhs(self) -> int:
        return int(self.force.shape[0])


def quat_to_rot(q: np.ndarray) -> np.ndarray:
    """Rotation matrices [nb,3,3] of unit quaternions q = (s, p1, p2, p3) [nb,4]."""
    s, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((q.shape[0], 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - s * z); R[:, 0, 2] = 2 * (x * z + s * y)
    R[:, 1, 0] = 2 * (x * y + s * z); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - s * x)
    R[:, 2, 0] = 2 * (x * z - s * y); R[:, 2, 1] = 2 * (y * z + s * x); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def icosahedron_vertices() -> np.ndarray:
    """The 12 vertices of a regular icosahedron on the unit sphere."""
    phi = (1.0 + np.sqrt(5.0)) / 2.0
    v = []
    for s1 in (1.0, -1.0):
        for s2 in (1.0, -1.0):
            v.append((0.0, s1, s2 * phi))
            v.append((s1, s2 * phi, 0.0))
            v.append((s2 * phi, 0.0, s1))
    v = np.array(v)
    return v / np.linalg.norm(v, axis=1, keepdims=True)


def shell_template(n_blobs: int = 42) -> np.ndarray:
    """Unit-sphere shell of 12, 42, 162 or 642 blobs: icosahedron vertices, then every subdivision adds the
    edge midpoints projected back to the sphere.  New points are appended after
    the old ones, so the 12- and 42-blob shells are prefixes of the finer ones."""
    levels = {12: 0, 42: 1, 162: 2, 642: 3}
    if n_blobs not in levels:
        raise ValueError("shell_template: 12, 42, 162 or 642 blobs")
    v = icosahedron_vertices()
    for _ in range(levels[n_blobs]):
        d = np.linalg.norm(v[:, None, :] - v[None, :, :], axis=2)
        edge = d[d > 1e-9].min()
        mids = []
        for i in range(v.shape[0]):
            for j in np.nonzero((d[i] < 1.2 * edge) & (np.arange(v.shape[0]) > i))[0]:
                m = 0.5 * (v[i] + v[j])
                mids.append(m / np.linalg.norm(m))
        v = np.concatenate([v, np.array(mids)], axis=0)
    assert v.shape == (n_blobs, 3)
    return v


def boomerang_template() -> np.ndarray:
    """15-blob L shape: corner blob at the origin, two 7-blob arms along +x and +y,
    blob spacing 2.1 a (BASELINE.json config 2; PAPER.md:750 defers the geometry to [68])."""
    t = [(0.0, 0.0, 0.0)]
    t += [(2.1 * m, 0.0, 0.0) for m in range(1, 8)]
    t += [(0.0, 2.1 * m, 0.0) for m in range(1, 8)]
    return np.array(t)


def _forces(rng, k: int, n: int) -> np.ndarray:
    return rng.standard_normal((k, n, 3))


def config1(seed: int = 0, n: int = 2000, k: int = 1) -> Workload:
    """Independent blobs in a box: x,y ~ U(0,60), z ~ U(1.2,20), then lambda ~ N(0,1)."""
    rng = np.random.default_rng(seed)
    x = rng.uniform(0.0, 60.0, n)
    y = rng.uniform(0.0, 60.0, n)
    z = rng.uniform(1.2, 20.0, n)
    pos = np.stack([x, y, z], axis=1)
    return Workload("cfg1_box2000" if n == 2000 else f"cfg1_box{n}", pos, _forces(rng, k, n),
                    precisions=("f64",), meta={"seed": seed})


def config2(seed: int = 0, n_bodies: int = 1000, k: int = 1, side: float = 400.0) -> Workload:
    """Boomerangs near the wall.  Draw order: quaternions N(0,1)[nb,4] (normalised),
    centre x ~ U(0,side), y ~ U(0,side), z = |N(0, std 2)| + 2.5, then lambda.
    The body 'centre' is the corner blob; every blob is then clamped to z >= 1.1.
    side = 400 is BASELINE.json's box; other values keep the number density when n_bodies changes
    (side = 400 sqrt(n_bodies / 1000): the scaling study of Table III, right)."""
    rng = np.random.default_rng(seed)
    q = rng.standard_normal((n_bodies, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    cx = rng.uniform(0.0, side, n_bodies)
    cy = rng.uniform(0.0, side, n_bodies)
    cz = np.abs(rng.normal(0.0, 2.0, n_bodies)) + 2.5
    tmpl = boomerang_template()
    R = quat_to_rot(q)
    pos = np.einsum("bij,tj->bti", R, tmpl) + np.stack([cx, cy, cz], axis=1)[:, None, :]
    pos = pos.reshape(-1, 3)
    pos[:, 2] = np.maximum(pos[:, 2], 1.1)
    n = pos.shape[0]
    return Workload(f"cfg2_boomerang{n}", pos, _forces(rng, k, n), blobs_per_body=15,
                    precisions=("f64", "f32"), meta={"seed": seed, "n_bodies": n_bodies})


def _shell_lattice(rng, side: int):
    """side x side spheres of 42 blobs, shell radius 3, lattice spacing 8 with jitter
    U(-0.5,0.5) in x and y, z ~ U(4.2,10); shells unrotated.  Draw order: jx, jy, z."""
    nb = side * side
    jx = rng.uniform(-0.5, 0.5, nb)
    jy = rng.uniform(-0.5, 0.5, nb)
    cz = rng.uniform(4.2, 10.0, nb)
    ii, jj = np.meshgrid(np.arange(side), np.arange(side), indexing="ij")
    cx = 8.0 * (ii.reshape(-1) + 0.5) + jx
    cy = 8.0 * (jj.reshape(-1) + 0.5) + jy
    tmpl = 3.0 * shell_template(42)
    pos = tmpl[None, :, :] + np.stack([cx, cy, cz], axis=1)[:, None, :]
    return pos.reshape(-1, 3)


def config3(seed: int = 0, side: int = 64, k: int = 1) -> Workload:
    """4,096 rigid 42-blob spheres = 172,032 blobs (side=64); then lambda."""
    rng = np.random.default_rng(seed)
    pos = _shell_lattice(rng, side)
    n = pos.shape[0]
    return Workload(f"cfg3_shells{n}", pos, _forces(rng, k, n), blobs_per_body=42,
                    precisions=("f32", "f64"), meta={"seed": seed, "n_bodies": side * side})


def config4(seed: int = 0, n: int = 1 << 20, k: int = 1) -> Workload:
    """Dense sedimented monolayer: x,y ~ U(0,3000), z ~ U(1.1,5), then lambda."""
    rng = np.random.default_rng(seed)
    x = rng.uniform(0.0, 3000.0, n)
    y = rng.uniform(0.0, 3000.0, n)
    z = rng.uniform(1.1, 5.0, n)
    pos = np.stack([x, y, z], axis=1)
    return Workload(f"cfg4_monolayer{n}", pos, _forces(rng, k, n), precisions=("f32",),
                    meta={"seed": seed})


def config5(seed: int = 0, side: int = 64, k: int = 8) -> Workload:
    """Geometry of config 3 with k = 8 simultaneous lambda vectors (same rng, forces drawn
    after the geometry); run through the wall and the free-space kernels."""
    rng = np.random.default_rng(seed)
    pos = _shell_lattice(rng, side)
    n = pos.shape[0]
    return Workload(f"cfg5_shells{n}_k{k}", pos, _forces(rng, k, n), blobs_per_body=42,
                    precisions=("f32",), variants=("wall", "free"),
                    meta={"seed": seed, "n_bodies": side * side})


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4, 5: config5}


def make(config: int, **kw) -> Workload:
    return CONFIGS[config](**kw)


@dataclass
class Bodies:
    """Rigid-body view of a workload: body p owns the contiguous blobs
    offsets[p] .. offsets[p+1]-1 and has the tracking point q[p]; F are applied forces/torques."""
    offsets: np.ndarray        # [n_bodies+1] int64
    q: np.ndarray              # [n_bodies,3] float64
    F: np.ndarray              # [n_bodies,6] float64 (f_p, tau_p), N(0,1)

    @property
    def n_bodies(self) -> int:
        return int(self.q.shape[0])


def bodies_of(w: Workload, seed: int = 1) -> Bodies:
    """Bodies of a rigid-body workload (configs 2, 3, 5).  Tracking point q_p: the first blob of
    the body (the boomerang's corner blob, config 2) / the mean of the body's blobs (the shell
    centre, configs 3 and 5).  F ~ N(0,1)[nb,6] comes from its own generator (`seed`), so the blob
    forces of the matvec workloads are unchanged."""
    bpb = w.blobs_per_body
    if bpb <= 1 or w.n_blobs % bpb:
        raise ValueError("workload has no rigid bodies")
    nb = w.n_blobs // bpb
    offsets = np.arange(nb + 1, dtype=np.int64) * bpb
    body = w.pos.reshape(nb, bpb, 3)
    q = body[:, 0, :].copy() if w.name.startswith("cfg2") else body.mean(axis=1)
    F = np.random.default_rng(seed).standard_normal((nb, 6))
    return Bodies(offsets, q, F)


def sample_rows(n: int, n_rows: int, seed: int = 12345) -> np.ndarray:
    """Seeded sorted sample of target rows used for parity / oracle timing at large N."""
    if n_rows >= n:
        return np.arange(n, dtype=np.int64)
    rng = np.random.default_rng(seed)
    return np.sort(rng.choice(n, size=n_rows, replace=False)).astype(np.int64)


def cylinder_template(n_rings: int = 10, per_ring: int = 6, radius: float = 1.2, spacing: float = 2.0) -> np.ndarray:
    """Blobs on the surface of a cylinder along x (rings of `per_ring` blobs, alternate rings turned by
    half a step): the surface-resolved rod of PAPER.md:641, scaled down.  Centre of mass at the origin."""
    pts = []
    for r in range(n_rings):
        x = (r - 0.5 * (n_rings - 1)) * spacing
        for s in range(per_ring):
            th = 2.0 * np.pi * (s + 0.5 * (r % 2)) / per_ring
            pts.append((x, radius * np.cos(th), radius * np.sin(th)))
    return np.array(pts)


def mixed_suspension(seed: int = 0, n_groups: int = 2):
    """Bodies of different sizes in one suspension (15-blob boomerangs, 42-blob shells of radius 3,
    60-blob cylinders), `n_groups` of each, on a jittered lattice of spacing 40a, random orientations,
    every blob at z >= 1.1a.  Returns (pos [N,3], Bodies, lambda [N,3]).  Exercises ragged offsets and
    both the shared-memory (3*blobs <= 162) and the global-memory factorisation paths."""
    rng = np.random.default_rng(seed)
    templates = [boomerang_template(), 3.0 * shell_template(42), cylinder_template()]
    pos, q, offsets = [], [], [0]
    slot = 0
    for g in range(n_groups):
        for t in templates:
            quat = rng.standard_normal(4)
            R = quat_to_rot((quat / np.linalg.norm(quat))[None, :])[0]
            c = np.array([40.0 * (slot % 4) + rng.uniform(-3, 3), 40.0 * (slot // 4) + rng.uniform(-3, 3), 0.0])
            body = t @ R.T
            c[2] = 1.1 - body[:, 2].min() + rng.uniform(0.2, 3.0)
            body = body + c
            pos.append(body); q.append(body.mean(axis=0)); offsets.append(offsets[-1] + body.shape[0])
            slot += 1
    pos = np.concatenate(pos, axis=0)
    b = Bodies(np.array(offsets, dtype=np.int64), np.array(q), rng.standard_normal((len(q), 6)))
    lam = rng.standard_normal(pos.shape)
    return pos, b, lam


def rods_near_wall(n_rods: int = 1000, phi: float = 0.1, h_over_d: float = 0.75, seed: int = 0, n_blobs: int = 21):
    """The suspension of Section V.D / Table III, minimally resolved: cylinders of
    aspect ratio L/D = 6.4, each `n_blobs` = 21 blobs of radius a = 1.02 R uniformly spaced along a segment
    of length L, parallel to the wall at centreline height H = h_over_d * D, at surface packing fraction
    phi.  The paper packs hard rectangles with a molecular-dynamics code; here L x D rectangles are placed
    by random sequential addition in a periodic square (no overlaps; fine for phi <= 0.3).  Units: a = 1.
    Returns (pos [n_rods * n_blobs, 3], Bodies)."""
    rng = np.random.default_rng(seed)
    R = 1.0 / 1.02; D = 2.0 * R; L = 6.4 * D
    side = np.sqrt(n_rods * L * D / phi)
    centres, angles = [], []
    corners = lambda c, th: c + np.array([[sx * L / 2 * np.cos(th) - sy * D / 2 * np.sin(th),
                                            sx * L / 2 * np.sin(th) + sy * D / 2 * np.cos(th)]
                                           for sx in (-1, 1) for sy in (-1, 1)])

    def overlap(c1, t1, c2, t2):                      # separating-axis test for two rectangles
        d = c2 - c1
        d -= side * np.round(d / side)                # periodic image
        if d @ d > (L * L + D * D):
            return False
        p1, p2 = corners(np.zeros(2), t1), corners(d, t2)
        for th in (t1, t1 + np.pi / 2, t2, t2 + np.pi / 2):
            ax = np.array([np.cos(th), np.sin(th)])
            a1, a2 = p1 @ ax, p2 @ ax
            if a1.max() < a2.min() or a2.max() < a1.min():
                return False
        return True

    cell = L + D
    ncell = max(1, int(side // cell))
    grid = {}
    while len(centres) < n_rods:
        c = rng.uniform(0.0, side, 2); th = rng.uniform(0.0, np.pi)
        key = (int(c[0] / side * ncell) % ncell, int(c[1] / side * ncell) % ncell)
        ok = True
        for dx in (-1, 0, 1):
            for dy in (-1, 0, 1):
                for j in grid.get(((key[0] + dx) % ncell, (key[1] + dy) % ncell), ()):
                    if overlap(c, th, centres[j], angles[j]):
                        ok = False
                        break
                if not ok:
                    break
            if not ok:
                break
        if ok:
            grid.setdefault(key, []).append(len(centres))
            centres.append(c); angles.append(th)
    s = (np.arange(n_blobs) - (n_blobs - 1) / 2.0) * (L / (n_blobs - 1))
    pos = np.empty((n_rods, n_blobs, 3))
    for i, (c, th) in enumerate(zip(centres, angles)):
        pos[i, :, 0] = c[0] + s * np.cos(th); pos[i, :, 1] = c[1] + s * np.sin(th); pos[i, :, 2] = h_over_d * D
    q = pos.mean(axis=1)
    F = np.random.default_rng(seed + 1).standard_normal((n_rods, 6))
    axis = np.stack([np.cos(angles), np.sin(angles), np.zeros(n_rods)], axis=1)
    F[:, 3:] -= np.sum(F[:, 3:] * axis, axis=1, keepdims=True) * axis       # no torque about the axis
    b = Bodies(np.arange(n_rods + 1, dtype=np.int64) * n_blobs, q, F)
    return pos.reshape(-1, 3), b


def sphere_lattice(n_side: int = 8, n_blobs: int = 42, phi: float = 0.09, seed: int = 0):
    """Section IV.D / Table I (right): n_side^3 spherical shells of `n_blobs` blobs
    (a/s = 1/2, geometric radius R_g = 1) on a finite simple cubic lattice in an unbounded fluid, at volume
    fraction phi = (4/3) pi R_h^3 / d^3 (d = lattice spacing; phi = 0.09 is d = 4 R_g = 3.6 R_h).
    Returns (pos, Bodies, a): random forces and torques on every sphere; the blob radius a."""
    rh_over_rg = {12: 1.2625, 42: 1.1220}[n_blobs]            # Table I (left), a/s = 1/2
    t = shell_template(n_blobs)
    dmat = np.linalg.norm(t[:, None] - t[None], axis=2)
    a = 0.5 * dmat[dmat > 1e-9].min()
    d = rh_over_rg * (4.0 * np.pi / (3.0 * phi)) ** (1.0 / 3.0)
    g = (np.arange(n_side) - (n_side - 1) / 2.0) * d
    c = np.stack(np.meshgrid(g, g, g, indexing="ij"), -1).reshape(-1, 3)
    pos = (c[:, None, :] + t[None, :, :]).reshape(-1, 3)
    F = np.random.default_rng(seed).standard_normal((c.shape[0], 6))
    return pos, Bodies(np.arange(c.shape[0] + 1, dtype=np.int64) * n_blobs, c, F), a
