"""Triangle-mesh generators.

Icosphere(L): regular icosahedron inscribed in the unit sphere, L rounds of
1->4 edge-midpoint subdivision, every new vertex re-projected to the unit
sphere; triangles counter-clockwise seen from outside, so the flat normal
points out of the bubble into the liquid.  Vertex / triangle
counts are 10*4^L+2 / 20*4^L -- the paper's own meshes have 642, 2562 and
10242 vertices.
"""
from __future__ import annotations

import functools
import numpy as np


def _icosahedron():
    t = (1.0 + 5.0 ** 0.5) / 2.0
    v = np.array(
        [
            [-1, t, 0], [1, t, 0], [-1, -t, 0], [1, -t, 0],
            [0, -1, t], [0, 1, t], [0, -1, -t], [0, 1, -t],
            [t, 0, -1], [t, 0, 1], [-t, 0, -1], [-t, 0, 1],
        ],
        dtype=np.float64,
    )
    v /= np.linalg.norm(v, axis=1, keepdims=True)
    f = np.array(
        [
            [0, 11, 5], [0, 5, 1], [0, 1, 7], [0, 7, 10], [0, 10, 11],
            [1, 5, 9], [5, 11, 4], [11, 10, 2], [10, 7, 6], [7, 1, 8],
            [3, 9, 4], [3, 4, 2], [3, 2, 6], [3, 6, 8], [3, 8, 9],
            [4, 9, 5], [2, 4, 11], [6, 2, 10], [8, 6, 7], [9, 8, 1],
        ],
        dtype=np.int64,
    )
    # make every face counter-clockwise seen from outside
    c = v[f].mean(axis=1)
    n = np.cross(v[f[:, 1]] - v[f[:, 0]], v[f[:, 2]] - v[f[:, 0]])
    flip = np.einsum("ij,ij->i", n, c) < 0
    f[flip] = f[flip][:, [0, 2, 1]]
    return v, f


def _subdivide(v, f):
    nv = v.shape[0]
    e = np.concatenate([f[:, [0, 1]], f[:, [1, 2]], f[:, [2, 0]]], axis=0)
    e.sort(axis=1)
    key = e[:, 0] * np.int64(nv) + e[:, 1]
    ukey, inv = np.unique(key, return_inverse=True)
    a = ukey // nv
    b = ukey % nv
    mid = v[a] + v[b]
    mid /= np.linalg.norm(mid, axis=1, keepdims=True)
    v2 = np.concatenate([v, mid], axis=0)
    nt = f.shape[0]
    m01 = nv + inv[:nt]
    m12 = nv + inv[nt:2 * nt]
    m20 = nv + inv[2 * nt:]
    f2 = np.concatenate(
        [
            np.stack([f[:, 0], m01, m20], axis=1),
            np.stack([f[:, 1], m12, m01], axis=1),
            np.stack([f[:, 2], m20, m12], axis=1),
            np.stack([m01, m12, m20], axis=1),
        ],
        axis=0,
    )
    return v2, f2


@functools.lru_cache(maxsize=None)
def _icosphere_cached(level: int):
    v, f = _icosahedron()
    for _ in range(level):
        v, f = _subdivide(v, f)
    v.setflags(write=False)
    f = f.astype(np.int32)
    f.setflags(write=False)
    return v, f


def icosphere(level: int):
    """Unit icosphere: (V[10*4^L+2, 3] float64, F[20*4^L, 3] int32)."""
    v, f = _icosphere_cached(int(level))
    return v.copy(), f.copy()


def deform_radial(v_unit, radius_fn):
    """Map unit-sphere vertices v -> r(theta, phi) * v (config 3)."""
    x, y, z = v_unit[:, 0], v_unit[:, 1], v_unit[:, 2]
    theta = np.arccos(np.clip(z, -1.0, 1.0))
    phi = np.arctan2(y, x)
    return v_unit * radius_fn(theta, phi)[:, None]


def cluster_mesh(level: int, centres, radii):
    """M copies of icosphere(level), scaled by radii[b] and moved to centres[b].

    Returns V[M*Nd, 3], F[M*Td, 3] int32, bubble_id[M*Nd] int32, and the unit
    template vertices tiled per bubble (angles for density recipes).
    No rotation of the template mesh.
    """
    v0, f0 = icosphere(level)
    centres = np.asarray(centres, dtype=np.float64).reshape(-1, 3)
    radii = np.asarray(radii, dtype=np.float64).reshape(-1)
    m = centres.shape[0]
    nd, td = v0.shape[0], f0.shape[0]
    V = (v0[None, :, :] * radii[:, None, None] + centres[:, None, :]).reshape(m * nd, 3)
    F = (f0[None, :, :].astype(np.int64) + (np.arange(m, dtype=np.int64) * nd)[:, None, None])
    F = F.reshape(m * td, 3).astype(np.int32)
    bid = np.repeat(np.arange(m, dtype=np.int32), nd)
    return np.ascontiguousarray(V), np.ascontiguousarray(F), bid


def lattice_cluster(level: int, nb: int, spacing: float, radius: float = 1.0):
    """The paper's own family: nb^3 equal bubbles on a regular grid with centre
    spacing 4*a0."""
    g = np.arange(nb, dtype=np.float64) * spacing
    cx, cy, cz = np.meshgrid(g, g, g, indexing="ij")
    centres = np.stack([cx.ravel(), cy.ravel(), cz.ravel()], axis=1)
    radii = np.full(centres.shape[0], radius)
    return cluster_mesh(level, centres, radii)
