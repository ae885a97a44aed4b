"""Independent numpy helpers for the oracle pins (test code only: shares nothing
with oracle/ or the CUDA library)."""
import numpy as np


def tri_areas_normals(V, F):
    e1 = V[F[:, 1]] - V[F[:, 0]]
    e2 = V[F[:, 2]] - V[F[:, 0]]
    cr = np.cross(e1, e2)
    nn = np.linalg.norm(cr, axis=1)
    return 0.5 * nn, cr / nn[:, None]


def interior_solid_angle(V, F, i):
    """Solid angle of the polyhedron interior seen from vertex i: the spherical
    polygon of the one-ring edge directions, area = sum(angles) - (n-2) pi."""
    tris = [t for t in F if i in t]
    # order the ring: triangle (i, a, b) counter-clockwise seen from outside
    nxt = {}
    for t in tris:
        k = list(t).index(i)
        a, b = t[(k + 1) % 3], t[(k + 2) % 3]
        nxt[a] = b
    start = next(iter(nxt))
    ring = [start]
    while nxt[ring[-1]] != start:
        ring.append(nxt[ring[-1]])
    u = V[ring] - V[i]
    u /= np.linalg.norm(u, axis=1, keepdims=True)
    n = len(ring)
    ang = 0.0
    for k in range(n):
        a, b, c = u[k - 1], u[k], u[(k + 1) % n]
        # interior angle at b of the spherical polygon: angle between the great
        # circle arcs b->a and b->c, i.e. between tangent vectors at b
        ta = a - np.dot(a, b) * b
        tc = c - np.dot(c, b) * b
        # signed angle from ta to tc about the axis b (the ring runs counter-clockwise
        # seen from outside, so the body lies on the side where this angle is the
        # interior one); reflex angles (> pi) occur at non-convex vertices
        w = np.arctan2(np.dot(b, np.cross(ta, tc)), np.dot(tc, ta))
        ang += w if w >= 0 else w + 2 * np.pi
    excess = ang - (n - 2) * np.pi
    # the ring is counter-clockwise seen from OUTSIDE, i.e. the polygon bounds the
    # set of directions pointing INTO the body when the vertex is convex
    return excess


def brute_triangle_integrals(tri, x, depth=5, ngl=12):
    """int_T lambda_a/(4 pi r) and int_T lambda_a N.(x-y)/(4 pi r^3) by uniform 4^depth
    subdivision with a collapsed tensor Gauss-Legendre rule on every piece (numpy)."""
    tri = np.asarray(tri, float).reshape(3, 3)
    x = np.asarray(x, float)
    N = np.cross(tri[1] - tri[0], tri[2] - tri[0])
    N /= np.linalg.norm(N)
    # barycentric corners of all sub-triangles
    corners = [np.eye(3)]
    for _ in range(depth):
        new = []
        for c in corners:
            a, b, d = c
            ab, bd, da = (a + b) / 2, (b + d) / 2, (d + a) / 2
            new += [np.array([a, ab, da]), np.array([b, bd, ab]), np.array([d, da, bd]), np.array([ab, bd, da])]
        corners = new
    B = np.array(corners)                       # [M, 3 corners, 3 bary]
    g, w = np.polynomial.legendre.leggauss(ngl)
    g = 0.5 * (g + 1); w = 0.5 * w
    s, t = np.meshgrid(g, g, indexing="ij")
    ws = (w[:, None] * w[None, :] * s).ravel()
    s = s.ravel(); t = t.ravel()
    loc = np.stack([1 - s, s * (1 - t), s * t], axis=1)      # [Q, 3] local bary in sub-triangle
    lam = np.einsum("qc,mcb->mqb", loc, B)                   # [M, Q, 3] root barycentrics
    y = lam @ tri                                            # [M, Q, 3]
    area = 0.5 * np.linalg.norm(np.cross(tri[1] - tri[0], tri[2] - tri[0]))
    jac = 2.0 * area / 4 ** depth
    d = x - y
    r = np.linalg.norm(d, axis=2)
    kS = ws[None, :] * jac / (4 * np.pi * r)
    kD = ws[None, :] * jac * (d @ N) / (4 * np.pi * r ** 3)
    WS = np.einsum("mq,mqb->b", kS, lam)
    WD = np.einsum("mq,mqb->b", kD, lam)
    return WS, WD
