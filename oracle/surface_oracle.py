"""CPU oracle of the steps either side of the solve in a time step:
vertex normals and areas, surface velocity, shape filter.

TEST INFRASTRUCTURE, NOT PRODUCT CODE (same rules as oracle/__init__.py): plain numpy in fp64,
every function the definition the paper prints, written out; nothing here is shared with the
CUDA library, and only tests/ and bench.py's cpu legs import it.

  vertex_geometry   Eq. 17: s_j = 1/3 sum_{k ni j} A_k,  n_j = m_j/|m_j|,  m_j = sum_{k ni j} N_k A_k
  surface_velocity  Eqs. 22-27: v_j = n_j q_j + (n x v)_j x n_j,
                    (n x v)_k A_k = 1/2 [ (r_k2 - r_k3) phi_k1 + (r_k3 - r_k1) phi_k2 + (r_k1 - r_k2) phi_k3 ]   (Eq. 26)
                    (n x v)_j = 1/(3 s_j) sum_{k ni j} (n x v)_k A_k                                            (Eq. 27)
  filter_matrix     Eqs. 37-42: F = G (G* G)^-1 G*, G_ij = Y_j(theta_i, phi_i), j = (n, m), n < p_f
  filter_apply      Eqs. 41, 43: xhat_l = F x_l for every bubble l and every surface function
  bubble_volumes    V_m of the polytropic gas law (Eq. 6; "volume" among the surface functions of PAPER.md:612):
                    the volume enclosed by the flat-triangle surface of bubble m, by the divergence theorem with the field r/3:
                    V_m = 1/3 sum_{k in bubble m} A_k N_k . c_k  (c_k the centroid; r . N is constant on a flat triangle)

Parity pinned by tests/test_oracle_pins.py (closed forms on the sphere, projector identities).
"""
from __future__ import annotations

import numpy as np
from scipy.special import sph_harm_y


def vertex_geometry(V, F):
    """(s [N], n [N,3], A [T], Ntri [T,3]) of Eq. 17."""
    V = np.asarray(V, dtype=np.float64)
    F = np.asarray(F, dtype=np.int64)
    e1 = V[F[:, 1]] - V[F[:, 0]]
    e2 = V[F[:, 2]] - V[F[:, 0]]
    cr = np.cross(e1, e2)
    A = 0.5 * np.linalg.norm(cr, axis=1)
    Ntri = cr / (2.0 * A)[:, None]
    N = V.shape[0]
    s = np.zeros(N)
    m = np.zeros((N, 3))
    for a in range(3):                       # sum over the triangles that hold vertex j at corner a
        np.add.at(s, F[:, a], A / 3.0)
        np.add.at(m, F[:, a], Ntri * A[:, None])
    n = m / np.linalg.norm(m, axis=1)[:, None]
    return s, n, A, Ntri


def bubble_volumes(V, F, bubble_id=None):
    """V_m = 1/3 sum_k A_k N_k . c_k over the triangles of bubble m (divergence theorem, F = r/3; N_k points out of the
    bubble).  The paper prints no formula for V_m (it only uses it in the gas law); for a
    closed flat-triangle surface this is its definition written out.  Returns [n_bubbles]."""
    V = np.asarray(V, dtype=np.float64)
    F = np.asarray(F, dtype=np.int64)
    _, _, A, Ntri = vertex_geometry(V, F)
    cen = (V[F[:, 0]] + V[F[:, 1]] + V[F[:, 2]]) / 3.0
    contrib = A * np.einsum("kd,kd->k", Ntri, cen) / 3.0
    if bubble_id is None:
        return np.array([contrib.sum()])
    b = np.asarray(bubble_id, dtype=np.int64)[F[:, 0]]
    vol = np.zeros(int(b.max()) + 1)
    np.add.at(vol, b, contrib)
    return vol


def surface_velocity(V, F, phi, q):
    """v [N,3]: v_j = n_j q_j + v_tj (Eq. 22), tangential part by the contour integrals of Eqs. 23-27."""
    V = np.asarray(V, dtype=np.float64)
    F = np.asarray(F, dtype=np.int64)
    phi = np.asarray(phi, dtype=np.float64)
    q = np.asarray(q, dtype=np.float64)
    s, n, _, _ = vertex_geometry(V, F)
    r1, r2, r3 = V[F[:, 0]], V[F[:, 1]], V[F[:, 2]]
    f1, f2, f3 = phi[F[:, 0]], phi[F[:, 1]], phi[F[:, 2]]
    nxvA = 0.5 * ((r2 - r3) * f1[:, None] + (r3 - r1) * f2[:, None] + (r1 - r2) * f3[:, None])    # Eq. 26 times A_k
    acc = np.zeros_like(V)
    for a in range(3):
        np.add.at(acc, F[:, a], nxvA)
    nxv = acc / (3.0 * s)[:, None]                                                                 # Eq. 27
    vt = np.cross(nxv, n)
    return n * q[:, None] + vt


def harmonic_matrix(theta, phi, p_f):
    """G [N_d, p_f^2] of Eq. 39 in the real orthonormal basis (the projector of Eq. 42 only depends on the span:
    {Re Y_n^m, Im Y_n^m} spans what {Y_n^m, m = -n..n} spans).  theta = polar angle, phi = azimuth."""
    theta = np.asarray(theta, dtype=np.float64)
    phi = np.asarray(phi, dtype=np.float64)
    cols = []
    for n in range(p_f):
        cols.append(np.real(sph_harm_y(n, 0, theta, phi)))
        for m in range(1, n + 1):
            y = sph_harm_y(n, m, theta, phi)
            cols.append(np.sqrt(2.0) * np.real(y))
            cols.append(np.sqrt(2.0) * np.imag(y))
    return np.stack(cols, axis=1)


def filter_matrix(theta, phi, p_f):
    """F = G (G* G)^-1 G* (Eq. 42) by least squares (Eq. 40)."""
    G = harmonic_matrix(theta, phi, p_f)
    Gp = np.linalg.lstsq(G, np.eye(G.shape[0]), rcond=None)[0]       # pseudoinverse G^(-1) of Eq. 40
    return G @ Gp


def filter_apply(Fm, x):
    """xhat[c, :] = F x[c, :] for every column c = (surface function, bubble): x is [n_cols, N_d] (Eqs. 41, 43)."""
    x = np.asarray(x, dtype=np.float64)
    return x @ Fm.T


def one_ring_first_five(F, N):
    """The five neighbours of every vertex used by the paraboloid fit ("when more than 5 neighbors are
    available, we use just 5" -- which five is not said; reading R32 of DESIGN.md): walk the triangles that hold the
    vertex in mesh order (triangle index, then corner index), and of each take the two other vertices in the
    triangle's cyclic order; keep the first five distinct ones.  Returns [N, 5] (-1 where a vertex has fewer)."""
    F = np.asarray(F, dtype=np.int64)
    ring = [[] for _ in range(N)]
    for k in range(F.shape[0]):
        for a in range(3):
            j = int(F[k, a])
            for b in (F[k, (a + 1) % 3], F[k, (a + 2) % 3]):
                b = int(b)
                if b not in ring[j] and len(ring[j]) < 5:
                    ring[j].append(b)
    out = -np.ones((N, 5), dtype=np.int64)
    for j, r in enumerate(ring):
        out[j, :len(r)] = r
    return out


def mean_curvature(V, F):
    """H_j = -B_j^(3) - B_j^(5) (Eq. 29) from the paraboloid z = B1 x + B2 y + B3 x^2 + B4 x y + B5 y^2 through five
    neighbours (Eq. 28), in a frame centred at r_j whose z axis is the vertex normal n_j of Eq. 17.  The sum B3 + B5 does
    not depend on the choice of the x, y axes.  Positive for a sphere with the normal out of the bubble: H = 1/R."""
    V = np.asarray(V, dtype=np.float64)
    N = V.shape[0]
    _, n, _, _ = vertex_geometry(V, F)
    ring = one_ring_first_five(F, N)
    H = np.zeros(N)
    for j in range(N):
        if ring[j].min() < 0:
            H[j] = np.nan
            continue
        z = n[j]
        a = np.array([1.0, 0.0, 0.0]) if abs(z[0]) < 0.9 else np.array([0.0, 1.0, 0.0])
        ex = np.cross(z, a); ex /= np.linalg.norm(ex)
        ey = np.cross(z, ex)
        d = V[ring[j]] - V[j]
        x, y, zz = d @ ex, d @ ey, d @ z
        Q = np.stack([x, y, x * x, x * y, y * y], axis=1)            # Eq. 28
        B = np.linalg.solve(Q, zz)
        H[j] = -B[2] - B[4]                                           # Eq. 29
    return H
