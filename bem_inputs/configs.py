"""The five BASELINE.json configurations as seeded synthetic inputs
(SURVEY.md §8(d) D1).  Seeds: 190501341 + cfg; the 2000-row parity sample uses
190501341 + 100 + cfg.  These stand in for the paper's own bubble clusters
(regular grids of 642-vertex bubbles); no dataset is used.
"""
from __future__ import annotations

import numpy as np

from .meshes import icosphere, cluster_mesh, deform_radial
from .sph import real_sph_harm, real_sph_harm_im

CONFIG_SEED0 = 190501341
N_CONFIGS = 5

# expansion order p, leaf size and near radius eta used with each config
CONFIG_PARAMS = {
    1: dict(p=8, leaf_size=64, eta=2.5),
    2: dict(p=10, leaf_size=64, eta=2.5),
    3: dict(p=10, leaf_size=64, eta=2.5),
    4: dict(p=10, leaf_size=96, eta=2.5),
    5: dict(p=12, leaf_size=256, eta=2.5),
}


def _angles(v_unit):
    theta = np.arccos(np.clip(v_unit[:, 2], -1.0, 1.0))
    phi = np.arctan2(v_unit[:, 1], v_unit[:, 0])
    return theta, phi


def _place_bubbles(rng, n, side, sigma, gap=1.1):
    """radii lognormal(0, sigma) drawn first, in order; centres by rejection:
    c ~ U(r, side-r)^3, accepted iff |c - c_j| >= gap (r + r_j) for all accepted j."""
    radii = rng.lognormal(mean=0.0, sigma=sigma, size=n)
    centres = np.zeros((n, 3))
    k = 0
    draws = 0
    while k < n:
        r = radii[k]
        c = rng.uniform(r, side - r, size=3)
        draws += 1
        if k == 0 or np.all(
            np.linalg.norm(centres[:k] - c, axis=1) >= gap * (r + radii[:k])
        ):
            centres[k] = c
            k += 1
        if draws > 200 * n:
            raise RuntimeError("bubble placement did not converge")
    return centres, radii


def make_config(cfg: int, n_bubbles: int | None = None):
    """Return dict(V, F, bubble_id, q, phi, p, leaf_size, eta, name).

    `n_bubbles` shrinks configs 4/5 (same recipe, same seed, fewer bubbles and
    a cube scaled to keep the number density) for tests that must run in seconds.
    """
    rng = np.random.default_rng(CONFIG_SEED0 + cfg)
    if cfg == 1:
        v0, F = icosphere(3)
        V = v0.copy()
        bid = np.zeros(V.shape[0], dtype=np.int32)
        th, ph = _angles(v0)
        q = real_sph_harm(3, 1, th, ph) + rng.uniform(-1e-2, 1e-2, size=V.shape[0])
        phi = np.ones(V.shape[0])
        name = "cfg1: sphere R=1, icosphere L3, 642 nodes"
    elif cfg == 2:
        g = np.arange(3, dtype=np.float64) * 3.0
        cx, cy, cz = np.meshgrid(g, g, g, indexing="ij")
        centres = np.stack([cx.ravel(), cy.ravel(), cz.ravel()], axis=1)
        radii = rng.uniform(0.9, 1.1, size=27)
        V, F, bid = cluster_mesh(4, centres, radii)
        q = rng.uniform(-1.0, 1.0, size=V.shape[0])
        phi = rng.uniform(-1.0, 1.0, size=V.shape[0])
        name = "cfg2: 27 bubbles 3x3x3, icosphere L4, 69,174 nodes"
    elif cfg == 3:
        v0, F = icosphere(7)
        rad = lambda t, p: 1.0 + 0.3 * real_sph_harm(4, 2, t, p) + 0.15 * real_sph_harm(6, 3, t, p)
        V = deform_radial(v0, rad)
        bid = np.zeros(V.shape[0], dtype=np.int32)
        th, ph = _angles(v0)
        phi = np.zeros(V.shape[0])
        for n in range(0, 9):
            for m in range(0, n + 1):
                a = rng.normal()
                phi += a * real_sph_harm(n, m, th, ph)
                if m > 0:
                    b = rng.normal()
                    phi += b * real_sph_harm_im(n, m, th, ph)
        q = rng.normal(size=V.shape[0])
        name = "cfg3: deformed bubble, icosphere L7, 163,842 nodes"
    elif cfg in (4, 5):
        n_full, side, sigma = (1000, 40.0, 0.25) if cfg == 4 else (4000, 64.0, 0.3)
        n = n_full if n_bubbles is None else int(n_bubbles)
        if n != n_full:
            side = side * (n / n_full) ** (1.0 / 3.0)
        centres, radii = _place_bubbles(rng, n, side, sigma)
        V, F, bid = cluster_mesh(3, centres, radii)
        q = rng.uniform(-1.0, 1.0, size=V.shape[0])
        phi = rng.uniform(-1.0, 1.0, size=V.shape[0])
        name = f"cfg{cfg}: {n} bubbles in cube {side:.3g}, icosphere L3, {V.shape[0]:,} nodes"
    else:
        raise ValueError("cfg must be 1..5")
    # unit-sphere template whose vertex angles every bubble of the config keeps (the correspondence point index ->
    # (theta, phi) of the shape filter); the bubbles follow each other in V, template order inside each
    template = {1: 3, 2: 4, 3: 7, 4: 3, 5: 3}[cfg]
    out = dict(V=np.ascontiguousarray(V), F=np.ascontiguousarray(F, dtype=np.int32),
               bubble_id=bid, q=q, phi=phi, name=name, cfg=cfg, template=icosphere(template)[0])
    out.update(CONFIG_PARAMS[cfg])
    return out


def sample_rows(cfg: int, n_nodes: int, n_rows: int = 2000):
    """The seeded random target rows of the large-config parity check."""
    rng = np.random.default_rng(CONFIG_SEED0 + 100 + cfg)
    n_rows = min(n_rows, n_nodes)
    return np.sort(rng.choice(n_nodes, n_rows, replace=False)).astype(np.int64)


def random_cube_points(n: int, seed: int):
    """Uniform random points in the unit cube with unit-scale monopole strengths:
    the workload of the paper's Tables 1-2."""
    rng = np.random.default_rng(seed)
    pts = rng.uniform(0.0, 1.0, size=(n, 3))
    strengths = rng.uniform(0.0, 1.0, size=n)
    return pts, strengths
