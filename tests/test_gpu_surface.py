"""Parity of the surface functions and the shape filter (include/bem.h: bem_surface_velocity,
bem_filter_*) with the numpy oracle (oracle/surface_oracle.py), element by element on seeded inputs.  fp64 on both
sides, different summation orders: tolerance 1e-12 relative for the surface functions, 1e-10 for the filter (it goes
through a Cholesky factorisation of G^T G on the device and a least-squares solve in the oracle)."""
import numpy as np
import pytest

import bem_inputs as bi
from bem_inputs.configs import make_config
from bem_inputs.sph import real_sph_harm
from oracle import surface_oracle as so

pytestmark = pytest.mark.gpu


def _bem():
    import paper_1905_01341_b200 as bem
    return bem


def _angles(v):
    return np.arccos(np.clip(v[:, 2] / np.linalg.norm(v, axis=1), -1, 1)), np.arctan2(v[:, 1], v[:, 0])


def _maxrel(a, b):
    return np.max(np.abs(a - b)) / np.max(np.abs(b))


@pytest.mark.parametrize("case", ["sphere", "deformed", "cluster"])
def test_surface_velocity_matches_oracle(case):
    rng = np.random.default_rng(190501341 + 31)
    if case == "sphere":
        V, F = bi.icosphere(3)
    elif case == "deformed":
        v, F = bi.icosphere(5)
        th, ph = _angles(v)
        V = (1.0 + 0.3 * real_sph_harm(4, 2, th, ph) + 0.15 * real_sph_harm(6, 3, th, ph))[:, None] * v
    else:
        c = make_config(4, n_bubbles=40)
        V, F = c["V"], c["F"]
    N = V.shape[0]
    phi, q = rng.uniform(-1, 1, N), rng.uniform(-1, 1, N)
    ctx = _bem().bem_create(V, F)
    v, n, s = np.full((N, 3), np.nan), np.full((N, 3), np.nan), np.full(N, np.nan)
    ctx.bem_surface_velocity(phi, q, v, n, s)
    so_s, so_n, _, _ = so.vertex_geometry(V, F)
    so_v = so.surface_velocity(V, F, phi, q)
    assert _maxrel(s, so_s) <= 1e-12 and _maxrel(n, so_n) <= 1e-12 and _maxrel(v, so_v) <= 1e-12
    # tangential part only (q = NULL), device pointers, twice the same bits
    import torch
    pd = torch.tensor(phi, device="cuda")
    v1, v2 = torch.empty(N, 3, dtype=torch.float64, device="cuda"), torch.empty(N, 3, dtype=torch.float64, device="cuda")
    ctx.bem_surface_velocity(pd, None, v1)
    ctx.bem_surface_velocity(pd, None, v2)
    torch.cuda.synchronize()
    assert torch.equal(v1, v2)
    assert _maxrel(v1.cpu().numpy(), so.surface_velocity(V, F, phi, np.zeros(N))) <= 1e-12
    # outputs may be left out one by one
    s2 = np.full(N, np.nan)
    ctx.bem_surface_velocity(None, None, None, None, s2)
    assert np.array_equal(s, s2)
    with pytest.raises(_bem().BemError):
        ctx.bem_surface_velocity(None, None, v)                     # velocity without phi
    ctx.bem_destroy()


def test_surface_velocity_rejects_point_clouds():
    pts = np.random.default_rng(3).uniform(size=(100, 3))
    ctx = _bem().bem_create_points(pts, pts)
    with pytest.raises(_bem().BemError):
        ctx.bem_surface_velocity(np.zeros(100), None, np.zeros((100, 3)))
    ctx.bem_destroy()


@pytest.mark.parametrize("lvl,p_f", [(3, 9), (3, 1), (2, 12), (4, 16)])
def test_filter_matches_oracle(lvl, p_f):
    """Eq. 41 / 43 on the coordinates and the potential of a cluster whose bubbles share the template angles."""
    rng = np.random.default_rng(190501341 + 32 + lvl)
    v, _ = bi.icosphere(lvl)
    th, ph = _angles(v)
    nd = v.shape[0]
    Fm = so.filter_matrix(th, ph, p_f)
    nb = 37                                                         # 4 x 37 = 148 columns: ragged last group of 8
    radii = rng.lognormal(0.0, 0.3, nb)
    cols = []
    for b in range(nb):
        Vb = radii[b] * (1.0 + 0.2 * real_sph_harm(3, 2, th, ph))[:, None] * v + rng.uniform(-20, 20, 3) + 1e-3 * rng.standard_normal((nd, 3))
        cols += [Vb[:, 0], Vb[:, 1], Vb[:, 2], rng.uniform(-1, 1, nd)]
    X = np.ascontiguousarray(np.stack(cols))
    ref = so.filter_apply(Fm, X)
    flt = _bem().bem_filter_create(th, ph, p_f)
    out = np.full_like(X, np.nan)
    flt.bem_filter_apply(X, X.shape[0], out)
    assert _maxrel(out, ref) <= 1e-10
    import torch
    xd = torch.tensor(X, device="cuda")
    flt.bem_filter_apply(xd, X.shape[0], xd)                        # in place, device pointers
    torch.cuda.synchronize()
    assert np.array_equal(xd.cpu().numpy(), out)
    flt.bem_filter_apply(xd, X.shape[0], xd)                        # a projector: filtering twice changes nothing
    torch.cuda.synchronize()
    assert _maxrel(xd.cpu().numpy(), out) <= 1e-11
    one = np.full(nd, np.nan)
    flt.bem_filter_apply(np.ascontiguousarray(X[5]), 1, one)
    assert np.array_equal(one, out[5])
    flt.bem_filter_apply(X, 0, out)                                 # empty batch
    flt.bem_filter_destroy()


def test_filter_large_batch_takes_the_tensor_path():
    """2048 columns and more run as two DMMA GEMMs (filter_apply_dmma): same tolerance against the oracle, ragged last
    warp (2051 columns), in place, and equal to the FMA kernel's result on a small batch of the same columns to rounding."""
    rng = np.random.default_rng(190501341 + 40)
    v, _ = bi.icosphere(3)
    th, ph = _angles(v)
    nd = v.shape[0]
    for p_f in (9, 4, 10):
        Fm = so.filter_matrix(th, ph, p_f)
        X = rng.standard_normal((2051, nd))
        ref = so.filter_apply(Fm, X)
        flt = _bem().bem_filter_create(th, ph, p_f)
        out = np.full_like(X, np.nan)
        flt.bem_filter_apply(X, X.shape[0], out)
        assert _maxrel(out, ref) <= 1e-10
        small = np.full((64, nd), np.nan)
        flt.bem_filter_apply(np.ascontiguousarray(X[:64]), 64, small)
        assert _maxrel(small, out[:64]) <= 1e-12
        import torch
        xd = torch.tensor(X, device="cuda")
        flt.bem_filter_apply(xd, X.shape[0], xd)
        torch.cuda.synchronize()
        assert np.array_equal(xd.cpu().numpy(), out)
        flt.bem_filter_destroy()


def test_filter_argument_checks():
    bem = _bem()
    v, _ = bi.icosphere(1)                                          # 42 points
    th, ph = _angles(v)
    for p_f in (0, 7, 17):                                          # p_f^2 must stay below n_d; p_f <= 16
        with pytest.raises(bem.BemError) as e:
            bem.bem_filter_create(th, ph, p_f)
        assert e.value.status == bem.BEM_ERR_INVALID_ARG
    with pytest.raises(bem.BemError) as e:                          # all points on one meridian: the band is not resolved
        bem.bem_filter_create(np.linspace(0.1, 3.0, 42), np.zeros(42), 4)
    assert e.value.status == bem.BEM_ERR_BAD_MESH


@pytest.mark.parametrize("case", ["sphere", "deformed", "cluster"])
def test_surface_curvature_matches_oracle(case):
    """Eqs. 28-29: same five neighbours on both sides (reading R32), the solution of a 5 x 5 system each: relative 1e-9
    (the systems have condition numbers up to ~1e4 on the finest meshes); 1/R on spheres within the paper's 1%."""
    if case == "sphere":
        v, F = bi.icosphere(3)
        V = 1.6 * v + 0.4
    elif case == "deformed":
        v, F = bi.icosphere(4)
        th, ph = _angles(v)
        V = (1.0 + 0.3 * real_sph_harm(4, 2, th, ph) + 0.15 * real_sph_harm(6, 3, th, ph))[:, None] * v
    else:
        c = make_config(4, n_bubbles=12)
        V, F = c["V"], c["F"]
    N = V.shape[0]
    ctx = _bem().bem_create(V, F)
    H = np.full(N, np.nan)
    ctx.bem_surface_curvature(H)
    ref = so.mean_curvature(V, F)
    assert np.all(np.isfinite(H)) and np.max(np.abs(H - ref)) <= 1e-9 * np.max(np.abs(ref))
    if case == "sphere":
        assert np.max(np.abs(1.6 * H - 1.0)) < 1e-2
    import torch
    hd = torch.empty(N, dtype=torch.float64, device="cuda")
    ctx.bem_surface_curvature(hd)
    torch.cuda.synchronize()
    assert np.array_equal(hd.cpu().numpy(), H)
    ctx.bem_destroy()


def test_bubble_volume_matches_oracle():
    """bem_bubble_volume against oracle bubble_volumes: a cluster of 40 polydisperse bubbles in a
    cube of side 40 (far from the origin: the kernel sums tetrahedra from a vertex of the bubble, the oracle uses
    A_k N_k . c_k / 3 about the origin -- different formulas, both exact for the polyhedron), a single mesh without
    ids, host and device outputs, the same bits on a second call, and the size check."""
    import torch
    bem = _bem()
    c = make_config(4, n_bubbles=40)
    V, F, bid = c["V"], c["F"], c["bubble_id"]
    ctx = bem.bem_create(V, F, bid)
    nb = int(bid.max()) + 1
    vo = so.bubble_volumes(V, F, bid)
    vh = np.full(nb, np.nan)
    ctx.bem_bubble_volume(vh)
    assert _maxrel(vh, vo) <= 1e-12 and (vh > 0).all()
    vd = torch.full((nb,), float("nan"), dtype=torch.float64, device="cuda")
    ctx.bem_bubble_volume(vd)
    assert np.array_equal(vd.cpu().numpy(), vh)
    with pytest.raises(bem.BemError):
        ctx.bem_bubble_volume(np.zeros(nb + 1))
    ctx.bem_destroy()
    # one bubble, no ids, shifted off the origin: translation must not cost digits
    v, f = bi.icosphere(4)
    ctx = bem.bem_create(0.7 * v + np.array([100.0, -50.0, 25.0]), f, None)
    one = np.zeros(1)
    ctx.bem_bubble_volume(one)
    assert abs(one[0] - so.bubble_volumes(0.7 * v, f)[0]) <= 1e-12 * one[0]
    assert 0.99 < one[0] / (4 * np.pi * 0.7 ** 3 / 3) < 1.0
    ctx.bem_destroy()
