"""Point clouds with dipoles, the FMM operators one chain at a time (SURVEY.md 8(c) pin P11) and the off-surface
evaluator (Eq. 11, r not on S), all through the C-ABI against the CPU oracle.  `pytest -m gpu`."""
import numpy as np
import pytest

import bem_inputs as bi
from bem_inputs.configs import make_config
import oracle

pytestmark = pytest.mark.gpu


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _bem():
    import paper_1905_01341_b200 as bem
    return bem


def _cloud_apply(src, tgt, m, d, p, leaf=64, **opts):
    ctx = _bem().bem_create_points(src, tgt)
    for k, v in opts.items():
        ctx.bem_set_option(k, v)
    ctx.bem_setup(p, leaf, 2.5)
    y = np.full(tgt.shape[0], np.nan)
    ctx.bem_apply(m, d, y)
    st = ctx.bem_get_stats()
    ctx.bem_destroy()
    assert np.isfinite(y).all()
    return y, st


# ------------------------------------------------------------------ dipole clouds
def test_dipole_cloud_direct_and_fmm():
    """bem_create_points with monopole and dipole sources (Eq. 13 in point form): direct mode to 1e-12, FMM at p = 12 to
    the north_star's 1e-5, each layer alone and both together; sources and targets coincide (r = 0 pairs skipped)."""
    rng = np.random.default_rng(31)
    n = 20000
    pts = rng.uniform(0, 1, size=(n, 3))
    m = rng.uniform(-1, 1, size=n)
    d = rng.normal(size=(n, 3)) * 0.02
    rows = np.sort(rng.choice(n, 400, replace=False))
    for mm, dd in ((m, d), (None, d), (m, None)):
        yo = oracle.point_sum(pts, mm, dd, pts[rows])
        y, _ = _cloud_apply(pts, pts, mm, dd, 12, mode=1)
        assert _rel(y[rows], yo) <= 1e-12
        y, st = _cloud_apply(pts, pts, mm, dd, 12)
        e = _rel(y[rows], yo)
        print("cloud", "m" if mm is not None else "-", "d" if dd is not None else "-", f"{e:.2e}", "lmax", st["lmax"])
        assert st["m2l_pairs"] > 0 and e <= 1e-5
    y32, _ = _cloud_apply(pts, pts, m, d, 12, p2p_precision=1)
    assert _rel(y32[rows], oracle.point_sum(pts, m, d, pts[rows])) <= 1e-5


# ------------------------------------------------------------------ P11: the operators, one chain at a time
def _two_clusters(rng, cs, ct, half, ns=60, nt=40):
    """ns sources in a small cube around cs, nt targets around ct, plus two zero-strength sources at the corners of the
    unit cube so that the octree's cube IS the unit cube and the box grid is known."""
    src = np.vstack([cs + rng.uniform(-half, half, size=(ns, 3)), [[0.0, 0.0, 0.0], [1.0, 1.0, 1.0]]])
    tgt = ct + rng.uniform(-half, half, size=(nt, 3))
    m = np.append(rng.uniform(0.5, 1.5, size=ns), [0.0, 0.0])
    d = np.vstack([rng.normal(size=(ns, 3)), np.zeros((2, 3))]) * 0.05
    return src, tgt, m, d


CHAINS = {
    # name: (lmax, source cluster centre, target cluster centre)
    "P2M-M2L-L2P at level 2": (2, [0.125, 0.125, 0.125], [0.875, 0.375, 0.625]),
    # level-3 boxes (1,1,1) and (6,2,5): their parents (0,0,0), (3,1,2) are not neighbours, so the pair meets at level 2.
    # M2M and L2L are exact on the degrees kept, so the truncation error is set by the distance of the clusters from the
    # LEVEL-2 centres (0.125, ..) and (0.875, 0.375, 0.625) -- corners of the level-3 boxes; the clusters sit next to them
    "P2M-M2M-M2L-L2L-L2P": (3, [0.135, 0.135, 0.135], [0.865, 0.365, 0.635]),
    # level-3 boxes (1,1,1) and (3,1,1): two apart, parents (0,0,0), (1,0,0) adjacent -> translated at level 3 itself
    "P2M-M2L-L2P at level 3": (3, [0.1875, 0.1875, 0.1875], [0.4375, 0.1875, 0.1875]),
    # a diagonal offset (2, -3, 3) between level-3 boxes of neighbouring parents: every azimuth and class of the M2L table
    "P2M-M2L-L2P, oblique offset": (3, [0.1875, 0.4375, 0.0625], [0.4375, 0.0625, 0.4375]),
}


@pytest.mark.parametrize("chain", list(CHAINS))
@pytest.mark.parametrize("p,tol", [(20, 1e-13), (16, 2e-12)])
def test_fmm_operator_chains(chain, p, tol):
    """SURVEY.md 8(c) pin P11: each FMM operator against the direct sum for ONE well-separated pair of boxes, monopole
    and dipole sources apart.  The clusters are much smaller than their boxes, so the truncation error at p = 16 / 20 is
    below rounding and what is left is the arithmetic of P2M, M2M, M2L, L2L, L2P themselves: a wrong coefficient, sign
    or index in any of them (the dipole gradient of P2M included) shows at O(1).  p = 20 runs the any-p kernels (plain
    FMA tiles), p = 16 the template kernels and the FP64 tensor tiles.  direct_pairs = 0 keeps the pair in the far field;
    the graded truncation of the M2L tiles is on (default) -- it must not cost accuracy here either."""
    lmax, cs, ct = CHAINS[chain]
    rng = np.random.default_rng(5)
    src, tgt, m, d = _two_clusters(rng, np.array(cs), np.array(ct), 0.008)
    for name, mm, dd in (("monopoles", m, None), ("dipoles", None, d), ("both", m, d)):
        yo = oracle.point_sum(src, mm, dd, tgt)
        y, st = _cloud_apply(src, tgt, mm, dd, p, lmax=lmax, direct_pairs=0, dipole_degrees=0)
        e = _rel(y, yo)
        print(f"{chain} p={p} {name}: {e:.2e} (m2l pairs {st['m2l_pairs']:.0f}, p2p pairs {st['p2p_pairs']:.0f})")
        assert st["lmax"] == lmax and st["m2l_pairs"] >= 1 and st["p2p_pairs"] == 0      # nothing reaches the targets directly
        assert e <= tol, (name, e)


def test_fmm_operator_chain_truncation_rate():
    """The same pair of boxes with clusters that FILL a fraction of their boxes: the error falls geometrically with p
    and dipoles sit above monopoles by about four degrees (they are one derivative of the same expansion)."""
    lmax, cs, ct = CHAINS["P2M-M2L-L2P at level 3"]
    rng = np.random.default_rng(6)
    src, tgt, m, d = _two_clusters(rng, np.array(cs), np.array(ct), 0.045, ns=200, nt=100)
    yoM, yoD = oracle.point_sum(src, m, None, tgt), oracle.point_sum(src, None, d, tgt)
    eM, eD = {}, {}
    for p in (4, 8, 12, 16):
        eM[p] = _rel(_cloud_apply(src, tgt, m, None, p, lmax=lmax, direct_pairs=0, dipole_degrees=0)[0], yoM)
        eD[p] = _rel(_cloud_apply(src, tgt, None, d, p, lmax=lmax, direct_pairs=0, dipole_degrees=0)[0], yoD)
    print("monopoles", {p: f"{e:.1e}" for p, e in eM.items()}, "dipoles", {p: f"{e:.1e}" for p, e in eD.items()})
    for a, b in ((4, 8), (8, 12), (12, 16)):
        assert eM[b] < 0.05 * eM[a] and eD[b] < 0.05 * eD[a]
    for p in eM:
        assert eD[p] > eM[p]
    for p in (4, 8, 12):                                     # about four degrees behind (R5')
        assert eD[p + 4] <= 10.0 * eM[p], (p, eD[p + 4], eM[p])


# ------------------------------------------------------------------ off-surface evaluation
def _shell_points(V, rng, n):
    """points at random distances 0.03 .. 2 from a star-shaped surface around the origin, inside and outside"""
    k = rng.choice(V.shape[0], n)
    s = np.concatenate([rng.uniform(0.3, 0.97, n // 3), rng.uniform(1.03, 3.0, n - n // 3)])
    jitter = rng.normal(size=(n, 3)) * 0.02
    return V[k] * s[:, None] + jitter


@pytest.mark.parametrize("name", ["sphere", "deformed"])
def test_evaluator_matches_oracle(name):
    rng = np.random.default_rng(41)
    V, F = bi.icosphere(3)
    if name == "deformed":
        V = bi.deform_radial(V, lambda t, p: 1 + 0.3 * bi.real_sph_harm(4, 2, t, p) + 0.15 * bi.real_sph_harm(6, 3, t, p))
    q, ph = rng.normal(size=V.shape[0]), rng.normal(size=V.shape[0])
    X = _shell_points(V, rng, 3000)
    bem = _bem()
    mesh = bem.bem_create(V, F, None)
    yo = {k: oracle.g3_evaluate(V, F, a, b, X, eta=2.5) for k, (a, b) in (("both", (q, ph)), ("S", (q, None)), ("D", (None, ph)))}
    for mode, p, tol in ((1, 8, 1e-12), (0, 12, 1e-5), (0, 24, 1e-8)):
        ev = bem.bem_create_evaluator(mesh, X)
        ev.bem_set_option("mode", mode)
        ev.bem_setup(p, 64, 2.5)
        for k, (a, b) in (("both", (q, ph)), ("S", (q, None)), ("D", (None, ph))):
            u = np.full(X.shape[0], np.nan)
            ev.bem_apply(a, b, u)
            e = _rel(u, yo[k])
            print(f"evaluator {name} mode {mode} p {p} {k}: {e:.2e}")
            assert np.isfinite(u).all() and e <= tol
        st = ev.bem_get_stats()
        assert st["csr_nnz"] > 0 and st["n_targets"] == X.shape[0] and st["n_sources"] == 3 * F.shape[0]
        ev.bem_destroy()
    mesh.bem_destroy()


def test_evaluator_greens_representation_and_errors():
    """Eq. 11: u = S[q] - D[phi] is -phi in the liquid and 0 inside the bubble for a harmonic exterior field
    (a point source inside); -D[1] is 1 inside and 0 outside.  On device tensors, with a mesh context that was never set up."""
    import torch
    bem = _bem()
    V, F = bi.icosphere(4)
    z = np.array([0.15, -0.1, 0.05])
    phi_at = lambda P: 1.0 / (4 * np.pi * np.linalg.norm(P - z, axis=1))
    r = V - z
    q = -(r * V).sum(1) / (4 * np.pi * np.linalg.norm(r, axis=1) ** 3)
    rng = np.random.default_rng(43)
    X = _shell_points(V, rng, 2000)
    inside = np.linalg.norm(X, axis=1) < 1.0
    mesh = bem.bem_create(V, F, None)
    ev = bem.bem_create_evaluator(mesh, X)
    ev.bem_setup(12, 64, 2.5)
    u = torch.empty(X.shape[0], dtype=torch.float64, device="cuda")
    ev.bem_apply(torch.tensor(q, device="cuda"), torch.tensor(phi_at(V), device="cuda"), u)
    expect = np.where(inside, 0.0, -phi_at(X))
    assert np.abs(u.cpu().numpy() - expect).max() <= 2e-3 * np.abs(expect).max()          # O(h^2) of the mesh
    ev.bem_apply(None, torch.ones(V.shape[0], dtype=torch.float64, device="cuda"), u)
    assert np.abs(u.cpu().numpy() - inside).max() <= 1e-3
    # what an evaluator does not do
    with pytest.raises(bem.BemError):
        ev.bem_solve(np.ones(V.shape[0]), np.zeros(V.shape[0]))
    with pytest.raises(bem.BemError):
        ev.bem_set_option("quadrature", 1)
    with pytest.raises(bem.BemError):
        bem.bem_create_evaluator(ev, X)                      # an evaluator has no mesh of its own
    assert "holds no mesh" in bem.load_library().bem_last_error(None).decode()
    ev.bem_destroy()
    mesh.bem_destroy()


def test_evaluator_outlives_its_mesh_context():
    """include/bem.h: the mesh context is read by bem_setup of the evaluator only.  Destroy it after the set-up, let another
    context of another size take its place on the heap, and the evaluator's products (host buffers: their staging is sized
    by the MESH's vertex count) must not change by a bit."""
    bem = _bem()
    V, F = bi.icosphere(3)
    rng = np.random.default_rng(47)
    X = _shell_points(V, rng, 1500)
    q, phi = rng.normal(size=V.shape[0]), rng.normal(size=V.shape[0])
    mesh = bem.bem_create(V, F, None)
    ev = bem.bem_create_evaluator(mesh, X)
    ev.bem_setup(10, 64, 2.5)
    mesh.bem_destroy()
    V2, F2 = bi.icosphere(2)
    others = [bem.bem_create(V2 * (1 + k), F2, None) for k in range(4)]      # same-sized heap blocks, other N and T
    u1 = np.full(X.shape[0], np.nan)
    ev.bem_apply(q, phi, u1)
    u2 = np.full(X.shape[0], np.nan)
    ev.bem_apply(q, phi, u2)
    st = ev.bem_get_stats()
    assert st["n_targets"] == X.shape[0] and st["n_sources"] == 3 * F.shape[0]
    assert np.array_equal(u1, u2)
    assert _rel(u1, oracle.g3_evaluate(V, F, q, phi, X, eta=2.5)) <= 1e-5
    ev.bem_destroy()
    for o in others:
        o.bem_destroy()


def test_evaluator_on_a_cluster_sampled_points():
    """Config 2 (27 bubbles, 69,174 nodes): the potential at 4000 points of the liquid between the bubbles."""
    c = make_config(2)
    rng = np.random.default_rng(44)
    X = rng.uniform(-1.0, 7.0, size=(12000, 3))
    cen = 3.0 * np.array([[i, j, k] for i in range(3) for j in range(3) for k in range(3)], float)
    dist = np.linalg.norm(X[:, None, :] - cen[None, :, :], axis=2).min(1)
    X = X[(dist > 1.15)][:4000]                              # in the liquid, at least 0.05 off every surface (radii <= 1.1)
    rows = np.sort(rng.choice(X.shape[0], 500, replace=False))
    yo = oracle.g3_evaluate(c["V"], c["F"], c["q"], c["phi"], X[rows], eta=c["eta"])
    bem = _bem()
    mesh = bem.bem_create(c["V"], c["F"], c["bubble_id"])
    ev = bem.bem_create_evaluator(mesh, X)
    ev.bem_setup(c["p"], c["leaf_size"], c["eta"])
    u = np.full(X.shape[0], np.nan)
    ev.bem_apply(c["q"], c["phi"], u)
    st = ev.bem_get_stats()
    ev.bem_destroy(); mesh.bem_destroy()
    e = _rel(u[rows], yo)
    print(f"evaluator cfg2: {e:.2e}, lmax {st['lmax']:.0f}, p_dipole {st['p_dipole']:.0f}")
    assert st["m2l_pairs"] > 0 and e <= 1e-5


# ------------------------------------------------------------------ robustness items of the round-1 review
def test_contexts_on_two_devices():
    """Kernel attributes (dynamic shared memory above 48 KB, carve-out) are per device: a context on a second GPU must
    launch the same kernels.  Skipped on a one-GPU box."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    bem = _bem()
    c = make_config(1)
    ys = []
    for dev in (0, 1):
        torch.cuda.set_device(dev)
        ctx = bem.bem_create(c["V"], c["F"], c["bubble_id"])
        ctx.bem_setup(12, 64, 2.5)
        y = np.zeros(c["V"].shape[0])
        ctx.bem_apply(c["q"], c["phi"], y)
        ctx.bem_destroy()
        ys.append(y)
    torch.cuda.set_device(0)
    assert np.array_equal(ys[0], ys[1])


def test_caller_graph_capture_with_fp32_pairs_and_no_warm_up():
    """bem_apply inside the caller's torch.cuda.graph capture as the FIRST product after p2p_precision = 1: the fp32
    source records were built when the option was set (never inside a product), so nothing allocates in the capture."""
    import torch
    bem = _bem()
    c = make_config(2)
    ctx = bem.bem_create(c["V"], c["F"], c["bubble_id"])
    stream = torch.cuda.Stream()
    ctx.bem_set_stream(stream.cuda_stream)
    ctx.bem_setup(c["p"], c["leaf_size"], c["eta"])
    ctx.bem_set_option("p2p_precision", 1)
    qd, pd = torch.tensor(c["q"], device="cuda"), torch.tensor(c["phi"], device="cuda")
    yd = torch.zeros_like(qd)
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=stream):
        ctx.bem_apply(qd, pd, yd)
    g.replay()
    torch.cuda.synchronize()
    y_graph = yd.cpu().numpy().copy()
    yd.zero_()
    ctx.bem_set_option("graph", 0)
    ctx.bem_apply(qd, pd, yd)
    torch.cuda.synchronize()
    ctx.bem_destroy()
    assert np.array_equal(y_graph, yd.cpu().numpy())
