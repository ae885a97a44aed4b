"""The adaptive octree (option tree = 1, reading R9 stage 2; csrc/adaptive.cu) against the CPU oracle at
the tolerances of the uniform tree, through the C-ABI.  `pytest -m gpu`."""
import numpy as np
import pytest

import bem_inputs as bi
from bem_inputs.configs import make_config, sample_rows
import oracle

pytestmark = pytest.mark.gpu


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _bem():
    import paper_1905_01341_b200 as bem
    return bem


def _run(c, rows, q="q", phi="phi", p=None, leaf=None, **opts):
    ctx = _bem().bem_create(c["V"], c["F"], c.get("bubble_id"))
    ctx.bem_set_option("tree", 1)
    for k, v in opts.items():
        ctx.bem_set_option(k, v)
    ctx.bem_setup(p or c["p"], leaf or c["leaf_size"], c["eta"])
    N = c["V"].shape[0]
    y, y2 = np.full(N, np.nan), np.full(N, np.nan)
    qq, pp = (None if q is None else c[q]), (None if phi is None else c[phi])
    ctx.bem_apply(qq, pp, y)
    ctx.bem_apply(qq, pp, y2)
    st = ctx.bem_get_stats()
    ctx.bem_destroy()
    assert np.isfinite(y).all() and np.array_equal(y, y2)                     # bit-reproducible
    return y, st


@pytest.mark.parametrize("n,nb", [(1, None), (2, None), (3, None), (4, 60), (5, 150)])
def test_adaptive_tree_meets_the_fmm_tolerances(n, nb):
    """North_star tolerance at the stated p (S - D <= 1e-5) and Table 1's for the single layer, on every config (4 and 5
    shrunken), with leaves on several levels; <= 1e-8 at p = 24 on configs 1-2."""
    c = make_config(n) if nb is None else make_config(n, n_bubbles=nb)
    N = c["V"].shape[0]
    rows = np.arange(N, dtype=np.int64) if N < 3000 else sample_rows(n, N, 1000)
    yo = oracle.g3_apply(c["V"], c["F"], c["q"], c["phi"], eta=c["eta"], rows=rows)
    yoS = oracle.g3_apply(c["V"], c["F"], c["q"], None, eta=c["eta"], rows=rows)
    y, st = _run(c, rows)
    yS, _ = _run(c, rows, phi=None)
    eB, eS = _rel(y[rows], yo), _rel(yS[rows], yoS)
    print(f"cfg{n} adaptive p={c['p']}: S {eS:.2e}, S-D {eB:.2e}; lmax {st['lmax']:.0f}, leaves {st['n_src_leaves']:.0f} / {st['n_tgt_leaves']:.0f}, "
          f"m2l pairs {st['m2l_pairs']:.0f}, point pairs {st['p2p_pairs']:.3e} ({st['p2p_pairs_executed']:.3e} executed)")
    table1 = {8: 1e-5, 10: 2.2e-6, 12: 5e-7}
    assert st["m2l_pairs"] > 0 and eB <= 1e-5 and eS <= 3.0 * table1[c["p"]]
    if n <= 2:
        yh, _ = _run(c, rows, p=24)
        assert _rel(yh[rows], yo) <= 1e-8


def test_adaptive_tree_depth_controls_and_quadratures():
    """leaf_size 1 .. huge, a capped depth (option lmax), a lower minimum level (leaves on MANY levels), direct_pairs off /
    all, and the paper's V1 quadrature (coincident source and target) all give the same product up to truncation."""
    c = make_config(1)
    N = c["V"].shape[0]
    rows = np.arange(N, dtype=np.int64)
    yo = oracle.g3_apply(c["V"], c["F"], c["q"], c["phi"], eta=c["eta"])
    for opts in (dict(leaf=1), dict(leaf=8), dict(leaf=100000), dict(leaf=16, lmax=3), dict(leaf=8, tree_min_level=2),
                 dict(leaf=24, tree_min_level=2, direct_pairs=0), dict(leaf=24, tree_min_level=2, direct_pairs=10 ** 9)):
        leaf = opts.pop("leaf")
        y, st = _run(c, rows, p=12, leaf=leaf, **opts)
        e = _rel(y, yo)
        print(f"leaf {leaf} {opts}: {e:.2e}, lmax {st['lmax']:.0f}, tgt leaves {st['n_tgt_leaves']:.0f}")
        assert e <= 3e-5                                      # the bound of test_fmm_leaf_size_one_and_huge (uniform tree, p = 12)
    yv = oracle.v1_apply(c["V"], c["F"], c["q"], c["phi"])
    y, _ = _run(c, rows, p=12, leaf=8, quadrature=1, tree_min_level=2)
    assert _rel(y, yv) <= 3e-5


def test_adaptive_tree_on_a_strongly_non_uniform_cloud():
    """Where the adaptive tree is for: 90% of the points in a ball of 1% of the cube's edge.  The uniform rule stops at the
    depth the MEAN population gives and leaves the ball in a handful of boxes; the adaptive tree keeps refining there.
    Both meet the tolerance; the adaptive one does it with a fraction of the point pairs."""
    rng = np.random.default_rng(77)
    n = 60000
    dense = 0.5 + 0.005 * rng.normal(size=(int(0.9 * n), 3))
    pts = np.vstack([dense, rng.uniform(0, 1, size=(n - dense.shape[0], 3))])
    m = rng.uniform(-1, 1, size=n)
    rows = np.sort(rng.choice(n, 300, replace=False))
    yo = oracle.monopole_sum(pts, m, pts[rows])
    res = {}
    for tree in (0, 1):
        ctx = _bem().bem_create_points(pts, pts)
        ctx.bem_set_option("tree", tree)
        ctx.bem_setup(12, 64, 2.5)
        y = np.full(n, np.nan)
        ctx.bem_apply(m, None, y)
        st = ctx.bem_get_stats()
        ctx.bem_destroy()
        res[tree] = (_rel(y[rows], yo), st["p2p_pairs"], st["lmax"], st["p2p_pairs_wx"])
        print(f"tree {tree}: error {res[tree][0]:.2e}, point pairs {st['p2p_pairs']:.3e} (W/X ranges {st['p2p_pairs_wx']:.3e}), "
              f"lmax {st['lmax']:.0f}, m2l pairs {st['m2l_pairs']:.0f}, m2m pairs {st['m2m_pairs']:.0f} -> {st['m2m_parents']:.0f} parents")
        assert 0 < st["m2m_parents"] <= st["m2m_pairs"] <= 8 * st["m2m_parents"]
    assert res[0][0] <= 1e-5 and res[1][0] <= 1e-5
    assert res[1][1] < 0.2 * res[0][1] and res[1][2] > res[0][2]
    # BEM_S_P2P_PAIRS_WX: the uniform tree has no W or X list; a graded cloud must have both, and they are part of the direct pairs
    assert res[0][3] == 0 and 0 < res[1][3] < res[1][1]


def test_adaptive_tree_evaluator_and_refusals():
    bem = _bem()
    V, F = bi.icosphere(3)
    rng = np.random.default_rng(5)
    q, ph = rng.normal(size=V.shape[0]), rng.normal(size=V.shape[0])
    X = V[rng.choice(V.shape[0], 1500)] * rng.uniform(1.05, 2.5, size=(1500, 1))
    mesh = bem.bem_create(V, F, None)
    ev = bem.bem_create_evaluator(mesh, X)
    ev.bem_set_option("tree", 1)
    ev.bem_setup(12, 32, 2.5)
    u = np.full(X.shape[0], np.nan)
    ev.bem_apply(q, ph, u)
    assert _rel(u, oracle.g3_evaluate(V, F, q, ph, X, eta=2.5)) <= 1e-5
    ev.bem_set_option("p2p_precision", 1)                      # fp32 pairs need leaves of one size
    with pytest.raises(bem.BemError):
        ev.bem_apply(q, ph, u)
    ev.bem_destroy(); mesh.bem_destroy()


@pytest.mark.parametrize("tree", [0, 1])
def test_side_stream_option_gives_the_same_bits(tree):
    """Option overlap = 1 (the row sums of the M2L stages on a side stream beside the near field, round 1's default) against
    the one-stream default, on device buffers, for both trees; and a context switched from the adaptive tree back to the
    uniform one gives the uniform tree's bits."""
    import torch
    bem = _bem()
    c = make_config(2)
    qd, pd = torch.tensor(c["q"], device="cuda"), torch.tensor(c["phi"], device="cuda")
    ctx = bem.bem_create(c["V"], c["F"], c["bubble_id"])
    ctx.bem_set_option("tree", tree)
    ctx.bem_setup(c["p"], c["leaf_size"], c["eta"])
    ys = []
    for ov in (0, 1, 0):
        ctx.bem_set_option("overlap", ov)
        yd = torch.empty_like(qd)
        ctx.bem_apply(qd, pd, yd)
        torch.cuda.synchronize()
        ys.append(yd.cpu().numpy())
    assert np.array_equal(ys[0], ys[1]) and np.array_equal(ys[0], ys[2])
    if tree == 1:
        ctx.bem_set_option("tree", 0)
        ctx.bem_setup(c["p"], c["leaf_size"], c["eta"])
        yd = torch.empty_like(qd)
        ctx.bem_apply(qd, pd, yd)
        ref = bem.bem_create(c["V"], c["F"], c["bubble_id"])
        ref.bem_setup(c["p"], c["leaf_size"], c["eta"])
        yr = torch.empty_like(qd)
        ref.bem_apply(qd, pd, yr)
        torch.cuda.synchronize()
        assert np.array_equal(yd.cpu().numpy(), yr.cpu().numpy())
        ref.bem_destroy()
    ctx.bem_destroy()


def test_adaptive_tree_full_size_config5_as_bench_times_it():
    """BASELINE.json config 5 at full size in the configuration bench.py times by default (tree = 1, leaf_size 350,
    device-resident q, phi, y) on the 2000 seeded rows of the north_star; bit-identical repeat; GMRES takes one more
    step through it (products without phi) and reduces the residual."""
    import torch
    bem = _bem()
    c = make_config(5)
    N = c["V"].shape[0]
    rows = sample_rows(5, N, 2000)
    yo = oracle.g3_apply(c["V"], c["F"], c["q"], c["phi"], eta=c["eta"], rows=rows)
    ctx = bem.bem_create(c["V"], c["F"], c["bubble_id"])
    ctx.bem_set_option("tree", 1)
    ctx.bem_setup(c["p"], 350, c["eta"])
    qd, pd = torch.tensor(c["q"], device="cuda"), torch.tensor(c["phi"], device="cuda")
    yd = torch.empty_like(qd)
    ctx.bem_apply(qd, pd, yd)
    y1 = yd.cpu().numpy()
    ctx.bem_apply(qd, pd, yd)
    assert np.array_equal(y1, yd.cpu().numpy())
    st = ctx.bem_get_stats()
    e = _rel(y1[rows], yo)
    print(f"cfg5 full size, adaptive: S-D on 2000 rows {e:.2e}; lmax {st['lmax']:.0f}, target leaves {st['n_tgt_leaves']:.0f}, "
          f"m2l pairs {st['m2l_pairs']:.0f}, point pairs {st['p2p_pairs']:.3e}")
    assert st["lmax"] > 6 and e <= 1e-5
    qs = torch.zeros_like(qd)
    status, it, rr = ctx.bem_solve(pd, qs, tol=1e-6, max_iter=3)
    assert it == 3 and rr < 1.0 and status == bem.BEM_ERR_NOT_CONVERGED      # unpreconditioned GMRES starts slowly here (0.93 after 3 steps)
    ctx.bem_destroy()


def test_degenerate_inputs_both_trees():
    """The smallest closed mesh (a tetrahedron: 4 vertices), one target, one source, all sources in one point's
    neighbourhood and coincident source/target clouds -- both trees, FMM and direct, against the oracle."""
    bem = _bem()
    V = np.array([[1.0, 1.0, 1.0], [1.0, -1.0, -1.0], [-1.0, 1.0, -1.0], [-1.0, -1.0, 1.0]])
    F = np.array([[0, 1, 2], [0, 3, 1], [0, 2, 3], [1, 3, 2]], dtype=np.int32)
    if np.dot(np.cross(V[1] - V[0], V[2] - V[0]), V[0] + V[1] + V[2]) < 0:
        F = F[:, [0, 2, 1]].copy()                           # outward orientation
    q, ph = np.array([1.0, -2.0, 0.5, 3.0]), np.array([0.3, 0.1, -0.7, 1.1])
    yo = oracle.g3_apply(V, F, q, ph, eta=2.5)
    for tree in (0, 1):
        for mode in (0, 1):
            ctx = bem.bem_create(V, F, None)
            ctx.bem_set_option("tree", tree); ctx.bem_set_option("mode", mode)
            ctx.bem_setup(6, 1, 2.5)
            y = np.full(4, np.nan)
            ctx.bem_apply(q, ph, y)
            ctx.bem_destroy()
            # FMM tolerance 1e-4, not the north_star's 1e-5: this mesh is set up at p = 6 (S - D then runs at 9, R5'), below every
            # stated p of BASELINE.json (8 / 10 / 12) -- the bound is Table 1's p = 8 column relaxed by the missing degrees
            # (DESIGN.md section 3 R5': about one digit per 2.5 degrees), and with 12 sources at leaf_size 1 nearly every
            # pair is a far pair, so the product IS the truncation error.  What the case checks is that a 4-vertex mesh
            # builds a tree and lists at all; accuracy at the stated p is tests/test_gpu_parity.py's.
            assert _rel(y, yo) <= (1e-12 if mode else 1e-4), (tree, mode, _rel(y, yo))
    rng = np.random.default_rng(9)
    src = rng.uniform(0, 1, size=(500, 3))
    m = rng.normal(size=500)
    for tgt in (np.array([[0.5, 0.5, 0.5]]), np.array([[5.0, -3.0, 2.0]]), src[:1].copy()):
        yo = oracle.monopole_sum(src, m, tgt)
        for tree in (0, 1):
            ctx = bem.bem_create_points(src, tgt)
            ctx.bem_set_option("tree", tree)
            ctx.bem_setup(12, 16, 2.5)
            y = np.full(1, np.nan)
            ctx.bem_apply(m, None, y)
            ctx.bem_destroy()
            assert abs(y[0] - yo[0]) <= 1e-5 * abs(yo[0]), (tree, tgt, y, yo)
    one = np.array([[0.25, 0.5, 0.75]])
    tg = rng.uniform(0, 1, size=(300, 3))
    yo = oracle.point_sum(one, np.array([2.0]), np.array([[0.1, -0.2, 0.3]]), tg)
    for tree in (0, 1):
        ctx = bem.bem_create_points(one, tg)
        ctx.bem_set_option("tree", tree)
        ctx.bem_setup(16, 8, 2.5)
        y = np.full(300, np.nan)
        ctx.bem_apply(np.array([2.0]), np.array([[0.1, -0.2, 0.3]]), y)
        ctx.bem_destroy()
        assert _rel(y, yo) <= 1e-6, (tree, _rel(y, yo))


def test_adaptive_tree_row_overflow_rebuilds_without_direct_far_pairs():
    """include/bem.h, option "direct_pairs": a target leaf of the adaptive tree may hold at most max_direct_ranges (256)
    direct source ranges.  Lower the limit until the library's own choice of direct far pairs no longer fits: an explicit
    direct_pairs is then refused, the default (-1) rebuilds the lists with every far pair translated -- the same lists as
    direct_pairs = 0 -- and still meets the tolerance."""
    bem = _bem()
    rng = np.random.default_rng(78)
    n = 30000
    dense = 0.5 + 0.005 * rng.normal(size=(int(0.9 * n), 3))
    pts = np.vstack([dense, rng.uniform(0, 1, size=(n - dense.shape[0], 3))])
    m = rng.uniform(-1, 1, size=n)
    rows = np.sort(rng.choice(n, 200, replace=False))
    yo = oracle.monopole_sum(pts, m, pts[rows])

    def run(direct_pairs, limit):
        ctx = bem.bem_create_points(pts, pts)
        ctx.bem_set_option("tree", 1)
        ctx.bem_set_option("direct_pairs", direct_pairs)
        ctx.bem_set_option("max_direct_ranges", limit)
        try:
            ctx.bem_setup(12, 8, 2.5)
            y = np.full(n, np.nan)
            ctx.bem_apply(m, None, y)
            return _rel(y[rows], yo), ctx.bem_get_stats()
        finally:
            ctx.bem_destroy()

    found = False
    for limit in (200, 160, 120, 90, 70, 50, 40):
        try:
            e0, st0 = run(0, limit)
        except bem.BemError:
            break                                            # even the plain lists no longer fit: nothing below will
        try:
            run(800, limit)
            continue                                         # the direct far pairs still fit under this limit
        except bem.BemError as ex:
            assert ex.status == bem.BEM_ERR_INVALID_ARG and "direct source ranges" in str(ex)
        e, st = run(-1, limit)
        print(f"limit {limit}: rebuilt, error {e:.2e}, m2l pairs {st['m2l_pairs']:.0f} (direct_pairs = 0: {st0['m2l_pairs']:.0f})")
        assert e <= 1e-5 and e0 <= 1e-5
        assert st["m2l_pairs"] == st0["m2l_pairs"] and st["p2p_pairs"] == st0["p2p_pairs"]
        found = True
        break
    assert found, "no limit separated the lists with and without direct far pairs"
