"""Parity of the CUDA path (through the C-ABI, paper_1905_01341_b200) with the CPU
oracle (oracle/), element by element on the same seeded inputs.

Tolerances (BASELINE.json north_star):
  direct-sum mode   relative L2 <= 1e-12   ("brute force" product)
  FMM mode          relative L2 <= tolerance at the stated p / <= 1e-8 at high p
                    (the paper's own check is the relative L2
                    error against direct evaluation at checkpoints)
All of these need a B200: `pytest -m gpu`.
"""
import numpy as np
import pytest

import bem_inputs as bi
from bem_inputs.configs import make_config, sample_rows
import oracle

pytestmark = pytest.mark.gpu

TOL_DIRECT = 1e-12


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _bem():
    import paper_1905_01341_b200 as bem
    return bem


def _ctx(c, mode=0, quad=0, p=None, leaf=None, eta=None, **opts):
    bem = _bem()
    ctx = bem.bem_create(c["V"], c["F"], c.get("bubble_id"))
    ctx.bem_set_option("mode", mode)
    ctx.bem_set_option("quadrature", quad)
    for k, v in opts.items():
        ctx.bem_set_option(k, v)
    ctx.bem_setup(p or c["p"], leaf or c["leaf_size"], eta or c["eta"])
    return ctx


def _apply(ctx, q, phi):
    y = np.full(ctx.n_vertices, np.nan)
    ctx.bem_apply(q, phi, y)
    assert np.isfinite(y).all()
    return y


_cfg_cache = {}


def cfg(n, **kw):
    key = (n, tuple(sorted(kw.items())))
    if key not in _cfg_cache:
        _cfg_cache[key] = make_config(n, **kw)
    return _cfg_cache[key]


_oracle_cache = {}


def oracle_rows(c, rows, quad=0, q="q", phi="phi"):
    key = (c["name"], quad, q, phi, len(rows), int(rows[0]), int(rows[-1]))
    if key not in _oracle_cache:
        qq = None if q is None else c[q]
        pp = None if phi is None else c[phi]
        if quad == 0:
            _oracle_cache[key] = oracle.g3_apply(c["V"], c["F"], qq, pp, eta=c["eta"], rows=rows)
        else:
            _oracle_cache[key] = oracle.v1_apply(c["V"], c["F"], qq, pp, rows=rows)
    return _oracle_cache[key]


# ------------------------------------------------------------------ direct-sum mode, <= 1e-12
@pytest.mark.parametrize("quad", [0, 1])
def test_direct_cfg1_all_rows(quad):
    c = cfg(1)
    rows = np.arange(c["V"].shape[0], dtype=np.int64)
    y = _apply(_ctx(c, mode=1, quad=quad), c["q"], c["phi"])
    assert _rel(y, oracle_rows(c, rows, quad)) <= TOL_DIRECT


@pytest.mark.parametrize("quad", [0, 1])
def test_direct_cfg2_sampled_rows(quad):
    c = cfg(2)
    rows = sample_rows(2, c["V"].shape[0], 2000)
    y = _apply(_ctx(c, mode=1, quad=quad), c["q"], c["phi"])
    assert _rel(y[rows], oracle_rows(c, rows, quad)) <= TOL_DIRECT


def test_direct_cfg3_sampled_rows():
    c = cfg(3)
    rows = sample_rows(3, c["V"].shape[0], 2000)
    y = _apply(_ctx(c, mode=1), c["q"], c["phi"])
    assert _rel(y[rows], oracle_rows(c, rows)) <= TOL_DIRECT


def test_direct_single_layers():
    """q = NULL or phi = NULL skips that layer (f, g of Eq. 45)."""
    c = cfg(1)
    rows = np.arange(c["V"].shape[0], dtype=np.int64)
    ctx = _ctx(c, mode=1)
    yS = _apply(ctx, c["q"], None)
    yD = _apply(ctx, None, c["phi"])
    assert _rel(yS, oracle_rows(c, rows, 0, "q", None)) <= TOL_DIRECT
    assert _rel(yD, oracle_rows(c, rows, 0, None, "phi")) <= TOL_DIRECT
    assert _rel(yS + yD, oracle_rows(c, rows)) <= TOL_DIRECT


@pytest.mark.parametrize("lvl,eta", [(0, 2.5), (1, 1.0), (2, 4.0), (2, 1e30)])
def test_direct_tiny_meshes_and_eta(lvl, eta):
    """12..162 vertices; eta = 1 (incident triangles only, mostly), 4, and infinity (every triangle exact)."""
    V, F = bi.icosphere(lvl)
    rng = np.random.default_rng(7 + lvl)
    V = V * np.array([1.0, 0.8, 1.3]) + np.array([5.0, -2.0, 0.5])      # ellipsoid off the origin
    q, phi = rng.normal(size=V.shape[0]), rng.normal(size=V.shape[0])
    c = dict(V=V, F=F, bubble_id=None, q=q, phi=phi, p=6, leaf_size=16, eta=eta, name=f"tiny{lvl}-{eta}")
    y = _apply(_ctx(c, mode=1), q, phi)
    yo = oracle.g3_apply(V, F, q, phi, eta=eta)
    assert _rel(y, yo) <= TOL_DIRECT


# ------------------------------------------------------------------ FMM mode
# Tolerances ("FMM tolerance").  The expansions are truncated to degrees
# 0..p-1 as the paper states.
#  * SINGLE layer (monopole sources -- the workload of the paper's Table 1):
#    within 3x of the value Table 1 prints at that p (1e-5 at p = 8, 5e-7 at p = 12; p = 10 by
#    geometric interpolation).
#  * Full operator S - D: the north_star's 1e-5 at the stated p (8, 10, 12) and 1e-8 at high p = 24.
#    Dipole sources lose accuracy against monopoles at equal truncation (R5': a dipole moment of degree l
#    scales like l a^(l-1); test_dipole_penalty_is_a_truncation_effect measures it: 3-4 degrees), so the library carries
#    products WITH dipoles 3 degrees higher below p = 12 (option dipole_degrees = -1, the default).  With
#    dipole_degrees = 0 -- the paper's convention, one truncation for everything -- the full operator at
#    p = 8, 10 only reaches TOL_FULL_PAPER_CONVENTION; that reading is NOT the default because it misses the north_star.
TABLE1 = {4: 7e-4, 8: 1e-5, 10: 2.2e-6, 12: 5e-7, 16: 3e-8, 20: 4e-9}      # tests/golden/table1_fmm_error.txt
TOL_S = {p: 3.0 * v for p, v in TABLE1.items()}
TOL_FULL = {8: 1e-5, 10: 1e-5, 12: 1e-5}                                    # BASELINE.json north_star
TOL_FULL_PAPER_CONVENTION = 1e-4                                            # dipole_degrees = 0 (measured 1.5e-5 .. 6e-5)
HIGH_P = 24


def _fmm_errors(c, rows, p, **opts):
    ctx = _ctx(c, p=p, **opts)
    yS = _apply(ctx, c["q"], None)
    yB = _apply(ctx, c["q"], c["phi"])
    eS = _rel(yS[rows], oracle_rows(c, rows, 0, "q", None))
    eB = _rel(yB[rows], oracle_rows(c, rows))
    st = ctx.bem_get_stats()
    ctx.bem_destroy()
    return eS, eB, st


@pytest.mark.parametrize("n", [1, 2, 3])
def test_fmm_stated_p(n):
    c = cfg(n)
    N = c["V"].shape[0]
    rows = np.arange(N, dtype=np.int64) if N < 3000 else sample_rows(n, N, 2000)
    eS, eB, st = _fmm_errors(c, rows, c["p"])
    print(f"cfg{n} p={c['p']}: single layer {eS:.2e}, S-D {eB:.2e}, lmax {st['lmax']:.0f}")
    assert st["lmax"] >= 3 and st["m2l_pairs"] > 0            # the far field really goes through the tree
    assert eS <= TOL_S[c["p"]]
    assert eB <= TOL_FULL[c["p"]]


@pytest.mark.parametrize("n", [1, 2, 3])
def test_fmm_stated_p_paper_convention(n):
    """dipole_degrees = 0: one truncation number for monopoles and dipoles, as PAPER.md:438 states it.  The single layer
    is unchanged (Table 1); the full operator stays within a decade of the north_star's figure and reaches it at p + 4."""
    c = cfg(n)
    N = c["V"].shape[0]
    rows = np.arange(N, dtype=np.int64) if N < 3000 else sample_rows(n, N, 2000)
    eS, eB, st = _fmm_errors(c, rows, c["p"], dipole_degrees=0)
    eS4, eB4, _ = _fmm_errors(c, rows, c["p"] + 4, dipole_degrees=0)
    print(f"cfg{n} dipole_degrees=0: p={c['p']}: single layer {eS:.2e}, S-D {eB:.2e}; p={c['p'] + 4}: {eS4:.2e}, {eB4:.2e}")
    assert st["p_dipole"] == c["p"]
    assert eS <= TOL_S[c["p"]] and eB <= TOL_FULL_PAPER_CONVENTION
    assert eB4 <= 1e-5 and eS4 <= 1e-5


@pytest.mark.parametrize("n,nb", [(2, None), (3, None), (4, 60)])
def test_dipole_penalty_is_a_truncation_effect(n, nb):
    """DESIGN.md R5' as a tested fact.  With ONE truncation number (dipole_degrees = 0) the relative error of the double
    layer alone (q = NULL) is 5-60x that of the single layer alone (phi = NULL) at every p, both fall at the same rate
    (2-3x per degree), and the double layer at p + 4 is as accurate as the single layer at p (within 3x) -- a constant
    shift in p, i.e. truncation, not a defect of the dipole path of P2M (whose formulas test_fmm_operator_chains pins
    to rounding)."""
    c = cfg(n) if nb is None else cfg(n, n_bubbles=nb)
    N = c["V"].shape[0]
    rows = sample_rows(n, N, 1000)
    yoS, yoD = oracle_rows(c, rows, 0, "q", None), oracle_rows(c, rows, 0, None, "phi")
    eS, eD = {}, {}
    for p in (6, 8, 10, 12, 14):
        ctx = _ctx(c, p=p, dipole_degrees=0)
        eS[p] = _rel(_apply(ctx, c["q"], None)[rows], yoS)
        eD[p] = _rel(_apply(ctx, None, c["phi"])[rows], yoD)
        ctx.bem_destroy()
    print(f"cfg{n}: S-only", {p: f"{e:.2e}" for p, e in eS.items()}, "D-only", {p: f"{e:.2e}" for p, e in eD.items()})
    for p in eS:
        assert 5.0 <= eD[p] / eS[p] <= 60.0, (p, eD[p] / eS[p])
    for a, b in ((6, 8), (8, 10), (10, 12), (12, 14)):
        assert 3.0 <= eS[a] / eS[b] <= 12.0 and 3.0 <= eD[a] / eD[b] <= 12.0, (a, b)
    for p in (6, 8, 10):
        assert eD[p + 4] <= 3.0 * eS[p], (p, eD[p + 4], eS[p])


@pytest.mark.parametrize("n", [1, 2, 3])
def test_fmm_high_p(n):
    c = cfg(n)
    N = c["V"].shape[0]
    rows = np.arange(N, dtype=np.int64) if N < 3000 else sample_rows(n, N, 2000)
    eS, eB, _ = _fmm_errors(c, rows, HIGH_P)
    print(f"cfg{n} p={HIGH_P}: single layer {eS:.2e}, S-D {eB:.2e}")
    assert eB <= 1e-8 and eS <= 1e-8


def test_fmm_error_decays_with_p_like_table1():
    """P9: the truncation convention (degrees 0..p-1) reproduces the decay of the paper's Table 1
     for monopole sources: same order of magnitude (within 5x) as every printed value -- the paper's
    points fill a cube, ours lie on bubble surfaces, so equality is not expected.  The bound is two-sided and 5x because
    SURVEY.md 8(c) pin P9 asks for "same order of magnitude as PAPER.md:464-471 (Table 1)", not for an upper bound: the
    first hardware run measured p = 4 at 1.4x ABOVE and p = 16 at 3x BELOW the printed values (surface data converge
    faster at high p), which a one-sided 3x bound misread as a failure."""
    c = cfg(2)
    rows = sample_rows(2, c["V"].shape[0], 1000)
    errs = {}
    for p in (4, 8, 12, 16, 20):
        errs[p] = _fmm_errors(c, rows, p)[0]
    print(errs)
    for p, e in errs.items():
        assert TABLE1[p] / 5.0 <= e <= 5.0 * TABLE1[p]
    assert all(errs[a] > errs[b] for a, b in ((4, 8), (8, 12), (12, 16), (16, 20)))


@pytest.mark.parametrize("n,nb", [(4, 60), (5, 150)])
def test_fmm_shrunken_clusters(n, nb):
    """Configs 4 and 5 with fewer bubbles (same recipe and seed): polydisperse leaves, ragged tails."""
    c = cfg(n, n_bubbles=nb)
    rows = sample_rows(n, c["V"].shape[0], 1500)
    eS, eB, st = _fmm_errors(c, rows, c["p"])
    print(f"cfg{n}/{nb} p={c['p']}: single layer {eS:.2e}, S-D {eB:.2e}, lmax {st['lmax']:.0f}")
    assert eS <= TOL_S[c["p"]] and eB <= TOL_FULL[c["p"]]


@pytest.mark.parametrize("quad", [0, 1])
def test_fmm_v1_and_g3_cfg1_lmax_sweep(quad):
    """The lists partition all pairs exactly once at every depth: the FMM result does not depend on
    l_max beyond truncation error."""
    c = cfg(1)
    rows = np.arange(c["V"].shape[0], dtype=np.int64)
    yo = oracle_rows(c, rows, quad)
    for lmax in (2, 3, 4, 5):
        y = _apply(_ctx(c, quad=quad, p=12, lmax=lmax), c["q"], c["phi"])
        assert _rel(y, yo) <= 3e-5, (lmax, _rel(y, yo))


def test_fmm_leaf_size_one_and_huge():
    c = cfg(1)
    rows = np.arange(c["V"].shape[0], dtype=np.int64)
    yo = oracle_rows(c, rows)
    for leaf in (1, 8, 100000):
        ctx = _ctx(c, p=12, leaf=leaf)
        y = _apply(ctx, c["q"], c["phi"])
        assert _rel(y, yo) <= 3e-5, (leaf, ctx.bem_get_stats()["lmax"], _rel(y, yo))


def test_fmm_every_truncation_number_cfg1():
    """Odd p (stored in the layout of the next even template bucket), the buckets themselves and the run-time-p
    kernels (p > 16): the single-layer error falls monotonically (to rounding) and follows Table 1's decay."""
    c = cfg(1)
    rows = np.arange(c["V"].shape[0], dtype=np.int64)
    yo = oracle_rows(c, rows, 0, "q", None)
    errs = {}
    for p in (1, 2, 3, 4, 5, 7, 9, 11, 13, 15, 16, 17, 19):
        ctx = _ctx(c, p=p, lmax=3, direct_pairs=0)             # uniform lists: the truncation error alone (the direct-pair
        errs[p] = _rel(_apply(ctx, c["q"], None), yo)           # threshold moves with the layout size of p)
        ctx.bem_destroy()
    print({p: f"{e:.2e}" for p, e in errs.items()})
    ps = sorted(errs)
    assert all(errs[b] < 1.05 * errs[a] for a, b in zip(ps, ps[1:]))
    assert errs[4] < 5e-3 and errs[9] < 3e-5 and errs[13] < 1e-6 and errs[17] < 5e-8 and errs[19] < 1e-8


def test_gemm_paths_agree():
    """Option gemm_path: the FP64 tensor tiles and the plain-FMA tiles compute the same translations."""
    c = cfg(2)
    ctx = _ctx(c, p=10)
    y0 = _apply(ctx, c["q"], c["phi"])
    ctx.bem_set_option("gemm_path", 1)
    y1 = _apply(ctx, c["q"], c["phi"])
    ctx.bem_destroy()
    assert _rel(y1, y0) <= 1e-13


# ------------------------------------------------------------------ point clouds: the paper's own Table 1 workload
def _cloud(n, seed):
    pts, m = bi.random_cube_points(n, seed)
    rows = np.sort(np.random.default_rng(seed + 1).choice(n, int(np.sqrt(n)), replace=False))     # sqrt(N) checkpoints
    return pts, m, rows


def test_point_cloud_direct_matches_oracle():
    pts, m, rows = _cloud(20000, 11)
    ctx = _bem().bem_create_points(pts, pts[rows])
    ctx.bem_set_option("mode", 1)
    ctx.bem_setup(8, 64, 2.5)
    y = np.full(len(rows), np.nan)
    ctx.bem_apply(m, None, y)
    ctx.bem_destroy()
    assert _rel(y, oracle.monopole_sum(pts, m, pts[rows])) <= TOL_DIRECT


def test_point_cloud_fmm_reproduces_table1():
    """PAPER.md:462-471, Table 1 (tests/golden/table1_fmm_error.txt): relative L2 error of the FMM product for N = 131,072
    uniform random monopoles in a cube, measured at sqrt(N) checkpoints against the direct sum -- the paper's own
    workload and protocol.  The paper does not state the distribution of the intensities (reading R27): with
    zero-mean intensities U(-1, 1) the errors reproduce every printed value within 4x; with positive intensities
    U(0, 1) the potential has a large smooth mean and the same absolute error is a 10-100x smaller relative error."""
    n = 131072
    pts, m01, rows = _cloud(n, 12)
    ctx = _bem().bem_create_points(pts, pts)
    res = {}
    for name, m in (("zero-mean", 2.0 * m01 - 1.0), ("positive", m01)):
        yo = oracle.monopole_sum(pts, m, pts[rows])
        errs = {}
        for p in (4, 8, 12, 16, 20):
            ctx.bem_setup(p, 64, 2.5)
            y = np.full(n, np.nan)
            ctx.bem_apply(m, None, y)
            errs[p] = _rel(y[rows], yo)
        res[name] = errs
        print(name, {p: f"{e:.2e}" for p, e in errs.items()}, "lmax", ctx.bem_get_stats()["lmax"])
    ctx.bem_destroy()
    for p, e in res["zero-mean"].items():
        assert TABLE1[p] / 4.0 <= e <= 4.0 * TABLE1[p], (p, e)
    for errs in res.values():
        ps = sorted(errs)
        assert all(errs[b] < errs[a] for a, b in zip(ps, ps[1:]))
    assert all(res["positive"][p] < res["zero-mean"][p] for p in res["positive"])


# ------------------------------------------------------------------ full-size configs 4 and 5, as bench.py runs them
@pytest.mark.parametrize("n,nrows", [(4, 2000), (5, 2000)])
def test_fmm_full_size_clusters_sampled_rows(n, nrows):
    """BASELINE.json configs 4 (642,000 nodes, p = 10) and 5 (2,568,000 nodes, p = 12) at full size, in the launch
    configuration bench.py times (same leaf_size, device-resident q, phi, y, two streams), on seeded sampled rows the
    oracle evaluates one by one (the paper's own check uses checkpoints)."""
    import torch
    c = cfg(n)
    N = c["V"].shape[0]
    rows = sample_rows(n, N, nrows)
    ctx = _ctx(c)
    qd, pd = torch.tensor(c["q"], device="cuda"), torch.tensor(c["phi"], device="cuda")
    yd = torch.empty_like(qd)
    ctx.bem_apply(qd, pd, yd)
    y1 = yd.cpu().numpy()
    ctx.bem_apply(qd, pd, yd)                                   # bit-reproducible with the side stream too
    assert np.array_equal(y1, yd.cpu().numpy())
    st = ctx.bem_get_stats()
    ctx.bem_destroy()
    e = _rel(y1[rows], oracle_rows(c, rows))
    print(f"cfg{n} full size p={c['p']} lmax {st['lmax']:.0f}: S-D on {nrows} rows {e:.2e}")
    assert np.isfinite(y1).all()
    assert e <= 1e-5                                             # north_star: <= 1e-5 at the stated p


# ------------------------------------------------------------------ single-precision near field (option p2p_precision = 1)
TABLE1_SINGLE = {4: 5e-4, 8: 8e-6, 12: 4e-7, 16: 2e-7, 20: 2e-7}             # tests/golden/table1_fmm_error_single.txt, N = 131,072


@pytest.mark.parametrize("n,nb", [(1, None), (2, None), (3, None), (4, 60), (5, 150)])
def test_mixed_precision_near_field_stated_p(n, nb):
    """SURVEY.md 8(f) #1 / PAPER.md:456-473: A^(sparse) X with fp32 pair arithmetic and fp64 accumulation.  At the stated
    p the product keeps the tolerances of the fp64 path ("up to p_fmm = 12 the accuracy of the MVP practically is not
    affected"), the serial (option timing) and the three-stream launch orders give the same bits, and at p = 24 what is
    left is the single-precision floor of the near field (the paper's Table 1 prints 5e-8 .. 2e-7 for it)."""
    c = cfg(n) if nb is None else cfg(n, n_bubbles=nb)
    N = c["V"].shape[0]
    rows = np.arange(N, dtype=np.int64) if N < 3000 else sample_rows(n, N, 1500)
    yo, yoS = oracle_rows(c, rows), oracle_rows(c, rows, 0, "q", None)
    ctx = _ctx(c, p2p_precision=1)
    yB, yS = _apply(ctx, c["q"], c["phi"]), _apply(ctx, c["q"], None)
    ctx.bem_set_option("timing", 1)
    yB_serial = _apply(ctx, c["q"], c["phi"])
    ctx.bem_set_option("timing", 0)
    ctx.bem_set_option("p2p_precision", 0)
    yB64 = _apply(ctx, c["q"], c["phi"])
    ctx.bem_destroy()
    eB, eS, e64 = _rel(yB[rows], yo), _rel(yS[rows], yoS), _rel(yB64[rows], yo)
    ctx = _ctx(c, p=HIGH_P, p2p_precision=1)
    floor = _rel(_apply(ctx, c["q"], c["phi"])[rows], yo)
    ctx.bem_destroy()
    print(f"cfg{n} p={c['p']} fp32 near field: single layer {eS:.2e}, S-D {eB:.2e} (fp64 near field {e64:.2e}); floor at p={HIGH_P}: {floor:.2e}")
    assert np.array_equal(yB, yB_serial)
    assert eS <= TOL_S[c["p"]] and eB <= TOL_FULL[c["p"]]
    assert eB <= 1.5 * e64 + 1e-6                               # practically not affected
    assert floor <= 2e-6


def test_mixed_precision_point_cloud_reproduces_table1_single_column():
    """PAPER.md:462-471, Table 1, "single" column at N = 131,072 (tests/golden/table1_fmm_error_single.txt): same workload
    and protocol as test_point_cloud_fmm_reproduces_table1.  Up to p = 12 the printed values are the truncation error
    (within 4x, as for the double column); at p = 16 and 20 the paper's error stops at 2e-7 -- the floor of ITS single
    precision kernel.  Ours must stop falling too (it cannot follow the double column) and stay at or below 4x that floor."""
    n = 131072
    pts, m01, rows = _cloud(n, 12)
    m = 2.0 * m01 - 1.0
    yo = oracle.monopole_sum(pts, m, pts[rows])
    ctx = _bem().bem_create_points(pts, pts)
    ctx.bem_set_option("p2p_precision", 1)
    errs = {}
    for p in (4, 8, 12, 16, 20):
        ctx.bem_setup(p, 64, 2.5)
        y = np.full(n, np.nan)
        ctx.bem_apply(m, None, y)
        errs[p] = _rel(y[rows], yo)
    ctx.bem_destroy()
    print("fp32 near field", {p: f"{e:.2e}" for p, e in errs.items()})
    for p in (4, 8, 12):                                        # the printed single and double values differ by <= 1.4x here
        hi = max(TABLE1_SINGLE[p], TABLE1[p] if p != 12 else 4e-7)
        assert TABLE1_SINGLE[p] / 4.0 <= errs[p] <= 4.0 * hi, (p, errs[p])
    for p in (16, 20):
        assert TABLE1[p] < errs[p] <= 4.0 * TABLE1_SINGLE[p], (p, errs[p])


# ------------------------------------------------------------------ sparse far pairs summed directly (option direct_pairs)
@pytest.mark.parametrize("n,nb,prec", [(2, None, 0), (5, 150, 0), (5, 150, 1), (4, 60, 0)])
def test_direct_pairs_thresholds(n, nb, prec):
    """Leaf-level M2L pairs with nt x ns <= threshold move to the near-field kernel (tree.cu): threshold 0 = the uniform
    lists of PAPER.md:440, -1 = cost model, 1e9 = every leaf-level far pair direct (up to 27 + 189 source segments per
    target leaf).  All three meet the FMM tolerance; the pair counts move as stated; the all-direct product is the most
    accurate (direct pairs are exact)."""
    c = cfg(n) if nb is None else cfg(n, n_bubbles=nb)
    N = c["V"].shape[0]
    rows = sample_rows(n, N, 1500)
    yo = oracle_rows(c, rows)
    res = {}
    for d in (0, -1, 10 ** 9):
        ctx = _ctx(c, direct_pairs=d, p2p_precision=prec)
        y = _apply(ctx, c["q"], c["phi"])
        st = ctx.bem_get_stats()
        ctx.bem_destroy()
        res[d] = (_rel(y[rows], yo), st["m2l_pairs"], st["p2p_pairs"])
        print(f"cfg{n} direct_pairs {d} prec {prec}: S-D {res[d][0]:.2e}, m2l pairs {res[d][1]:.0f}, point pairs {res[d][2]:.3e}")
    for d in res:
        assert res[d][0] <= TOL_FULL[c["p"]]
    assert res[0][1] > res[-1][1] > res[10 ** 9][1] and res[0][2] < res[-1][2] < res[10 ** 9][2]
    assert res[10 ** 9][0] <= res[0][0] * 1.05


@pytest.mark.parametrize("quad", [0, 1])
def test_options_combine_on_v1_and_g3(quad):
    """fp32 pairs and direct far pairs with both quadratures: V1 has coincident source and target (j = i),
    which the fp32 kernel and the all-direct lists must skip as the fp64 kernel does."""
    c = cfg(1)
    rows = np.arange(c["V"].shape[0], dtype=np.int64)
    yo = oracle_rows(c, rows, quad)
    base = None
    for opts in (dict(), dict(direct_pairs=10 ** 9), dict(p2p_precision=1), dict(p2p_precision=1, direct_pairs=10 ** 9)):
        ctx = _ctx(c, quad=quad, p=12, lmax=3, **opts)
        y = _apply(ctx, c["q"], c["phi"])
        ctx.bem_destroy()
        e = _rel(y, yo)
        print(f"quad {quad} {opts}: {e:.2e}")
        assert e <= 1e-5
        base = e if base is None else base
        assert e <= 1.5 * base + 2e-6


def test_point_cloud_options_and_coincident_points():
    """Point clouds where sources and targets are the same points (r = 0 pairs are skipped) with fp32 pairs and with
    every leaf-level far pair summed directly."""
    pts, m01, rows = _cloud(30000, 21)
    m = 2.0 * m01 - 1.0
    yo = oracle.monopole_sum(pts, m, pts[rows])
    for opts in (dict(), dict(p2p_precision=1), dict(direct_pairs=10 ** 9), dict(p2p_precision=1, direct_pairs=10 ** 9)):
        ctx = _bem().bem_create_points(pts, pts)
        for k, v in opts.items():
            ctx.bem_set_option(k, v)
        ctx.bem_setup(12, 64, 2.5)
        y = np.full(len(pts), np.nan)
        ctx.bem_apply(m, None, y)
        ctx.bem_destroy()
        assert np.isfinite(y).all()
        e = _rel(y[rows], yo)
        print(opts, f"{e:.2e}")
        assert e <= 1e-5
