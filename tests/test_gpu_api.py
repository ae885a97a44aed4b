"""Boundary behaviour of the C-ABI on a real device: validation, error codes, host/device
pointers, determinism, invariances (pin P10), bem_solve (pins P7, P8).  `pytest -m gpu`."""
import numpy as np
import pytest

import bem_inputs as bi
from bem_inputs.configs import make_config
from bem_inputs.sph import real_sph_harm
import oracle

pytestmark = pytest.mark.gpu


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _bem():
    import paper_1905_01341_b200 as bem
    return bem


def _mk(V, F, bid=None, mode=0, quad=0, p=10, leaf=32, eta=2.5, **opts):
    ctx = _bem().bem_create(V, F, bid)
    ctx.bem_set_option("mode", mode)
    ctx.bem_set_option("quadrature", quad)
    for k, v in opts.items():
        ctx.bem_set_option(k, v)
    ctx.bem_setup(p, leaf, eta)
    return ctx


def _apply(ctx, q, phi):
    y = np.full(ctx.n_vertices, np.nan)
    ctx.bem_apply(q, phi, y)
    return y


# ------------------------------------------------------------------ bem_create validation
def test_create_rejects_bad_meshes():
    bem = _bem()
    V, F = bi.icosphere(1)
    with pytest.raises(bem.BemError) as e:            # inward orientation: negative volume
        bem.bem_create(V, F[:, [0, 2, 1]])
    assert e.value.status == bem.BEM_ERR_BAD_MESH
    with pytest.raises(bem.BemError) as e:            # a hole: two triangles removed
        bem.bem_create(V, F[:-2])
    assert e.value.status == bem.BEM_ERR_BAD_MESH
    Fb = F.copy(); Fb[3, 1] = V.shape[0]              # index out of range
    with pytest.raises(bem.BemError) as e:
        bem.bem_create(V, Fb)
    assert e.value.status == bem.BEM_ERR_BAD_MESH
    Fb = F.copy(); Fb[5] = Fb[5][[1, 0, 2]]           # one flipped triangle: edge used twice in one direction
    with pytest.raises(bem.BemError) as e:
        bem.bem_create(V, Fb)
    assert e.value.status == bem.BEM_ERR_BAD_MESH
    Vb = V.copy(); Vb[F[0, 1]] = Vb[F[0, 0]]          # zero-area triangle
    with pytest.raises(bem.BemError) as e:
        bem.bem_create(Vb, F)
    assert e.value.status == bem.BEM_ERR_BAD_MESH
    with pytest.raises(bem.BemError) as e:            # empty mesh
        bem.bem_create(np.zeros((0, 3)), np.zeros((0, 3), dtype=np.int32))
    assert e.value.status == bem.BEM_ERR_INVALID_ARG
    # a triangle that joins two bubbles
    c = make_config(4, n_bubbles=2)
    bid = c["bubble_id"].copy(); bid[c["F"][0, 0]] = 1 - bid[c["F"][0, 0]]
    with pytest.raises(bem.BemError) as e:
        bem.bem_create(c["V"], c["F"], bid)
    assert e.value.status == bem.BEM_ERR_BAD_MESH
    # one inverted bubble among two is caught by the per-bubble volume
    V2, F2, bid2 = c["V"], c["F"].copy(), c["bubble_id"]
    second = bid2[F2[:, 0]] == 1
    F2[second] = F2[second][:, [0, 2, 1]]
    with pytest.raises(bem.BemError) as e:
        bem.bem_create(V2, F2, bid2)
    assert e.value.status == bem.BEM_ERR_BAD_MESH


def test_setup_apply_argument_errors():
    bem = _bem()
    V, F = bi.icosphere(2)
    ctx = bem.bem_create(V, F)
    y = np.zeros(V.shape[0]); q = np.ones(V.shape[0])
    with pytest.raises(bem.BemError) as e:
        ctx.bem_apply(q, None, y)
    assert e.value.status == bem.BEM_ERR_NOT_SETUP
    for bad in ((0, 8, 2.5), (33, 8, 2.5), (8, 0, 2.5), (8, 8, 0.5)):
        with pytest.raises(bem.BemError) as e:
            ctx.bem_setup(*bad)
        assert e.value.status == bem.BEM_ERR_INVALID_ARG
    with pytest.raises(bem.BemError) as e:
        ctx.bem_set_option("no_such_option", 1)
    assert e.value.status == bem.BEM_ERR_INVALID_ARG
    ctx.bem_setup(6, 16, 2.5)
    with pytest.raises(bem.BemError) as e:            # y aliases q
        ctx.bem_apply(q, None, q)
    assert e.value.status == bem.BEM_ERR_INVALID_ARG
    ctx.bem_apply(None, None, y)                      # both densities absent: y = 0
    assert np.all(y == 0.0)
    ctx.bem_destroy()
    ctx.bem_destroy()                                 # idempotent


# ------------------------------------------------------------------ pointers, streams, determinism
@pytest.mark.parametrize("mode", [0, 1])
def test_host_and_device_pointers_agree_bitwise_and_runs_repeat(mode):
    import torch
    c = make_config(4, n_bubbles=12)
    ctx = _mk(c["V"], c["F"], c["bubble_id"], mode=mode)
    yh = _apply(ctx, c["q"], c["phi"])
    qd = torch.tensor(c["q"], device="cuda"); pd = torch.tensor(c["phi"], device="cuda")
    yd = torch.empty_like(qd)
    s = torch.cuda.Stream()
    ctx.bem_set_stream(s.cuda_stream)
    with torch.cuda.stream(s):
        ctx.bem_apply(qd, pd, yd)
        y1 = yd.cpu().numpy().copy()
        ctx.bem_apply(qd, pd, yd)
    s.synchronize()
    y2 = yd.cpu().numpy()
    assert np.array_equal(y1, yh)                     # same kernels, same order of sums
    assert np.array_equal(y1, y2)                     # no atomics on the data path: bit-reproducible
    # mixed: host q, device phi
    ym = torch.empty_like(qd)
    ctx.bem_apply(c["q"], pd, ym)
    assert np.array_equal(ym.cpu().numpy(), yh)


# ------------------------------------------------------------------ invariances (P10)
def test_invariances_fmm():
    c = make_config(4, n_bubbles=8)
    V, F, bid, q, phi = c["V"], c["F"], c["bubble_id"], c["q"], c["phi"]
    p = 16
    tol = 5e-6                                          # FMM truncation at p = 16 (tree placement changes)
    y = _apply(_mk(V, F, bid, p=p), q, phi)
    # linearity
    ctx = _mk(V, F, bid, p=p)
    yS, yD = _apply(ctx, q, None), _apply(ctx, None, phi)
    assert _rel(yS + yD, y) < 1e-13
    assert _rel(_apply(ctx, 3.0 * q, -2.0 * phi), 3.0 * yS - 2.0 * yD) < 1e-13
    # rigid motion
    rng = np.random.default_rng(3)
    Q, _ = np.linalg.qr(rng.normal(size=(3, 3)))
    if np.linalg.det(Q) < 0:
        Q[:, 0] = -Q[:, 0]
    V2 = V @ Q.T + np.array([100.0, -50.0, 7.0])
    assert _rel(_apply(_mk(V2, F, bid, p=p), q, phi), y) < tol
    # scaling lengths by a: S scales by a, D is unchanged
    a = 3.7
    ctx = _mk(a * V, F, bid, p=p)
    assert _rel(_apply(ctx, q, None), a * yS) < tol
    assert _rel(_apply(ctx, None, phi), yD) < tol
    # permutation of vertex and triangle order
    pv = rng.permutation(V.shape[0]); inv = np.empty_like(pv); inv[pv] = np.arange(V.shape[0])
    pt = rng.permutation(F.shape[0])
    V3 = V[pv]; F3 = inv[F[pt]].astype(np.int32); b3 = bid[pv]
    y3 = _apply(_mk(V3, F3, b3, p=p), q[pv], phi[pv])
    assert _rel(y3, y[pv]) < tol


def test_direct_permutation_is_exact_to_rounding():
    c = make_config(4, n_bubbles=3)
    V, F, bid, q, phi = c["V"], c["F"], c["bubble_id"], c["q"], c["phi"]
    y = _apply(_mk(V, F, bid, mode=1), q, phi)
    rng = np.random.default_rng(5)
    pv = rng.permutation(V.shape[0]); inv = np.empty_like(pv); inv[pv] = np.arange(V.shape[0])
    pt = rng.permutation(F.shape[0])
    y3 = _apply(_mk(V[pv], inv[F[pt]].astype(np.int32), bid[pv], mode=1), q[pv], phi[pv])
    assert _rel(y3, y[pv]) < 1e-13


# ------------------------------------------------------------------ free term and bem_solve
def test_free_term_is_solid_angle():
    """c_i = 1 + (D.1)_i = 1 - Omega_in/(4 pi) (reading R6; pin P2 on the oracle side)."""
    V, F = bi.icosphere(2)
    ctx = _mk(V, F, mode=1, eta=1e30)
    cf = ctx.bem_get_free_term()
    D1 = -oracle.g3_apply(V, F, None, np.ones(V.shape[0]), eta=1e30)
    assert np.abs(cf - (1.0 + D1)).max() < 1e-13
    ctx2 = _mk(V, F, mode=1, free_term=1)
    assert np.all(ctx2.bem_get_free_term() == 0.5)


@pytest.mark.parametrize("mode", [1, 0])
def test_solve_matches_dense_lu_of_the_oracle(mode):
    """P8: tiny mesh; S, D, c from the oracle's dense rows, q by LU."""
    V, F = bi.icosphere(2)
    V = V * np.array([1.0, 1.2, 0.9])
    N = V.shape[0]
    rng = np.random.default_rng(11)
    phi = rng.normal(size=N)
    S, D = oracle.g3_dense(V, F, eta=2.5)
    cfree = 1.0 + D @ np.ones(N)
    q_ref = np.linalg.solve(S, -cfree * phi + D @ phi)
    ctx = _mk(V, F, mode=mode, p=24, leaf=8, lmax=3)
    q = np.zeros(N)
    st, it, rr = ctx.bem_solve(phi, q, tol=1e-11, max_iter=N)
    assert st == 0 and rr <= 1e-11 and it <= N
    tol = 1e-8 if mode == 1 else 2e-6           # cond(S) ~ 33 times the residual / FMM truncation
    assert _rel(q, q_ref) < tol
    # warm start from the answer: converges at once
    st, it2, rr2 = ctx.bem_solve(phi, q, use_q_as_x0=True, tol=1e-8, max_iter=N)
    assert st == 0 and it2 <= 1
    # restarted GMRES reaches the same answer
    ctx.bem_set_option("gmres_restart", 10)
    q2 = np.zeros(N)
    st, it3, rr3 = ctx.bem_solve(phi, q2, tol=1e-9, max_iter=2000)
    assert st == 0 and _rel(q2, q_ref) < 1e-5


def test_solve_not_converged_returns_last_iterate():
    bem = _bem()
    c = make_config(4, n_bubbles=4)
    ctx = _mk(c["V"], c["F"], c["bubble_id"])
    q = np.zeros(c["V"].shape[0])
    st, it, rr = ctx.bem_solve(c["phi"], q, tol=1e-14, max_iter=3)
    assert st == bem.BEM_ERR_NOT_CONVERGED and it == 3 and 0 < rr < 1 and np.isfinite(q).all() and np.abs(q).max() > 0
    # the reported residual is the true residual of the returned iterate, checked by the oracle
    rows = np.arange(0, c["V"].shape[0], 7, dtype=np.int64)
    V, F = c["V"], c["F"]
    Dphi = -oracle.g3_apply(V, F, None, c["phi"], rows=rows)
    D1 = -oracle.g3_apply(V, F, None, np.ones(V.shape[0]), rows=rows)
    b = -(1.0 + D1) * c["phi"][rows] + Dphi
    r = b - oracle.g3_apply(V, F, q, None, rows=rows)
    assert abs(np.linalg.norm(r) / np.linalg.norm(b) - rr) < 0.05 * rr


def test_solve_sphere_dirichlet_to_neumann():
    """P7: on the sphere of radius R, phi = Y_n^m gives q = -(n+1)/R Y_n^m up to O(h^2)."""
    v0, F = bi.icosphere(3)
    R = 1.5
    V = R * v0
    th = np.arccos(np.clip(v0[:, 2], -1, 1)); ph = np.arctan2(v0[:, 1], v0[:, 0])
    ctx = _mk(V, F, p=12, leaf=32)
    for n, m, tol in ((1, 0, 2e-2), (3, 1, 5e-2)):
        Y = real_sph_harm(n, m, th, ph)
        q = np.zeros(V.shape[0])
        st, it, rr = ctx.bem_solve(Y, q, tol=1e-8, max_iter=200)
        assert st == 0
        assert _rel(q, -(n + 1) / R * Y) < tol


def test_timings_and_stats():
    import torch
    c = make_config(4, n_bubbles=20)
    ctx = _mk(c["V"], c["F"], c["bubble_id"], timing=1)
    st = ctx.bem_get_stats()
    N = c["V"].shape[0]
    assert st["n_targets"] == N and st["n_sources"] == 3 * c["F"].shape[0]
    assert st["csr_nnz"] > 6 * N and st["p2p_pairs"] > 0 and st["m2l_pairs"] > 0 and st["kernel_launches_per_apply"] >= 7
    qd = torch.tensor(c["q"], device="cuda"); yd = torch.empty_like(qd)
    ctx.bem_apply(qd, qd, yd)
    t = ctx.bem_get_timings()
    assert t["total"] > 0 and abs(sum(v for k, v in t.items() if k != "total") - t["total"]) < 0.2 * t["total"] + 0.05
    assert ctx.bem_fp64_peak() > 1000.0           # GFLOP/s


def test_solve_diagonal_preconditioner_same_solution_fewer_iterations():
    """Option precond = 1 (right scaling by S_ii) solves the same system: same q to the tolerance, and on a
    polydisperse cluster (config 4 recipe, radii spread 3x) in fewer iterations."""
    c = make_config(4, n_bubbles=12)
    V, F, bid, phi = c["V"], c["F"], c["bubble_id"], c["phi"]
    ctx = _mk(V, F, bid, p=12)
    res = {}
    for pre in (0, 1):
        ctx.bem_set_option("precond", pre)
        q = np.zeros(V.shape[0])
        st, it, rr = ctx.bem_solve(phi, q, tol=1e-8, max_iter=400)
        assert st == 0 and rr <= 1e-8
        res[pre] = (q, it)
    ctx.bem_destroy()
    print("iterations", res[0][1], res[1][1])
    assert _rel(res[1][0], res[0][0]) <= 1e-5          # cond(S) ~ 1e2-1e3 times the residual tolerance
    assert res[1][1] < res[0][1]


def test_non_default_stream_and_option_toggles_between_products():
    """bem_set_stream with a torch side stream: same bits as on the default stream; p2p_precision, reduce_ctas, p2p_ctas
    and timing may change between products without a new bem_setup (include/bem.h)."""
    import torch
    c = make_config(4, n_bubbles=30)
    ctx = _bem().bem_create(c["V"], c["F"], c["bubble_id"])
    ctx.bem_setup(c["p"], c["leaf_size"], c["eta"])
    qd, pd = torch.tensor(c["q"], device="cuda"), torch.tensor(c["phi"], device="cuda")
    y0 = torch.empty_like(qd)
    ctx.bem_apply(qd, pd, y0)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    ctx.bem_set_stream(side.cuda_stream)
    y1 = torch.empty_like(qd)
    with torch.cuda.stream(side):
        ctx.bem_apply(qd, pd, y1)
    side.synchronize()
    assert torch.equal(y0, y1)
    outs = {}
    for prec in (1, 0, 1):
        ctx.bem_set_option("p2p_precision", prec)
        for rc, pc, tm in ((0, 0, 0), (3, 2, 0), (16, 6, 0), (0, 0, 1)):
            ctx.bem_set_option("reduce_ctas", rc); ctx.bem_set_option("p2p_ctas", pc); ctx.bem_set_option("timing", tm)
            y = torch.empty_like(qd)
            with torch.cuda.stream(side):
                ctx.bem_apply(qd, pd, y)
            side.synchronize()
            outs.setdefault(prec, []).append(y.clone())
    # CUDA graph replay (option graph, default on): the third and later products with the same pointers are one launch
    ctx.bem_set_option("p2p_precision", 0); ctx.bem_set_option("timing", 0); ctx.bem_set_option("reduce_ctas", 0); ctx.bem_set_option("p2p_ctas", 0)
    yg = torch.empty_like(qd)
    for prec in (0, 1):
        ctx.bem_set_option("p2p_precision", prec)
        for rep in range(5):
            yg.fill_(float("nan"))
            with torch.cuda.stream(side):
                ctx.bem_apply(qd, pd, yg)
                ctx.bem_apply(qd, None, y1)                         # a second cached product in between
            side.synchronize()
            assert torch.equal(yg, outs[prec][0]), (prec, rep)
    ctx.bem_set_option("graph", 0)
    with torch.cuda.stream(side):
        ctx.bem_apply(qd, pd, yg)
    side.synchronize()
    assert torch.equal(yg, outs[1][0])
    # bem_setup itself on the (non-blocking) side stream: same lists, same bits
    st0 = ctx.bem_get_stats()
    ctx2 = _bem().bem_create(c["V"], c["F"], c["bubble_id"])
    ctx2.bem_set_stream(side.cuda_stream)
    with torch.cuda.stream(side):
        ctx2.bem_setup(c["p"], c["leaf_size"], c["eta"])
        y2 = torch.empty_like(qd)
        ctx2.bem_apply(qd, pd, y2)
    side.synchronize()
    st2 = ctx2.bem_get_stats()
    for k in ("p2p_pairs", "m2l_pairs", "csr_nnz", "lmax", "n_src_leaves", "n_tgt_leaves"):
        assert st0[k] == st2[k], k
    assert torch.equal(y2, y0)
    ctx2.bem_destroy()
    ctx.bem_set_stream(0)
    ctx.bem_destroy()
    for prec, ys in outs.items():
        assert all(torch.equal(ys[0], y) for y in ys)               # launch configuration never changes the bits
    assert torch.equal(outs[0][0], y0)
    rel = float(torch.linalg.norm(outs[1][0] - y0) / torch.linalg.norm(y0))
    assert 0 < rel < 5e-6


def test_solve_with_single_precision_pairs_reaches_the_same_solution():
    c = make_config(4, n_bubbles=20)
    ctx = _bem().bem_create(c["V"], c["F"], c["bubble_id"])
    ctx.bem_setup(12, c["leaf_size"], c["eta"])
    ctx.bem_set_option("precond", 1)
    N = c["V"].shape[0]
    sols = []
    for prec in (0, 1):
        ctx.bem_set_option("p2p_precision", prec)
        q = np.zeros(N)
        st, it, rr = ctx.bem_solve(c["phi"], q, tol=1e-6, max_iter=500)
        print("p2p_precision", prec, "status", st, "iterations", it, "relres", rr)
        assert st == 0 and rr <= 1e-6
        sols.append((q, it))
    ctx.bem_destroy()
    (q0, it0), (q1, it1) = sols
    assert abs(it0 - it1) <= 2
    assert np.linalg.norm(q1 - q0) / np.linalg.norm(q0) < 1e-3    # cond(S) times (tolerance + the 1e-6 perturbation of the operator)


def test_apply_inside_a_callers_cuda_graph():
    """A caller may capture bem_apply into a CUDA graph of its own (torch.cuda.graph): the library then launches kernel by
    kernel into that capture instead of starting one of its own."""
    import torch
    c = make_config(1)
    ctx = _bem().bem_create(c["V"], c["F"], c["bubble_id"])
    ctx.bem_setup(c["p"], c["leaf_size"], c["eta"])
    qd, pd = torch.tensor(c["q"], device="cuda"), torch.tensor(c["phi"], device="cuda")
    y0, y1 = torch.empty_like(qd), torch.empty_like(qd)
    ctx.bem_apply(qd, pd, y0)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    ctx.bem_set_stream(side.cuda_stream)
    with torch.cuda.stream(side):
        ctx.bem_apply(qd, pd, y1)                                    # warm: every lazy allocation and attribute is made
    side.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=side):
        ctx.bem_apply(qd, pd, y1)
    for _ in range(3):
        y1.fill_(float("nan"))
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(y0, y1)
    ctx.bem_set_stream(0)
    ctx.bem_destroy()
