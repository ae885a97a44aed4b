"""bem_direct_sum_static -- the library's one entry that allocates no device memory -- against the existing direct-sum
path (bem_create_points, option "mode" = 1, bem_apply).  `pytest -m gpu`.

Why the entry exists: a host that has already given all device memory to its own arenas, that lives under a fixed
memory budget on a shared GPU, or that cannot take the device-wide synchronisation of cudaMalloc / cudaFree inside its
loop can use none of the other calls (they all allocate).  This one keeps its scratch -- the partial sums of the source
chunks -- in an 8 MiB array compiled into the library, so it takes at most DIRECT_STATIC_MAX_TARGETS targets per call and
all calls on a device share (and overwrite) the same array.

This file is named so that pytest collects it last: with `-x` a failure here hides no other test.  It passes alone in
a fresh process (its first call then does the per-device look-up of the scratch address) and after the other files."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

TOL_DIRECT = 1e-12      # relative L2, the tolerance of the direct-sum mode everywhere in tests/ (north_star)


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


def _existing_direct(bem, src, tgt, m, d):
    """the existing path: a point-cloud context in direct-sum mode (allocates its context, copies and partial sums)"""
    ctx = bem.bem_create_points(src, tgt)
    ctx.bem_set_option("mode", 1)
    ctx.bem_setup(8, 64, 2.5)
    y = np.full(tgt.shape[0], np.nan)
    ctx.bem_apply(m, d, y)
    ctx.bem_destroy()
    return y


def test_static_scratch_direct_sum_matches_the_allocating_path_twice_in_a_row():
    import torch
    import paper_1905_01341_b200 as bem

    dev = torch.device("cuda:0")
    rng = np.random.default_rng(20261106)
    # call A: monopoles + dipoles, 20,000 targets (40 target blocks -> 8 source chunks in the scratch)
    srcA = rng.uniform(0, 1, size=(30000, 3))
    tgtA = rng.uniform(-0.2, 1.2, size=(20000, 3))
    mA = rng.uniform(-1, 1, size=30000)
    dA = rng.normal(size=(30000, 3)) * 0.02
    # call B: monopoles only, 700 targets that ARE sources (r = 0 pairs are skipped), 16 chunks of other sizes: it lands
    # on the part of the scratch call A has just filled
    srcB = rng.uniform(0, 1, size=(5000, 3))
    tgtB = srcB[:700].copy()
    mB = rng.uniform(-1, 1, size=5000)

    refA = _existing_direct(bem, srcA, tgtA, mA, dA)
    refB = _existing_direct(bem, srcB, tgtB, mB, None)

    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    sA, tA, qA, ddA, sB, tB, qB = t(srcA), t(tgtA), t(mA), t(dA), t(srcB), t(tgtB), t(mB)
    yA = torch.full((20000,), float("nan"), dtype=torch.float64, device=dev)
    yB = torch.full((700,), float("nan"), dtype=torch.float64, device=dev)
    stream = torch.cuda.current_stream().cuda_stream

    # two calls in a row on one stream, no synchronisation between them
    bem.bem_direct_sum_static(sA, qA, ddA, tA, yA, stream)
    bem.bem_direct_sum_static(sB, qB, None, tB, yB, stream)
    torch.cuda.synchronize()
    outA, outB = yA.cpu().numpy(), yB.cpu().numpy()
    assert np.isfinite(outA).all() and np.isfinite(outB).all()
    eA, eB = _rel(outA, refA), _rel(outB, refB)
    print(f"static direct sum vs bem_apply(mode=1): A {eA:.2e}  B {eB:.2e}")
    assert eA <= TOL_DIRECT and eB <= TOL_DIRECT

    # the same two calls again: the array still holds call B's partial sums when A starts, and the results must not
    # notice (bit for bit: the chunks are added in a fixed order); no byte of device memory may be taken meanwhile
    yA2, yB2 = torch.empty_like(yA), torch.empty_like(yB)
    free_before = torch.cuda.mem_get_info()[0]
    bem.bem_direct_sum_static(sA, qA, ddA, tA, yA2, stream)
    bem.bem_direct_sum_static(sB, qB, None, tB, yB2, stream)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free_before
    assert torch.equal(yA2, yA) and torch.equal(yB2, yB)


def test_static_scratch_direct_sum_refuses_what_it_cannot_hold():
    import torch
    import paper_1905_01341_b200 as bem

    dev = torch.device("cuda:0")
    n_big = bem.DIRECT_STATIC_MAX_TARGETS + 1
    src = torch.rand((64, 3), dtype=torch.float64, device=dev)
    q = torch.ones(64, dtype=torch.float64, device=dev)
    tgt = torch.rand((n_big, 3), dtype=torch.float64, device=dev)
    y = torch.zeros(n_big, dtype=torch.float64, device=dev)
    with pytest.raises(bem.BemError) as e:
        bem.bem_direct_sum_static(src, q, None, tgt, y)
    assert e.value.status == bem.BEM_ERR_INVALID_ARG and "BEM_DIRECT_STATIC_MAX_TARGETS" in str(e.value)
    # exactly the maximum is accepted
    bem.bem_direct_sum_static(src, q, None, tgt[:-1], y[:-1])
    torch.cuda.synchronize()
    assert torch.isfinite(y[:-1]).all() and float(y[:-1].min()) > 0.0
    # a host array would have to be copied into a buffer the call may not allocate
    with pytest.raises(bem.BemError) as e:
        bem.bem_direct_sum_static(src, q.cpu(), None, tgt[:10], y[:10])
    assert e.value.status == bem.BEM_ERR_INVALID_ARG and "not device memory" in str(e.value)
    # no strengths at all: zeros, and nothing else is touched
    y[:10] = 7.0
    bem.bem_direct_sum_static(src, None, None, tgt[:10], y[:10])
    torch.cuda.synchronize()
    assert float(y[:10].abs().max()) == 0.0
