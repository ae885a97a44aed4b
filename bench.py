#!/usr/bin/env python
"""bench.py -- one JSON line for the BEM matrix-vector product (BASELINE.json metric:
"BEM MVP ms/apply vs N nodes; P2P Gpairs/s; M2L/SpMV % of FP64/HBM roofline").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

A step = one bem_apply (the whole hot path: lift, P2M, M2M, M2L, L2L, L2P, P2P, correction SpMV)
on a seeded synthetic bubble cluster.  Default workload: config 5 of BASELINE.json (4000 bubbles,
2,568,000 nodes, p = 12, fp64) -- the >= 2.5M-node cluster the north_star's target names.

  value     ms per bem_apply with q, phi, y resident in HBM (CUDA events on the context's stream)
  e2e       the same call with HOST buffers: H2D of q and phi, D2H of y inside the timed region
  roofline  the dominant kernel (on config 5 the near-field pair kernel p2p_leaf_kernel, FP64 ALU bound) against the
            DFMA loop measured in the same run; the other kernels with their own roofs under "kernels"
  sweep     (default run only) configs 1-4 timed the same way: the metric is ms/apply VERSUS N nodes
  cpu_baseline  the CPU oracle, timed on a bounded sample of target rows of the same workload

The path does not shard (BASELINE.json: one GPU, no collectives): --gpus N runs N independent
replicas, one per rank ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from bem_inputs.configs import make_config, sample_rows  # noqa: E402

METRIC = "bem_apply_ms"
UNIT = "ms"
# nominal FP64 FMA peak of B200 for the "alu" roofline: 148 SMs x 64 FP64
# FMA lanes per SM per clock x 2 flop x 1.965 GHz (clocks.max.sm)
FP64_NOMINAL_GFLOPS = 148 * 64 * 2 * 1.965


def ncu_traffic(kernel, cfg):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` from the committed ncu --set full capture:
    profiles/traffic.json names the commit and the command it came from.  None when there is no capture of this kernel
    on this config (the file says which config it was taken on)."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
        if int(t.get("config", -1)) != int(cfg):
            return None
        v = t["kernels"].get(kernel)
        return None if v is None else float(v["dram_bytes"])
    except Exception:
        return None


def workload_name(c):
    return c["name"]


def use_adaptive_tree(args):
    """The adaptive octree (option tree = 1) is the faster one on config 5 (21.4 against 22.2 ms) and within
    1% of the uniform one elsewhere: auto = adaptive on config 5 with fp64 pairs (fp32 pairs need the uniform tree)."""
    if args.direct:
        return False
    return (args.tree == "adaptive" or (args.tree == "auto" and args.config == 5 and args.p2p_precision == 64)
            or any(o.replace(" ", "") == "tree=1" for o in args.opt))


def bench_leaf_size(args, c):
    """leaf_size of the run: the config's, or 350 for the adaptive tree on config 5 (measured optimum; the uniform tree of
    config 5 has l_max = 6 for any leaf_size between 171 and 678)."""
    if args.leaf_size:
        return int(args.leaf_size)
    return 350 if (args.config == 5 and use_adaptive_tree(args)) else int(c["leaf_size"])


def p_with_dipoles(args, p):
    """The truncation a product WITH phi executes (include/bem.h option "dipole_degrees"; R5'): the stated p is the
    truncation of the monopole (single-layer) products; dipole sources carry 3 more degrees below p = 12 unless the option
    says otherwise.  Direct mode has no truncation.  run_gpu checks this against the library's own BEM_S_P_DIPOLE."""
    if args.direct:
        return int(p)
    dd = None
    for o in args.opt:
        k, _, v = o.replace(" ", "").partition("=")
        if k == "dipole_degrees":
            dd = int(float(v))
    if dd is None or dd < 0:
        dd = 3 if p < 12 else 0
    return int(min(32, p + dd))


def workload_config(c, args, p):
    """The keys that name the workload -- the SAME dict in the b200 arm and in the reference arm (the CPU oracle computes
    the same discretised operator on the same inputs); what only the GPU run knows (tree depth, launch mode, device bytes)
    goes to the line's "run" key."""
    N, T = int(c["V"].shape[0]), int(c["F"].shape[0])
    cloud = bool(c.get("cloud"))
    return dict(workload=workload_name(c), operator="y = S[q] - D[phi] (G3 quadrature + near correction)" if not cloud else "monopole sum",
                p=int(p), p_executed_with_phi=(int(p) if cloud else p_with_dipoles(args, p)),
                p_note="p = truncation of the products without dipoles (S[q], every GMRES iteration); S[q] - D[phi] runs at p_executed_with_phi",
                n_nodes=N, n_triangles=T, n_sources=(N if cloud else 3 * T), leaf_size=bench_leaf_size(args, c),
                eta=c["eta"], parallelism="replicas only" if args.gpus > 1 else "1 gpu",
                l2="working set larger than L2" if N >= 100000 else "flushed between iterations (512 MB write)")


def cloud_config(n, seed=190501341 + 6):
    """Config 6 (not in BASELINE.json): the paper's own Tables 1-2 workload -- n monopoles placed
    randomly and uniformly in the unit cube, sources = receivers, intensities U(-1, 1), p = 12."""
    from bem_inputs.configs import random_cube_points
    pts, m = random_cube_points(n, seed)
    return dict(V=pts, F=np.zeros((0, 3), np.int32), bubble_id=None, q=2.0 * m - 1.0, phi=None, p=12, leaf_size=256, eta=2.5,
                cfg=6, cloud=True, name=f"cfg6: {n:,} uniform random monopoles in the unit cube (paper Tables 1-2)")


def lattice_config(nb, seed=190501341 + 7):
    """Config 7 (not in BASELINE.json): the paper's own scaling family and the workload of its Table 3 -- nb^3 equal bubbles
    (icosphere L3, 642 vertices, a0 = 1) on a regular grid with centre spacing 4 a0;
    nb = 12 -> N = 1,109,376, nb = 16 -> N = 2,629,632.  q, phi ~ U(-1, 1)."""
    from bem_inputs.meshes import lattice_cluster, icosphere
    V, F, bid = lattice_cluster(3, nb, 4.0, 1.0)
    rng = np.random.default_rng(seed)
    N = V.shape[0]
    return dict(V=np.ascontiguousarray(V), F=np.ascontiguousarray(F, dtype=np.int32), bubble_id=bid, q=rng.uniform(-1, 1, N),
                phi=rng.uniform(-1, 1, N), p=12, leaf_size=256, eta=2.5, cfg=7, template=icosphere(3)[0],
                name=f"cfg7: {nb}x{nb}x{nb} regular cluster, spacing 4 a0, icosphere L3, {N:,} nodes (paper Table 3 family)")


def get_config(args):
    if args.config == 7:
        return lattice_config(args.lattice_nb)
    return cloud_config(args.cloud_points) if args.config == 6 else make_config(args.config)


def oracle_sample(c, seconds_target=15.0):
    """Time the oracle, as it stands, on a bounded sample of target rows; extrapolate to all rows
    (rows are independent: the paper extrapolates its CPU brute-force reference the same way)."""
    import oracle
    V, F, q, phi = c["V"], c["F"], c["q"], c["phi"]
    N = V.shape[0]
    cores = oracle.num_threads()
    if c.get("cloud"):
        nsrc = N
        run = lambda rows: oracle.monopole_sum(V, q, V[rows])
    else:
        nsrc = 3 * F.shape[0]
        run = lambda rows: oracle.g3_apply(V, F, q, phi, eta=c["eta"], rows=rows)
    probe = sample_rows(c["cfg"], N, min(N, 4 * cores))
    t0 = time.perf_counter()
    run(probe)
    dt = max(time.perf_counter() - t0, 1e-4)
    nrows = int(min(N, max(len(probe), seconds_target / dt * len(probe))))
    rows = sample_rows(c["cfg"], N, nrows)
    t0 = time.perf_counter()
    y = run(rows)
    dt = time.perf_counter() - t0
    ms_full = dt * 1e3 * N / len(rows)
    return dict(value=ms_full, unit=UNIT, cores=cores, kind="oracle",
                sample=f"{len(rows)} of {N} target rows x all {nsrc} sources in {dt:.2f} s, scaled by N/rows",
                ns_per_pair=dt * 1e9 / (len(rows) * float(nsrc))), rows, y


def run_reference(args):
    """--impl reference: the CPU oracle on the same config/metric; each step is one bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = get_config(args)
    per_step = []
    info = None
    for i in range(args.warmup + args.steps):
        info, _, _ = oracle_sample(c, seconds_target=args.ref_seconds)
        if i >= args.warmup:
            per_step.append(info["value"])
    v = float(np.mean(per_step))
    line = dict(impl="reference", metric=METRIC, value=v, unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                warmup=args.warmup, ms_per_step=v, higher_is_better=False, scaling="weak", vs_baseline=None,
                dtype="f64", data="synthetic", config=workload_config(c, args, args.p or c["p"]),
                ratio_note="this arm is the plain O(N^2) direct sum of the oracle: a b200 / reference ratio is 'FMM on a GPU vs direct sum "
                           "on host cores' and says nothing about kernel quality (the roofline fractions do)",
                cpu_baseline=dict(value=v, unit=UNIT, cores=info["cores"], kind="oracle", sample=info["sample"]),
                e2e=dict(value=v, unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)
    print(json.dumps(line), flush=True)


class ClockSampler:
    """nvidia-smi clocks + throttle reasons during the timed region (B200_PROFILING.md)."""

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except Exception:
            self.p = None

    def stop(self):
        if self.p is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.f.read().splitlines():
            parts = [x.strip() for x in ln.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1]))
            except ValueError:
                continue
            for nme, v in zip(names, parts[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        os.unlink(self.f.name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=float(max(mx)) if mx else None,
                    samples=len(sm), reasons=sorted(reasons))


def run_sweep(args, bem, torch, stream):
    """The other points of "ms/apply vs N nodes" (BASELINE.json metric): configs 1-4 with the library's defaults at each
    config's own p and leaf_size, timed like the headline (device-resident value, end-to-end with host buffers) and checked
    against the oracle on seeded rows (all rows on config 1).  A failure is recorded, it does not cost the headline."""
    import oracle
    out = []
    fbuf = torch.empty(512 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda")

    def timed(fn, steps, flush):
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in evs:
            if flush:
                fbuf.fill_(1.0)
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in evs)

    for k in (1, 2, 3, 4):
        try:
            c = make_config(k)
            V, F = c["V"], c["F"]
            N = V.shape[0]
            ctx = bem.bem_create(V, F, c["bubble_id"])
            ctx.bem_set_stream(stream.cuda_stream)
            ctx.bem_setup(c["p"], c["leaf_size"], c["eta"])
            st = ctx.bem_get_stats()
            qd, pd = torch.tensor(c["q"], device="cuda"), torch.tensor(c["phi"], device="cuda")
            yd = torch.empty_like(qd)
            qh, ph = torch.tensor(c["q"]).pin_memory(), torch.tensor(c["phi"]).pin_memory()
            yh = torch.empty(N, dtype=torch.float64).pin_memory()
            n_it = max(3, min(args.steps, 10))
            for _ in range(3):
                ctx.bem_apply(qd, pd, yd)
            flush = N < 100000
            ms = timed(lambda: ctx.bem_apply(qd, pd, yd), n_it, flush) / n_it
            for _ in range(2):
                ctx.bem_apply(qh, ph, yh)
            e2e = timed(lambda: ctx.bem_apply(qh, ph, yh), n_it, flush) / n_it
            y = yd.cpu().numpy()
            rows = sample_rows(c["cfg"], N, N if N < 3000 else args.sweep_rows)
            yo = oracle.g3_apply(V, F, c["q"], c["phi"], eta=c["eta"], rows=rows)
            out.append(dict(config=k, workload=c["name"], n_nodes=int(N), p=int(c["p"]), p_executed_with_phi=int(st["p_dipole"]),
                            leaf_size=int(c["leaf_size"]), lmax=int(st["lmax"]), ms=ms, e2e_ms=e2e, steps=n_it,
                            parity_rel_l2_vs_oracle=float(np.linalg.norm(y[rows] - yo) / np.linalg.norm(yo)), parity_rows=int(len(rows)),
                            l2="flushed between iterations (512 MB write)" if flush else "working set larger than L2"))
            ctx.bem_destroy()
            del qd, pd, yd
        except Exception as e:  # noqa: BLE001
            out.append(dict(config=k, error=repr(e)[:300]))
    return out


def run_gpu(args):
    import torch
    import paper_1905_01341_b200 as bem

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the BEM library has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    c = get_config(args)
    V, F = c["V"], c["F"]
    N, T = V.shape[0], F.shape[0]
    p = args.p or c["p"]
    # bem_apply replays a CUDA graph on any stream but the legacy default one (option "graph"): one launch instead of 20-40,
    # which pays on the launch-bound small meshes (config 1: 0.104 -> 0.079 ms); on the large configs the product is
    # kernel-bound and measured 1-3% faster launched kernel by kernel on the default stream.  auto = side stream below 200k nodes
    stream = torch.cuda.current_stream()
    if args.stream == "side" or (args.stream == "auto" and N < 200000):
        stream = torch.cuda.Stream()
        torch.cuda.set_stream(stream)

    t0 = time.perf_counter()
    ctx = bem.bem_create_points(V, V) if c.get("cloud") else bem.bem_create(V, F, c["bubble_id"])
    ctx.bem_set_stream(stream.cuda_stream)
    ctx.bem_set_option("mode", 1 if args.direct else 0)
    adaptive = use_adaptive_tree(args)
    if adaptive:
        ctx.bem_set_option("tree", 1)
    if args.lmax:
        ctx.bem_set_option("lmax", args.lmax)
    if args.no_graph:
        ctx.bem_set_option("graph", 0)
    if args.p2p_precision == 32:
        ctx.bem_set_option("p2p_precision", 1)
    if args.direct_pairs is not None:
        ctx.bem_set_option("direct_pairs", args.direct_pairs)
    if args.p2p_ctas:
        ctx.bem_set_option("p2p_ctas", args.p2p_ctas)
    if args.reduce_ctas:
        ctx.bem_set_option("reduce_ctas", args.reduce_ctas)
    for kv in args.opt:
        k, v = kv.split("=")
        ctx.bem_set_option(k, float(v))
    ctx.bem_setup(p, bench_leaf_size(args, c), c["eta"])
    torch.cuda.synchronize()
    setup_wall_ms = (time.perf_counter() - t0) * 1e3
    stats = ctx.bem_get_stats()

    cloud = bool(c.get("cloud"))
    qd = torch.tensor(c["q"], device="cuda"); pd = None if cloud else torch.tensor(c["phi"], device="cuda")
    yd = torch.empty_like(qd)
    qh = torch.tensor(c["q"]).pin_memory(); ph = None if cloud else torch.tensor(c["phi"]).pin_memory()
    yh = torch.empty(N, dtype=torch.float64).pin_memory()

    # L2 policy: the working set of one apply (sources, expansions, lists, CSR) is far above the 126 MB L2 for
    # configs 3-5; for the small configs a 512 MB buffer is rewritten between timed iterations.
    flush = N < 100000
    fbuf = torch.empty(512 * 1024 * 1024 // 8, dtype=torch.float64, device="cuda") if flush else None

    def timed(fn, steps):
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        for a, b in evs:
            if fbuf is not None:
                fbuf.fill_(1.0)
            a.record(stream)
            fn()
            b.record(stream)
        torch.cuda.synchronize()
        return sum(a.elapsed_time(b) for a, b in evs)

    for _ in range(max(args.warmup, 3)):
        ctx.bem_apply(qd, pd, yd)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    total_ms = timed(lambda: ctx.bem_apply(qd, pd, yd), args.steps)
    barrier()
    # end to end: host (pinned) q, phi -> y host, copies inside the call
    for _ in range(2):
        ctx.bem_apply(qh, ph, yh)
    barrier()
    e2e_ms = timed(lambda: ctx.bem_apply(qh, ph, yh), args.steps)
    barrier()
    clocks = sampler.stop() if sampler else None
    if dist is not None:
        t = torch.tensor([total_ms, e2e_ms], device="cuda", dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms, e2e_ms = t.tolist()
    ms = total_ms / args.steps
    e2e = e2e_ms / args.steps
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # per-kernel-class breakdown (CUDA events inside bem_apply, on the context's stream), averaged
    ctx.bem_set_option("timing", 1)
    acc = None
    nb = max(3, min(args.steps, 10))
    for _ in range(nb):
        if fbuf is not None:
            fbuf.fill_(1.0)
        ctx.bem_apply(qd, pd, yd)
        t = ctx.bem_get_timings()
        acc = t if acc is None else {k: acc[k] + t[k] for k in t}
    ctx.bem_set_option("timing", 0)
    tm = {k: v / nb for k, v in acc.items()}
    dfma = ctx.bem_fp64_peak()
    dmma = ctx.bem_fp64_tensor_peak()
    hbm = None
    try:
        hbm = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]
    except Exception:
        pass
    hbm_peak, hbm_src = (hbm, "measured") if hbm else (6650.0, "fallback")

    # ---- roofline of the dominant kernel + the other kernels the metric names
    # FP64 pipe: 148 SMs x 64 lanes x 1.965 GHz = 18.6 T instr/s; an FMA counts 2 flop, so the flop peak is 37.2 TFLOP/s.
    # P2P: 17 FP64 instructions per pair (9 DFMA + 5 DMUL + 3 DADD = 26 flop; SASS count).
    P2P_INSTR, P2P_FLOP = 17.0, 26.0
    if not args.direct and not any(o.replace(" ", "") == "p2p_exact=1" for o in args.opt):
        # FMM mode: ONE Newton step after the hardware seed (option p2p_exact = 0): 8 DFMA + 5 DMUL + 3 DADD per pair
        P2P_INSTR, P2P_FLOP = 16.0, 24.0
    slot_peak = FP64_NOMINAL_GFLOPS / 2e3                      # T instr/s
    f32 = args.p2p_precision == 32 and not args.direct
    if f32:
        # fp32 pairs (p2p_f32.cu): 12 FP32-pipe instructions (6 FFMA + 3 FMUL + 3 FADD = 18 flop) + 1 MUFU.RSQ per pair;
        # FP32 pipes: 148 SMs x 128 lanes x 1.965 GHz = 37.2 T instr/s
        P2P_INSTR, P2P_FLOP = 12.0, 18.0
        slot_peak = 2.0 * FP64_NOMINAL_GFLOPS / 2e3
    nre = stats["exp_stride"] / 2.0
    kernels = {}
    p2p_s = tm["p2p"] * 1e-3
    kernels["p2p"] = dict(ms=tm["p2p"], pairs=stats["p2p_pairs"], pairs_executed=stats["p2p_pairs_executed"],
                          executed_note="source lists are padded to rounds of 128: pairs / pairs_executed of the kernel's work is useful",
                          pairs_wx=stats["p2p_pairs_wx"], wx_share=(stats["p2p_pairs_wx"] / stats["p2p_pairs"]) if stats["p2p_pairs"] else None,
                          wx_note="adaptive tree: pairs of W-list and X-list ranges, which the library sums directly instead of M2P / P2L (0 on the uniform tree)",
                          gpairs_per_s=stats["p2p_pairs"] / p2p_s / 1e9 if p2p_s > 0 else None,
                          tflops=stats["p2p_pairs"] * P2P_FLOP / p2p_s / 1e12 if p2p_s > 0 else None,
                          fp64_slot_frac=stats["p2p_pairs"] * P2P_INSTR / p2p_s / 1e12 / slot_peak if p2p_s > 0 else None,
                          note=("12 FP32 instr (18 flop) + 1 MUFU.RSQ per pair; fp64_slot_frac here = share of the FP32 pipes' issue slots (nominal 37.2 T instr/s)"
                                if f32 else "%d FP64 instr / %d flop per pair; slot_frac = share of the FP64 pipe's issue slots (nominal 18.6 T instr/s)" % (P2P_INSTR, P2P_FLOP)))
    if not args.direct:
        m2l_s = tm["m2l"] * 1e-3
        exec_flop = stats["m2l_flop"]                             # two blocks of (4 KE)^2 MACs per pair, KE = k-steps of the pair's truncation class
        dense_flop = stats["m2l_pairs"] * 2.0 * p ** 4            # the dense p^2 x p^2 translation of SURVEY.md 8(d)
        kernels["m2l"] = dict(ms=tm["m2l"], pairs=stats["m2l_pairs"], executed_tflops=exec_flop / m2l_s / 1e12,
                              dense_equivalent_tflops=dense_flop / m2l_s / 1e12,
                              frac_of_measured_dmma_peak=exec_flop / m2l_s / 1e9 / dmma, frac_of_nominal_fp64_peak=exec_flop / m2l_s / 1e9 / FP64_NOMINAL_GFLOPS,
                              note="executed = the graded-truncation count the library reports (BEM_S_M2L_FLOP): per pair two blocks of (4 KE)^2 "
                                   "multiply-adds, KE = k-steps of the pair's truncation class (full order: 4 nre^2 flop, nre = %d); dense-equivalent = 2 p^4" % int(nre))
        red_bytes = stats["m2l_row_bytes"]
        kernels["reduce"] = dict(ms=tm["l2l_reduce"], gbs=red_bytes / (tm["l2l_reduce"] * 1e-3) / 1e9,
                                 frac_hbm=red_bytes / (tm["l2l_reduce"] * 1e-3) / 1e9 / hbm_peak, bytes=red_bytes,
                                 note="bytes = the packed translated rows the sums read (BEM_S_M2L_ROW_BYTES: 16 bytes x the dofs each pair's "
                                      "truncation class carries); the L2L tiles and sums run in the same timing class and their rows are not counted")
        # P2M is FP64-ALU bound: FP64 SASS instructions of p2m_kernel_t<P, DIP> per (lane, source) -- static count of
        # DFMA + DMUL + DADD in the kernel (cuobjdump -sass); the 32-entry row sums execute 4x their static 8, so it is a lower bound
        P2M_FP64 = {(8, 0): 323, (8, 1): 617, (10, 0): 499, (10, 1): 967, (12, 0): 690, (12, 1): 1372, (14, 0): 930, (14, 1): 1866,
                    (16, 0): 1207, (16, 1): 2450}
        p_run = int(stats["p_dipole"]) if pd is not None else int(p)
        key = (max(8, p_run + (p_run & 1)), 0 if pd is None else 1)
        ins = P2M_FP64.get(key)
        p2m_s = tm["p2m"] * 1e-3
        kernels["p2m"] = dict(ms=tm["p2m"], msources_per_s=stats["n_sources"] / p2m_s / 1e6, bound="alu",
                              fp64_instr_per_source=ins,
                              fp64_slot_frac_lower_bound=(stats["n_sources"] * ins / p2m_s / 1e12 / (FP64_NOMINAL_GFLOPS / 2e3)) if ins else None,
                              note="FP64 instructions per source: static SASS count of p2m_kernel_t<%d, %s>; slots against the nominal 18.6 T instr/s; "
                                   "idle lanes of ragged leaves not counted" % (key[0], "dipoles" if key[1] else "monopoles"))
        # tree passes that only move data (north_star: "achieved HBM GB/s for SpMV and tree passes, each against the B200 peak");
        # algorithmic bytes per unit as stated in DESIGN.md section 8
        nst = stats["exp_stride"]
        tree = dict(
            lift=(80.0 * stats["n_sources"], "80 B per source (weights 32, vertex ids 16, strengths written 32); the densities (16 N B) stay in L2 and are not counted"),
            m2m=(8.0 * nst * (stats["m2m_pairs"] + stats["m2m_parents"]), "one child expansion read per (child, parent) translation, one parent expansion written (8 nst B each)"),
            l2p=(32.0 * N + 8.0 * nst * stats["n_tgt_leaves"], "24 B position + 8 B result per target, one local expansion (8 nst B) per target leaf"))
        for name, (nbytes, what) in tree.items():
            t_s = tm[name] * 1e-3
            if t_s > 0:
                kernels[name] = dict(ms=tm[name], bytes=nbytes, gbs=nbytes / t_s / 1e9, frac_hbm=nbytes / t_s / 1e9 / hbm_peak, note=what)
        kernels["l2l"] = dict(note="runs inside the 'reduce' timing class (L2L tiles + sums follow the M2L sums of each level): no separate figure")
    spmv_bytes = 20.0 * stats["csr_nnz"] + 32.0 * N
    kernels["spmv"] = dict(ms=tm["spmv"], gbs=spmv_bytes / (tm["spmv"] * 1e-3) / 1e9, frac_hbm=spmv_bytes / (tm["spmv"] * 1e-3) / 1e9 / hbm_peak,
                           hbm_peak_gbs=hbm_peak, hbm_peak_source=hbm_src, bytes=spmv_bytes)
    common = dict(peak_source="measured in this run: register-resident DFMA loop (bem_fp64_peak) %.1f TFLOP/s, DMMA loop %.1f TFLOP/s; "
                              "MEASURED_PEAKS.json has no FP64 entry; derived nominal for context: 148 SMs x 64 FP64 lanes/clk x 2 flop x 1.965 GHz = %.1f"
                              % (dfma / 1e3, dmma / 1e3, FP64_NOMINAL_GFLOPS / 1e3),
                  measured_dfma_tflops=dfma / 1e3, measured_dmma_tflops=dmma / 1e3, derived_nominal_tflops=FP64_NOMINAL_GFLOPS / 1e3)
    if f32 and tm["p2p"] >= tm["m2l"]:
        k = kernels["p2p"]
        peak32 = 2.0 * FP64_NOMINAL_GFLOPS / 1e3
        roof = dict(kernel="p2p_leaf_kernel_f32", bound="alu", achieved=k["tflops"], peak=peak32, unit="TFLOP/s", frac=k["tflops"] / peak32,
                    fp32_slot_frac=k["fp64_slot_frac"], traffic=None, algorithmic="18 flop (12 FP32 instructions) + 1 MUFU per pair x %d pairs" % stats["p2p_pairs"],
                    ms=tm["p2p"], share_of_step=tm["p2p"] / tm["total"],
                    peak_source="derived: 148 SMs x 128 FP32 lanes/clk x 2 flop x 1.965 GHz")
    elif args.direct or tm["p2p"] >= tm["m2l"]:
        k = kernels["p2p"]
        # two conventions, both printed: "flop" counts an FMA as 2 and a DMUL / DADD as 1 (so a kernel of 8 FMA + 8 others
        # cannot pass 0.75); "slots" counts FP64 instructions against the pipe's issue rate and is what ncu's
        # sm__pipe_fp64_cycles_active measures.  frac is the flop convention against the MEASURED DFMA loop.
        roof = dict(kernel="p2p_direct_kernel" if args.direct else "p2p_leaf_kernel", bound="alu", achieved=k["tflops"],
                    peak=dfma / 1e3, unit="TFLOP/s", frac=k["tflops"] / (dfma / 1e3), frac_convention="flop / measured DFMA-loop flop rate",
                    frac_of_derived_nominal=k["tflops"] / (FP64_NOMINAL_GFLOPS / 1e3),
                    fp64_slot_frac=k["fp64_slot_frac"], fp64_slot_frac_of_measured=k["fp64_slot_frac"] * FP64_NOMINAL_GFLOPS / dfma,
                    traffic=ncu_traffic("p2p_direct_kernel" if args.direct else "p2p_leaf_kernel", args.config),
                    algorithmic="%d flop (%d FP64 instructions) per pair x %d pairs" % (P2P_FLOP, P2P_INSTR, stats["p2p_pairs"]), ms=tm["p2p"],
                    share_of_step=tm["p2p"] / tm["total"], **common)
    else:
        k = kernels["m2l"]
        roof = dict(kernel="translate_dmma", bound="tensor", achieved=k["executed_tflops"], peak=dmma / 1e3, unit="TFLOP/s",
                    frac=k["frac_of_measured_dmma_peak"], traffic=ncu_traffic("translate_dmma", args.config),
                    algorithmic="4 nre^2 flop per M2L pair x %d pairs (FP64 DMMA; peak = DMMA loop measured in this run)" % stats["m2l_pairs"],
                    ms=tm["m2l"], share_of_step=tm["m2l"] / tm["total"], **common)
    breakdown = {k: round(v, 4) for k, v in tm.items()}

    # parity in the same run + the oracle timed beside it (bounded sample of rows)
    cpu, rows, yo = oracle_sample(c, seconds_target=args.ref_seconds)
    y = yd.cpu().numpy()
    # north_star: "on large configs the check runs over 2000 seeded random target rows" (all rows below 3000 nodes).  The oracle
    # is TIMED on the bounded sample above and then evaluates the rest of the 2000 rows untimed (--parity-rows 0: the timed sample only)
    n_par = N if N < 3000 else min(N, args.parity_rows)
    if n_par > len(rows):
        import oracle
        rows = sample_rows(c["cfg"], N, n_par)
        yo = (oracle.monopole_sum(V, c["q"], V[rows]) if cloud else oracle.g3_apply(V, F, c["q"], c["phi"], eta=c["eta"], rows=rows))
    parity = float(np.linalg.norm(y[rows] - yo) / np.linalg.norm(yo))
    parity_rows = int(len(rows))

    # the paper's "single precision on GPU" option for A^(sparse) X, measured beside the fp64 default
    mixed = None
    if not args.direct and not f32 and not adaptive:                            # fp32 pairs need leaves of one size (uniform tree)
        ctx.bem_set_option("p2p_precision", 1)
        for _ in range(3):
            ctx.bem_apply(qd, pd, yd)
        torch.cuda.synchronize()
        mixed_ms = timed(lambda: ctx.bem_apply(qd, pd, yd), args.steps) / args.steps
        ym = yd.cpu().numpy()
        ctx.bem_set_option("timing", 1)
        ctx.bem_apply(qd, pd, yd)
        tmix = ctx.bem_get_timings()
        ctx.bem_set_option("timing", 0)
        ctx.bem_set_option("p2p_precision", 0)
        mixed = dict(option="p2p_precision = 1: near-field pairs in fp32 (leaf-relative positions), sums in fp64; far field and correction fp64",
                     value=mixed_ms, unit=UNIT, p2p_ms=tmix["p2p"], p2p_gpairs_per_s=stats["p2p_pairs"] / (tmix["p2p"] * 1e-3) / 1e9,
                     parity_rel_l2_vs_oracle=float(np.linalg.norm(ym[rows] - yo) / np.linalg.norm(yo)),
                     rel_l2_vs_fp64_path=float(np.linalg.norm(ym - y) / np.linalg.norm(y)))

    # the uniform tree of PAPER.md:440 (the library default) beside the adaptive one, with its fp32-pair variant
    uniform = None
    if adaptive:
        cu = bem.bem_create(V, F, c["bubble_id"])
        cu.bem_set_stream(stream.cuda_stream)
        if args.lmax:
            cu.bem_set_option("lmax", args.lmax)
        cu.bem_setup(p, args.leaf_size or c["leaf_size"], c["eta"])          # the config's own leaf_size
        su = cu.bem_get_stats()
        for _ in range(3):
            cu.bem_apply(qd, pd, yd)
        torch.cuda.synchronize()
        u_ms = timed(lambda: cu.bem_apply(qd, pd, yd), args.steps) / args.steps
        yu = yd.cpu().numpy()
        cu.bem_set_option("timing", 1)
        cu.bem_apply(qd, pd, yd)
        tu = cu.bem_get_timings()
        cu.bem_set_option("timing", 0)
        cu.bem_set_option("p2p_precision", 1)
        for _ in range(3):
            cu.bem_apply(qd, pd, yd)
        torch.cuda.synchronize()
        u32_ms = timed(lambda: cu.bem_apply(qd, pd, yd), args.steps) / args.steps
        yu32 = yd.cpu().numpy()
        cu.bem_destroy()
        uniform = dict(option="tree = 0: uniform depth l_max, the paper's tree (PAPER.md:440) and the library default", value=u_ms, unit=UNIT,
                       lmax=int(su["lmax"]), breakdown_ms={k: round(v, 4) for k, v in tu.items()}, m2l_pairs=int(su["m2l_pairs"]),
                       p2p_pairs=su["p2p_pairs"], device_bytes=int(su["device_bytes"] - stats["device_bytes"]),
                       device_bytes_note="BEM_S_DEVICE_BYTES counts every live context of the process: the headline context's bytes are subtracted",
                       parity_rel_l2_vs_oracle=float(np.linalg.norm(yu[rows] - yo) / np.linalg.norm(yo)),
                       with_fp32_pairs=dict(value=u32_ms, unit=UNIT,
                                            parity_rel_l2_vs_oracle=float(np.linalg.norm(yu32[rows] - yo) / np.linalg.norm(yo))))

    # the steps either side of the solve in a time step: surface velocity, shape filter
    extras = None
    if not cloud and not args.direct:
        vd = torch.empty(N, 3, dtype=torch.float64, device="cuda")
        ctx.bem_surface_velocity(pd, qd, vd)
        torch.cuda.synchronize()
        sv_ms = timed(lambda: ctx.bem_surface_velocity(pd, qd, vd), args.steps) / args.steps
        hd = torch.empty(N, dtype=torch.float64, device="cuda")
        ctx.bem_surface_curvature(hd)
        torch.cuda.synchronize()
        cv_ms = timed(lambda: ctx.bem_surface_curvature(hd), args.steps) / args.steps
        vol_ms = None
        if c["bubble_id"] is not None:
            vb = torch.empty(int(np.max(c["bubble_id"])) + 1, dtype=torch.float64, device="cuda")
            ctx.bem_bubble_volume(vb)
            torch.cuda.synchronize()
            vol_ms = timed(lambda: ctx.bem_bubble_volume(vb), args.steps) / args.steps
        extras = dict(surface_velocity_ms=sv_ms, surface_curvature_ms=cv_ms, bubble_volume_ms=vol_ms,
                      surface_note="normals, areas, velocity (Eq. 17, Eqs. 22-27) and curvature (Eqs. 28-29), one thread per vertex; "
                                   "bubble volumes (gas law, PAPER.md:108-115), one warp per bubble: together the 'Surface' row of the paper's Table 3")
        tmpl = c.get("template")
        if tmpl is not None and 81 < tmpl.shape[0] <= 2600:         # all bubbles share the angles of one template mesh
            th = np.arccos(np.clip(tmpl[:, 2], -1, 1)); ph = np.arctan2(tmpl[:, 1], tmpl[:, 0])
            nd, p_f = tmpl.shape[0], 9
            flt = bem.bem_filter_create(th, ph, p_f)
            nbub = N // nd
            X = torch.cat([torch.tensor(np.ascontiguousarray(V.T), device="cuda").reshape(3 * nbub, nd), pd.reshape(nbub, nd)]).contiguous()
            Y = torch.empty_like(X)
            flt.bem_filter_apply(X, X.shape[0], Y, stream.cuda_stream)
            torch.cuda.synchronize()
            f_ms = timed(lambda: flt.bem_filter_apply(X, X.shape[0], Y, stream.cuda_stream), args.steps) / args.steps
            flop = 4.0 * p_f * p_f * nd * X.shape[0]
            extras.update(filter_ms=f_ms, filter_columns=int(X.shape[0]), filter_bandwidth=p_f, filter_points_per_bubble=int(nd),
                          filter_tflops=flop / (f_ms * 1e-3) / 1e12, filter_frac_of_fp64_peak=flop / (f_ms * 1e-3) / 1e9 / FP64_NOMINAL_GFLOPS,
                          filter_note="xhat = G (G^+ x) on x, y, z, phi of every bubble: 4 p_f^2 N_d flop per column; the paper's dense F x would be 2 N_d^2")
            flt.bem_filter_destroy()

    # bem_solve: config 4 asks for exactly 30 iterations at tol 1e-6 (BASELINE.json), config 5 for a solve to tol 1e-6;
    # --solve-iters -1 (default) = 30, or 400 on config 5 (it converges in ~220 / ~150 iterations)
    solve = None
    max_it = args.solve_iters if args.solve_iters >= 0 else (400 if args.config == 5 else 30)
    if max_it > 0 and not cloud:
        solve = {}
        runs = [("unpreconditioned (paper)", 0, 0), ("diagonal S_ii (option precond)", 1, 0)]
        if not args.direct and not f32 and not adaptive:
            runs.append(("diagonal S_ii, fp32 pairs (options precond, p2p_precision)", 1, 1))
        for name, pre, prec in runs:
            ctx.bem_set_option("precond", pre)
            if not args.direct:
                ctx.bem_set_option("p2p_precision", 1 if (prec or f32) else 0)
            qs = torch.zeros_like(qd)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            st, it, rr = ctx.bem_solve(pd, qs, tol=args.solve_tol, max_iter=max_it)
            torch.cuda.synchronize()
            ms_s = (time.perf_counter() - t0) * 1e3
            solve[name] = dict(ms=ms_s, iterations=it, relres=rr, tol=args.solve_tol, max_iter=max_it,
                               status=bem.STATUS_NAMES[st], ms_per_iteration=ms_s / max(it, 1))
            if pre == 0 and prec == 0:
                q_cold = qs.clone()
                if args.solve_check_rows > 0 and not cloud:
                    # the residual of the returned q recomputed by the ORACLE on seeded rows:
                    # b_i = -c_i phi_i + (D phi)_i with c_i = 1 + (D.1)_i, r_i = b_i - (S q)_i -- three oracle products
                    import oracle
                    rr_rows = sample_rows(c["cfg"], N, args.solve_check_rows)
                    qh_s = qs.cpu().numpy()
                    o = lambda a, b: oracle.g3_apply(V, F, a, b, eta=c["eta"], rows=rr_rows)
                    t0o = time.perf_counter()
                    cfree = 1.0 - o(None, np.ones(N))
                    b_rows = -cfree * c["phi"][rr_rows] - o(None, c["phi"])
                    res_rows = b_rows - o(qh_s, None)
                    solve[name]["relres_by_oracle_on_rows"] = float(np.linalg.norm(res_rows) / np.linalg.norm(b_rows))
                    solve[name]["oracle_rows"] = int(len(rr_rows))
                    solve[name]["oracle_check_s"] = time.perf_counter() - t0o
        # the paper's regime: every time step starts GMRES from the previous step's solution and needs
        # 2-10 iterations.  Perturb phi by 1% (seeded) and solve again from the cold solution of the unperturbed phi.
        if not cloud and "unpreconditioned (paper)" in solve and solve["unpreconditioned (paper)"]["status"] == "BEM_OK":
            ctx.bem_set_option("precond", 0)
            rng = np.random.default_rng(190501341 + 200 + int(c["cfg"]))
            pd2 = pd * torch.tensor(1.0 + 0.01 * rng.uniform(-1.0, 1.0, N), device="cuda")
            qw = q_cold.clone()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            st, it, rr = ctx.bem_solve(pd2, qw, use_q_as_x0=True, tol=args.solve_tol, max_iter=max_it)
            torch.cuda.synchronize()
            ms_s = (time.perf_counter() - t0) * 1e3
            solve["warm start, phi perturbed by 1% (unpreconditioned)"] = dict(ms=ms_s, iterations=it, relres=rr, tol=args.solve_tol,
                                                                                status=bem.STATUS_NAMES[st], ms_per_iteration=ms_s / max(it, 1))
            # the same with a SMOOTH change, which is what a time step does to phi: phi + 0.01 Re Y_2^1 on every bubble
            tmpl = c.get("template")
            if tmpl is not None and N % tmpl.shape[0] == 0:
                from bem_inputs.sph import real_sph_harm
                th = np.arccos(np.clip(tmpl[:, 2] / np.linalg.norm(tmpl, axis=1), -1, 1)); az = np.arctan2(tmpl[:, 1], tmpl[:, 0])
                bump = np.tile(0.01 * real_sph_harm(2, 1, th, az), N // tmpl.shape[0])
                pd3 = pd + torch.tensor(bump, device="cuda")
                qw = q_cold.clone()
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                st, it, rr = ctx.bem_solve(pd3, qw, use_q_as_x0=True, tol=args.solve_tol, max_iter=max_it)
                torch.cuda.synchronize()
                ms_s = (time.perf_counter() - t0) * 1e3
                solve["warm start, phi + 0.01 Re Y_2^1 on every bubble (unpreconditioned)"] = dict(
                    ms=ms_s, iterations=it, relres=rr, tol=args.solve_tol, status=bem.STATUS_NAMES[st], ms_per_iteration=ms_s / max(it, 1))
        solve["note"] = ("the stopping test runs on the FMM operator: a tol below its truncation error (parity_rel_l2_vs_oracle) is met in the "
                         "library's norm but not in the oracle's (relres_by_oracle_on_rows)")
        ctx.bem_set_option("precond", 0)
        if not args.direct:
            ctx.bem_set_option("p2p_precision", 1 if f32 else 0)

    cfg_d = workload_config(c, args, p)
    if not cloud and not args.direct:
        cfg_d["p_executed_with_phi"] = int(stats["p_dipole"])         # the library's own word (equals the rule of p_with_dipoles)
    sweep = run_sweep(args, bem, torch, stream) if (args.sweep and args.config == 5 and world == 1 and not args.direct) else None

    line = dict(metric=METRIC, value=ms, unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3), ms_per_step=ms,
                higher_is_better=False, scaling="weak", vs_baseline=None, dtype="f64 (near-field pairs f32)" if f32 else "f64", data="synthetic",
                config=cfg_d, sweep=sweep,
                run=dict(mode="direct" if args.direct else "fmm", tree="adaptive" if adaptive else "uniform", p2p_precision="fp32 pairs, fp64 sums" if f32 else "fp64",
                         p_dipole=int(stats["p_dipole"]), lmax=int(stats["lmax"]), n_src_leaves=int(stats["n_src_leaves"]),
                         n_tgt_leaves=int(stats["n_tgt_leaves"]),
                         launch="CUDA graph replay" if (stream.cuda_stream != 0 and not args.no_graph) else "kernel by kernel",
                         device_bytes=int(stats["device_bytes"]), options=args.opt),
                e2e=dict(value=e2e, unit=UNIT, h2d_bytes_per_step=(8 if cloud else 16) * N, d2h_bytes_per_step=8 * N),
                gpu_launches=int(stats["kernel_launches_per_apply"]) * args.steps,
                clocks=clocks, roofline=roof, cpu_baseline=cpu, parity_rel_l2_vs_oracle=parity, parity_rows=parity_rows,
                breakdown_ms=breakdown, kernels=kernels, setup_ms=stats["setup_ms"], setup_wall_ms=setup_wall_ms,
                m2l_pairs=int(stats["m2l_pairs"]), solve=solve, mixed_precision_option=mixed, uniform_tree_option=uniform, time_step_extras=extras,
                paper_context=("paper Table 2 (PAPER.md:479-490): at N=1,048,576, p=12 the FMM+GPU (double) product is 2309x faster than the CPU "
                               "brute force and the brute-force GPU (double) 33x, Xeon 5660 + Tesla K20" if cloud else
                               "paper Table 3 (PAPER.md:606): 1 MVP = 4.0 s at N=2,629,632, p=12, double, Xeon 5660 x12 cores + Tesla K20"))
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--config", type=int, default=5, help="BASELINE.json config 1..5 (default 5: 2.57M nodes); 6 = point cloud (paper Tables 1-2); 7 = regular nb^3 cluster (paper Table 3)")
    ap.add_argument("--cloud-points", type=int, default=1048576, help="config 6: number of points")
    ap.add_argument("--lattice-nb", type=int, default=16, help="config 7: bubbles per edge of the regular cluster (paper: 1..16)")
    ap.add_argument("--p", type=int, default=0)
    ap.add_argument("--leaf-size", type=int, default=0)
    ap.add_argument("--lmax", type=int, default=0)
    ap.add_argument("--direct", action="store_true", help="direct-sum mode (configs 1-3)")
    ap.add_argument("--p2p-precision", type=int, default=64, choices=[64, 32],
                    help="near-field pair arithmetic: 64 = fp64 (default, the measured mode), 32 = fp32 pairs with fp64 accumulation (PAPER.md:456-473)")
    ap.add_argument("--stream", default="auto", choices=["auto", "default", "side"],
                    help="stream of the products: the legacy default stream, or a side stream (CUDA-graph replay); auto = side below 200k nodes")
    ap.add_argument("--no-graph", action="store_true", help="launch bem_apply kernel by kernel instead of replaying its CUDA graph")
    ap.add_argument("--direct-pairs", type=int, default=None,
                    help="leaf-level far pairs with nt x ns <= this are summed directly instead of translated (default: library cost model; 0: off)")
    ap.add_argument("--p2p-ctas", type=int, default=0, help="fp32 near field: CTAs per SM of its persistent grid (0: library default)")
    ap.add_argument("--reduce-ctas", type=int, default=0, help="CTAs per SM of the persistent row-sum passes (0: library cost model)")
    ap.add_argument("--tree", default="auto", choices=["auto", "uniform", "adaptive"],
                    help="octree: uniform depth (the paper's), adaptive (option tree = 1), auto = adaptive on config 5 with fp64 pairs (measured faster)")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE", help="any bem_set_option key (repeatable), set before bem_setup")
    ap.add_argument("--solve-iters", type=int, default=-1, help="also run bem_solve with this max_iter (0: skip; -1: 30, or 400 = to convergence on config 5)")
    ap.add_argument("--solve-tol", type=float, default=1e-6)
    ap.add_argument("--parity-rows", type=int, default=2000, help="seeded rows of the parity check against the oracle (0: the timed sample only)")
    ap.add_argument("--solve-check-rows", type=int, default=400,
                    help="rows on which the ORACLE recomputes the residual of the first bem_solve (three oracle products; 0: skip)")
    ap.add_argument("--ref-seconds", type=float, default=12.0, help="CPU time budget of one oracle sample")
    ap.add_argument("--no-sweep", dest="sweep", action="store_false",
                    help="skip the configs 1-4 points that the default config-5 run appends (\"ms/apply vs N nodes\")")
    ap.add_argument("--sweep-rows", type=int, default=500, help="seeded oracle rows of each sweep point (all rows below 3000 nodes)")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
