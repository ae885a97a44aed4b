// The C-ABI boundary (include/bem.h): context, bem_create, bem_setup, bem_apply and the
// small query calls.  bem_solve lives in solve.cu.
#include "common.cuh"
#include "harmonics.cuh"

#include <chrono>
#include <cmath>

namespace bem {
// mesh.cu
void validate_mesh(bem_ctx *c);
void compute_geometry(bem_ctx *c);
void build_sources(bem_ctx *c, const uint32_t *order);
void source_points(bem_ctx *c, dvec<double> &xyz);
// nearfield.cu
void build_correction(bem_ctx *c);
void build_empty_correction(bem_ctx *c);
// tree.cu
void boxset_sort(BoxSet &bs, const double *xyz, int64_t n, const double cube_min[3], double cube_side, int counts[22], cudaStream_t s);
void boxset_build(BoxSet &bs, int lmax, const int counts[22], cudaStream_t s);
void build_lists(bem_ctx *c);
// adaptive.cu
int adaptive_source_flags(bem_ctx *c, bool *want_deeper);
void build_adaptive(bem_ctx *c);
// translate.cu
void build_matrices(bem_ctx *c, FmmLayout &L);
void pack_scratch(bem_ctx *c);
void launch_stage(bem_ctx *c, const Stage &st, int cls_gemm, int cls_reduce);
void launch_stage_gemm(bem_ctx *c, const Stage &st, int which, cudaStream_t stream);
void launch_stage_reduce(bem_ctx *c, const Stage &st, cudaStream_t stream, int ctas_per_sm);
void launch_p2m(bem_ctx *c);
void launch_l2p(bem_ctx *c, const int32_t *leaf_of);
// p2p.cu
void launch_lift(bem_ctx *c, const double *q, const double *phi);
void launch_p2p_direct(bem_ctx *c);
void launch_p2p_leaves(bem_ctx *c);
void launch_spmv_combine(bem_ctx *c, const double *q, const double *phi, double *y);
// p2p_f32.cu
void launch_p2p_leaves_f32(bem_ctx *c, cudaStream_t stream, int ctas_per_sm, int leaf0, int leaf1, int part);
void ensure_p2p_f32(bem_ctx *c);

const bem_ctx *mesh_of(const bem_ctx *c) { return c->parent ? c->parent : c; }

bool is_device_ptr(const void *p)
{
    if (!p) return true;
    cudaPointerAttributes a;
    cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

template <class F>
static bem_status guarded(bem_ctx *c, F &&f)
{
    try {
        if (c) CUDA_TRY(cudaSetDevice(c->device));
        f();
        return BEM_OK;
    } catch (const Error &e) {
        if (c) c->err = e.what();
        cudaGetLastError();
        return e.status;
    } catch (const std::exception &e) {
        if (c) c->err = e.what();
        return BEM_ERR_CUDA;
    } catch (...) {
        if (c) c->err = "unknown error";
        return BEM_ERR_CUDA;
    }
}

__global__ void gather_targets(const double *V, const uint32_t *perm, int64_t N, double *tgt, uint32_t *inv)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= N) return;
    const uint32_t i = perm[e];
    tgt[3 * e] = V[3 * (int64_t)i]; tgt[3 * e + 1] = V[3 * (int64_t)i + 1]; tgt[3 * e + 2] = V[3 * (int64_t)i + 2];
    inv[i] = (uint32_t)e;
}
__global__ void fill_const(double *v, int64_t n, double a)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v[i] = a;
}
// c_i = 1 - y_i where y = bem_apply(0, 1) = -D.1   (reading R6)
__global__ void free_term_kernel(const double *y, int64_t n, double *c)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) c[i] = 1.0 - y[i];
}

// ------------------------------------------------------------------ V1 diagonal (a3')
// natural-order vertex weights (s, s n) come from lift_w through the engine permutation
__global__ void v1_scatter_normals(const double4 *lw, const int4 *lv, int64_t N, double *s, double *nrm)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= N) return;
    const int j = lv[e].x;
    const double4 w = lw[e];
    s[j] = w.x;
    nrm[3 * (int64_t)j] = w.y / w.x; nrm[3 * (int64_t)j + 1] = w.z / w.x; nrm[3 * (int64_t)j + 2] = w.w / w.x;
}
__global__ void v1_rhs(const double *V, const double *nrm, int64_t N, int axis, double r0, double *q, double *phi)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    q[i] = nrm[3 * i + axis];
    phi[i] = V[3 * i + axis] - r0;
}
// M_ii = -1/2 + y0_i ;  L_ii = - sum_a n_i^a y^a_i + y0_i n_i.(r_i - r0)     (Eqs. 19-21)
__global__ void v1_diag(const double *V, const double *nrm, const double *y0, const double *yx, const double *yy, const double *yz,
                        int64_t N, double r0x, double r0y, double r0z, double *dL, double *dM)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double nx = nrm[3 * i], ny = nrm[3 * i + 1], nz = nrm[3 * i + 2];
    dM[i] = -0.5 + y0[i];
    dL[i] = -(nx * yx[i] + ny * yy[i] + nz * yz[i]) +
            y0[i] * (nx * (V[3 * i] - r0x) + ny * (V[3 * i + 1] - r0y) + nz * (V[3 * i + 2] - r0z));
}

// ------------------------------------------------------------------ truncation layouts
static void init_layout(FmmLayout &L, int p)
{
    L.p = p;
    // template buckets of the P2M / L2P / DMMA kernels: the even degrees 4 .. 16, and 11 and 13 (what p = 8 and 10 become
    // with three more degrees for the dipoles)
    L.pl = p > 16 ? p : (p == 11 || p == 13) ? p : std::max(4, 2 * ((p + 1) / 2));
    L.nre = lay_nre(L.pl);
    L.nst = lay_nst(L.pl);
}
void activate_layout(bem_ctx *c, int i)
{
    const FmmLayout &L = c->lay[i];
    c->lay_active = i;
    c->p = L.p; c->pl = L.pl; c->nre = L.nre; c->nst = L.nst;
    c->mats.p = L.mats.get(); c->rot.p = L.rot.get(); c->kinfo.p = L.kinfo.get();
    c->mat_ne.p = L.mat_ne.get(); c->mat_cls.p = L.mat_cls.get(); c->mat_w.p = L.mat_w.get();
    c->m2l_row_bytes = L.m2l_row_bytes;
}
// executed work of the M2L tiles of one product with this layout (bem_get_stats), from the pairs per matrix
static void layout_stats(const bem_ctx *c, FmmLayout &L)
{
    L.m2l_flop = L.m2l_row_bytes = 0;
    const bool dmma = c->gemm_path == 0 && L.pl <= 16;             // the plain-FMA tiles run every matrix in full
    for (int m = 0; m < MAT_L2L; ++m) {
        const double kr = dmma ? 4.0 * ke_of(L.pl - L.mat_cls_host[m]) : (double)L.nre;
        L.m2l_flop += c->m2l_hist[m] * 4.0 * kr * kr;
        L.m2l_row_bytes += c->m2l_hist[m] * 16.0 * L.mat_w_host[m];
    }
}

// ------------------------------------------------------------------ apply (device pointers)
void mark(bem_ctx *c, int cls)
{
    if (!c->timing) return;
    if (c->ev_n == (int)c->ev.size()) {
        cudaEvent_t e;
        CUDA_TRY(cudaEventCreate(&e));
        c->ev.push_back(e);
        c->ev_cls.push_back(cls);
    }
    c->ev_cls[c->ev_n] = cls;
    CUDA_TRY(cudaEventRecord(c->ev[c->ev_n++], c->stream));
}

// CTAs per SM of the persistent side-stream sums: enough for them to end just before the pair kernel does.  Model: fp64
// pairs at 700 Gpairs/s, fp32 pairs at 1400 (with 4 CTAs per SM of the pair kernel resident, 6 CTAs of the sums still
// fit); the sums at 4 TB/s with >= 16 CTAs per SM, in proportion below that (measured on configs 4 and 5).
static int reduce_ctas_for(const bem_ctx *c)
{
    if (c->reduce_ctas > 0) return c->reduce_ctas;
    const bool f32 = c->p2p_precision == 1;
    const double t_p2p = (double)c->p2p_pairs / (f32 ? 1400e9 : 700e9);
    const double t_sum = c->m2l_row_bytes / 4e12;
    const int k = (int)std::ceil(16.0 * 1.3 * t_sum / std::max(t_p2p, 1e-9));
    return std::max(3, std::min(k, f32 ? 6 : 16));
}

void apply_device(bem_ctx *c, const double *q, const double *phi, double *y)
{
    c->ev_n = 0;
    if (c->mode == 0) activate_layout(c, (phi && c->n_lay > 1) ? 1 : 0);      // products with dipoles carry more degrees (option dipole_degrees)
    if (c->mode == 0 && c->p2p_precision == 1) {
        if (c->adaptive) throw Error(BEM_ERR_INVALID_ARG, "p2p_precision = 1 needs the uniform tree (option tree = 0): its fp32 positions are relative to leaves of one size");
        ensure_p2p_f32(c);
    }
    mark(c, -1);
    launch_lift(c, q, phi);
    mark(c, BEM_T_LIFT);
    if (c->mode == 1) {
        launch_p2p_direct(c);
        mark(c, BEM_T_P2P);
    } else {
        const int lmax = c->sb.lmax;
        launch_p2m(c);
        mark(c, BEM_T_P2M);
        for (int l = lmax - 1; l >= 2; --l) launch_stage(c, c->m2m[l], BEM_T_M2M, BEM_T_M2M);
        if (c->timing || !c->side || !c->overlap) {
            // one stream, class by class (option "timing": the per-class event times add up to the total)
            for (int l = 2; l <= lmax; ++l) launch_stage(c, c->m2l[l], BEM_T_M2L, BEM_T_L2L_REDUCE);
            for (int l = 3; l <= lmax; ++l) launch_stage(c, c->l2l[l], BEM_T_L2L_REDUCE, BEM_T_L2L_REDUCE);
            launch_l2p(c, c->tb.leaf_of.get());
            mark(c, BEM_T_L2P);
            if (c->p2p_precision == 1) launch_p2p_leaves_f32(c, c->stream, 8, 0, c->tb.nbox[lmax], 0);
            else launch_p2p_leaves(c);
            mark(c, BEM_T_P2P);
        } else {
            // The M2L tiles of every level only read multipole expansions: issue them all, then fork.  The per-level
            // sums of the translated rows (HBM-bound, independent of each other) run on a high-priority side stream
            // while the near field (P2P: FP64-bound, no HBM traffic) runs on the main stream; after the join the short
            // downward pass L(l) += L2L L(l-1) and L2P follow on the main stream.
            cudaStream_t main = c->stream;
            for (int l = 2; l <= lmax; ++l) launch_stage_gemm(c, c->m2l[l], TILES_ALL, main);
            CUDA_TRY(cudaEventRecord(c->ev_fork, main));
            CUDA_TRY(cudaStreamWaitEvent(c->side, c->ev_fork, 0));
            for (int l = lmax; l >= 2; --l) launch_stage_reduce(c, c->m2l[l], c->side, reduce_ctas_for(c));
            CUDA_TRY(cudaEventRecord(c->ev_join, c->side));
            // fp32 pairs: a persistent grid of a few CTAs per SM (80 registers each) so that the CTAs of the sums still fit
            if (c->p2p_precision == 1) launch_p2p_leaves_f32(c, main, c->p2p_ctas > 0 ? c->p2p_ctas : 4, 0, c->tb.nbox[lmax], 0);
            else launch_p2p_leaves(c);
            CUDA_TRY(cudaStreamWaitEvent(main, c->ev_join, 0));
            for (int l = 3; l <= lmax; ++l) launch_stage(c, c->l2l[l], BEM_T_L2L_REDUCE, BEM_T_L2L_REDUCE);
            launch_l2p(c, c->tb.leaf_of.get());
        }
    }
    launch_spmv_combine(c, q, phi, y);
    mark(c, BEM_T_SPMV);
    c->ev_valid = c->timing != 0;
}

static void drop_graphs(bem_ctx *c)
{
    for (auto &g : c->graphs) if (g.exec) cudaGraphExecDestroy(g.exec);
    c->graphs.clear();
}

// bem_apply with device pointers: replay a captured graph when the same product was asked for before
static void apply_device_cached(bem_ctx *c, const double *q, const double *phi, double *y)
{
    // the legacy default stream cannot be captured; option "timing" records events between the kernels
    if (!c->use_graph || c->timing || c->stream == nullptr || c->stream == cudaStreamLegacy) { apply_device(c, q, phi, y); return; }
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(c->stream, &cap) != cudaSuccess || cap != cudaStreamCaptureStatusNone) {
        cudaGetLastError();
        apply_device(c, q, phi, y);                                          // the caller is capturing this stream: become part of ITS graph
        return;
    }
    for (auto &g : c->graphs) {
        if (g.q != q || g.phi != phi || g.y != y || g.stream != c->stream) continue;
        if (g.exec) { CUDA_TRY(cudaGraphLaunch(g.exec, c->stream)); return; }
        if (c->mode == 0 && c->p2p_precision == 1) ensure_p2p_f32(c);       // allocations stay outside the capture
        c->has_dipole = phi != nullptr;
        cudaGraph_t graph = nullptr;
        CUDA_TRY(cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal));
        try {
            apply_device(c, q, phi, y);
        } catch (...) {
            cudaStreamEndCapture(c->stream, &graph);
            if (graph) cudaGraphDestroy(graph);
            cudaGetLastError();
            throw;
        }
        CUDA_TRY(cudaStreamEndCapture(c->stream, &graph));
        cudaGraphExec_t exec = nullptr;
        const cudaError_t e = cudaGraphInstantiate(&exec, graph, 0);
        cudaGraphDestroy(graph);
        CUDA_TRY(e);
        g.exec = exec;
        CUDA_TRY(cudaGraphLaunch(g.exec, c->stream));
        return;
    }
    if (c->graphs.size() >= 8) {                                             // keep the cache small: drop the oldest entry
        if (c->graphs.front().exec) cudaGraphExecDestroy(c->graphs.front().exec);
        c->graphs.erase(c->graphs.begin());
    }
    c->graphs.push_back({q, phi, y, c->stream, 1, nullptr});
    apply_device(c, q, phi, y);
}

static void setup_impl(bem_ctx *c, int p, int leaf_size, double eta)
{
    drop_graphs(c);
    cudaStream_t s = c->stream;
    const auto t0 = std::chrono::steady_clock::now();
    c->ready = false;
    c->have_diag = false;
    c->have_cfree = false;
    c->p_user = p;
    init_layout(c->lay[0], p);
    // Products with dipole sources lose about 3.5 degrees of accuracy against monopoles at equal truncation (a dipole moment
    // of degree l scales like l a^(l-1); measured: DESIGN.md R5'), so they carry dd more degrees.  -1 = the measured table:
    // 3 degrees below p = 12 (S - D then meets the north_star's 1e-5 at the stated p of every BASELINE config), none from 12 on.
    const int dd = c->dipole_degrees >= 0 ? c->dipole_degrees : (p < 12 ? 3 : 0);
    const int p_dip = std::min(P_MAX, p + dd);
    c->n_lay = (p_dip > p && c->mode == 0) ? 2 : 1;
    if (c->n_lay == 2) init_layout(c->lay[1], p_dip);
    activate_layout(c, 0);
    c->leaf_size = leaf_size;
    c->eta = eta;
    if (c->quadrature < 2) compute_geometry(c);
    if (c->quadrature == 3 && !c->parent->triA.p) {              // an evaluator uses the areas and normals of its parent's mesh
        CUDA_TRY(cudaSetDevice(c->parent->device));
        struct StreamSwap {                                      // the parent's geometry is computed on the evaluator's stream;
            bem_ctx *ctx; cudaStream_t saved;                    // its own stream comes back whatever compute_geometry throws
            StreamSwap(bem_ctx *x, cudaStream_t t) : ctx(x), saved(x->stream) { x->stream = t; }
            ~StreamSwap() { ctx->stream = saved; }
        };
        {
            StreamSwap swap(c->parent, s);
            compute_geometry(c->parent);
        }
        CUDA_TRY(cudaStreamSynchronize(s));
    }
    const int64_t N = c->N;
    c->ns = (c->quadrature == 0 || c->quadrature == 3) ? 3 * mesh_of(c)->T : (c->quadrature == 2 ? c->np : N);

    {
        // unit-cube scaling (reading R11): cube centred on the bounding box, side = largest extent (1 + 1e-9)
        dvec<double> bb;
        bb.alloc(6);
        bbox3(c->V.get(), N, bb.get(), s);
        double hb[6];
        d2h_sync(hb, bb.get(), sizeof hb, s);
        if (c->quadrature >= 2) {                           // the cube holds sources and targets
            double hs[6];
            if (c->quadrature == 2) bbox3(c->P.get(), c->np, bb.get(), s);
            else bbox3(c->parent->V.get(), c->parent->N, bb.get(), s);          // Gauss points lie inside the box of the vertices
            d2h_sync(hs, bb.get(), sizeof hs, s);
            for (int d = 0; d < 3; ++d) { hb[d] = std::min(hb[d], hs[d]); hb[3 + d] = std::max(hb[3 + d], hs[3 + d]); }
        }
        double side = 0;
        for (int d = 0; d < 3; ++d) side = std::max(side, hb[3 + d] - hb[d]);
        side *= (1.0 + 1e-9);
        if (!(side > 0)) side = 1.0;
        for (int d = 0; d < 3; ++d) c->cube_min[d] = 0.5 * (hb[d] + hb[3 + d]) - 0.5 * side;
        c->cube_side = side;

    }
    const double side = c->cube_side;
    if (c->mode == 1) {
        build_sources(c, nullptr);
        c->tgt_pos.alloc(3 * N);
        CUDA_TRY(cudaMemcpyAsync(c->tgt_pos.get(), c->V.get(), 3 * N * sizeof(double), cudaMemcpyDeviceToDevice, s));
        const int tb = cdiv(N, 512);
        int nsplit = cdiv(148 * 14, tb);             // >= 14 CTAs (56 warps) per SM: the pair loop is latency-bound below that
        nsplit = std::max(1, std::min(nsplit, 64));
        nsplit = (int)std::max<int64_t>(1, std::min<int64_t>(nsplit, c->ns / 256));
        c->nsplit = nsplit;
        c->ypart.alloc((size_t)nsplit * N);
        c->launches_per_apply = 3;
    } else {
        dvec<double> sxyz;
        source_points(c, sxyz);
        int cs[22], ct[22];
        boxset_sort(c->sb, sxyz.get(), c->ns, c->cube_min, side, cs, s);
        sxyz.free();
        boxset_sort(c->tb, c->V.get(), N, c->cube_min, side, ct, s);
        // depth: smallest level >= 2 whose mean non-empty source-box population <= leaf_size (reading R9)
        int lmax = 2;
        while (lmax < MAX_LEVEL && (double)c->ns / (double)cs[lmax] > (double)leaf_size) ++lmax;
        if (c->force_lmax >= 2) lmax = std::min(c->force_lmax, MAX_LEVEL);
        if (c->adaptive) {
            // adaptive tree: build the source boxes down to a probe depth (option lmax caps it), flag what exists under the
            // rule "subdivide a box that holds more than leaf_size sources", and keep the levels that hold an existing box
            c->ad.lmin = c->tree_min_level >= 2 ? std::min(c->tree_min_level, lmax) : lmax;
            if (c->force_lmax >= 2) c->ad.lmin = std::min(c->ad.lmin, lmax);
            int lprobe = c->force_lmax >= 2 ? lmax : std::min(MAX_LEVEL, lmax + 3);
            int deep = 2;
            for (;;) {                                            // deepen the probe while the rule still wants to subdivide
                bool more = false;
                boxset_build(c->sb, lprobe, cs, s);
                deep = adaptive_source_flags(c, &more);
                if (!more || c->force_lmax >= 2 || lprobe >= MAX_LEVEL) break;
                lprobe = std::min(MAX_LEVEL, lprobe + 3);
            }
            if (deep < lprobe) { boxset_build(c->sb, deep, cs, s); adaptive_source_flags(c, nullptr); }
            lmax = deep;
            for (int l = lmax + 1; l <= MAX_LEVEL; ++l) {
                c->sb.bkey[l].free(); c->sb.child[l].free(); c->sb.parent[l].free(); c->sb.nbox[l] = 0;
                c->ad.s_ex[l].free(); c->ad.s_sub[l].free(); c->ad.s_pbeg[l].free();
            }
            c->sb.child[lmax].free();
        } else {
            c->ad = Adaptive();                                   // a context that was adaptive before: drop its tables
            boxset_build(c->sb, lmax, cs, s);
        }
        boxset_build(c->tb, lmax, ct, s);
        build_sources(c, c->sb.perm.get());
        c->tgt_pos.alloc(3 * N);
        c->tgt_inv.alloc(N);
        gather_targets<<<cdiv(N, 256), 256, 0, s>>>(c->V.get(), c->tb.perm.get(), N, c->tgt_pos.get(), c->tgt_inv.get());
        KERNEL_CHECK();
        for (int i = 0; i < c->n_lay; ++i) build_matrices(c, c->lay[i]);
        activate_layout(c, 0);
        const int nst_max = c->lay[c->n_lay - 1].nst;
        c->Mexp.alloc((size_t)c->sb.total() * nst_max);
        c->Lexp.alloc((size_t)c->tb.total() * nst_max);
        {
            // leaf-level far pairs that cost less summed directly than translated (option "direct_pairs").  One M2L pair +
            // its row sum costs ~1.35 us at p = 12 (nre = 80) whatever the boxes hold, one point pair ~1.4 ns in a full
            // leaf and several times that in the sparsely filled leaves these pairs come from; measured optimum on configs
            // 4 and 5: nt x ns <= 800 (nre / 80)^2 (flat between half and 1.5x that)
            const double w = 800.0 * (double)c->nre * (double)c->nre / 6400.0;
            c->direct_max_eff = c->direct_max >= 0 ? c->direct_max : (int64_t)w;
        }
        if (c->adaptive) {
            try {
                build_adaptive(c);
            } catch (const Error &) {
                // A target leaf met more direct source ranges than the pair kernel's segment table holds (SEG_MAX).  With a small
                // leaf_size the cost model above moves up to 189 leaf-level far pairs per leaf from the M2L list to the direct
                // list, which leaves few slots for the coarser leaves next to the ancestors of a leaf in a strongly graded
                // cloud.  When that choice was the library's (direct_pairs = -1), build the lists again with every far pair
                // translated: a row then holds at most the 27 neighbours of the leaf and of each ancestor.  An explicit
                // direct_pairs is the caller's to lower: the refusal stands.
                if (!c->ad.row_overflow || c->direct_max >= 0 || c->direct_max_eff == 0) throw;
                c->direct_max_eff = 0;
                build_adaptive(c);
            }
        } else build_lists(c);
        pack_scratch(c);
        for (int i = 0; i < c->n_lay; ++i) layout_stats(c, c->lay[i]);
        activate_layout(c, 0);
        c->nsplit = 2;                                  // far field (L2P) and near field (P2P) partial sums
        c->ypart.alloc(2 * N);
        if (!c->side) {
            CUDA_TRY(cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, c->device));
            int lo = 0, hi = 0;
            CUDA_TRY(cudaDeviceGetStreamPriorityRange(&lo, &hi));
            CUDA_TRY(cudaStreamCreateWithPriority(&c->side, cudaStreamNonBlocking, hi));
            CUDA_TRY(cudaEventCreateWithFlags(&c->ev_fork, cudaEventDisableTiming));
            CUDA_TRY(cudaEventCreateWithFlags(&c->ev_join, cudaEventDisableTiming));
        }
        c->p2p_counter.alloc(4);                         // [0], [1] fp32 pair kernel, [2] P2M: leaf counters of the persistent grids
        c->src_pos_f.free();
        c->src_str_f.free();
        int launches = 2 /*lift, p2m*/ + 3 /*l2p, p2p, spmv*/;
        for (int l = lmax - 1; l >= 2; --l) launches += 2;
        for (int l = 2; l <= lmax; ++l) launches += l > 2 ? 4 : 2;     // M2L tiles + sum; L2L tiles + sum
        c->launches_per_apply = launches;
    }

    if (c->quadrature == 0 || c->quadrature == 3) build_correction(c);
    else build_empty_correction(c);
    if (c->mode == 0 && c->p2p_precision == 1 && !c->adaptive) ensure_p2p_f32(c);
    c->ready = true;
    if (c->quadrature >= 2) {                               // point cloud, evaluator: no free term, no solve
        CUDA_TRY(cudaStreamSynchronize(s));
        c->setup_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
        return;
    }

    dvec<double> ones, y0;
    ones.alloc(N);
    y0.alloc(N);
    fill_const<<<cdiv(N, 256), 256, 0, s>>>(ones.get(), N, 1.0);
    KERNEL_CHECK();
    struct TimingOff {                                           // products made inside bem_setup are not timed; restored on every exit
        bem_ctx *c; int saved;
        explicit TimingOff(bem_ctx *cc) : c(cc), saved(cc->timing) { c->timing = 0; }
        ~TimingOff() { c->timing = saved; }
    } timing_off(c);
    if (c->quadrature == 1) {
        // the paper's four products for the singular diagonal, pair j = i skipped
        dvec<double> sv, nrm, qv, pv, ya[3];
        sv.alloc(N); nrm.alloc(3 * N); qv.alloc(N); pv.alloc(N);
        v1_scatter_normals<<<cdiv(N, 256), 256, 0, s>>>(c->lift_w.get(), c->lift_vid.get(), N, sv.get(), nrm.get());
        KERNEL_CHECK();
        apply_device(c, nullptr, ones.get(), y0.get());
        const double r0[3] = {c->cube_min[0] + 0.5 * c->cube_side, c->cube_min[1] + 0.5 * c->cube_side, c->cube_min[2] + 0.5 * c->cube_side};
        for (int a = 0; a < 3; ++a) {
            ya[a].alloc(N);
            v1_rhs<<<cdiv(N, 256), 256, 0, s>>>(c->V.get(), nrm.get(), N, a, r0[a], qv.get(), pv.get());
            KERNEL_CHECK();
            apply_device(c, qv.get(), pv.get(), ya[a].get());
        }
        c->diagL.alloc(N);
        c->diagM.alloc(N);
        v1_diag<<<cdiv(N, 256), 256, 0, s>>>(c->V.get(), nrm.get(), y0.get(), ya[0].get(), ya[1].get(), ya[2].get(), N,
                                             r0[0], r0[1], r0[2],
                                             c->diagL.get(), c->diagM.get());
        KERNEL_CHECK();
        CUDA_TRY(cudaStreamSynchronize(s));
        c->have_diag = true;
    }
    // free term of bem_solve
    c->cfree.alloc(N);
    if (c->free_term == 1) {
        fill_const<<<cdiv(N, 256), 256, 0, s>>>(c->cfree.get(), N, 0.5);
        KERNEL_CHECK();
    } else {
        apply_device(c, nullptr, ones.get(), y0.get());
        free_term_kernel<<<cdiv(N, 256), 256, 0, s>>>(y0.get(), N, c->cfree.get());
        KERNEL_CHECK();
    }
    CUDA_TRY(cudaStreamSynchronize(s));
    c->have_cfree = true;
    c->setup_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
}

// register-resident DFMA loop: 8 independent chains per thread
__global__ void dfma_loop(double *out, int iters, double a, double b)
{
    double x0 = threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5, x6 = x0 + 6, x7 = x0 + 7;
    for (int i = 0; i < iters; ++i) {
        x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
        x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}

// register-resident DMMA loop: 8 independent m8n8k4 accumulator tiles per warp
__global__ void dmma_loop(double *out, int iters, double a, double b)
{
    double c[8][2];
    for (int i = 0; i < 8; ++i) { c[i][0] = threadIdx.x; c[i][1] = i; }
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int i = 0; i < 8; ++i)
            asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                         : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
    for (int i = 0; i < 8; ++i) s += c[i][0] + c[i][1];
    out[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <class K>
static double time_loop(bem_ctx *c, K kern, double flop_per_thread_iter)
{
    cudaDeviceProp prop;
    CUDA_TRY(cudaGetDeviceProperties(&prop, c->device));
    const int blocks = prop.multiProcessorCount * 8, threads = 256, iters = 20000;
    dvec<double> out;
    out.alloc((size_t)blocks * threads);
    cudaEvent_t e0, e1;
    CUDA_TRY(cudaEventCreate(&e0));
    CUDA_TRY(cudaEventCreate(&e1));
    double best = 0;
    for (int rep = 0; rep < 4; ++rep) {
        CUDA_TRY(cudaEventRecord(e0, c->stream));
        kern<<<blocks, threads, 0, c->stream>>>(out.get(), iters, 0.999999, 1e-9);
        KERNEL_CHECK();
        CUDA_TRY(cudaEventRecord(e1, c->stream));
        CUDA_TRY(cudaEventSynchronize(e1));
        float ms;
        CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
        const double gf = flop_per_thread_iter * iters * (double)blocks * threads / (ms * 1e6);
        if (rep > 0) best = std::max(best, gf);
    }
    cudaEventDestroy(e0);
    cudaEventDestroy(e1);
    return best;
}

}  // namespace bem

using namespace bem;

// message of this thread's last failed bem_create / bem_create_points / bem_create_evaluator (no context exists to hold it)
static thread_local std::string g_create_error = "null context";

extern "C" {

bem_status bem_create(const double *vertices, int64_t n_vertices, const int32_t *triangles, int64_t n_triangles,
                      const int32_t *bubble_id, bem_ctx **out)
{
    if (!out) return BEM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!vertices || !triangles || n_vertices < 4 || n_triangles < 4 || n_vertices > 2000000000ll || n_triangles > 700000000ll)
        return BEM_ERR_INVALID_ARG;
    bem_ctx *c = new (std::nothrow) bem_ctx();
    if (!c) return BEM_ERR_OOM;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { delete c; cudaGetLastError(); return BEM_ERR_CUDA; }
    cudaGetDevice(&c->device);
    c->N = n_vertices;
    c->T = n_triangles;
    bem_status st = guarded(c, [&]() {
        c->V.alloc(3 * c->N);
        c->F.alloc(3 * c->T);
        CUDA_TRY(cudaMemcpy(c->V.get(), vertices, 3 * c->N * sizeof(double), cudaMemcpyDefault));
        CUDA_TRY(cudaMemcpy(c->F.get(), triangles, 3 * c->T * sizeof(int32_t), cudaMemcpyDefault));
        if (bubble_id) {
            c->bid.alloc(c->N);
            CUDA_TRY(cudaMemcpy(c->bid.get(), bubble_id, c->N * sizeof(int32_t), cudaMemcpyDefault));
        }
        validate_mesh(c);
    });
    if (st != BEM_OK) {
        g_create_error = c->err;                                  // bem_last_error(NULL) returns it (this thread's last failed create)
        delete c;
        return st;
    }
    *out = c;
    return BEM_OK;
}

bem_status bem_create_points(const double *sources, int64_t n_sources, const double *targets, int64_t n_targets, bem_ctx **out)
{
    if (!out) return BEM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!sources || !targets || n_sources < 1 || n_targets < 1 || n_sources > 2000000000ll || n_targets > 2000000000ll)
        return BEM_ERR_INVALID_ARG;
    bem_ctx *c = new (std::nothrow) bem_ctx();
    if (!c) return BEM_ERR_OOM;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { delete c; cudaGetLastError(); return BEM_ERR_CUDA; }
    cudaGetDevice(&c->device);
    c->N = n_targets;
    c->T = 0;
    c->np = n_sources;
    c->quadrature = 2;
    bem_status st = guarded(c, [&]() {
        c->V.alloc(3 * c->N);
        c->P.alloc(3 * c->np);
        CUDA_TRY(cudaMemcpy(c->V.get(), targets, 3 * c->N * sizeof(double), cudaMemcpyDefault));
        CUDA_TRY(cudaMemcpy(c->P.get(), sources, 3 * c->np * sizeof(double), cudaMemcpyDefault));
    });
    if (st != BEM_OK) { g_create_error = c->err; delete c; return st; }
    *out = c;
    return BEM_OK;
}

bem_status bem_create_evaluator(bem_ctx *mesh_ctx, const double *targets, int64_t n_targets, bem_ctx **out)
{
    if (!out) return BEM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!mesh_ctx || !targets || n_targets < 1 || n_targets > 2000000000ll) return BEM_ERR_INVALID_ARG;
    if (mesh_ctx->quadrature >= 2 || mesh_ctx->T == 0) {
        mesh_ctx->err = "bem_create_evaluator: the context holds no mesh";
        g_create_error = mesh_ctx->err;                           // no context is returned: bem_last_error(NULL) is where a caller looks
        return BEM_ERR_INVALID_ARG;
    }
    bem_ctx *c = new (std::nothrow) bem_ctx();
    if (!c) return BEM_ERR_OOM;
    c->device = mesh_ctx->device;
    c->stream = mesh_ctx->stream;
    c->parent = mesh_ctx;
    c->mesh_N = mesh_ctx->N;                                      // bem_apply sizes q and phi with these and never reads the parent
    c->mesh_T = mesh_ctx->T;
    c->N = n_targets;
    c->T = 0;
    c->quadrature = 3;
    bem_status st = guarded(c, [&]() {
        c->V.alloc(3 * c->N);
        CUDA_TRY(cudaMemcpy(c->V.get(), targets, 3 * c->N * sizeof(double), cudaMemcpyDefault));
    });
    if (st != BEM_OK) { g_create_error = c->err; delete c; return st; }
    *out = c;
    return BEM_OK;
}

bem_status bem_set_option(bem_ctx *c, const char *key, double value)
{
    if (!c || !key) return BEM_ERR_INVALID_ARG;
    const int v = (int)value;
    drop_graphs(c);
    if (!strcmp(key, "graph")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->use_graph = v; return BEM_OK; }
    if (!strcmp(key, "quadrature")) { if ((v != 0 && v != 1) || c->quadrature >= 2) return BEM_ERR_INVALID_ARG; c->quadrature = v; c->ready = false; }
    else if (!strcmp(key, "mode")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->mode = v; c->ready = false; }
    else if (!strcmp(key, "free_term")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->free_term = v; c->ready = false; }
    else if (!strcmp(key, "gmres_restart")) { if (v < 0) return BEM_ERR_INVALID_ARG; c->gmres_restart = v; }
    else if (!strcmp(key, "lmax")) { if (v != 0 && (v < 2 || v > MAX_LEVEL)) return BEM_ERR_INVALID_ARG; c->force_lmax = v; c->ready = false; }
    else if (!strcmp(key, "timing")) { c->timing = v != 0; }
    else if (!strcmp(key, "reduce_ctas")) { if (v < 0 || v > 32) return BEM_ERR_INVALID_ARG; c->reduce_ctas = v; }
    else if (!strcmp(key, "m2l_rows16")) { c->m2l_rows16 = v != 0; }
    else if (!strcmp(key, "precond")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->precond = v; }
    else if (!strcmp(key, "p2p_precision")) {
        if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG;
        c->p2p_precision = v;
        // the fp32 source records are built HERE (or at the end of bem_setup), never inside a product: a product may run
        // inside a stream capture of the caller, where an allocation is not allowed
        if (v == 1 && c->ready && c->mode == 0 && !c->adaptive) return guarded(c, [&]() { ensure_p2p_f32(c); CUDA_TRY(cudaStreamSynchronize(c->stream)); });
    }
    else if (!strcmp(key, "max_direct_ranges")) { if (v < 1 || v > 256) return BEM_ERR_INVALID_ARG; c->seg_limit = v; c->ready = false; }
    else if (!strcmp(key, "direct_pairs")) { if (value < -1 || value > 1e9) return BEM_ERR_INVALID_ARG; c->direct_max = (int64_t)value; c->ready = false; }
    else if (!strcmp(key, "p2p_ctas")) { if (v < 0 || v > 16) return BEM_ERR_INVALID_ARG; c->p2p_ctas = v; }
    else if (!strcmp(key, "m2l_order_radius")) { if (!(value >= 0 && value < 1.0)) return BEM_ERR_INVALID_ARG; c->m2l_order_radius = value; c->ready = false; }
    else if (!strcmp(key, "m2l_order_extra")) { if (v < -8 || v > 8) return BEM_ERR_INVALID_ARG; c->m2l_order_extra = v; c->ready = false; }
    else if (!strcmp(key, "dipole_degrees")) { if (v < -1 || v > 16) return BEM_ERR_INVALID_ARG; c->dipole_degrees = v; c->ready = false; }
    else if (!strcmp(key, "tree_min_level")) { if (v != 0 && (v < 2 || v > MAX_LEVEL)) return BEM_ERR_INVALID_ARG; c->tree_min_level = v; c->ready = false; }
    else if (!strcmp(key, "tree")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->adaptive = v; c->ready = false; }
    else if (!strcmp(key, "p2p_exact")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->p2p_exact = v; }
    else if (!strcmp(key, "reduce_stream")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->reduce_stream = v; }
    else if (!strcmp(key, "overlap")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->overlap = v; }
    else if (!strcmp(key, "gemm_path")) { if (v != 0 && v != 1) return BEM_ERR_INVALID_ARG; c->gemm_path = v; }
    else { c->err = std::string("unknown option: ") + key; return BEM_ERR_INVALID_ARG; }
    return BEM_OK;
}

bem_status bem_set_stream(bem_ctx *c, void *cuda_stream)
{
    if (!c) return BEM_ERR_INVALID_ARG;
    drop_graphs(c);
    c->stream = (cudaStream_t)cuda_stream;
    return BEM_OK;
}

bem_status bem_setup(bem_ctx *c, int p, int leaf_size, double near_radius)
{
    if (!c) return BEM_ERR_INVALID_ARG;
    if (p < 1 || p > 32 || leaf_size < 1 || !(near_radius >= 1.0)) {
        c->err = "bem_setup: need 1 <= p <= 32, leaf_size >= 1, near_radius >= 1";
        return BEM_ERR_INVALID_ARG;
    }
    return guarded(c, [&]() { setup_impl(c, p, leaf_size, near_radius); });
}

bem_status bem_apply(bem_ctx *c, const double *q, const double *phi, double *y)
{
    if (!c || !y) return BEM_ERR_INVALID_ARG;
    if (!c->ready) { c->err = "bem_apply before bem_setup"; return BEM_ERR_NOT_SETUP; }
    if (y == q || y == phi) { c->err = "bem_apply: y aliases an input"; return BEM_ERR_INVALID_ARG; }
    return guarded(c, [&]() {
        // lengths: q, phi are per mesh vertex (an evaluator: of its parent's mesh); a point cloud takes one monopole and
        // one dipole VECTOR per source; y is per target
        const size_t bytes = c->N * sizeof(double);
        const size_t nv = c->quadrature == 3 ? c->mesh_N : c->N;    // an evaluator's mesh context may be gone by now (bem.h)
        const size_t nq = c->quadrature == 2 ? c->np : nv, nphi = c->quadrature == 2 ? 3 * c->np : nv;
        const size_t qbytes = nq * sizeof(double), pbytes = nphi * sizeof(double);
        const bool hq = !is_device_ptr(q), hp = !is_device_ptr(phi), hy = !is_device_ptr(y);
        const double *dq = q, *dp = phi;
        double *dy = y;
        if (hq) { if (!c->stage_q.p) c->stage_q.alloc(nq); CUDA_TRY(cudaMemcpyAsync(c->stage_q.get(), q, qbytes, cudaMemcpyHostToDevice, c->stream)); dq = c->stage_q.get(); }
        if (hp) { if (!c->stage_phi.p) c->stage_phi.alloc(nphi); CUDA_TRY(cudaMemcpyAsync(c->stage_phi.get(), phi, pbytes, cudaMemcpyHostToDevice, c->stream)); dp = c->stage_phi.get(); }
        if (hy) { if (!c->stage_y.p) c->stage_y.alloc(c->N); dy = c->stage_y.get(); }
        if (hq || hp || hy) apply_device(c, dq, dp, dy);
        else apply_device_cached(c, dq, dp, dy);
        if (hy) CUDA_TRY(cudaMemcpyAsync(y, dy, bytes, cudaMemcpyDeviceToHost, c->stream));
        if (hq || hp || hy) CUDA_TRY(cudaStreamSynchronize(c->stream));
    });
}

bem_status bem_get_timings(bem_ctx *c, double *ms_out, int n)
{
    if (!c || !ms_out || n < 1) return BEM_ERR_INVALID_ARG;
    if (!c->ev_valid || c->ev_n < 2) { c->err = "no timed bem_apply yet (set option timing = 1)"; return BEM_ERR_NOT_SETUP; }
    return guarded(c, [&]() {
        CUDA_TRY(cudaStreamSynchronize(c->stream));
        double t[BEM_T_COUNT] = {0};
        float ms;
        for (int k = 1; k < c->ev_n; ++k) {
            CUDA_TRY(cudaEventElapsedTime(&ms, c->ev[k - 1], c->ev[k]));
            if (c->ev_cls[k] >= 0 && c->ev_cls[k] < BEM_T_TOTAL) t[c->ev_cls[k]] += ms;
        }
        CUDA_TRY(cudaEventElapsedTime(&ms, c->ev[0], c->ev[c->ev_n - 1]));
        t[BEM_T_TOTAL] = ms;
        for (int k = 0; k < n && k < BEM_T_COUNT; ++k) ms_out[k] = t[k];
    });
}

bem_status bem_get_stats(const bem_ctx *c, double *out, int n)
{
    if (!c || !out || n < 1) return BEM_ERR_INVALID_ARG;
    if (!c->ready) return BEM_ERR_NOT_SETUP;
    double s[BEM_S_COUNT] = {0};
    s[BEM_S_N_TARGETS] = (double)c->N;
    s[BEM_S_N_SOURCES] = (double)c->ns;
    s[BEM_S_CSR_NNZ] = (double)c->nnz;
    s[BEM_S_NEAR_TRIANGLES] = (double)c->near_tris;
    s[BEM_S_SETUP_MS] = c->setup_ms;
    s[BEM_S_DEVICE_BYTES] = (double)g_device_bytes.load();
    s[BEM_S_EXP_STRIDE] = c->lay[c->n_lay - 1].nst;
    s[BEM_S_KERNEL_LAUNCHES_PER_APPLY] = c->launches_per_apply;
    if (c->mode == 0) {
        s[BEM_S_LMAX] = c->sb.lmax;
        s[BEM_S_N_SRC_LEAVES] = c->adaptive ? c->ad.n_src_leaves : c->sb.nbox[c->sb.lmax];
        s[BEM_S_N_TGT_LEAVES] = c->adaptive ? c->ad.n_tleaf : c->tb.nbox[c->tb.lmax];
        s[BEM_S_P2P_PAIRS] = (double)c->p2p_pairs;
        s[BEM_S_P2P_PAIRS_EXECUTED] = (double)c->p2p_pairs_exec;
        s[BEM_S_M2L_PAIRS] = (double)c->m2l_pairs;
        const FmmLayout &Lf = c->lay[c->n_lay - 1];           // the layout of a full product (q and phi)
        s[BEM_S_M2L_FLOP] = Lf.m2l_flop;
        s[BEM_S_M2L_ROW_BYTES] = Lf.m2l_row_bytes;
        s[BEM_S_P_DIPOLE] = Lf.p;
        s[BEM_S_P2P_PAIRS_WX] = c->adaptive ? (double)c->p2p_pairs_wx : 0.0;
        for (const bem::Stage &st : c->m2m) {
            s[BEM_S_M2M_PAIRS] += (double)st.npairs;
            if (st.npairs > 0) s[BEM_S_M2M_PARENTS] += (double)(st.n_list >= 0 ? st.n_list : st.ntgt);
        }
        s[BEM_S_N_SRC_BOXES] = c->sb.total();
        s[BEM_S_N_TGT_BOXES] = c->tb.total();
    } else {
        s[BEM_S_P2P_PAIRS] = s[BEM_S_P2P_PAIRS_EXECUTED] = (double)c->N * (double)c->ns;
    }
    for (int k = 0; k < n && k < BEM_S_COUNT; ++k) out[k] = s[k];
    return BEM_OK;
}

bem_status bem_get_free_term(bem_ctx *c, double *c_out)
{
    if (!c || !c_out) return BEM_ERR_INVALID_ARG;
    if (!c->ready || !c->have_cfree) return BEM_ERR_NOT_SETUP;
    return guarded(c, [&]() {
        CUDA_TRY(cudaMemcpyAsync(c_out, c->cfree.get(), c->N * sizeof(double), cudaMemcpyDefault, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
    });
}

bem_status bem_fp64_peak(bem_ctx *c, double *gflops_out)
{
    if (!c || !gflops_out) return BEM_ERR_INVALID_ARG;
    return guarded(c, [&]() { *gflops_out = time_loop(c, dfma_loop, 2.0 * 8.0); });
}

bem_status bem_fp64_tensor_peak(bem_ctx *c, double *gflops_out)
{
    if (!c || !gflops_out) return BEM_ERR_INVALID_ARG;
    return guarded(c, [&]() { *gflops_out = time_loop(c, dmma_loop, 8.0 * 512.0 / 32.0); });
}

const char *bem_last_error(const bem_ctx *c) { return c ? c->err.c_str() : g_create_error.c_str(); }

void bem_destroy(bem_ctx *c)
{
    if (!c) return;
    cudaSetDevice(c->device);
    drop_graphs(c);
    for (cudaEvent_t e : c->ev) cudaEventDestroy(e);
    if (c->ev_fork) cudaEventDestroy(c->ev_fork);
    if (c->ev_join) cudaEventDestroy(c->ev_join);
    if (c->side) cudaStreamDestroy(c->side);
    delete c;
}

}  // extern "C"
