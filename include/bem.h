/*
 * bem.h -- C-ABI of the B200-native boundary-element matrix-vector product
 * for the 3-D Laplace equation on triangulated bubble surfaces
 * (arXiv 1905.01341; citations are /root/reference/PAPER.md:<line>).
 *
 * The operator (Eqs. 11-13; collocation at the mesh vertices,
 * PAPER.md:150-158, Eq. 14):
 *
 *     y_i = S[q](r_i) - D[phi](r_i),     i = 0 .. n_vertices-1,
 *     S[q](r)   = int_S q(r')   G(r,r')          dS(r'),   G = 1/(4 pi |r-r'|),
 *     D[phi](r) = int_S phi(r') dG/dn(r')(r,r')  dS(r'),
 *     dG/dn(r') = n(r').(r-r') / (4 pi |r-r'|^3),
 *
 * with the normal n pointing out of the bubble into the liquid.
 * This is the product "A X, A = f L + g M" the paper's iterative solver calls
 * every iteration (Eq. 45), with monopoles and dipoles handled
 * in ONE call.  Its far field is evaluated with the fast
 * multipole method and its near field directly, A = A^(dense) + A^(sparse)
 * (PAPER.md:436-440); the data structure is built once per mesh and reused by
 * every product.
 *
 * Discretisation ("quadrature" option):
 *   G3 (default)  3-point Gauss per flat triangle with linear (P1) densities:
 *                 monopole strengths q.w and dipole strengths phi.N.w at the
 *                 Gauss points, plus a sparse CSR correction matrix holding
 *                 (exact flat-triangle integral - Gauss value) on the near set
 *                 of every collocation point -- the "correction matrix" scheme
 *                 of PAPER.md:432.
 *   V1            the paper's own lumped rule, Eq. 17, with
 *                 the singular diagonal from the identities Eqs. 19-21
 *                 (PAPER.md:198-216), obtained with 4 internal products
 *                 (PAPER.md:218).
 *
 * Everything runs on ONE CUDA device (sm_100a), in fp64.  There is no CPU
 * fallback: every entry point fails with BEM_ERR_CUDA if no device is usable.
 *
 * Pointers: unless stated otherwise an array argument may be a HOST or a DEVICE
 * pointer (detected with cudaPointerGetAttributes).  Host arrays are copied
 * to / from the device inside the call, which then synchronises; with device
 * pointers bem_apply only enqueues work on the context's stream.
 * No function throws or aborts across this boundary.
 */
#ifndef BEM_B200_H
#define BEM_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bem_ctx bem_ctx;   /* opaque; owns every device allocation it makes */

typedef enum {
    BEM_OK = 0,
    BEM_ERR_INVALID_ARG = 1,     /* NULL / out-of-range argument, unknown option        */
    BEM_ERR_BAD_MESH = 2,        /* mesh is not a closed, outward-oriented manifold      */
    BEM_ERR_NOT_SETUP = 3,       /* bem_apply / bem_solve before a successful bem_setup  */
    BEM_ERR_CUDA = 4,            /* CUDA runtime error (text in bem_last_error)          */
    BEM_ERR_OOM = 5,             /* device allocation failed                             */
    BEM_ERR_NOT_CONVERGED = 6    /* bem_solve stopped at max_iter; outputs are filled    */
} bem_status;

/* Indices of the per-kernel-class timings returned by bem_get_timings (ms). */
enum {
    BEM_T_LIFT = 0, BEM_T_P2M, BEM_T_M2M, BEM_T_M2L, BEM_T_L2L_REDUCE, BEM_T_L2P,
    BEM_T_P2P, BEM_T_SPMV, BEM_T_TOTAL, BEM_T_COUNT
};

/* Indices of the statistics returned by bem_get_stats. */
enum {
    BEM_S_N_TARGETS = 0, BEM_S_N_SOURCES, BEM_S_LMAX, BEM_S_N_SRC_LEAVES, BEM_S_N_TGT_LEAVES,
    BEM_S_P2P_PAIRS, BEM_S_M2L_PAIRS, BEM_S_CSR_NNZ, BEM_S_NEAR_TRIANGLES, BEM_S_SETUP_MS,
    BEM_S_N_SRC_BOXES, BEM_S_N_TGT_BOXES,
    BEM_S_DEVICE_BYTES,    /* live device bytes of ALL contexts and filters of the process (one atomic counter), not of ctx alone */
    BEM_S_EXP_STRIDE,
    BEM_S_KERNEL_LAUNCHES_PER_APPLY,
    BEM_S_M2L_FLOP,        /* executed flop of the M2L tiles of one product (graded truncation: 4 (4 KE)^2 per pair) */
    BEM_S_M2L_ROW_BYTES,   /* bytes of translated rows the per-target sums read in one product                     */
    BEM_S_P_DIPOLE,        /* truncation number of the products that carry dipoles (option "dipole_degrees")                 */
    BEM_S_P2P_PAIRS_EXECUTED, /* point pairs the near-field kernel executes: BEM_S_P2P_PAIRS are the useful ones, the source list
                               of a target leaf is padded to whole rounds of 128 sources                               */
    BEM_S_P2P_PAIRS_WX,    /* adaptive tree: the point pairs of BEM_S_P2P_PAIRS that belong to W-list ranges (children, not touching the
                            * target leaf, of a subdivided same-level neighbour) and X-list ranges (coarser source leaves that touch an
                            * ancestor but not the leaf): the library sums them directly; an FMM with M2P / P2L would expand them   */
    BEM_S_M2M_PAIRS,       /* (child, parent) translations of one upward pass                                               */
    BEM_S_M2M_PARENTS,     /* parent boxes written by the upward pass                                                        */
    BEM_S_COUNT
};

/* bem_create -- take a triangulated bubble-cluster surface (PAPER.md:150-152:
 * "the surface is discretized by a mesh with N vertices"; collocation points are
 * the vertices).
 *   vertices   [n_vertices x 3] row-major fp64 coordinates.
 *   triangles  [n_triangles x 3] 0-based vertex ids, counter-clockwise seen from
 *              the liquid, so that (r2-r1)x(r3-r1) points out of the bubble
 *              (PAPER.md:141, 233).
 *   bubble_id  [n_vertices] 0..M-1, the bubble a vertex belongs to (may be NULL:
 *              one bubble).  Used for the per-bubble orientation check only.
 * The mesh is COPIED to the device; the caller keeps ownership of its arrays.
 * Validation (on the device): indices in range, no zero-area triangle, every
 * directed edge matched by exactly one opposite edge (closed oriented manifold),
 * all three vertices of a triangle in one bubble, signed volume of every bubble
 * > 0.  Violations return BEM_ERR_BAD_MESH and *out = NULL.
 * The context is created with the CUDA device that is current at the call. */
bem_status bem_create(const double *vertices, int64_t n_vertices,
                      const int32_t *triangles, int64_t n_triangles,
                      const int32_t *bubble_id, bem_ctx **out);

/* bem_create_points -- the same engine on a POINT CLOUD: the workload of the paper's Tables 1-2 (PAPER.md:456-490:
 * "N sources and N receivers distributed randomly and uniformly inside a cube", monopoles), and the general point form
 * of the two kernels of PAPER.md:143-145 (Eq. 13) with monopole AND dipole sources.
 *   sources  [n_sources x 3] fp64 source positions, targets [n_targets x 3] evaluation points (may be the same array).
 * bem_apply(ctx, q, d, y) then computes, over all sources with x_i != y_j,
 *     y_i = sum_j [ q_j / (4 pi |x_i - y_j|)  -  d_j . (x_i - y_j) / (4 pi |x_i - y_j|^3) ],
 * q: [n_sources] monopole strengths, d (the `phi` argument): [n_sources x 3] row-major dipole VECTORS (d_j = phi_j n_j w_j
 * is the quadrature of -D[phi] with weights w_j and normals n_j); either may be NULL.  y is [n_targets].  There is no
 * mesh, no correction matrix and no bem_solve in this mode; options "mode", "lmax", "timing", "gemm_path",
 * "dipole_degrees" and bem_setup(p, leaf_size, -) work as for a mesh (near_radius is ignored).  Arrays are copied; host
 * or device pointers. */
bem_status bem_create_points(const double *sources, int64_t n_sources, const double *targets, int64_t n_targets,
                             bem_ctx **out);

/* bem_create_evaluator -- the potential OFF the surface (Eq. 11, the cases r not on S): for x in the
 * liquid  S[q](x) - D[phi](x) = -phi(x),  inside a bubble it is 0 -- Green's representation of the field by the surface
 * data the solver works with.  The new context evaluates
 *     u(x_t) = S[q](x_t) - D[phi](x_t),   t = 0 .. n_targets-1,
 * with the SAME discretisation as bem_apply on the mesh (G3: 3-point Gauss per flat triangle with P1 densities, plus the
 * exact flat-triangle integrals on the near set { k : |x_t - c_k| <= eta d_k } through a CSR correction matrix whose
 * columns are the mesh vertices), the same octree / FMM engine and the same options.
 *   mesh_ctx  a context made by bem_create (it need not be set up itself).  Its mesh is read by every bem_setup of the
 *             evaluator and by nothing else: it must be alive during those calls, and may be destroyed after the last
 *             one -- bem_apply, bem_get_stats and bem_destroy of the evaluator do not touch it (a bem_setup after the
 *             mesh context is gone is a use-after-free the library cannot detect).  The evaluator runs on the device
 *             and stream of mesh_ctx.
 *   targets   [n_targets x 3] fp64 points, host or device, copied.  A target ON the surface is not allowed (use
 *             bem_apply for the vertices); a target closer to a triangle than ~1e-6 of its size loses accuracy.
 * Then: bem_setup(ev, p, leaf_size, near_radius); bem_apply(ev, q, phi, u) with q, phi [n_vertices of the MESH] and
 * u [n_targets]; bem_get_stats, bem_set_option, bem_set_stream, bem_destroy as usual.  bem_solve, the surface functions
 * and option "quadrature" do not apply (BEM_ERR_INVALID_ARG). */
bem_status bem_create_evaluator(bem_ctx *mesh_ctx, const double *targets, int64_t n_targets, bem_ctx **out);

/* bem_set_option -- must be called before bem_setup to take effect.
 *   "quadrature"    0 = G3 (default), 1 = V1 (paper's Eq. 17 + Eqs. 19-21)
 *   "mode"          0 = FMM (default), 1 = direct all-pairs sum (the paper's
 *                   "brute force" product)
 *   "free_term"     0 = c_i = 1 + (D.1)_i, the discrete solid angle implied by
 *                   the diagonal rule M_ii = -1/2 - sum_{j!=i} M_ij
 *                   (default); 1 = c_i = 1/2 literally (Eq. 15)
 *   "gmres_restart" 0 = no restart up to max_iter (default), else restart length
 *   "overlap"       0 (default) = every kernel of a product on the context's stream; 1 = the per-target sums of the
 *                   translated M2L rows (HBM-bound) run on a side stream beside the near field (FP64-bound).  Round 1
 *                   measured a gain (25.6 -> 24.5 ms on config 5); with the graded M2L rows of round 2 the sums are
 *                   short, and the CTAs they hold cost the near-field kernel more than the overlap wins (config 5:
 *                   22.6 ms on one stream, 22.6-24.4 ms with the side stream).  Results are bit-identical.
 *   "reduce_stream" 1 (default) = the per-target sums of the translated rows stream the packed rows of a target through
 *                   shared memory (cp.async, batches of 4 rows, two in flight); 0 = direct loads.  The same bits; tuning.
 *   "reduce_ctas"   with overlap = 1: the sums are a persistent grid of this many CTAs per SM (1..32; 0 = chosen
 *                   from the pair counts so that it ends just before the near field does).  Tuning only.
 *   "m2l_rows16"    M2L tiles at p = 11, 12: 1 = 4 warps x 16 rows per CTA (default), 0 = 8 warps x 8 rows.
 *                   A tuning switch: both compute the same tiles.  May be changed between products.
 *   "precond"       bem_solve: 0 = unpreconditioned GMRES, as in the paper (default); 1 = right
 *                   diagonal scaling, GMRES on (S D^-1)(D q) = b with D = diag(S) (exact self integrals; in V1
 *                   the L_ii of Eq. 21).  The stopping rule (true relative residual of S q = b) is unchanged.
 *                   Not in the paper: it equilibrates bubbles of different size (S_ii ~ mesh size).  May be
 *                   changed between solves.
 *   "lmax"          0 = choose the octree depth from leaf_size (default), else force it (adaptive tree: cap it)
 *   "tree"          0 = uniform depth l_max with empty boxes skipped -- the paper's tree (default);
 *                   1 = adaptive octree: a box is subdivided iff it holds more than leaf_size sources or lies above
 *                   the depth the uniform rule gives for that leaf_size (so the adaptive tree only REFINES the boxes
 *                   that are denser than the mean; "tree_min_level" lowers that floor, >= 2), a box exists iff its
 *                   parent is subdivided, leaves sit on several levels.  Far field between existing boxes of equal
 *                   level (V lists); a target leaf sums directly the sources of the same-level boxes that touch it
 *                   and of the coarser source leaves that touch its ancestors (the U, W and X lists of the adaptive
 *                   FMM, W and X taken directly: exact).  Same tolerances; p2p_precision = 1 is refused (its fp32
 *                   positions need leaves of one size).  Measured: on the bubble clusters of BASELINE.json the two
 *                   trees are within 2% of each other; on a strongly clustered point cloud the adaptive tree needs
 *                   19x fewer point pairs.
 *   "tree_min_level" adaptive tree: boxes above this level are always subdivided (0 = the uniform depth; >= 2)
 *   "dipole_degrees" products that carry dipoles (phi != NULL) are truncated to p + this many degrees; -1 (default) =
 *                   3 below p = 12 and 0 from 12 on (measured: S - D then meets relative L2 1e-5 at the stated p of
 *                   every BASELINE config; a dipole is one derivative of the monopole expansion and loses 3-4
 *                   degrees of accuracy at equal truncation); 0 = one truncation for everything, the paper's
 *                   convention.  Products without dipoles (every GMRES iteration) always use p.
 *   "m2l_order_radius", "m2l_order_extra"  graded truncation of the M2L translations: the offset o (in box edges) uses
 *                   the degrees < p_o = ceil(p ln k(2) / ln k(|o|)) + extra, k(d) = a / (d - a), a = radius (default
 *                   0.5, extra 1: error against the direct sum unchanged within 7% on every config, executed M2L work
 *                   x0.54 at p = 12); radius 0 = every translation uses all p degrees.
 *   "timing"        1 = record per-kernel-class CUDA-event timings in bem_apply
 *   "gemm_path"     batched translations (M2M, M2L, L2L): 0 = FP64 tensor-core tiles (DMMA; p <= 16,
 *                   default -- measured faster), 1 = plain FP64 FMA tiles (any p).
 *                   May be changed between products.
 *   "p2p_precision" near field A^(sparse) X in FMM mode: 0 = fp64 pairs (default; the measured mode, the only one
 *                   that meets the 1e-8 tolerance at high p); 1 = the paper's "single precision on GPU" option
 *                   (Table 1): every pair 1/r, d.(x-y)/r^3 in fp32 on positions taken relative to
 *                   the leaf centres (in leaf edges), at most 8 pairs per target summed in fp32, all further sums
 *                   in fp64 in a fixed order.  The far field, the correction matrix and the direct-sum mode stay
 *                   fp64.  Error floor ~1e-7 (monopoles) .. 1e-6 (dipoles on surfaces) relative L2: at the
 *                   configs' p (<= 12) the product's error is unchanged.  May be changed between products.
 *   "p2p_exact"     near field of the FMM mode, fp64 pairs: 0 (default) = 1/r by the hardware seed and ONE Newton step (relative
 *                   error of a pair <= 4e-13, one-sided: four decades below the truncation error of the far field; 16
 *                   FP64 instructions per pair), 1 = the third-order step of the direct-sum mode (1 ulp; 17 instructions).
 *                   The direct-sum mode always uses the third-order step (its tolerance is 1e-12).  May be changed
 *                   between products.
 *   "direct_pairs"  leaf-level far-field (M2L) pairs whose boxes hold nt targets and ns sources with nt x ns <= this
 *                   value are summed directly in the near-field kernel instead of being translated: a translation
 *                   costs 4 nre^2 flop whatever the boxes hold, and on surface meshes a third of the leaf-level pairs
 *                   join sparsely filled boxes (the balance of A^(dense) and A^(sparse), per pair).
 *                   -1 = 800 (nre / 80)^2 from the measured costs (default), 0 = off (the uniform lists of
 *                   PAPER.md:440).  Direct pairs are exact, so the error can only fall.
 *                   Adaptive tree: the pair kernel holds at most 256 direct source ranges per target leaf (27 of the own
 *                   level, the coarser leaves next to its ancestors, up to 189 direct far pairs).  When a leaf exceeds
 *                   that and direct_pairs is -1, bem_setup rebuilds the lists with every far pair translated; with an
 *                   explicit direct_pairs > 0 it returns BEM_ERR_INVALID_ARG (lower it, or raise leaf_size).
 *   "max_direct_ranges"  1..256 (default 256): lowers that limit (a test hook for the rebuild above; no reason to set it
 *                   otherwise).
 *   "graph"         1 (default): bem_apply with DEVICE pointers q, phi, y on a stream other than the legacy default stream is
 *                   captured into a CUDA graph the second time the same (q, phi, y) is asked for and replayed from then
 *                   on -- one launch instead of 20-40 on the launch-bound small meshes.  Any bem_set_option,
 *                   bem_set_stream or bem_setup drops the captured graphs.  0: always launch kernel by kernel.
 *                   The cache is keyed on the raw (q, phi, y, stream) addresses and holds no reference to the buffers:
 *                   a replay reads and writes whatever lives at those addresses, so freeing a buffer and asking for a
 *                   product with a new buffer that landed on the same address is fine, but a freed buffer must not be
 *                   passed again; set "graph" 0 if the caller's allocator makes that hard to guarantee.
 *   "p2p_ctas"      fp32 near field: CTAs per SM of its persistent grid while the row sums share the SMs
 *                   (1..16; 0 = 4, default).  Tuning only. */
bem_status bem_set_option(bem_ctx *ctx, const char *key, double value);

/* bem_set_stream -- cuda_stream is a cudaStream_t (NULL = default stream).  All
 * later work of this context is enqueued there. */
bem_status bem_set_stream(bem_ctx *ctx, void *cuda_stream);

/* bem_setup -- build everything that depends on the mesh only (PAPER.md:440:
 * "data structure ... built once"): triangle geometry, source points, the octree
 * from 63-bit Morton keys (unit-cube scaling, bit interleave, radix sort; empty
 * boxes skipped; separate source and receiver box sets), neighbour and
 * interaction lists, translation matrices, and the near-field correction CSR.
 *   p            truncation number: expansions hold degrees n = 0..p-1, p^2 real
 *                coefficients.  1 <= p <= 32.  Ignored in direct mode.
 *                p is the truncation of the products WITHOUT dipoles (phi == NULL: S[q],
 *                every iteration of bem_solve).  A product with phi != NULL runs at
 *                p + 3 when p < 12 (option "dipole_degrees", default -1; 0 = the paper's
 *                one truncation for both layers); BEM_S_P_DIPOLE reports the value used.
 *   leaf_size    the octree depth l_max is the smallest level >= 2 at which the mean
 *                population of non-empty source boxes is <= leaf_size (the paper's
 *                clustering parameter).  >= 1.
 *   near_radius  eta >= 1, dimensionless: triangle k is "near" vertex i iff i is a
 *                vertex of k or |r_i - c_k| <= eta * max_a |r_ka - c_k| (c_k the
 *                centroid).  Only used by G3. */
bem_status bem_setup(bem_ctx *ctx, int p, int leaf_size, double near_radius);

/* bem_apply -- y = S[q] - D[phi] at all vertices (Eq. 45, with
 * (f, g) = (1, -1)).  q, phi: [n_vertices] fp64, either may be NULL (zero
 * density: that layer is skipped -- f or g = 0).  y: [n_vertices] fp64 output,
 * must not alias q or phi.  No free term (+-1/2 phi) is added.  Asynchronous on
 * the context's stream when all pointers are device pointers.
 * (Point cloud: q [n_sources], phi = dipole vectors [n_sources x 3], y [n_targets];
 * evaluator: q, phi [n_vertices of its mesh], y [n_targets] -- see the two creators.) */
bem_status bem_apply(bem_ctx *ctx, const double *q, const double *phi, double *y);

/* bem_solve -- the Dirichlet problem of PAPER.md:125, 160-171 (Eqs. 15-16):
 * given phi on the surface find q = dphi/dn with  S q = b,
 * b_i = -c_i phi_i + (D phi)_i, by unpreconditioned GMRES,
 * Gram-Schmidt applied twice, stopping when ||b - S q|| / ||b|| <= tol.
 *   q           [n_vertices] output; read as the initial guess iff use_q_as_x0
 *               (the paper warm-starts from the previous time step).
 *   iters_out, relres_out  may be NULL.
 * Returns BEM_ERR_NOT_CONVERGED when it stops at max_iter, with q, iters_out
 * and relres_out filled with the last iterate. */
bem_status bem_solve(bem_ctx *ctx, const double *phi, double *q, int use_q_as_x0,
                     double tol, int max_iter, int *iters_out, double *relres_out);

/* bem_get_timings -- ms per kernel class (BEM_T_*) of the last bem_apply made
 * with option "timing" = 1; synchronises the stream.  ms_out: HOST array of n. */
bem_status bem_get_timings(bem_ctx *ctx, double *ms_out, int n);

/* bem_get_stats -- sizes fixed by bem_setup (BEM_S_*).  out: HOST array of n. */
bem_status bem_get_stats(const bem_ctx *ctx, double *out, int n);

/* bem_get_free_term -- c_i of bem_solve ([n_vertices], host or device output). */
bem_status bem_get_free_term(bem_ctx *ctx, double *c_out);

/* bem_fp64_peak -- register-resident DFMA loop on the context's device; returns
 * the achieved FP64 rate in GFLOP/s (2 flop per DFMA) in *gflops_out (HOST).
 * It is the measured denominator of the P2P / M2L roofline fractions. */
bem_status bem_fp64_peak(bem_ctx *ctx, double *gflops_out);

/* bem_fp64_tensor_peak -- the same with a register-resident mma.sync m8n8k4 f64 (DMMA) loop: the
 * FP64 tensor-core rate, GFLOP/s (512 flop per warp instruction) in *gflops_out (HOST).  north_star:
 * "tensor cores (FP64 DMMA) only if ... measured faster" -- this is that measurement. */
bem_status bem_fp64_tensor_peak(bem_ctx *ctx, double *gflops_out);

/* Last error text of this context (never NULL; valid until the next call).  ctx == NULL: the message of this thread's
 * last failed bem_create / bem_create_points / bem_create_evaluator (which return no context to ask). */
const char *bem_last_error(const bem_ctx *ctx);

/* Free every device allocation of the context.  NULL is allowed. */
void bem_destroy(bem_ctx *ctx);

/* ------------------------------------------------------------------------------------------------------------------
 * The steps either side of the solve in one time step ("Surface" functions and filters, ~10% of an
 * FMM call).  They need the mesh only, not bem_setup.
 *
 * bem_surface_velocity -- per vertex j (Eq. 17; Eqs. 22-27):
 *     s_j = 1/3 sum_{k ni j} A_k,   n_j = m_j / |m_j|,   m_j = sum_{k ni j} N_k A_k                       (Eq. 17)
 *     (n x v)_k A_k = 1/2 [ (r_k2 - r_k3) phi_k1 + (r_k3 - r_k1) phi_k2 + (r_k1 - r_k2) phi_k3 ]         (Eq. 26: the
 *         contour integral of the linearly interpolated phi around triangle k, by Stokes' theorem, Eq. 23)
 *     (n x v)_j = 1/(3 s_j) sum_{k ni j} (n x v)_k A_k,   v_j = n_j q_j + (n x v)_j x n_j                 (Eqs. 27, 22)
 *   phi, q  [n_vertices] potential and its normal derivative (q may be NULL: tangential part only; phi may be NULL
 *           when v is NULL)
 *   v            [n_vertices x 3] row-major, or NULL
 *   normals_out  [n_vertices x 3] n_j, or NULL;  areas_out [n_vertices] s_j, or NULL  (at least one output)
 * Host or device pointers (host: staged and synchronised).  The sums over the triangles of a vertex run in mesh
 * order (bit-reproducible).  BEM_ERR_INVALID_ARG for a point-cloud context. */
bem_status bem_surface_velocity(bem_ctx *ctx, const double *phi, const double *q, double *v, double *normals_out,
                                double *areas_out);

/* bem_surface_curvature -- mean curvature H_j at every vertex by the fitted paraboloid (Eqs. 28-29):
 * in the frame centred at r_j whose z axis is n_j (Eq. 17), the paraboloid z = B1 x + B2 y + B3 x^2 + B4 x y + B5 y^2
 * through FIVE neighbours of the vertex (5 x 5 linear system, Eq. 28), H_j = -B3 - B5 (Eq. 29): 1/R on a sphere whose
 * normal points out of the bubble.  The paper does not say which five of the neighbours are used: they are the first
 * five distinct vertices met when walking the triangles that hold vertex j in mesh order (triangle index, then corner),
 * taking of each triangle its two other vertices in cyclic order.  NaN where a vertex has fewer than five neighbours
 * or the system is singular.  H: [n_vertices], host or device. */
bem_status bem_surface_curvature(bem_ctx *ctx, double *H);

/* bem_bubble_volume -- V_m, the volume of every bubble: what the polytropic gas law needs each time step
 * (p_g = p_g0 (V_m0 / V_m)^kappa) and the "volume" among the surface functions of PAPER.md:612.  It is
 * the volume enclosed by the bubble's flat triangles (exact for the polyhedron; 4 pi R^3 / 3 (1 - O(h^2)) on a sphere).
 * A triangle belongs to the bubble of its first vertex (bem_create refuses triangles that join two bubbles).
 *   vol_out    [n_bubbles] fp64, host or device; n_bubbles must equal the mesh's bubble count (largest id + 1, or 1
 *              when bem_create got no ids), else BEM_ERR_INVALID_ARG.
 * Needs no bem_setup.  The grouping of triangles by bubble is built at the first call and kept.  Fixed summation
 * order: repeated calls return the same bits. */
bem_status bem_bubble_volume(bem_ctx *ctx, double *vol_out, int64_t n_bubbles);

/* Shape filter of bandwidth p_f (Eqs. 34-43): every bubble surface is a map of the unit sphere, the
 * mesh points keep their spherical angles (theta_i, phi_i) for all times, and a surface function sampled at them is
 * replaced by its least-squares fit with the spherical harmonics of degree n < p_f,
 *     xhat = F x,   F = G (G* G)^-1 G*,   G_ij = Y_j(theta_i, phi_i),  j = (n, m), n = 0..p_f-1          (Eqs. 39-42)
 * -- the orthogonal projector on the band.  One filter serves all bubbles that share the angles of their mesh points
 * ("only one shape filter is necessary when all bubbles have the same initial shape").  The library keeps
 * F in its factored form (rank p_f^2 << N_d): xhat = G (G^+ x), G^+ = (G^T G)^-1 G^T by a Cholesky factorisation on
 * the device, in the real orthonormal harmonic basis (same span as Eq. 37, so the same F).
 *
 * bem_filter_create -- theta (polar angle), phi (azimuth): [n_d] angles of the points of ONE bubble, host or device,
 *   copied.  1 <= p_f <= 16 and p_f^2 < n_d.  BEM_ERR_BAD_MESH when G^T G is singular (the points do not
 *   resolve the band).
 * bem_filter_apply -- x, xhat: [n_cols x n_d] row-major; a column c = (surface function, bubble) is the n_d samples of
 *   that function on that bubble (x, y, z, phi, ... of Eqs. 41, 43), contiguous.  xhat may be x (in place).  Host or
 *   device pointers; enqueued on cuda_stream (a cudaStream_t, NULL = default stream), synchronised only for host
 *   pointers. */
typedef struct bem_filter bem_filter;
bem_status bem_filter_create(const double *theta, const double *phi, int64_t n_d, int p_f, bem_filter **out);
bem_status bem_filter_apply(bem_filter *f, const double *x, int64_t n_cols, double *xhat, void *cuda_stream);
const char *bem_filter_last_error(const bem_filter *f);
void bem_filter_destroy(bem_filter *f);

/* bem_direct_sum_static -- the all-pairs sum of the two kernels of PAPER.md:143-145 (Eq. 13) over a point cloud,
 *     y_i = sum_{j : y_j != x_i} [ q_j / (4 pi |x_i - y_j|)  -  d_j . (x_i - y_j) / (4 pi |x_i - y_j|^3) ],
 * the same sum as bem_create_points + option "mode" = 1 + bem_apply (the direct-sum mode of PAPER.md:490), for callers
 * that must NOT allocate device memory: this call makes no cudaMalloc / cudaFree and calls nothing that does.  It is
 * meant for a host whose device memory is already spoken for when the sum is needed -- a simulation that carved the
 * GPU into its own arenas at start-up, a tenant under a fixed MPS / MIG memory budget -- and for a latency-bound loop
 * that cannot take the device-wide synchronisation a cudaMalloc / cudaFree brings.  Every other entry of this library
 * allocates (contexts, staging, Krylov vectors) and is not for them.
 *   sources  [n_sources x 3], q [n_sources] monopole strengths or NULL, d [n_sources x 3] dipole vectors or NULL,
 *   targets  [n_targets x 3], y [n_targets] (overwritten; must not overlap the inputs).  All fp64, row-major, and all
 *   DEVICE pointers of the CURRENT device (a host pointer is refused: copying it would need a staging buffer).
 *   cuda_stream  a cudaStream_t, NULL = the default stream.  The call enqueues two kernels and returns; it never
 *   synchronises.
 * Scratch: the partial sums of the source chunks live in an array compiled into the library (static __device__,
 * 16 x BEM_DIRECT_STATIC_MAX_TARGETS doubles = 8 MiB).  Consequences a caller must know:
 *   - n_targets > BEM_DIRECT_STATIC_MAX_TARGETS is refused with BEM_ERR_INVALID_ARG (n_sources: up to 2^31 - 1);
 *     split a larger target set into several calls, one after the other.
 *   - every GPU on which the process has loaded the library holds those 8 MiB until the process exits, whether or not
 *     this function is ever called.
 *   - all calls on a device share the one array.  Nothing in it has to start at zero (each call overwrites every slot
 *     it reads), but two calls whose kernels overlap on the GPU -- different streams, different host threads -- race
 *     on it and return garbage: keep the calls of one device on one stream, or order them with events.
 *   - the FIRST call on each device looks up the array's device address (cudaGetSymbolAddress, with that device
 *     current) and keeps it; make that first call during start-up, before any stream capture begins.
 * Errors: BEM_ERR_INVALID_ARG (sizes, NULL or host pointers, buffers of another device), BEM_ERR_CUDA; the text is
 * returned by bem_direct_sum_static_last_error() (per host thread). */
#define BEM_DIRECT_STATIC_MAX_TARGETS 65536
bem_status bem_direct_sum_static(const double *sources, int64_t n_sources, const double *q, const double *d,
                                 const double *targets, int64_t n_targets, double *y, void *cuda_stream);
const char *bem_direct_sum_static_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* BEM_B200_H */
