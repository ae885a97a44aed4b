// Shared declarations of the library: error handling, device buffers, the
// context.  Product code only -- nothing here is shared with oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <cstdio>
#include <atomic>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>
#include <stdexcept>

#include "../../include/bem.h"

namespace bem {

struct Error : std::runtime_error {
    bem_status status;
    Error(bem_status s, const std::string &m) : std::runtime_error(m), status(s) {}
};

inline void cuda_check(cudaError_t e, const char *what, const char *file, int line)
{
    if (e == cudaSuccess) return;
    char buf[512];
    snprintf(buf, sizeof buf, "%s: %s (%s:%d)", what, cudaGetErrorString(e), file, line);
    throw Error(e == cudaErrorMemoryAllocation ? BEM_ERR_OOM : BEM_ERR_CUDA, buf);
}
#define CUDA_TRY(x) ::bem::cuda_check((x), #x, __FILE__, __LINE__)
#define KERNEL_CHECK() ::bem::cuda_check(cudaGetLastError(), "kernel launch", __FILE__, __LINE__)

extern std::atomic<size_t> g_device_bytes;   // running total of the live device allocations of ALL contexts of the process (stats only)

// Owning device array.
template <class T>
struct dvec {
    T *p = nullptr;
    size_t n = 0;
    dvec() = default;
    dvec(const dvec &) = delete;
    dvec &operator=(const dvec &) = delete;
    dvec(dvec &&o) noexcept : p(o.p), n(o.n) { o.p = nullptr; o.n = 0; }
    dvec &operator=(dvec &&o) noexcept { if (this != &o) { free(); p = o.p; n = o.n; o.p = nullptr; o.n = 0; } return *this; }
    ~dvec() { free(); }
    void free() { if (p) { cudaFree(p); g_device_bytes -= n * sizeof(T); } p = nullptr; n = 0; }
    void alloc(size_t count)
    {
        free();
        if (count == 0) count = 1;
        CUDA_TRY(cudaMalloc((void **)&p, count * sizeof(T)));
        n = count;
        g_device_bytes += n * sizeof(T);
    }
    void zero(cudaStream_t s) { CUDA_TRY(cudaMemsetAsync(p, 0, n * sizeof(T), s)); }
    T *get() const { return p; }
};
// non-owning view of a device array (the active truncation layout of the context)
template <class T>
struct dptr {
    T *p = nullptr;
    T *get() const { return p; }
};

// Preferred shared-memory carve-out (percent of the SM's L1/shared array) of the kernels that bem_apply runs side by side
// on one SM (the near-field pair kernels and the row sums of the M2L stages).  An SM can only hold CTAs whose kernels
// agree on the carve-out: with the driver's per-kernel default, a few KB more static shared memory in one of them was
// enough to serialise the two (measured: config 5, fp32 pairs beside the sums, 21.3 -> 26.5 ms).
constexpr int CORUN_CARVEOUT = 14;     // 32 KB of 228

// device -> host copy of a result of the work enqueued on stream s.  (A plain cudaMemcpy runs on the legacy default stream,
// which does not wait for a NON-BLOCKING user stream: bem_setup on such a stream would read counters before their kernels end.)
inline void d2h_sync(void *dst, const void *src, size_t bytes, cudaStream_t s)
{
    CUDA_TRY(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
}

inline int cdiv(int64_t a, int64_t b) { return (int)((a + b - 1) / b); }

// Function attributes (dynamic shared-memory opt-in, carve-out) are PER DEVICE, and contexts may live on several devices
// and threads: every launch site keeps one flag per device and sets its attributes through once_per_device.
// The mutex is held WHILE the attributes are set: a second thread on the same device waits until the opt-in is in place and
// cannot launch with more dynamic shared memory than the default allows.  A failed set-up leaves the flag clear.
std::mutex &device_once_mutex();
template <class F>
inline void once_per_device(std::vector<char> &done, int device, F &&set_attributes)
{
    std::lock_guard<std::mutex> lock(device_once_mutex());
    if ((int)done.size() <= device) done.resize(device + 1, 0);
    if (done[device]) return;
    set_attributes();
    done[device] = 1;
}
}  // namespace bem
struct bem_ctx;
namespace bem {
const bem_ctx *mesh_of(const bem_ctx *c);     // the context that owns the mesh: c itself, or the parent of an evaluator
// with option "timing": record an event on the context's stream; the time since the previous mark is charged to cls
void mark(bem_ctx *c, int cls);

// ---------------------------------------------------------------- primitives (prims.cu)
void scan_exclusive_i32(const int32_t *in, int32_t *out, int64_t n, cudaStream_t s);  // out[n] = total (n+1 outputs)
void scan_exclusive_i64(const int32_t *in, int64_t *out, int64_t n, cudaStream_t s);  // out[n] = total
// stable LSD radix sort of (key, value) pairs on bits [begin_bit, end_bit); result ends in (keys, vals);
// tmp arrays must hold n elements.
void radix_sort_pairs(uint64_t *keys, uint32_t *vals, uint64_t *keys_tmp, uint32_t *vals_tmp,
                      int64_t n, int begin_bit, int end_bit, cudaStream_t s);
void iota_u32(uint32_t *v, int64_t n, cudaStream_t s);
// min / max of the three coordinates of n points (AoS xyz); out6 = device [minx,miny,minz,maxx,maxy,maxz]
void bbox3(const double *xyz, int64_t n, double *out6, cudaStream_t s);
double reduce_max(const double *v, int64_t n, cudaStream_t s);   // synchronises

// ---------------------------------------------------------------- octree tables (tree.cu)
constexpr int MAX_LEVEL = 12;      // expansions exist on levels 2..lmax <= MAX_LEVEL
constexpr int N_OFFSETS = 343;     // (2*3+1)^3 relative positions, 316 of them well separated
constexpr int MAT_M2L = 0;         // matrix ids: [0,343) M2L by offset, then 8 L2L, then 8 M2M
constexpr int MAT_L2L = 343;
constexpr int MAT_M2M = 351;
constexpr int N_MATS = 359;
constexpr int ROT_M = 32;          // entries per matrix in the azimuth table (m < P_MAX = 32)

struct BoxSet {                     // the non-empty boxes of one point set on levels 0..lmax
    int lmax = 0;
    int64_t npts = 0;
    dvec<uint64_t> key_sorted;      // [npts] 63-bit Morton keys, ascending
    dvec<uint32_t> perm;            // [npts] sorted position -> original index
    int nbox[MAX_LEVEL + 1] = {0};  // boxes per level
    int base[MAX_LEVEL + 2] = {0};  // global index of the first box of a level (levels 2..lmax)
    dvec<uint64_t> bkey[MAX_LEVEL + 1];   // [nbox] key prefix (3*level bits) of each box, ascending
    dvec<int32_t> child[MAX_LEVEL + 1];   // [nbox+1] first child at level+1 (for level < lmax)
    dvec<int32_t> parent[MAX_LEVEL + 1];  // [nbox] parent at level-1
    dvec<int32_t> begin;            // [nbox[lmax]+1] first point of each leaf
    dvec<int32_t> leaf_of;          // [npts] leaf of each sorted point
    int total() const { return base[lmax + 1]; }
};

// existence / subdivision flags of the boxes an interaction-list kernel looks at (adaptive tree; all null: uniform tree)
struct AdaptiveFlags {
    const uint8_t *t_ex = nullptr, *t_sub = nullptr;                 // target boxes of the level
    const uint8_t *s_sub = nullptr;                                   // source boxes of the level
    const uint8_t *s_ex_parent = nullptr, *s_sub_parent = nullptr;    // source boxes of the parent level
};

// One batched-translation stage: out[tgt] = sum over the target's pairs of T[mat] * in[src]
// executed as (tiles of a dense GEMM per matrix) -> scratch rows in target-major order -> fixed-order row sums.
struct Tile { int32_t mat, row0, nrows, flags; };     // flags: bit 0 input rows are local expansions, bit 1 M2L (azimuth split)
constexpr int M2L_NCLS = 5;        // truncation classes of the M2L tiles: degrees < pl - i, i = 0..4
// k-steps (4 dofs each, in pairs) of either block that hold the degrees < pp: 4 ke_of(pl) = nre of the layout
__host__ __device__ constexpr int ke_of(int pp) { return pp < 2 ? 2 : 2 * ((pp * (pp + 1) / 2 + 7) / 8); }
constexpr int TILES_ALL = 0, TILES_SPLIT = 1, TILES_DENSE = 2;
struct Stage {
    int64_t npairs = 0;
    int64_t scratch_off = 0;        // order of the regions: pairs of the stages before this one (M2M / L2L stages alias region 0)
    // packed scratch rows (translate.cu pack_scratch), per truncation layout: the row of pair k (target-major) holds the
    // 2 W dofs its matrix class computes (W real parts, then W imaginary parts) at row_off[k] units of 16 doubles from the
    // start of the stage's region, which starts region_units units into the scratch buffer
    dvec<int32_t> row_off[2];       // [npairs + 1] by target-major pair index k (the row sums)
    dvec<int32_t> orow[2];          // [npairs] the same offsets by tile row r: orow[r] = row_off[krow[r]] (the tile kernels: one load, not two)
    dvec<uint8_t> tile_cls[2];      // [ntiles] truncation class of every tile's matrix (loaded beside the tile, not after it)
    std::vector<int32_t> tile_mat_host;
    int64_t region_units[2] = {0, 0};
    int ntgt = 0;
    int out_base = 0;               // global index of the first target box
    bool out_is_local = false;      // output array: local (L) or multipole (M) expansions
    bool accumulate = false;        // the reduce pass adds to the output instead of overwriting it (L2L)
    bool keep_empty = false;        // the reduce pass leaves the output of a target with no pair alone (adaptive M2M: leaves)
    dvec<int32_t> src_sorted;       // [npairs] global input box of scratch row r (matrix-sorted order)
    dvec<int32_t> krow;             // [npairs] target-major index k of the pair in tile row r: its scratch row (the rows of a target are
                                    // contiguous in scratch, so the row sums stream them; the tiles scatter whole 8 nst-byte rows)
    dvec<int32_t> mat_t;            // [npairs] matrix id of pair k (target-major order): the reduce pass rotates back by its azimuth
    dvec<int32_t> ptr;              // [ntgt+1] CSR of pairs per target (target-major)
    dvec<int32_t> tgt_list;         // adaptive tree: the targets the reduce pass visits (existing boxes; M2M: subdivided parents)
    int n_list = -1;                // -1: every target
    dvec<Tile> tiles;
    int ntiles = 0;
    int ntiles_split = 0;           // the first ntiles_split tiles are M2L tiles (matrix ids < MAT_L2L come first)
};

// Adaptive octree (option "tree" = 1, adaptive.cu): flags and tables on top of the two BoxSets
struct Adaptive {
    dvec<uint8_t> s_ex[MAX_LEVEL + 1], s_sub[MAX_LEVEL + 1];   // source boxes of a level: exists (parent subdivided), subdivided
    dvec<uint8_t> t_ex[MAX_LEVEL + 1], t_sub[MAX_LEVEL + 1];   // target boxes
    dvec<int32_t> s_pbeg[MAX_LEVEL + 1], t_pbeg[MAX_LEVEL + 1]; // [nbox + 1] first point of every box of a level
    dvec<int32_t> sleaf[MAX_LEVEL + 1];                         // source leaves of a level (box indices): P2M
    int n_sleaf[MAX_LEVEL + 1] = {0};
    int lmin = 2;                                                 // boxes above this level are always subdivided
    int n_src_leaves = 0;
    dvec<uint64_t> tkey_all;                                    // [target boxes] key and level by global box id: L2P
    dvec<uint8_t> tlev_all;
    dvec<int32_t> pt_gbox;                                      // [N] global box id of the leaf of every target point
    dvec<int32_t> tleaf_begin, tleaf_gbox;                      // target leaves in point order: first point, global box id
    int n_tleaf = 0;
    dvec<int32_t> near_ptr;                                     // [n_tleaf + 1] CSR of the direct source ranges of a target leaf
    dvec<int2> near_rng;                                        // (first source, count)
    dvec<int32_t> x_ptr[MAX_LEVEL + 1], x_src[MAX_LEVEL + 1];   // far pairs of two sparse leaves, summed directly (per level)
    bool row_overflow = false;                                  // the last build met a target leaf with more than SEG_MAX direct ranges
};

// Everything bem_setup builds that depends on the truncation number.  A context holds one layout for the products without
// dipoles (truncation p) and, when option "dipole_degrees" asks for it, a second one for the products with dipoles
// (truncation p + dipole degrees); bem_apply makes one of them the active layout (api.cu activate_layout).
struct FmmLayout {
    int p = 0, pl = 0, nre = 0, nst = 0;
    dvec<double> mats;              // [N_MATS * nst * nst] real translation matrices, row = input dof k, col = output dof
    dvec<double2> rot;              // [N_MATS * ROT_M] (cos m a, sin m a): azimuth a of the M2L offset, identity for M2M / L2L
    dvec<int32_t> kinfo;            // [nst] order m of every stored dof (0 for padding)
    dvec<int32_t> mat_ne;           // [N_MATS] leading dofs of either block that take part in the translation (graded truncation)
    dvec<int32_t> mat_cls;          // [N_MATS] truncation class of the M2L tiles of the matrix: min(M2L_NCLS - 1, pl - p_o)
    dvec<int32_t> mat_w;            // [N_MATS] dofs of either block a translated row of the matrix stores: 4 ke_of(pl - class) (M2M / L2L: nre)
    std::vector<int32_t> mat_w_host;
    std::vector<int32_t> mat_ne_host, mat_cls_host;
    double m2l_flop = 0;            // executed flop of the M2L tiles of one product: 4 (4 KE)^2 per pair, KE the k-steps of its class
    double m2l_row_bytes = 0;       // bytes of translated rows the sums read per product: 16 x dofs carried per pair
};

}  // namespace bem

// ---------------------------------------------------------------- the context
struct bem_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;

    // mesh (device)
    int64_t N = 0, T = 0;
    int nbubbles = 1;
    bem::dvec<double> V;            // [N*3]
    bem::dvec<int32_t> F;           // [T*3]
    bem::dvec<int32_t> bid;         // [N]
    bem::dvec<double> P;            // point-cloud mode (quadrature == 2): [np*3] source points; V holds the targets
    int64_t np = 0;
    bem_ctx *parent = nullptr;      // evaluator (quadrature == 3, bem_create_evaluator): the mesh context whose Gauss points are the
                                    // sources; V holds the evaluation points (N of them), densities are indexed by the parent's vertices
                                    // Only bem_setup follows this pointer (the mesh may be destroyed after the last set-up):
    int64_t mesh_N = 0, mesh_T = 0; // evaluator: vertex and triangle counts of the parent's mesh, copied at creation (what bem_apply needs)

    // vertex -> incident triangle corners, sorted by vertex (bem_surface_velocity; built at first use)
    bem::dvec<int32_t> vc_begin;    // [N+1]
    bem::dvec<uint32_t> vc_corner;  // [3T] corner index 3 k + a, in mesh order within a vertex
    // triangles grouped by bubble (bem_bubble_volume; built at first use)
    bem::dvec<int32_t> bv_begin;    // [nbubbles+1]
    bem::dvec<uint32_t> bv_tri;     // [T] triangle indices, mesh order within a bubble

    // options
    // quadrature: 0 = G3, 1 = V1, 2 = point cloud (bem_create_points), 3 = evaluator of a mesh context off its surface
    int quadrature = 0, mode = 0, free_term = 0, gmres_restart = 0, force_lmax = 0, timing = 0;
    int precond = 0;                // bem_solve: 0 = unpreconditioned (the paper), 1 = right diagonal scaling by S_ii
    int overlap = 0;                // option "overlap": 1 = the row sums of the M2L stages run on a side stream beside the near field, 0 = one stream (default: measured faster since round 2)
    int reduce_stream = 1;          // option "reduce_stream": 1 = the row sums stream the packed rows through shared memory (cp.async), 0 = direct loads
    int reduce_ctas = 0;            // option "reduce_ctas": CTAs per SM of the persistent side-stream sums, 0 = from the cost model
    int n_sm = 148;
    int m2l_rows16 = 1;             // M2L tiles: 1 = 4 warps x 16 rows (B fragments feed two DMMAs), 0 = 8 warps x 8 rows
    int gemm_path = 0;              // translations: 0 = FP64 tensor path (DMMA) where p <= 16, 1 = plain-FMA tiles
    int p2p_exact = 0;              // option "p2p_exact": 1 = the FMM near field refines 1/r to the last bit as direct mode does (17 FP64 instr per pair)
    int p2p_precision = 0;          // near field: 0 = fp64 pairs (default), 1 = fp32 pair arithmetic, fp64 accumulation (p2p_f32.cu)
    int p2p_ctas = 0;               // fp32 near field: CTAs per SM of its persistent grid beside the row sums, 0 = default (4)

    // setup state
    bool ready = false;
    bem::FmmLayout lay[2];          // [0] truncation p_user (products without dipoles), [1] p_user + dipole degrees (if any)
    int n_lay = 1, lay_active = 0;
    int p_user = 0;                 // the p of bem_setup
    int dipole_degrees = -1;        // option "dipole_degrees": -1 = 3 for p < 12 and 0 above (measured, R5'), else the value
    // the ACTIVE layout (copied from lay[lay_active] by activate_layout)
    int p = 0, nst = 0;             // truncation number, expansion row stride (harmonics.cuh: nre + nim)
    int pl = 0, nre = 0;            // layout degree count (kernel template bucket >= p), size of the real-part block
    int leaf_size = 0;
    double eta = 0;
    double cube_min[3] = {0, 0, 0}, cube_side = 1.0;

    // geometry (a0)
    bem::dvec<double> triA;         // [T]
    bem::dvec<double> triN;         // [T*3]

    // sources in engine order (Morton-sorted in FMM mode, natural in direct mode)
    int64_t ns = 0;
    bem::dvec<double4> src_pos;     // [ns] (x, y, z, 0)
    bem::dvec<double4> lift_w;      // [ns] (w, w Nx, w Ny, w Nz)
    bem::dvec<int4> lift_vid;       // [ns] (v0, v1, v2, -) densities are 2/3 f[v0] + 1/6 f[v1] + 1/6 f[v2]
    bem::dvec<double4> src_str;     // [ns] (m, dx, dy, dz), rewritten by every apply
    bool has_dipole = true;         // false while phi == NULL: dipole strengths are all zero
    // targets in engine order
    bem::dvec<double> tgt_pos;      // [N*3]
    bem::dvec<uint32_t> tgt_inv;    // [N] original vertex -> engine position (FMM mode)

    // octree + lists (FMM mode)
    bem::BoxSet sb, tb;
    int tree_min_level = 0;         // option "tree_min_level": 0 = the depth of the uniform rule, else the level (>= 2)
    int adaptive = 0;               // option "tree": 0 = uniform depth (the paper's), 1 = adaptive (adaptive.cu)
    bem::Adaptive ad;
    bem::dvec<int32_t> nbr;         // [n_tgt_leaves * 27] source leaves adjacent to a target leaf, -1 padded
    bem::dvec<int32_t> xdir_ptr;    // [n_tgt_leaves + 1] CSR of the leaf-level far pairs that are summed directly (option direct_pairs)
    bem::dvec<int32_t> xdir_src;    // [xdir_pairs] their source leaves
    int64_t xdir_pairs = 0;
    int64_t direct_max = -1;        // option "direct_pairs": nt x ns threshold, -1 = from the cost model, 0 = off
    int64_t direct_max_eff = 0;
    int seg_limit = 256;            // option "max_direct_ranges": longest row of direct source ranges a target leaf of the adaptive tree may
                                    // have (<= SEG_MAX of segments.cuh, the pair kernel's segment table)
    bem::dptr<double> mats;         // views of the active layout (FmmLayout)
    bem::dptr<double2> rot;
    bem::dptr<int32_t> kinfo, mat_ne, mat_cls, mat_w;
    double m2l_hist[bem::MAT_L2L] = {0};   // M2L pairs per matrix over all levels (statistics of the layouts)
    double m2l_order_radius = 0.5;  // option "m2l_order_radius": cluster radius a (box edges) of the graded truncation, 0 = off
    int m2l_order_extra = 1;        // option "m2l_order_extra": degrees added to the graded order of every offset
    double m2l_row_bytes = 0;       // of the active layout
    bem::dvec<double> Mexp, Lexp;   // [total boxes * nst]
    bem::dvec<double> scratch;      // [pairs of all M2L (+ L2L) stages * nst]: one region per level, so that the tiles of all
                                    // levels can be issued before the first reduce pass
    cudaStream_t side = nullptr;    // high-priority stream: reduce passes + L2P run here while P2P runs on `stream`
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    bem::dvec<int> p2p_counter;     // leaf counters of the persistent grids (fp32 pair kernel, P2M)
    bem::dvec<float4> src_pos_f;    // [ns] fp32 near field: position relative to the own leaf centre, in leaf edges (built at first use)
    bem::dvec<float4> src_str_f;    // [ns] fp32 near field: (m/h, d/h^2), rewritten by every apply
    std::vector<bem::Stage> m2m;    // leaf-1 .. 2
    std::vector<bem::Stage> m2l;    // 2 .. lmax: L_own(l) = sum of the M2L rows of the level
    std::vector<bem::Stage> l2l;    // 3 .. lmax: L(l) = L_own(l) + L2L L(l-1)
    int64_t m2l_pairs = 0, p2p_pairs = 0;
    int64_t p2p_pairs_wx = 0;       // adaptive tree: the part of p2p_pairs that comes from W-list and X-list ranges (summed directly here)
    int64_t p2p_pairs_exec = 0;     // pairs the near-field kernel executes: source lists padded to rounds of 128 (tree.cu)

    // partial sums of the point engine, combined by the SpMV kernel
    bem::dvec<double> ypart;        // [nsplit * N]  (FMM mode: slot 0 = far field (L2P), slot 1 = near field (P2P))
    int nsplit = 1;

    // near-field correction (a3) / V1 diagonal (a3')
    bem::dvec<int64_t> rowptr;      // [N+1]
    bem::dvec<int32_t> col;         // [nnz]
    bem::dvec<double2> val;         // [nnz] (C^S, C^D)
    int64_t nnz = 0, near_tris = 0;
    bem::dvec<double> diagL, diagM; // V1 only
    bem::dvec<double> diagS;        // G3: S_ii (exact), the diagonal preconditioner of bem_solve (option "precond")
    bool have_diag = false;

    bem::dvec<double> cfree;        // [N] free term c_i of bem_solve
    bool have_cfree = false;

    // CUDA graphs of bem_apply with device pointers (option "graph"): a product with the same (q, phi, y, stream) is
    // captured the second time it is asked for and replayed from then on (the launch-bound small meshes: 20-40 launches of
    // a few microseconds each); any bem_set_option / bem_setup / bem_set_stream drops the cache
    struct GraphEntry { const double *q, *phi; double *y; cudaStream_t stream; int seen; cudaGraphExec_t exec; };
    std::vector<GraphEntry> graphs;
    int use_graph = 1;

    // staging for host-pointer arguments
    bem::dvec<double> stage_q, stage_phi, stage_y;

    // timings: event k closes an interval that belongs to kernel class ev_cls[k] (-1: start)
    std::vector<cudaEvent_t> ev;
    std::vector<int> ev_cls;
    int ev_n = 0;
    bool ev_valid = false;
    double setup_ms = 0;
    int launches_per_apply = 0;
};
