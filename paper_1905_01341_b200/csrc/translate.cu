// Steps a5-a9: P2M, M2M, M2L, L2L, L2P on box-scaled real
// solid-harmonic expansions ("multipole and local expansions
// ... spherical harmonics ... truncated to the first p_fmm degrees"; the
// translations are "dense" p^2 x p^2 operators here, batched as GEMMs).
//
// Every translation of one kind and one relative position uses the SAME real
// p^2 x p^2 matrix on every level (box-scaled coefficients, harmonics.cuh), so
// a stage is:  rows of input expansions gathered by pair, sorted by matrix ->
// tiles of a dense fp64 GEMM (matrix staged in shared memory, reused by 64
// pairs) -> one scratch row per pair -> per-target sums of its rows in a fixed
// order (no atomics; results are bit-reproducible).
#include "common.cuh"
#include "harmonics.cuh"
#include "morton.cuh"

#include <cmath>
#include <mutex>

namespace bem {

// ------------------------------------------------------------------ matrices (setup)
__host__ __device__ inline int tab_len(int deg_excl) { return deg_excl * (deg_excl + 1) / 2; }

// one thread per matrix: its harmonic table.  An M2L offset (ox, oy, oz) is first turned about the z axis
// into the xz-plane, T' = (sqrt(ox^2 + oy^2), 0, oz): there every I_n^m(T') is REAL, so the real p^2 x p^2
// matrix splits into a (real parts -> real parts) and an (imaginary -> imaginary) block -- half the flops.
// The azimuth is applied to the coefficients instead: Mt'_j^k = e^{ik a} Mt_j^k going in (gather of the tile
// kernels) and Lt_l^m = e^{im a} Lt'_l^m coming out (reduce pass), a = atan2(oy, ox).
__global__ void harmonic_tables(int p, double *tab_re, double *tab_im, int stride)
{
    const int m = blockIdx.x * blockDim.x + threadIdx.x;
    if (m >= N_MATS) return;
    double *re = tab_re + (size_t)m * stride, *im = tab_im + (size_t)m * stride;
    if (m < MAT_L2L) {
        const int ox = m % 7 - 3, oy = (m / 7) % 7 - 3, oz = m / 49 - 3;
        if (max(max(abs(ox), abs(oy)), abs(oz)) < 2) return;          // adjacent offsets are never used
        eval_I(sqrt((double)(ox * ox + oy * oy)), 0.0, (double)oz, 2 * p - 1, re, im);
    } else {
        const int o = (m - MAT_L2L) & 7;                               // child octant: bit set -> +1/2
        eval_R((o & 1) ? 0.5 : -0.5, (o & 2) ? 0.5 : -0.5, (o & 4) ? 0.5 : -0.5, p, re, im);
    }
}
// mats[m][k][c] = T_m[c][k]  (row = input dof, column = output dof); padding dofs and degrees >= p are zero
__global__ void fill_matrices(int p, int nre, int nst, const double *tab_re, const double *tab_im, int stride, const int32_t *mat_ne, double *mats)
{
    const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t per = (int64_t)nst * nst;
    if (idx >= per * N_MATS) return;
    const int m = (int)(idx / per);
    const int k = (int)((idx % per) / nst), cc = (int)(idx % nst);
    double v = 0.0;
    const double *re = tab_re + (size_t)m * stride, *im = tab_im + (size_t)m * stride;
    if (m < MAT_L2L) {
        const int ox = m % 7 - 3, oy = (m / 7) % 7 - 3, oz = m / 49 - 3;
        // graded truncation: only the leading mat_ne[m] dofs of either part take part (build_matrices)
        const int ne = mat_ne[m];
        if (max(max(abs(ox), abs(oy)), abs(oz)) >= 2 && ((k < nre) == (cc < nre)) && (k < nre ? k : k - nre) < ne && (cc < nre ? cc : cc - nre) < ne)
            v = m2l_entry(re, im, p, nre, cc, k);
    } else if (m < MAT_M2M) v = l2l_entry(re, im, p, nre, cc, k);
    else v = m2m_entry(re, im, p, nre, cc, k);
    mats[idx] = v;
}

void build_matrices(bem_ctx *c, FmmLayout &L)
{
    const int p = L.p, nst = L.nst;
    const int stride = tab_len(2 * p - 1);
    dvec<double> tre, tim;
    tre.alloc((size_t)N_MATS * stride);
    tim.alloc((size_t)N_MATS * stride);
    tre.zero(c->stream);
    tim.zero(c->stream);
    harmonic_tables<<<cdiv(N_MATS, 64), 64, 0, c->stream>>>(p, tre.get(), tim.get(), stride);
    KERNEL_CHECK();
    // Graded truncation of the M2L translations by separation (option "m2l_order_radius" = a > 0, in box edges).  The
    // truncation error of a translation over the offset o falls like kappa(o)^p, kappa = a / (|o| - a) for clusters of
    // radius a; the nearest offsets (|o| = 2) set the error of the product, and an offset further away reaches the same
    // error with p_o = ceil(p ln kappa(2) / ln kappa(|o|)) + extra degrees (option "m2l_order_extra").  Only the leading
    // mat_ne[m] = p_o (p_o + 1) / 2 dofs of the real-part block (= of the imaginary-part block) of matrix m are non-zero,
    // and the M2L tile kernels run the k-steps and n-tiles of class min(M2L_NCLS - 1, pl - p_o) only.  a = 0: p_o = p.
    std::vector<int32_t> ne(N_MATS, L.nre), cls(N_MATS, 0);
    for (int m = 0; m < MAT_L2L; ++m) {
        const int ox = m % 7 - 3, oy = (m / 7) % 7 - 3, oz = m / 49 - 3;
        int po = p;
        if (c->m2l_order_radius > 0 && std::max(std::max(std::abs(ox), std::abs(oy)), std::abs(oz)) >= 2) {
            const double a = c->m2l_order_radius, d = std::sqrt((double)(ox * ox + oy * oy + oz * oz));
            const double k2 = a / (2.0 - a), kd = a / (d - a);
            po = (int)std::ceil(p * std::log(k2) / std::log(kd) - 1e-9) + c->m2l_order_extra;
            po = std::max(std::min(po, p), std::min(p, 2));
        }
        ne[m] = std::min(L.nre, po * (po + 1) / 2);
        cls[m] = std::max(0, std::min(M2L_NCLS - 1, L.pl - po));
    }
    L.mat_ne_host = ne;
    L.mat_cls_host = cls;
    std::vector<int32_t> mw(N_MATS, L.nre);                          // dofs per block a translated row stores (a multiple of 8)
    for (int m = 0; m < MAT_L2L; ++m) mw[m] = std::min(L.nre, 4 * ke_of(L.pl - cls[m]));
    L.mat_w_host = mw;
    L.mat_w.alloc(N_MATS);
    CUDA_TRY(cudaMemcpyAsync(L.mat_w.get(), mw.data(), N_MATS * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
    L.mat_ne.alloc(N_MATS);
    L.mat_cls.alloc(N_MATS);
    CUDA_TRY(cudaMemcpyAsync(L.mat_ne.get(), ne.data(), N_MATS * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaMemcpyAsync(L.mat_cls.get(), cls.data(), N_MATS * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
    const int64_t tot = (int64_t)N_MATS * nst * nst;
    L.mats.alloc(tot);
    fill_matrices<<<cdiv(tot, 256), 256, 0, c->stream>>>(p, L.nre, nst, tre.get(), tim.get(), stride, L.mat_ne.get(), L.mats.get());
    KERNEL_CHECK();
    // azimuth table (cos m a, sin m a) and the per-dof table (m, partner = the other part of the same (l, m), part)
    std::vector<double2> rot((size_t)N_MATS * ROT_M);
    for (int m = 0; m < N_MATS; ++m) {
        double a = 0.0;
        if (m < MAT_L2L) {
            const int ox = m % 7 - 3, oy = (m / 7) % 7 - 3;
            if (ox != 0 || oy != 0) a = atan2((double)oy, (double)ox);
        }
        for (int k = 0; k < ROT_M; ++k) rot[(size_t)m * ROT_M + k] = make_double2(cos(k * a), sin(k * a));
    }
    L.rot.alloc(rot.size());
    CUDA_TRY(cudaMemcpyAsync(L.rot.get(), rot.data(), rot.size() * sizeof(double2), cudaMemcpyHostToDevice, c->stream));
    std::vector<int32_t> kin(nst);
    for (int k = 0; k < nst; ++k) {
        int l, m, part;
        kin[k] = real_decode(k, L.pl, L.nre, &l, &m, &part) ? m : 0;
    }
    L.kinfo.alloc(nst);
    CUDA_TRY(cudaMemcpyAsync(L.kinfo.get(), kin.data(), nst * sizeof(int32_t), cudaMemcpyHostToDevice, c->stream));
    CUDA_TRY(cudaStreamSynchronize(c->stream));
}

// e^{i m a} applied to one coefficient (re, im) in place:  Re' = cos Re - sin Im,  Im' = cos Im + sin Re
__device__ __forceinline__ void azimuth(double2 cs, double &re, double &im)
{
    const double r = fma(cs.x, re, -cs.y * im);
    im = fma(cs.x, im, cs.y * re);
    re = r;
}

// ------------------------------------------------------------------ batched GEMM (a6, a7, a8)
// scratch[row0 + r][:] = in[src_sorted[row0 + r]][:] * mats[tile.mat]   for r < tile.nrows
// (M2L tiles: the input row is first turned by the azimuth of the offset, see harmonic_tables)
// Plain-FMA version (any p; the fallback for p > 16 and option gemm_path = 1).
// CTA: 64 rows x 64 columns, K in chunks of 8; thread: 4 rows x 4 columns (columns strided by 16).
constexpr int GEMM_TM = 64, GEMM_TN = 64, GEMM_KC = 8, GEMM_THREADS = 256;

__global__ void __launch_bounds__(GEMM_THREADS)
translate_gemm(const Tile *__restrict__ tiles, const int32_t *__restrict__ src_sorted,
               const double *__restrict__ Mexp, const double *__restrict__ Lexp,
               const double *__restrict__ mats, const int32_t *__restrict__ kinfo, const double2 *__restrict__ rot,
               int nst, const int32_t *__restrict__ orow_t, const int32_t *__restrict__ mat_w,
               double *__restrict__ scratch)
{
    __shared__ double As[GEMM_KC][GEMM_TM + 4];
    __shared__ double Bs[GEMM_KC][GEMM_TN];
    __shared__ int rows[GEMM_TM];
    const Tile tile = tiles[blockIdx.x];
    const int n0 = blockIdx.y * GEMM_TN;
    const double *in = (tile.flags & 1) ? Lexp : Mexp;
    const bool split = (tile.flags & 2) != 0;
    const double *B = mats + (size_t)tile.mat * nst * nst;
    const double2 *rcs = rot + (size_t)tile.mat * ROT_M;
    if (threadIdx.x < GEMM_TM) rows[threadIdx.x] = threadIdx.x < tile.nrows ? src_sorted[tile.row0 + threadIdx.x] : -1;
    __syncthreads();
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    double acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = 0.0;
    // loaders: A: thread -> (row = tid/4, two k's), B: thread -> (k = tid/32, two columns)
    const int ar = threadIdx.x >> 2, ak = (threadIdx.x & 3) * 2;
    const int bk = threadIdx.x >> 5, bc = (threadIdx.x & 31) * 2;
    const int arow = rows[ar];
    for (int k0 = 0; k0 < nst; k0 += GEMM_KC) {
        double2 av = make_double2(0.0, 0.0), bv = make_double2(0.0, 0.0);
        if (arow >= 0) {
            const double *ap = in + (size_t)arow * nst;
            av = *reinterpret_cast<const double2 *>(ap + k0 + ak);
            if (split) {                                        // partner = the other part of the same (l, m), nre away
                const int nre = nst >> 1, k = k0 + ak;
                const bool im = k >= nre;
                const double2 w = *reinterpret_cast<const double2 *>(ap + (im ? k - nre : k + nre));
                const double2 c0 = rcs[kinfo[k]], c1 = rcs[kinfo[k + 1]];
                double re0 = im ? w.x : av.x, im0 = im ? av.x : w.x, re1 = im ? w.y : av.y, im1 = im ? av.y : w.y;
                azimuth(c0, re0, im0);
                azimuth(c1, re1, im1);
                av.x = im ? im0 : re0;
                av.y = im ? im1 : re1;
            }
        }
        if (n0 + bc < nst) bv = *reinterpret_cast<const double2 *>(B + (size_t)(k0 + bk) * nst + n0 + bc);
        __syncthreads();
        As[ak][ar] = av.x; As[ak + 1][ar] = av.y;
        Bs[bk][bc] = bv.x; Bs[bk][bc + 1] = bv.y;
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < GEMM_KC; ++kk) {
            double a[4], b[4];
#pragma unroll
            for (int i = 0; i < 4; ++i) a[i] = As[kk][ty * 4 + i];
#pragma unroll
            for (int j = 0; j < 4; ++j) b[j] = Bs[kk][tx + 16 * j];
#pragma unroll
            for (int i = 0; i < 4; ++i)
#pragma unroll
                for (int j = 0; j < 4; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const int r = ty * 4 + i;
        if (r >= tile.nrows) continue;
        // packed row: the W leading dofs of the real parts, then of the imaginary parts (W = nre for M2M / L2L)
        double *out = scratch + (size_t)orow_t[tile.row0 + r] * 16;
        const int W = mat_w[tile.mat], nre = nst >> 1;
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const int col = n0 + tx + 16 * j;
            if (col < nst) {
                const int part = col >= nre, cc = col - part * nre;
                if (cc < W) out[part * W + cc] = acc[i][j];
            }
        }
    }
}

// ------------------------------------------------------------------ the same product on the FP64 tensor path
// Measured on B200 (profiles/): mma.sync m8n8k4 f64 (SASS DMMA) sustains 37.15 TFLOP/s, a register-resident
// DFMA loop 33.9; more important, one DMMA needs ONE 8-byte shared-memory operand per thread for 512 flop per
// warp, so the GEMM is no longer bound by shared-memory operand traffic.
//
// CTA = 8 warps = 64 scratch rows (pairs) of one matrix.  Each warp owns 8 rows and keeps their whole A
// operand (8 x nst input coefficients, gathered straight from global memory and, for M2L, turned by the
// azimuth of the offset in registers: the two parts of a coefficient sit in a[s] and a[s + KSH] of the same
// lane) as 2 KSH m8n8k4 A-fragments; the matrix streams through shared memory in chunks of up to DM_NT
// n-tiles (cp.async, double buffered), shared by the 8 warps.
// KSH = k-steps (4 dofs each) of the real-part block = of the imaginary-part block.  An M2L matrix is block
// diagonal in that split: its real-part columns only take the real-part k-steps and its imaginary-part
// columns the others -- KSH^2 DMMA per warp instead of 2 KSH^2.
// M2M / L2L matrices (8 + 8 of them, a few % of the work) are dense and take all k-steps.
constexpr int DM_NT = 5;             // n-tiles (8 columns of B) per chunk = independent accumulator chains per warp
constexpr int DM_S = 46;             // row stride of a chunk in doubles: 2 x 46 = 12 (mod 16) -> conflict-free fragment loads
constexpr int DM_NT_DENSE = 2;       // dense (M2M / L2L) tiles: twice the rows, so narrower chunks with row stride
constexpr int DM_S_DENSE = 22;       // 2 x 22 = 12 (mod 16); 2 nre x 22 doubles fit the nre x 46 buffer of the split tiles
constexpr int DM_THREADS = 256;

__device__ __forceinline__ void cp_async16(void *smem, const void *gmem)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gmem));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N)); }

__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                 : "+d"(c0), "+d"(c1)
                 : "d"(a), "d"(b));
}

// one chunk of NT n-tiles over the k-steps [KB, KE): cur = chunk buffer, whose row 0 is dof 4 KR
template <int KS, int KB, int KE, int KR, int NT, int S>
__device__ __forceinline__ void dm_chunk_nt(const double (&a)[KS], const double *cur, int lr, int lk, bool rvalid, double *orow_c0)
{
    const double *bp = cur + 2 * lk * S + lr;          // dof of fragment position (s, lk): 8 (s / 2) + 2 lk + (s & 1)
    double c[NT][2];
#pragma unroll
    for (int j = 0; j < NT; ++j) c[j][0] = c[j][1] = 0.0;
#pragma unroll
    for (int s = KB; s < KE; ++s) {
        const double *b = bp + (8 * ((s - KR) >> 1) + ((s - KR) & 1)) * S;
#pragma unroll
        for (int j = 0; j < NT; ++j) dmma884(c[j][0], c[j][1], a[s], b[8 * j]);
    }
    if (rvalid) {
#pragma unroll
        for (int j = 0; j < NT; ++j) *reinterpret_cast<double2 *>(orow_c0 + 8 * j) = make_double2(c[j][0], c[j][1]);
    }
}
template <int KS, int KB, int KE, int KR>
__device__ __forceinline__ void dm_chunk(const double (&a)[KS], const double *cur, int nt, int lr, int lk,
                                         bool rvalid, double *orow_c0)
{
    switch (nt) {                                               // warp-uniform
    case 5: dm_chunk_nt<KS, KB, KE, KR, 5, DM_S>(a, cur, lr, lk, rvalid, orow_c0); break;
    case 4: dm_chunk_nt<KS, KB, KE, KR, 4, DM_S>(a, cur, lr, lk, rvalid, orow_c0); break;
    case 3: dm_chunk_nt<KS, KB, KE, KR, 3, DM_S>(a, cur, lr, lk, rvalid, orow_c0); break;
    case 2: dm_chunk_nt<KS, KB, KE, KR, 2, DM_S>(a, cur, lr, lk, rvalid, orow_c0); break;
    default: dm_chunk_nt<KS, KB, KE, KR, 1, DM_S>(a, cur, lr, lk, rvalid, orow_c0); break;
    }
}
template <int KS>
__device__ __forceinline__ void dm_chunk_dense(const double (&a)[KS], const double *cur, int nt, int lr, int lk,
                                               bool rvalid, double *orow_c0)
{
    if (nt == 2) dm_chunk_nt<KS, 0, KS, 0, 2, DM_S_DENSE>(a, cur, lr, lk, rvalid, orow_c0);
    else dm_chunk_nt<KS, 0, KS, 0, 1, DM_S_DENSE>(a, cur, lr, lk, rvalid, orow_c0);
}

template <int KSH>
__global__ void __launch_bounds__(DM_THREADS)
translate_dmma(const Tile *__restrict__ tiles, const int32_t *__restrict__ src_sorted,
               const double *__restrict__ Mexp, const double *__restrict__ Lexp,
               const double *__restrict__ mats, const int32_t *__restrict__ kinfo, const double2 *__restrict__ rot,
               const int32_t *__restrict__ orow_t, double *__restrict__ scratch)
{
    extern __shared__ __align__(16) double dm_smem[];          // [2][NRE][DM_S] (dense tiles: [2][2 NRE][DM_S_DENSE])
    __shared__ double2 cs_k[4 * KSH];                          // (cos, sin)(m_k a) of every real-part dof k
    constexpr int KS = 2 * KSH, NRE = 4 * KSH, NST = 4 * KS;
    constexpr int NTH = KSH / 2;                               // n-tiles (8 columns) of one block
    const Tile tile = tiles[blockIdx.x];
    const double *in = (tile.flags & 1) ? Lexp : Mexp;
    const bool split = (tile.flags & 2) != 0;
    const int brows = split ? NRE : NST;                       // rows of B a chunk needs
    double *Bs0 = dm_smem, *Bs1 = dm_smem + NRE * DM_S;
    const int bstride = split ? DM_S : DM_S_DENSE;
    const double *B = mats + (size_t)tile.mat * NST * NST;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int lr = lane >> 2, lk = lane & 3;                   // fragment row / k (A), n / k (B)
    const int row = warp * 8 + lr;
    const bool rvalid = row < tile.nrows;

    // chunks of balanced width: per block of ntb n-tiles, ceil(ntb / DM_NT) chunks
    const int ntb = split ? NTH : 2 * NTH;                      // n-tiles per block (dense: one block = everything)
    const int wmax = split ? DM_NT : DM_NT_DENSE;
    const int cpb = (ntb + wmax - 1) / wmax;                    // chunks per block
    const int cw = (ntb + cpb - 1) / cpb;                       // chunk width in n-tiles
    const int nchunks = split ? 2 * cpb : cpb;
    auto chunk = [&](int ch, int &blk, int &t0, int &nt) {
        blk = ch >= cpb;
        const int cl = blk ? ch - cpb : ch;
        t0 = blk * NTH + cw * cl;
        nt = min(cw, blk * NTH + ntb - t0);
    };
    auto issue = [&](int ch, double *dst) {
        int blk, t0, nt;
        chunk(ch, blk, t0, nt);
        const int c0 = 8 * t0, per_row = 4 * nt;                // 16-byte pieces per row
        const int k0 = blk ? NRE : 0;                           // the block's own rows (dense: all rows)
        for (int i = threadIdx.x; i < brows * per_row; i += DM_THREADS) {
            const int k = i / per_row, j = (i % per_row) * 2;
            cp_async16(dst + k * bstride + j, B + (size_t)(k0 + k) * NST + c0 + j);
        }
        cp_async_commit();
    };
    issue(0, Bs0);
    if (split) {
        for (int k = threadIdx.x; k < NRE; k += DM_THREADS) cs_k[k] = __ldg(rot + (size_t)tile.mat * ROT_M + __ldg(kinfo + k));
    }

    // A operand -> registers.  K is permuted so that the fragments of the k-steps 2j and 2j+1 of a lane are the
    // two ADJACENT dofs 8j + 2 lk and 8j + 2 lk + 1: one 16-byte load per pair of k-steps.
    double a[KS];
    {
        const int arow = rvalid ? src_sorted[tile.row0 + row] : -1;
        const double2 *ap = reinterpret_cast<const double2 *>(in + (size_t)(arow < 0 ? 0 : arow) * NST) + lk;
#pragma unroll
        for (int j = 0; j < KS / 2; ++j) {
            const double2 v = arow >= 0 ? ap[4 * j] : make_double2(0.0, 0.0);
            a[2 * j] = v.x;
            a[2 * j + 1] = v.y;
        }
    }
    double *orow = scratch + (size_t)(rvalid ? orow_t[tile.row0 + row] : 0) * 16 + 2 * lk;     // dense rows are full rows

    for (int ch = 0; ch < nchunks; ++ch) {
        double *cur = (ch & 1) ? Bs1 : Bs0;
        cp_async_wait<0>();
        __syncthreads();                                        // chunk ch landed; everyone left chunk ch-1; cs_k visible
        if (ch == 0 && split) {
#pragma unroll
            for (int s = 0; s < KSH; ++s) azimuth(cs_k[8 * (s >> 1) + 2 * lk + (s & 1)], a[s], a[s + KSH]);
        }
        if (ch + 1 < nchunks) issue(ch + 1, (ch & 1) ? Bs0 : Bs1);
        int blk, t0, nt;
        chunk(ch, blk, t0, nt);
        // chunk buffers hold the block's rows from row 0: the imaginary block reads its k-steps KSH.. at rows 0..
        if (!split) dm_chunk_dense<KS>(a, cur, nt, lr, lk, rvalid, orow + 8 * t0);
        else if (blk == 0) dm_chunk<KS, 0, KSH, 0>(a, cur, nt, lr, lk, rvalid, orow + 8 * t0);
        else dm_chunk<KS, KSH, KS, KSH>(a, cur, nt, lr, lk, rvalid, orow + 8 * t0);
    }
}

// M2L tiles only (block-diagonal matrix): the lean version of the kernel above.  A warp holds ONE half of its
// A operand at a time -- the rotated real parts while it runs the real-part columns, then (rows gathered again,
// L2 hits) the rotated imaginary parts for the imaginary-part columns: 2 KSH instead of 4 KSH registers for A,
// so three CTAs (24 warps) fit an SM instead of two and the row gather of one CTA hides behind the DMMAs of the
// others (ncu on the two-CTA version: tensor pipe 65% active, 30% of the samples in the gather prologue).
//
// Graded truncation (build_matrices): a tile of class i runs only the KE = ke_of(PL - i) k-steps and KE / 2 n-tiles
// of either block that hold the degrees < PL - i; KSH = ke_of(PL) is the layout (row stride, place of the imaginary
// parts).  Every class is its own fully unrolled body (the k-loop must stay free of branches: the B fragments of the
// next k-steps are loaded while the DMMAs of this one run), selected per tile by a CTA-uniform switch.
template <int KSH, int KE>
__device__ __forceinline__ void m2l_body8(const Tile &tile, const int32_t *__restrict__ src_sorted, const double *__restrict__ Mexp,
                                          const double *__restrict__ mats, const int32_t *__restrict__ kinfo, const double2 *__restrict__ rot,
                                          const int32_t *__restrict__ orow_t, double *__restrict__ scratch,
                                          double *dm_smem, double2 *cs_k)
{
    constexpr int NRE = 4 * KSH, NST = 2 * NRE;               // layout of the stored rows and matrices
    constexpr int KR = 4 * KE;                                 // dofs of either block that take part
    constexpr int NTH = KE / 2;                                // n-tiles (8 columns) of one block
    constexpr int CPB = (NTH + DM_NT - 1) / DM_NT;             // chunks per block
    constexpr int CW = (NTH + CPB - 1) / CPB;                  // chunk width in n-tiles
    double *Bs0 = dm_smem, *Bs1 = dm_smem + KR * DM_S;
    const double *B = mats + (size_t)tile.mat * NST * NST;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int lr = lane >> 2, lk = lane & 3;
    const int row = warp * 8 + lr;
    const bool rvalid = row < tile.nrows;

    auto issue = [&](int ch, double *dst) {
        const int blk = ch >= CPB, cl = blk ? ch - CPB : ch;
        const int t0 = CW * cl, nt = min(CW, NTH - t0);
        const int c0 = blk * NRE + 8 * t0, per_row = 4 * nt, k0 = blk * NRE;
        for (int i = threadIdx.x; i < KR * per_row; i += DM_THREADS) {
            const int k = i / per_row, j = (i % per_row) * 2;
            cp_async16(dst + k * DM_S + j, B + (size_t)(k0 + k) * NST + c0 + j);
        }
        cp_async_commit();
    };
    issue(0, Bs0);
    for (int k = threadIdx.x; k < KR; k += DM_THREADS) cs_k[k] = __ldg(rot + (size_t)tile.mat * ROT_M + __ldg(kinfo + k));
    const int arow = rvalid ? src_sorted[tile.row0 + row] : -1;
    const double2 *ap = reinterpret_cast<const double2 *>(Mexp + (size_t)(arow < 0 ? 0 : arow) * NST) + lk;
    double *orow = scratch + (size_t)(rvalid ? orow_t[tile.row0 + row] : 0) * 16 + 2 * lk;   // packed row: 2 KR dofs
    double a[KE];

    for (int ch = 0; ch < 2 * CPB; ++ch) {
        double *cur = (ch & 1) ? Bs1 : Bs0;
        const int blk = ch >= CPB, cl = blk ? ch - CPB : ch;
        cp_async_wait<0>();
        __syncthreads();                                        // chunk ch landed; everyone left chunk ch-1; cs_k visible
        if (ch + 1 < 2 * CPB) issue(ch + 1, (ch & 1) ? Bs0 : Bs1);
        if (cl == 0) {                                          // first chunk of a block: this block's half of A
#pragma unroll
            for (int j = 0; j < KE / 2; ++j) {
                double2 re = make_double2(0.0, 0.0), im = re;
                if (arow >= 0) { re = ap[4 * j]; im = ap[4 * j + NRE / 2]; }
                const double2 c0 = cs_k[8 * j + 2 * lk], c1 = cs_k[8 * j + 2 * lk + 1];
                if (blk == 0) { a[2 * j] = fma(c0.x, re.x, -c0.y * im.x); a[2 * j + 1] = fma(c1.x, re.y, -c1.y * im.y); }
                else { a[2 * j] = fma(c0.x, im.x, c0.y * re.x); a[2 * j + 1] = fma(c1.x, im.y, c1.y * re.y); }
            }
        }
        const int t0 = CW * cl, nt = min(CW, NTH - t0);
        dm_chunk<KE, 0, KE, 0>(a, cur, nt, lr, lk, rvalid, orow + blk * KR + 8 * t0);
    }
}

constexpr int M2L_NCLS_K = M2L_NCLS;
static_assert(M2L_NCLS_K == 5, "the switches below list the classes");

template <int PL>
__global__ void __launch_bounds__(DM_THREADS, (ke_of(PL) <= 20 ? 3 : 2))
translate_dmma_split(const Tile *__restrict__ tiles, const int32_t *__restrict__ src_sorted,
                     const double *__restrict__ Mexp, const double *__restrict__ mats, const uint8_t *__restrict__ mat_cls,
                     const int32_t *__restrict__ kinfo, const double2 *__restrict__ rot, const int32_t *__restrict__ orow_t,
                     double *__restrict__ scratch)
{
    constexpr int KSH = ke_of(PL);
    extern __shared__ __align__(16) double dm_smem[];          // [2][NRE][DM_S]
    __shared__ double2 cs_k[4 * KSH];                          // (cos, sin)(m_k a) of every real-part dof k
    const Tile tile = tiles[blockIdx.x];
    switch (mat_cls[blockIdx.x]) {                              // truncation class of the tile's matrix (CTA-uniform; per-tile table)
    case 0: m2l_body8<KSH, ke_of(PL)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    case 1: m2l_body8<KSH, ke_of(PL - 1)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    case 2: m2l_body8<KSH, ke_of(PL - 2)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    case 3: m2l_body8<KSH, ke_of(PL - 3)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    default: m2l_body8<KSH, ke_of(PL - 4)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    }
}

// Same, 4 warps x 16 rows: every B fragment read from shared memory feeds TWO DMMAs (the two 8-row groups of the
// warp).  ncu on the 8 x 8-row version: LSU wavefronts 55% with the tensor pipe at 65% -- the fragment loads
// (2 wavefronts per DMMA), the cp.async fills, the row gather and the stores share one pipe.
constexpr int DM16_THREADS = 128;
template <int KE, int NT>
__device__ __forceinline__ void dm16_chunk_nt(const double (&a0)[KE], const double (&a1)[KE], const double *cur, int lr, int lk,
                                              bool v0, bool v1, double *o0, double *o1)
{
    const double *bp = cur + 2 * lk * DM_S + lr;
    double c0[NT][2], c1[NT][2];
#pragma unroll
    for (int j = 0; j < NT; ++j) c0[j][0] = c0[j][1] = c1[j][0] = c1[j][1] = 0.0;
#pragma unroll
    for (int s = 0; s < KE; ++s) {
        const double *b = bp + (8 * (s >> 1) + (s & 1)) * DM_S;
#pragma unroll
        for (int j = 0; j < NT; ++j) {
            const double bv = b[8 * j];
            dmma884(c0[j][0], c0[j][1], a0[s], bv);
            dmma884(c1[j][0], c1[j][1], a1[s], bv);
        }
    }
#pragma unroll
    for (int j = 0; j < NT; ++j) {
        if (v0) *reinterpret_cast<double2 *>(o0 + 8 * j) = make_double2(c0[j][0], c0[j][1]);
        if (v1) *reinterpret_cast<double2 *>(o1 + 8 * j) = make_double2(c1[j][0], c1[j][1]);
    }
}

template <int KSH, int KE>
__device__ __forceinline__ void m2l_body16(const Tile &tile, const int32_t *__restrict__ src_sorted, const double *__restrict__ Mexp,
                                           const double *__restrict__ mats, const int32_t *__restrict__ kinfo, const double2 *__restrict__ rot,
                                           const int32_t *__restrict__ orow_t, double *__restrict__ scratch,
                                           double *dm_smem, double2 *cs_k)
{
    constexpr int NRE = 4 * KSH, NST = 2 * NRE;
    constexpr int KR = 4 * KE;
    constexpr int NTH = KE / 2;
    constexpr int CPB = (NTH + DM_NT - 1) / DM_NT;
    constexpr int CW = (NTH + CPB - 1) / CPB;
    double *Bs0 = dm_smem, *Bs1 = dm_smem + KR * DM_S;
    const double *B = mats + (size_t)tile.mat * NST * NST;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int lr = lane >> 2, lk = lane & 3;
    const int row0 = warp * 16 + lr, row1 = row0 + 8;
    const bool v0 = row0 < tile.nrows, v1 = row1 < tile.nrows;

    auto issue = [&](int ch, double *dst) {
        const int blk = ch >= CPB, cl = blk ? ch - CPB : ch;
        const int t0 = CW * cl, nt = min(CW, NTH - t0);
        const int c0 = blk * NRE + 8 * t0, per_row = 4 * nt, k0 = blk * NRE;
        for (int i = threadIdx.x; i < KR * per_row; i += DM16_THREADS) {
            const int k = i / per_row, j = (i % per_row) * 2;
            cp_async16(dst + k * DM_S + j, B + (size_t)(k0 + k) * NST + c0 + j);
        }
        cp_async_commit();
    };
    issue(0, Bs0);
    for (int k = threadIdx.x; k < KR; k += DM16_THREADS) cs_k[k] = __ldg(rot + (size_t)tile.mat * ROT_M + __ldg(kinfo + k));
    const int ar0 = v0 ? src_sorted[tile.row0 + row0] : -1, ar1 = v1 ? src_sorted[tile.row0 + row1] : -1;
    const double2 *ap0 = reinterpret_cast<const double2 *>(Mexp + (size_t)(ar0 < 0 ? 0 : ar0) * NST) + lk;
    const double2 *ap1 = reinterpret_cast<const double2 *>(Mexp + (size_t)(ar1 < 0 ? 0 : ar1) * NST) + lk;
    double *o0 = scratch + (size_t)(v0 ? orow_t[tile.row0 + row0] : 0) * 16 + 2 * lk;      // packed rows: 2 KR dofs
    double *o1 = scratch + (size_t)(v1 ? orow_t[tile.row0 + row1] : 0) * 16 + 2 * lk;
    double a0[KE], a1[KE];

    for (int ch = 0; ch < 2 * CPB; ++ch) {
        double *cur = (ch & 1) ? Bs1 : Bs0;
        const int blk = ch >= CPB, cl = blk ? ch - CPB : ch;
        cp_async_wait<0>();
        __syncthreads();
        if (ch + 1 < 2 * CPB) issue(ch + 1, (ch & 1) ? Bs0 : Bs1);
        if (cl == 0) {
#pragma unroll
            for (int j = 0; j < KE / 2; ++j) {
                const double2 z = make_double2(0.0, 0.0);
                const double2 re0 = ar0 >= 0 ? ap0[4 * j] : z, im0 = ar0 >= 0 ? ap0[4 * j + NRE / 2] : z;
                const double2 re1 = ar1 >= 0 ? ap1[4 * j] : z, im1 = ar1 >= 0 ? ap1[4 * j + NRE / 2] : z;
                const double2 c0 = cs_k[8 * j + 2 * lk], c1 = cs_k[8 * j + 2 * lk + 1];
                if (blk == 0) {
                    a0[2 * j] = fma(c0.x, re0.x, -c0.y * im0.x); a0[2 * j + 1] = fma(c1.x, re0.y, -c1.y * im0.y);
                    a1[2 * j] = fma(c0.x, re1.x, -c0.y * im1.x); a1[2 * j + 1] = fma(c1.x, re1.y, -c1.y * im1.y);
                } else {
                    a0[2 * j] = fma(c0.x, im0.x, c0.y * re0.x); a0[2 * j + 1] = fma(c1.x, im0.y, c1.y * re0.y);
                    a1[2 * j] = fma(c0.x, im1.x, c0.y * re1.x); a1[2 * j + 1] = fma(c1.x, im1.y, c1.y * re1.y);
                }
            }
        }
        const int t0 = CW * cl, nt = min(CW, NTH - t0), oc = blk * KR + 8 * t0;
        switch (nt) {
        case 5: dm16_chunk_nt<KE, 5>(a0, a1, cur, lr, lk, v0, v1, o0 + oc, o1 + oc); break;
        case 4: dm16_chunk_nt<KE, 4>(a0, a1, cur, lr, lk, v0, v1, o0 + oc, o1 + oc); break;
        case 3: dm16_chunk_nt<KE, 3>(a0, a1, cur, lr, lk, v0, v1, o0 + oc, o1 + oc); break;
        case 2: dm16_chunk_nt<KE, 2>(a0, a1, cur, lr, lk, v0, v1, o0 + oc, o1 + oc); break;
        default: dm16_chunk_nt<KE, 1>(a0, a1, cur, lr, lk, v0, v1, o0 + oc, o1 + oc); break;
        }
    }
}

template <int PL>
__global__ void __launch_bounds__(DM16_THREADS, 3)
translate_dmma_split16(const Tile *__restrict__ tiles, const int32_t *__restrict__ src_sorted,
                       const double *__restrict__ Mexp, const double *__restrict__ mats, const uint8_t *__restrict__ mat_cls,
                       const int32_t *__restrict__ kinfo, const double2 *__restrict__ rot, const int32_t *__restrict__ orow_t,
                     double *__restrict__ scratch)
{
    constexpr int KSH = ke_of(PL);
    extern __shared__ __align__(16) double dm_smem[];          // [2][NRE][DM_S]
    __shared__ double2 cs_k[4 * KSH];
    const Tile tile = tiles[blockIdx.x];
    switch (mat_cls[blockIdx.x]) {
    case 0: m2l_body16<KSH, ke_of(PL)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    case 1: m2l_body16<KSH, ke_of(PL - 1)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    case 2: m2l_body16<KSH, ke_of(PL - 2)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    case 3: m2l_body16<KSH, ke_of(PL - 3)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    default: m2l_body16<KSH, ke_of(PL - 4)>(tile, src_sorted, Mexp, mats, kinfo, rot, orow_t, scratch, dm_smem, cs_k); break;
    }
}

// attributes of a kernel are per device: one flag per device, set under this mutex (common.cuh once_per_device)
std::mutex &device_once_mutex()
{
    static std::mutex mu;
    return mu;
}

template <int PL>
static void launch_dmma(bem_ctx *c, const Stage &st, int which, cudaStream_t stream, double *scratch)
{
    constexpr int KSH = ke_of(PL);
    const size_t smem = (size_t)2 * 4 * KSH * DM_S * sizeof(double);
    static std::vector<char> attr_done;
    once_per_device(attr_done, c->device, [&]() {
        CUDA_TRY(cudaFuncSetAttribute(translate_dmma<KSH>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CUDA_TRY(cudaFuncSetAttribute(translate_dmma_split<PL>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        if (PL == 12) CUDA_TRY(cudaFuncSetAttribute(translate_dmma_split16<(PL == 12 ? PL : 4)>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    });
    if (which != TILES_DENSE && st.ntiles_split > 0) {
        if (PL == 12 && c->m2l_rows16)                           // measured: pays at p = 11, 12 (cfg 5), not at p <= 10 (cfg 4)
            translate_dmma_split16<(PL == 12 ? PL : 4)><<<st.ntiles_split, DM16_THREADS, smem, stream>>>(
                st.tiles.get(), st.src_sorted.get(), c->Mexp.get(), c->mats.get(), st.tile_cls[c->lay_active].get(), c->kinfo.get(), c->rot.get(), st.orow[c->lay_active].get(), scratch);
        else
            translate_dmma_split<PL><<<st.ntiles_split, DM_THREADS, smem, stream>>>(st.tiles.get(), st.src_sorted.get(), c->Mexp.get(),
                                                                                   c->mats.get(), st.tile_cls[c->lay_active].get(), c->kinfo.get(), c->rot.get(),
                                                                                   st.orow[c->lay_active].get(), scratch);
    }
    if (which != TILES_SPLIT && st.ntiles > st.ntiles_split)
        translate_dmma<KSH><<<st.ntiles - st.ntiles_split, DM_THREADS, smem, stream>>>(st.tiles.get() + st.ntiles_split, st.src_sorted.get(),
                                                                                      c->Mexp.get(), c->Lexp.get(), c->mats.get(),
                                                                                      c->kinfo.get(), c->rot.get(),
                                                                                      st.orow[c->lay_active].get(), scratch);
}

// out[out_base + t][:] = sum_{k in ptr[t]..ptr[t+1]} e^{i m a_k} scratch[k][:]   (fixed order; a_k = azimuth of
// pair k's matrix, the identity for M2M / L2L pairs).  One CTA per target box, one thread per coefficient (l, m):
// it reads the real and the imaginary part (nre apart) of every row once and writes both.
constexpr int RED_CHUNK = 192;     // pairs of a target staged at a time (an M2L list holds at most 189)
__global__ void __launch_bounds__(160)
translate_reduce(const int32_t *__restrict__ ptr, const int32_t *__restrict__ mat_t, const int32_t *__restrict__ mat_ne,
                 const int32_t *__restrict__ mat_w, const int32_t *__restrict__ row_off, const double *__restrict__ scratch, const int32_t *__restrict__ kinfo, const double2 *__restrict__ rot,
                 int nre, int accumulate, int ntgt, const int32_t *__restrict__ list, double *__restrict__ out)
{
    // accumulate: 0 = overwrite (an empty list writes zeros), 1 = add to the output, 2 = overwrite but leave the output of an
    // empty list alone (adaptive tree: a parent without children is a leaf whose multipoles P2M wrote).
    // A row of a graded (truncated) translation holds the leading mat_ne[matrix] dofs only; the rest of the scratch row was
    // never written.  (matrix id | dofs << 16) of the target's pairs is staged in shared memory so that the row loads do
    // not wait for a global load of their predicate.
    __shared__ int s_mt[RED_CHUNK + 8], s_off[RED_CHUNK + 8], s_w[RED_CHUNK + 8];   // matrix | dofs << 16, row offset (16 doubles), dofs per block stored
    const int nst = 2 * nre;
    for (int ti = blockIdx.x; ti < ntgt; ti += gridDim.x) {         // grid < ntgt: a persistent pass (see launch_stage_reduce)
        const int t = list ? list[ti] : ti;                            // adaptive tree: only the boxes that exist are visited
        const int b = ptr[t], e = ptr[t + 1];
        double *o = out + (size_t)t * nst;
        if (b == e && accumulate == 0)
            for (int cc = threadIdx.x; cc < nst; cc += blockDim.x) o[cc] = 0.0;
        for (int k0 = b; k0 < e; k0 += RED_CHUNK) {                 // one round for every list the library builds
            const int n = min(RED_CHUNK, e - k0);
            __syncthreads();
            for (int i = threadIdx.x; i < n; i += blockDim.x) {
                const int mt = mat_t[k0 + i];
                s_mt[i] = mt | (__ldg(mat_ne + mt) << 16);
                s_off[i] = row_off[k0 + i];
                s_w[i] = __ldg(mat_w + mt);
            }
            __syncthreads();
            for (int cc = threadIdx.x; cc < nre; cc += blockDim.x) {
                const int m = kinfo[cc];
                const double *base = scratch + cc;
                double sr = 0.0, si = 0.0;
                // (a branch-free version that issues the 16 loads of 8 rows before using the first, reading the rows that do
                // not carry dof cc at a dummy offset, measured SLOWER: 3.77 against 2.84 ms on config 5)
                if (m == 0) {
#pragma unroll 8
                    for (int i = 0; i < n; ++i)
                        if (cc < (s_mt[i] >> 16)) sr += base[(size_t)s_off[i] * 16];
                } else {
#pragma unroll 8
                    for (int i = 0; i < n; ++i) {
                        const int mt = s_mt[i];
                        if (cc < (mt >> 16)) {
                            const double *row = base + (size_t)s_off[i] * 16;
                            double vr = row[0], vi = row[s_w[i]];
                            azimuth(__ldg(rot + (size_t)(mt & 0xffff) * ROT_M + m), vr, vi);
                            sr += vr;
                            si += vi;
                        }
                    }
                }
                if (accumulate == 1 || k0 > b) { sr += o[cc]; si += o[cc + nre]; }
                o[cc] = sr;
                o[cc + nre] = si;
            }
        }
    }
}

// The same sums with the rows STREAMED through shared memory (option "reduce_stream", default): the packed rows of a target
// are one contiguous byte range of the scratch (row offsets are a prefix sum in target-major order), so batches of
// RS_ROWS rows are copied whole by cp.async, two batches in flight, while the previous batch is summed from shared memory --
// the copies carry no predicate and no address arithmetic per dof, and many are in flight per thread.  Same order of the
// additions as translate_reduce: the same bits.
constexpr int RS_ROWS = 4;
constexpr int RS_STAGES = 2;        // batches in flight.  Measured on config 5 (ms of the sums + L2L class; direct loads: 2.88): two stages, 128 threads, rows 2 / 4 / 8 / 16: 2.57 / 2.22 / 2.65 / 3.78; four stages x 4 rows: 2.86; two stages, 96 threads, rows 3 / 4: 2.21 / 2.15 -- what counts is how many CTAs an SM holds
constexpr int RS_THREADS = 128;
__global__ void __launch_bounds__(RS_THREADS)
translate_reduce_stream(const int32_t *__restrict__ ptr, const int32_t *__restrict__ mat_t, const int32_t *__restrict__ mat_ne,
                        const int32_t *__restrict__ mat_w, const int32_t *__restrict__ row_off, const double *__restrict__ scratch,
                        const int32_t *__restrict__ kinfo, const double2 *__restrict__ rot,
                        int nre, int accumulate, int ntgt, const int32_t *__restrict__ list, double *__restrict__ out)
{
    extern __shared__ __align__(16) double rs_buf[];                  // [RS_STAGES][RS_ROWS * nst]
    __shared__ int s_mt[RED_CHUNK + 8], s_off[RED_CHUNK + 8], s_w[RED_CHUNK + 8];
    const int nst = 2 * nre;
    const int bufsz = RS_ROWS * nst;
    for (int ti = blockIdx.x; ti < ntgt; ti += gridDim.x) {
        const int t = list ? list[ti] : ti;
        const int b = ptr[t], e = ptr[t + 1];
        double *o = out + (size_t)t * nst;
        if (b == e && accumulate == 0)
            for (int cc = threadIdx.x; cc < nst; cc += blockDim.x) o[cc] = 0.0;
        for (int k0 = b; k0 < e; k0 += RED_CHUNK) {
            const int n = min(RED_CHUNK, e - k0);
            __syncthreads();
            for (int i = threadIdx.x; i <= n; i += blockDim.x) {
                s_off[i] = row_off[k0 + i];                              // row_off has npairs + 1 entries
                if (i < n) { const int mt = mat_t[k0 + i]; s_mt[i] = mt | (__ldg(mat_ne + mt) << 16); s_w[i] = __ldg(mat_w + mt); }
            }
            __syncthreads();
            const int nb = (n + RS_ROWS - 1) / RS_ROWS;
            auto issue = [&](int bi) {                                   // rows [bi RS_ROWS, ..) of the chunk: one contiguous range
                const int i0 = bi * RS_ROWS, i1 = min(n, i0 + RS_ROWS);
                const double *src = scratch + (size_t)s_off[i0] * 16;
                const int pieces = (s_off[i1] - s_off[i0]) * 8;          // 16-byte pieces
                double *dst = rs_buf + (bi % RS_STAGES) * bufsz;
                for (int q = threadIdx.x; q < pieces; q += blockDim.x) cp_async16(dst + 2 * q, src + 2 * q);
            };
            double sr = 0.0, si = 0.0;                                   // blockDim >= nre: one dof per thread
            const int cc = threadIdx.x;
            const int m = cc < nre ? kinfo[cc] : 0;
            for (int j = 0; j < RS_STAGES - 1; ++j) { if (j < nb) issue(j); cp_async_commit(); }
            for (int bi = 0; bi < nb; ++bi) {
                if (bi + RS_STAGES - 1 < nb) issue(bi + RS_STAGES - 1);  // into the buffer batch bi - 1 left (barrier below)
                cp_async_commit();                                       // one group per iteration, empty at the tail
                cp_async_wait<RS_STAGES - 1>();
                __syncthreads();                                         // batch bi is in shared memory
                if (cc < nre) {
                    const int i0 = bi * RS_ROWS, i1 = min(n, i0 + RS_ROWS);
                    const double *buf = rs_buf + (bi % RS_STAGES) * bufsz;
                    const int base = s_off[i0];
                    for (int i = i0; i < i1; ++i) {
                        const int mt = s_mt[i];
                        if (cc < (mt >> 16)) {
                            const double *row = buf + (s_off[i] - base) * 16;
                            double vr = row[cc], vi = row[s_w[i] + cc];
                            if (m != 0) { azimuth(__ldg(rot + (size_t)(mt & 0xffff) * ROT_M + m), vr, vi); si += vi; }
                            sr += vr;
                        }
                    }
                }
                __syncthreads();                                         // everyone left batch bi before it is overwritten
            }
            if (cc < nre) {
                if (accumulate == 1 || k0 > b) { sr += o[cc]; si += o[cc + nre]; }
                o[cc] = sr;
                o[cc + nre] = si;
            }
        }
    }
}


// ------------------------------------------------------------------ packed scratch rows (setup)
__global__ void gather_i32(const int32_t *idx, const int32_t *v, int64_t n, int32_t *out)
{
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r < n) out[r] = v[idx[r]];
}
__global__ void row_units(const int32_t *mat_t, int64_t n, const int32_t *mat_w, int32_t *u)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < n) u[k] = mat_w[mat_t[k]] >> 3;                       // 2 W doubles = W / 8 units of 16 doubles
}
// Row offsets of every stage for every truncation layout, and the scratch buffer.  The M2L stages of all levels have their
// own regions (their tiles are all issued before the first sum when option overlap = 1); M2M and L2L stages run when no
// M2L row is alive and alias the start of the buffer.
void pack_scratch(bem_ctx *c)
{
    cudaStream_t s = c->stream;
    int64_t need = 1;
    for (int i = 0; i < c->n_lay; ++i) {
        const FmmLayout &L = c->lay[i];
        int64_t region = 0, top = 0;
        auto pack = [&](Stage &st, bool own_region) {
            if (st.ntgt == 0 && st.npairs == 0) return;
            const int64_t n = st.npairs;
            st.row_off[i].alloc(n + 1);
            dvec<int32_t> u;
            u.alloc(n);
            if (n > 0) { row_units<<<cdiv(n, 256), 256, 0, s>>>(st.mat_t.get(), n, L.mat_w.get(), u.get()); KERNEL_CHECK(); }
            scan_exclusive_i32(u.get(), st.row_off[i].get(), n, s);
            int total = 0;
            d2h_sync(&total, st.row_off[i].get() + n, sizeof(int), s);
            st.orow[i].alloc(n);
            if (n > 0) { gather_i32<<<cdiv(n, 256), 256, 0, s>>>(st.krow.get(), st.row_off[i].get(), n, st.orow[i].get()); KERNEL_CHECK(); }
            std::vector<uint8_t> tc(st.tile_mat_host.size());
            for (size_t t = 0; t < tc.size(); ++t) tc[t] = (uint8_t)L.mat_cls_host[st.tile_mat_host[t]];
            st.tile_cls[i].alloc(tc.size());
            if (!tc.empty()) {
                CUDA_TRY(cudaMemcpyAsync(st.tile_cls[i].get(), tc.data(), tc.size(), cudaMemcpyHostToDevice, s));
                CUDA_TRY(cudaStreamSynchronize(s));
            }
            st.region_units[i] = own_region ? region : 0;
            if (own_region) region += total;
            top = std::max(top, (own_region ? region : (int64_t)total));
        };
        for (auto &st : c->m2l) pack(st, true);
        for (auto &st : c->m2m) pack(st, false);
        for (auto &st : c->l2l) pack(st, false);
        need = std::max(need, top);
    }
    c->scratch.alloc((size_t)need * 16);
}

// the tiles of a stage (which = all, only the M2L tiles, only the dense M2M / L2L tiles) on `stream`
void launch_stage_gemm(bem_ctx *c, const Stage &st, int which, cudaStream_t stream)
{
    const int first = which == TILES_DENSE ? st.ntiles_split : 0;
    const int last = which == TILES_SPLIT ? st.ntiles_split : st.ntiles;
    if (st.ntgt == 0 || last <= first) return;
    double *scratch = c->scratch.get() + (size_t)st.region_units[c->lay_active] * 16;
    const int pl = c->pl;
    if (c->gemm_path == 1 || pl > 16) {                         // plain-FMA tiles: p > 16, or forced (option "gemm_path")
        dim3 grid(last - first, cdiv(c->nst, GEMM_TN));
        translate_gemm<<<grid, GEMM_THREADS, 0, stream>>>(st.tiles.get() + first, st.src_sorted.get(), c->Mexp.get(), c->Lexp.get(),
                                                          c->mats.get(), c->kinfo.get(), c->rot.get(), c->nst,
                                                          st.orow[c->lay_active].get(), c->mat_w.get(), scratch);
    }
    else if (pl == 4) launch_dmma<4>(c, st, which, stream, scratch);     // layout degree -> ke_of(pl) = nre / 4 k-steps per block
    else if (pl == 6) launch_dmma<6>(c, st, which, stream, scratch);
    else if (pl == 8) launch_dmma<8>(c, st, which, stream, scratch);
    else if (pl == 10) launch_dmma<10>(c, st, which, stream, scratch);
    else if (pl == 11) launch_dmma<11>(c, st, which, stream, scratch);
    else if (pl == 13) launch_dmma<13>(c, st, which, stream, scratch);
    else if (pl == 12) launch_dmma<12>(c, st, which, stream, scratch);
    else if (pl == 14) launch_dmma<14>(c, st, which, stream, scratch);
    else launch_dmma<16>(c, st, which, stream, scratch);
    KERNEL_CHECK();
}

// ctas_per_sm > 0: a PERSISTENT pass of at most that many CTAs per SM looping over the targets.  The hardware does
// not backfill an SM with blocks of a lower-priority grid while a higher-priority grid still has blocks waiting, and
// serves equal priorities in arrival order; only a grid whose blocks are ALL resident at once leaves the rest of the
// machine to the kernel of the other stream (measured: DESIGN.md section 6).
void launch_stage_reduce(bem_ctx *c, const Stage &st, cudaStream_t stream, int ctas_per_sm)
{
    if (st.ntgt == 0) return;
    double *out = (st.out_is_local ? c->Lexp.get() : c->Mexp.get()) + (size_t)st.out_base * c->nst;
    const int nvisit = st.n_list >= 0 ? st.n_list : st.ntgt;
    if (nvisit == 0) return;
    const int grid = ctas_per_sm > 0 ? std::min(nvisit, c->n_sm * ctas_per_sm) : nvisit;
    static std::vector<char> attr_done;
    once_per_device(attr_done, c->device, [&]() {                       // same carve-out as the pair kernels it runs beside (common.cuh)
        CUDA_TRY(cudaFuncSetAttribute(translate_reduce, cudaFuncAttributePreferredSharedMemoryCarveout, CORUN_CARVEOUT));
    });
    if (c->reduce_stream && c->nre <= RS_THREADS) {                    // rows streamed through shared memory (cp.async)
        const size_t smem = (size_t)RS_STAGES * RS_ROWS * c->nst * sizeof(double);
        static std::vector<char> attr2_done;
        once_per_device(attr2_done, c->device, [&]() {
            CUDA_TRY(cudaFuncSetAttribute(translate_reduce_stream, cudaFuncAttributeMaxDynamicSharedMemorySize, RS_STAGES * RS_ROWS * 2 * RS_THREADS * (int)sizeof(double)));
        });
        translate_reduce_stream<<<grid, std::max(64, ((c->nre + 31) / 32) * 32), smem, stream>>>(
            st.ptr.get(), st.mat_t.get(), c->mat_ne.get(), c->mat_w.get(), st.row_off[c->lay_active].get(),
            c->scratch.get() + (size_t)st.region_units[c->lay_active] * 16,
            c->kinfo.get(), c->rot.get(), c->nre, st.accumulate ? 1 : (st.keep_empty ? 2 : 0), nvisit, st.n_list >= 0 ? st.tgt_list.get() : nullptr, out);
        KERNEL_CHECK();
        return;
    }
    translate_reduce<<<grid, std::min(160, ((c->nre + 31) / 32) * 32), 0, stream>>>(
        st.ptr.get(), st.mat_t.get(), c->mat_ne.get(), c->mat_w.get(), st.row_off[c->lay_active].get(),
        c->scratch.get() + (size_t)st.region_units[c->lay_active] * 16,
        c->kinfo.get(), c->rot.get(), c->nre, st.accumulate ? 1 : (st.keep_empty ? 2 : 0), nvisit, st.n_list >= 0 ? st.tgt_list.get() : nullptr, out);
    KERNEL_CHECK();
}

// one stage start to end on the context's stream
void launch_stage(bem_ctx *c, const Stage &st, int cls_gemm, int cls_reduce)
{
    if (st.ntgt == 0) return;
    launch_stage_gemm(c, st, TILES_ALL, c->stream);
    if (st.ntiles > 0) mark(c, cls_gemm);
    launch_stage_reduce(c, st, c->stream, 0);
    mark(c, cls_reduce);
}

// ------------------------------------------------------------------ P2M (a5)
// Mt_l^m = sum_s [ (m_s/h) conj R_l^m(a) - (1/h^2) d_s . grad conj R_l^m(a) ],  a = (y_s - c)/h, with
// d.grad R_l^m = d_z R_{l-1}^m + 1/2 (d_x - i d_y) R_{l-1}^{m+1} - 1/2 (d_x + i d_y) R_{l-1}^{m-1}.
// One warp per source leaf; lane = source (32 at a time).  Each lane builds the harmonics row by
// row (degree l from degrees l-1, l-2); the 2l+1 real values of a row go through shared memory so
// that lane k sums value k over the 32 sources -- a fixed-order sum, no atomics.
constexpr int P2M_WARPS_G = 4;

__global__ void __launch_bounds__(P2M_WARPS_G * 32)
p2m_kernel(const int32_t *__restrict__ sbegin, const uint64_t *__restrict__ skey, const int32_t *__restrict__ list, int nleaf, int level,
           double cmx, double cmy, double cmz, double h,
           const double4 *__restrict__ spos, const double4 *__restrict__ sstr, int p, int nre, int nst, double *__restrict__ Mout)
{
    extern __shared__ double sm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    int leaf = blockIdx.x * P2M_WARPS_G + warp;
    if (leaf >= nleaf) return;
    if (list) leaf = list[leaf];
    double *tbl = sm + (size_t)warp * (2 * p - 1) * 33;            // [2l+1 values][33]
    uint32_t ix, iy, iz;
    morton_decode(skey[leaf], &ix, &iy, &iz);
    const double cx = cmx + (ix + 0.5) * h, cy = cmy + (iy + 0.5) * h, cz = cmz + (iz + 0.5) * h;
    const double ih = 1.0 / h;
    const int s0 = sbegin[leaf], s1 = sbegin[leaf + 1];
    double *M = Mout + (size_t)leaf * nst;
    for (int cidx = lane; cidx < nst; cidx += 32) M[cidx] = 0.0;
    __syncwarp();
    double pre[P_MAX + 2], pim[P_MAX + 2], qre[P_MAX + 2], qim[P_MAX + 2], cre[P_MAX + 2], cim[P_MAX + 2];
    for (int base = s0; base < s1; base += 32) {
        const int s = base + lane;
        const bool valid = s < s1;
        double ax = 0, ay = 0, az = 0, mh = 0, dx = 0, dy = 0, dz = 0;
        if (valid) {
            const double4 ps = spos[s], st = sstr[s];
            ax = (ps.x - cx) * ih; ay = (ps.y - cy) * ih; az = (ps.z - cz) * ih;
            mh = st.x * ih; dx = st.y * ih * ih; dy = st.z * ih * ih; dz = st.w * ih * ih;
        }
        const double r2 = ax * ax + ay * ay + az * az;
        for (int l = 0; l < p; ++l) {
            // row l of R from rows l-1 (p*) and l-2 (q*)
            if (l == 0) { cre[0] = 1.0; cim[0] = 0.0; }
            else {
                for (int m = 0; m < l; ++m) {
                    double vr = (2 * l - 1) * az * pre[m], vi = (2 * l - 1) * az * pim[m];
                    if (m <= l - 2) { vr -= r2 * qre[m]; vi -= r2 * qim[m]; }
                    const double inv = 1.0 / ((double)(l - m) * (double)(l + m));
                    cre[m] = vr * inv; cim[m] = vi * inv;
                }
                const double f = -1.0 / (2.0 * l);
                cre[l] = f * (ax * pre[l - 1] - ay * pim[l - 1]);
                cim[l] = f * (ax * pim[l - 1] + ay * pre[l - 1]);
            }
            // coefficient values of this source for degree l
            for (int m = 0; m <= l; ++m) {
                double gr = 0.0, gi = 0.0;
                if (l > 0) {
                    const double Cr = (m <= l - 1) ? pre[m] : 0.0, Ci = (m <= l - 1) ? pim[m] : 0.0;
                    const double Ar = (m + 1 <= l - 1) ? pre[m + 1] : 0.0, Ai = (m + 1 <= l - 1) ? pim[m + 1] : 0.0;
                    double Br, Bi;
                    if (m >= 1) { Br = pre[m - 1]; Bi = pim[m - 1]; }
                    else if (l - 1 >= 1) { Br = -pre[1]; Bi = pim[1]; }       // R_{l-1}^{-1} = -conj R_{l-1}^{1}
                    else { Br = 0.0; Bi = 0.0; }
                    gr = dz * Cr + 0.5 * (dx * Ar + dy * Ai) - 0.5 * (dx * Br - dy * Bi);
                    gi = dz * Ci + 0.5 * (dx * Ai - dy * Ar) - 0.5 * (dx * Bi + dy * Br);
                }
                const double vr = mh * cre[m] - gr, vi = -(mh * cim[m] - gi);   // conj
                if (m == 0) tbl[lane] = valid ? vr : 0.0;
                else { tbl[(2 * m - 1) * 33 + lane] = valid ? vr : 0.0; tbl[(2 * m) * 33 + lane] = valid ? vi : 0.0; }
            }
            __syncwarp();
            for (int k = lane; k < 2 * l + 1; k += 32) {
                double sum = 0.0;
                for (int j = 0; j < 32; ++j) sum += tbl[k * 33 + j];
                M[real_idx(l, (k + 1) >> 1, (k > 0 && !(k & 1)) ? 1 : 0, nre)] += sum;
            }
            __syncwarp();
            for (int m = 0; m <= l; ++m) { qre[m] = pre[m]; qim[m] = pim[m]; pre[m] = cre[m]; pim[m] = cim[m]; }
        }
    }
}

void launch_p2m_generic(bem_ctx *c, int lmax, int nleaf, const int32_t *list, const int32_t *sbegin)
{
    const BoxSet &sb = c->sb;
    if (nleaf == 0) return;
    const double h = c->cube_side / (double)(1 << lmax);
    const size_t smem = (size_t)P2M_WARPS_G * (2 * c->p - 1) * 33 * sizeof(double);
    if (smem > 48 * 1024) CUDA_TRY(cudaFuncSetAttribute(p2m_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    p2m_kernel<<<cdiv(nleaf, P2M_WARPS_G), P2M_WARPS_G * 32, smem, c->stream>>>(
        sbegin, sb.bkey[lmax].get(), list, nleaf, lmax, c->cube_min[0], c->cube_min[1], c->cube_min[2], h,
        c->src_pos.get(), c->src_str.get(), c->p, c->nre, c->nst, c->Mexp.get() + (size_t)sb.base[lmax] * c->nst);
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ L2P (a9)
// Phi(x) = sum_l [ Lt_l^0 R_l^0(b) + 2 sum_{m>0} ( Re Lt_l^m Re R_l^m(b) + Im Lt_l^m Im R_l^m(b) ) ],  b = (x - c)/h.
// One thread per target; threads of a warp mostly share the leaf, so coefficient loads are broadcasts.
__global__ void __launch_bounds__(128)
l2p_kernel(const double *__restrict__ tgt, int64_t nt, const int32_t *__restrict__ leaf_of, const uint64_t *__restrict__ tkey,
           const uint8_t *__restrict__ lev_all, double cmx, double cmy, double cmz, double h, int p, int nre, int nst,
           const double *__restrict__ Lleaf, double *__restrict__ y)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nt) return;
    const int leaf = leaf_of[t];
    if (lev_all) h = ldexp(h, -(int)lev_all[leaf]);               // adaptive tree: global box ids, h = cube side
    uint32_t ix, iy, iz;
    morton_decode(tkey[leaf], &ix, &iy, &iz);
    const double ih = 1.0 / h;
    const double bx = (tgt[3 * t] - (cmx + (ix + 0.5) * h)) * ih;
    const double by = (tgt[3 * t + 1] - (cmy + (iy + 0.5) * h)) * ih;
    const double bz = (tgt[3 * t + 2] - (cmz + (iz + 0.5) * h)) * ih;
    const double r2 = bx * bx + by * by + bz * bz;
    const double *L = Lleaf + (size_t)leaf * nst;
    double pre[P_MAX + 2], pim[P_MAX + 2], qre[P_MAX + 2], qim[P_MAX + 2], cre[P_MAX + 2], cim[P_MAX + 2];
    double phi = 0.0;
    for (int l = 0; l < p; ++l) {
        if (l == 0) { cre[0] = 1.0; cim[0] = 0.0; }
        else {
            for (int m = 0; m < l; ++m) {
                double vr = (2 * l - 1) * bz * pre[m], vi = (2 * l - 1) * bz * pim[m];
                if (m <= l - 2) { vr -= r2 * qre[m]; vi -= r2 * qim[m]; }
                const double inv = 1.0 / ((double)(l - m) * (double)(l + m));
                cre[m] = vr * inv; cim[m] = vi * inv;
            }
            const double f = -1.0 / (2.0 * l);
            cre[l] = f * (bx * pre[l - 1] - by * pim[l - 1]);
            cim[l] = f * (bx * pim[l - 1] + by * pre[l - 1]);
        }
        const double *Lre = L + l * (l + 1) / 2, *Lim = Lre + nre;
        double row = Lre[0] * cre[0];
        for (int m = 1; m <= l; ++m) row += 2.0 * (Lre[m] * cre[m] + Lim[m] * cim[m]);
        phi += row;
        for (int m = 0; m <= l; ++m) { qre[m] = pre[m]; qim[m] = pim[m]; pre[m] = cre[m]; pim[m] = cim[m]; }
    }
    y[t] = phi;
}

void launch_l2p_generic(bem_ctx *c, const int32_t *leaf_of)
{
    const BoxSet &tb = c->tb;
    const int lmax = tb.lmax;
    const double h = c->cube_side / (double)(1 << lmax);
    if (c->adaptive)
        l2p_kernel<<<cdiv(c->N, 128), 128, 0, c->stream>>>(c->tgt_pos.get(), c->N, c->ad.pt_gbox.get(), c->ad.tkey_all.get(), c->ad.tlev_all.get(),
                                                           c->cube_min[0], c->cube_min[1], c->cube_min[2], c->cube_side, c->p, c->nre, c->nst,
                                                           c->Lexp.get(), c->ypart.get());
    else
    l2p_kernel<<<cdiv(c->N, 128), 128, 0, c->stream>>>(c->tgt_pos.get(), c->N, leaf_of, tb.bkey[lmax].get(), nullptr,
                                                       c->cube_min[0], c->cube_min[1], c->cube_min[2], h, c->p, c->nre, c->nst,
                                                       c->Lexp.get() + (size_t)tb.base[lmax] * c->nst, c->ypart.get());
    KERNEL_CHECK();
}

}  // namespace bem
