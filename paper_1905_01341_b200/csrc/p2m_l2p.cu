// Steps a5 (P2M) and a9 (L2P) of DESIGN.md with the truncation number as a template parameter:
// the solid-harmonic recurrences (harmonics.cuh) are fully unrolled, so the two
// rows of R_l^m a step needs live in registers (the run-time-p kernels in translate.cu keep them in
// local memory and remain the fallback for p > 16).
//
//   P2M  Mt_l^m = sum_s [ (m_s/h) conj R_l^m(a) - (1/h^2) d_s . grad conj R_l^m(a) ],  a = (y_s - c)/h,
//        d.grad R_l^m = d_z R_{l-1}^m + 1/2 (d_x - i d_y) R_{l-1}^{m+1} - 1/2 (d_x + i d_y) R_{l-1}^{m-1}
//   L2P  Phi(x) = sum_l [ Lt_l^0 R_l^0(b) + 2 sum_{m>0} ( Re Lt_l^m Re R_l^m(b) + Im Lt_l^m Im R_l^m(b) ) ],  b = (x - c)/h
// (expansions truncated to degrees 0..p-1; the dense part of the product).
#include "common.cuh"
#include "harmonics.cuh"
#include "morton.cuh"
#include <algorithm>

namespace bem {

// Rows of the expansion are flushed through shared memory in groups of at most 64 real values.
__host__ __device__ constexpr int grp_start(int l)
{
    int s = 0;
    for (int r = 0; r <= l; ++r)
        if ((r + 1) * (r + 1) - s * s > 64) s = r;
    return s;
}
__host__ __device__ constexpr int grp_index(int l)
{
    int s = 0, g = 0;
    for (int r = 0; r <= l; ++r)
        if ((r + 1) * (r + 1) - s * s > 64) { s = r; ++g; }
    return g;
}

// row l of R (into R*[l&1], overwriting row l-2) from row l-1 (R*[(l-1)&1]); all indices compile-time after unrolling
template <int P>
__device__ __forceinline__ void next_row(int l, double ax, double ay, double az, double r2, double (&Rre)[2][P], double (&Rim)[2][P])
{
    const int cur = l & 1, prv = cur ^ 1;
    if (l == 0) { Rre[0][0] = 1.0; Rim[0][0] = 0.0; return; }
    const double zl = (double)(2 * l - 1) * az;
#pragma unroll
    for (int m = 0; m < P; ++m) {
        if (m < l) {
            double vr = zl * Rre[prv][m], vi = zl * Rim[prv][m];
            if (m <= l - 2) { vr = fma(-r2, Rre[cur][m], vr); vi = fma(-r2, Rim[cur][m], vi); }
            const double inv = 1.0 / ((double)(l - m) * (double)(l + m));
            Rre[cur][m] = vr * inv;
            Rim[cur][m] = m == 0 ? 0.0 : vi * inv;
        }
    }
    const double f = -1.0 / (2.0 * l);
    Rre[cur][l] = f * (ax * Rre[prv][l - 1] - ay * Rim[prv][l - 1]);
    Rim[cur][l] = f * (ax * Rim[prv][l - 1] + ay * Rre[prv][l - 1]);
}

// ------------------------------------------------------------------ P2M
// One warp per source leaf, lane = source (32 at a time).  Each lane's p^2 values go through a
// [64][33] shared-memory table, group of rows by group; lane k then sums value k over the 32
// sources in a fixed order (no atomics) into a register accumulator.
#ifndef P2M_MINB
#define P2M_MINB 3
#endif
constexpr int P2M_WARPS = 4;
constexpr int P2M_TBL = 64 * 33;

template <int P, bool DIP>
__global__ void __launch_bounds__(P2M_WARPS * 32, P2M_MINB)
p2m_kernel_t(const int32_t *__restrict__ sbegin, const uint64_t *__restrict__ skey, const int32_t *__restrict__ list, int nleaf,
             double cmx, double cmy, double cmz, double h,
             const double4 *__restrict__ spos, const double4 *__restrict__ sstr, int p, int nst, double *__restrict__ Mout,
             int *__restrict__ counter)
{
    extern __shared__ double sm[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    double *tbl = sm + (size_t)warp * P2M_TBL;
    // persistent warps: leaf sizes differ by an order of magnitude on polydisperse clusters, and with one leaf per warp of a
    // 4-warp CTA the SM ran at 7 of its 12 warps on average (ncu); every warp now takes the next leaf from a counter
    for (;;) {
    int leaf = 0;
    if (lane == 0) leaf = atomicAdd(counter, 1);
    leaf = __shfl_sync(0xffffffffu, leaf, 0);
    if (leaf >= nleaf) return;
    if (list) leaf = list[leaf];                                  // adaptive tree: the leaves of this level are a subset of its boxes
    uint32_t ix, iy, iz;
    morton_decode(skey[leaf], &ix, &iy, &iz);
    const double cx = cmx + (ix + 0.5) * h, cy = cmy + (iy + 0.5) * h, cz = cmz + (iz + 0.5) * h;
    const double ih = 1.0 / h;
    const int s0 = sbegin[leaf], s1 = sbegin[leaf + 1];
    constexpr int NG = grp_index(P - 1) + 1;
    double acc[2 * NG];
#pragma unroll
    for (int i = 0; i < 2 * NG; ++i) acc[i] = 0.0;

    for (int base = s0; base < s1; base += 32) {
        const int s = base + lane;
        double ax = 0, ay = 0, az = 0, mh = 0, dx = 0, dy = 0, dz = 0;    // idle lanes carry zero strengths
        if (s < s1) {
            const double4 ps = spos[s], st = sstr[s];
            ax = (ps.x - cx) * ih; ay = (ps.y - cy) * ih; az = (ps.z - cz) * ih;
            mh = st.x * ih; dx = st.y * ih * ih; dy = st.z * ih * ih; dz = st.w * ih * ih;
        }
        const double r2 = ax * ax + ay * ay + az * az;
        const double hx = 0.5 * dx, hy = 0.5 * dy;
        double Rre[2][P], Rim[2][P];
#pragma unroll
        for (int l = 0; l < P; ++l) {
            next_row<P>(l, ax, ay, az, r2, Rre, Rim);
            const int cur = l & 1, prv = cur ^ 1;
            const int g0 = grp_start(l) * grp_start(l);               // expansion index of the group's first value
            double *col = tbl + (l * l - g0) * 33 + lane;
#pragma unroll
            for (int m = 0; m < P; ++m) {
                if (m <= l) {
                    double gr = 0.0, gi = 0.0;
                    if (DIP && l > 0) {
                        const double Cr = (m <= l - 1) ? Rre[prv][m] : 0.0, Ci = (m <= l - 1) ? Rim[prv][m] : 0.0;
                        const double Ar = (m + 1 <= l - 1) ? Rre[prv][m + 1] : 0.0, Ai = (m + 1 <= l - 1) ? Rim[prv][m + 1] : 0.0;
                        double Br = 0.0, Bi = 0.0;
                        if (m >= 1) { Br = Rre[prv][m - 1]; Bi = Rim[prv][m - 1]; }
                        else if (l - 1 >= 1) { Br = -Rre[prv][1]; Bi = Rim[prv][1]; }      // R_{l-1}^{-1} = -conj R_{l-1}^{1}
                        gr = fma(hx, Ar - Br, fma(hy, Ai + Bi, dz * Cr));           // hx = dx / 2, hy = dy / 2
                        gi = fma(hx, Ai - Bi, fma(-hy, Ar + Br, dz * Ci));
                    }
                    const double vr = fma(mh, Rre[cur][m], -gr), vi = fma(-mh, Rim[cur][m], gi);   // conj
                    if (m == 0) col[0] = vr;
                    else { col[(2 * m - 1) * 33] = vr; col[(2 * m) * 33] = vi; }
                }
            }
            const bool last = (l == P - 1) || (grp_start(l + 1) != grp_start(l));
            if (last) {
                const int nval = (l + 1) * (l + 1) - g0, g = grp_index(l);
                __syncwarp();
#pragma unroll
                for (int slot = 0; slot < 2; ++slot) {
                    const int k = lane + 32 * slot;
                    if (32 * slot < nval && k < nval) {
                        const double *rowp = tbl + k * 33;
                        double sum = 0.0;
#pragma unroll 8
                        for (int j = 0; j < 32; ++j) sum += rowp[j];
                        acc[2 * g + slot] += sum;
                    }
                }
                __syncwarp();
            }
        }
    }
    // group-local value k of group g is (l, m, part) in degree-major order l^2 + (0 | 2m-1 | 2m); store it at its
    // place in the split layout (harmonics.cuh); everything else of the row (padding, degrees >= p) is zero
    double *M = Mout + (size_t)leaf * nst;
    constexpr int NRE = ((P * (P + 1) / 2 + 7) / 8) * 8;
    for (int k = lane; k < nst; k += 32) M[k] = 0.0;
    __syncwarp();
#pragma unroll
    for (int l = 0; l < P; ++l) {
        const bool last = (l == P - 1) || (grp_start(l + 1) != grp_start(l));
        if (last) {
            const int g0 = grp_start(l) * grp_start(l), nval = (l + 1) * (l + 1) - g0, g = grp_index(l);
#pragma unroll
            for (int slot = 0; slot < 2; ++slot) {
                const int k = lane + 32 * slot;
                if (32 * slot < nval && k < nval) {
                    const int o = g0 + k;
                    int ll = (int)sqrt((double)o);
                    while (ll * ll > o) --ll;
                    while ((ll + 1) * (ll + 1) <= o) ++ll;
                    const int r = o - ll * ll, m = (r + 1) >> 1, part = (r > 0 && !(r & 1)) ? 1 : 0;
                    if (ll < p) M[real_idx(ll, m, part, NRE)] = acc[2 * g + slot];
                }
            }
        }
    }
    __syncwarp();
    }
}

// level / nleaf / list / sbegin: the leaves of one level (uniform tree: all boxes of level lmax, list = null)
template <int P>
static void p2m_launch(bem_ctx *c, int lmax, int nleaf, const int32_t *list, const int32_t *sbegin)
{
    const BoxSet &sb = c->sb;
    if (nleaf == 0) return;
    const double h = c->cube_side / (double)(1 << lmax);
    const size_t smem = (size_t)P2M_WARPS * P2M_TBL * sizeof(double);
    static std::vector<char> attr_done;
    once_per_device(attr_done, c->device, [&]() {
        CUDA_TRY(cudaFuncSetAttribute(p2m_kernel_t<P, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        CUDA_TRY(cudaFuncSetAttribute(p2m_kernel_t<P, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    });
    auto kern = c->has_dipole ? p2m_kernel_t<P, true> : p2m_kernel_t<P, false>;
    CUDA_TRY(cudaMemsetAsync(c->p2p_counter.get() + 2, 0, sizeof(int), c->stream));
    const int grid = std::max(1, std::min(cdiv(nleaf, P2M_WARPS), P2M_MINB * c->n_sm));     // the CTAs that fit an SM (registers, shared memory)
    kern<<<grid, P2M_WARPS * 32, smem, c->stream>>>(
        sbegin, sb.bkey[lmax].get(), list, nleaf, c->cube_min[0], c->cube_min[1], c->cube_min[2], h,
        c->src_pos.get(), c->src_str.get(), c->p, c->nst, c->Mexp.get() + (size_t)sb.base[lmax] * c->nst, c->p2p_counter.get() + 2);
    KERNEL_CHECK();
}

void launch_p2m_generic(bem_ctx *c, int level, int nleaf, const int32_t *list, const int32_t *sbegin);   // translate.cu

static void launch_p2m_level(bem_ctx *c, int level, int nleaf, const int32_t *list, const int32_t *sbegin)
{
    const int p = c->pl;                                          // the layout degree: the kernels store rows of its size
    if (p == 11) p2m_launch<11>(c, level, nleaf, list, sbegin);
    else if (p == 13) p2m_launch<13>(c, level, nleaf, list, sbegin);
    else if (p <= 4) p2m_launch<4>(c, level, nleaf, list, sbegin);
    else if (p <= 6) p2m_launch<6>(c, level, nleaf, list, sbegin);
    else if (p <= 8) p2m_launch<8>(c, level, nleaf, list, sbegin);
    else if (p <= 10) p2m_launch<10>(c, level, nleaf, list, sbegin);
    else if (p <= 12) p2m_launch<12>(c, level, nleaf, list, sbegin);
    else if (p <= 14) p2m_launch<14>(c, level, nleaf, list, sbegin);
    else if (p <= 16) p2m_launch<16>(c, level, nleaf, list, sbegin);
    else launch_p2m_generic(c, level, nleaf, list, sbegin);
}

void launch_p2m(bem_ctx *c)
{
    if (!c->adaptive) { launch_p2m_level(c, c->sb.lmax, c->sb.nbox[c->sb.lmax], nullptr, c->sb.begin.get()); return; }
    for (int l = 2; l <= c->sb.lmax; ++l)                         // adaptive tree: the source leaves of every level
        launch_p2m_level(c, l, c->ad.n_sleaf[l], c->ad.sleaf[l].get(), c->ad.s_pbeg[l].get());
}

// ------------------------------------------------------------------ L2P
// One thread per target; threads of a warp mostly share the leaf, so coefficient loads are broadcasts.
template <int P>
__global__ void __launch_bounds__(128)
l2p_kernel_t(const double *__restrict__ tgt, int64_t nt, const int32_t *__restrict__ leaf_of, const uint64_t *__restrict__ tkey,
             const uint8_t *__restrict__ lev_all, double cmx, double cmy, double cmz, double h, int p, int nst,
             const double *__restrict__ Lleaf, double *__restrict__ y)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nt) return;
    const int leaf = leaf_of[t];
    if (lev_all) h = ldexp(h, -(int)lev_all[leaf]);              // adaptive tree: leaf_of / tkey / Lleaf are indexed by the global box id; h = cube side
    uint32_t ix, iy, iz;
    morton_decode(tkey[leaf], &ix, &iy, &iz);
    const double ih = 1.0 / h;
    const double bx = (tgt[3 * t] - (cmx + (ix + 0.5) * h)) * ih;
    const double by = (tgt[3 * t + 1] - (cmy + (iy + 0.5) * h)) * ih;
    const double bz = (tgt[3 * t + 2] - (cmz + (iz + 0.5) * h)) * ih;
    const double r2 = bx * bx + by * by + bz * bz;
    const double *L = Lleaf + (size_t)leaf * nst;
    double Rre[2][P], Rim[2][P];
    double phi = 0.0;
#pragma unroll
    for (int l = 0; l < P; ++l) {
        next_row<P>(l, bx, by, bz, r2, Rre, Rim);
        if (l < p) {
            const int cur = l & 1;
            constexpr int NRE = ((P * (P + 1) / 2 + 7) / 8) * 8;
            const double *Lre = L + l * (l + 1) / 2, *Lim = Lre + NRE;                        // split layout (harmonics.cuh)
            double row = 0.0;
#pragma unroll
            for (int m = 1; m < P; ++m)
                if (m <= l) row = fma(__ldg(Lre + m), Rre[cur][m], fma(__ldg(Lim + m), Rim[cur][m], row));
            phi += fma(2.0, row, __ldg(Lre) * Rre[cur][0]);
        }
    }
    y[t] = phi;
}

template <int P>
static void l2p_launch(bem_ctx *c, const int32_t *leaf_of)
{
    const BoxSet &tb = c->tb;
    const int lmax = tb.lmax;
    const double h = c->cube_side / (double)(1 << lmax);
    if (c->adaptive)
        l2p_kernel_t<P><<<cdiv(c->N, 128), 128, 0, c->stream>>>(c->tgt_pos.get(), c->N, c->ad.pt_gbox.get(), c->ad.tkey_all.get(), c->ad.tlev_all.get(),
                                                                c->cube_min[0], c->cube_min[1], c->cube_min[2], c->cube_side, c->p, c->nst,
                                                                c->Lexp.get(), c->ypart.get());
    else
    l2p_kernel_t<P><<<cdiv(c->N, 128), 128, 0, c->stream>>>(c->tgt_pos.get(), c->N, leaf_of, tb.bkey[lmax].get(), nullptr,
                                                            c->cube_min[0], c->cube_min[1], c->cube_min[2], h, c->p, c->nst,
                                                            c->Lexp.get() + (size_t)tb.base[lmax] * c->nst, c->ypart.get());
    KERNEL_CHECK();
}

void launch_l2p_generic(bem_ctx *c, const int32_t *leaf_of);   // translate.cu

void launch_l2p(bem_ctx *c, const int32_t *leaf_of)
{
    const int p = c->pl;
    if (p == 11) l2p_launch<11>(c, leaf_of);
    else if (p == 13) l2p_launch<13>(c, leaf_of);
    else if (p <= 4) l2p_launch<4>(c, leaf_of);
    else if (p <= 6) l2p_launch<6>(c, leaf_of);
    else if (p <= 8) l2p_launch<8>(c, leaf_of);
    else if (p <= 10) l2p_launch<10>(c, leaf_of);
    else if (p <= 12) l2p_launch<12>(c, leaf_of);
    else if (p <= 14) l2p_launch<14>(c, leaf_of);
    else if (p <= 16) l2p_launch<16>(c, leaf_of);
    else launch_l2p_generic(c, leaf_of);
}

}  // namespace bem
