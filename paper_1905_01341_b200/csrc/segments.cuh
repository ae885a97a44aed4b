// The source list of one target leaf in the near-field kernels (p2p.cu, p2p_f32.cu): the sources of its (up to 27)
// neighbouring source leaves and of the leaf-level far boxes that are summed directly (tree.cu, option direct_pairs;
// up to 189), treated as ONE concatenated list of S sources.  Segment k is a source leaf: its first source seg_s0[k]
// and the prefix sums seg_pre[k] of the leaf sizes; entries beyond the last segment hold S so that a search never
// leaves the list.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bem {

constexpr int SEG_MAX = 256;          // 27 + 189 segments (uniform tree), rounded up; the longest CSR row an adaptive tree may have

// called by warp 0 of the CTA; per_segment(k, b) is called by the lane that owns segment k (b = source leaf or -1)
template <class F>
__device__ __forceinline__ void build_segments(int lane, int leaf, const int32_t *__restrict__ nbr, const int32_t *__restrict__ xptr,
                                               const int32_t *__restrict__ xsrc, const int32_t *__restrict__ sbegin,
                                               int *seg_s0, int *seg_pre, int *seg_n, F per_segment)
{
    const int x0 = xptr ? xptr[leaf] : 0, nx = xptr ? xptr[leaf + 1] - x0 : 0;
    const int nseg = 27 + nx;
    int run = 0;
    for (int base = 0; base < nseg; base += 32) {
        const int e = base + lane;
        int b = -1;
        if (e < 27) b = nbr[(int64_t)leaf * 27 + e];
        else if (e < nseg) b = xsrc[x0 + e - 27];
        int s0 = 0, cnt = 0;
        if (b >= 0) { s0 = sbegin[b]; cnt = sbegin[b + 1] - s0; }
        int inc = cnt;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
        if (e < SEG_MAX) { seg_s0[e] = s0; seg_pre[e + 1] = run + inc; per_segment(e, b); }
        run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) { seg_pre[0] = 0; *seg_n = nseg; }
    for (int e = ((nseg + 31) & ~31) + lane; e < SEG_MAX; e += 32) seg_pre[e + 1] = run;
}

// adaptive tree (adaptive.cu): the source list of a target leaf is a CSR row of (first source, count) ranges -- the boxes of
// its own level that touch it, the coarser source leaves that touch its ancestors, and the far leaves summed directly
__device__ __forceinline__ void build_segments_csr(int lane, int leaf, const int32_t *__restrict__ near_ptr, const int2 *__restrict__ near_rng,
                                                   int *seg_s0, int *seg_pre, int *seg_n)
{
    const int x0 = near_ptr[leaf], nseg = min(near_ptr[leaf + 1] - x0, SEG_MAX);     // bem_setup refuses longer rows
    int run = 0;
    for (int base = 0; base < nseg; base += 32) {
        const int e = base + lane;
        int2 r = make_int2(0, 0);
        if (e < nseg) r = near_rng[x0 + e];
        int inc = r.y;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
        if (e < SEG_MAX) { seg_s0[e] = r.x; seg_pre[e + 1] = run + inc; }
        run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) { seg_pre[0] = 0; *seg_n = nseg; }
    for (int e = ((nseg + 31) & ~31) + lane; e < SEG_MAX; e += 32) seg_pre[e + 1] = run;
}

// last k with seg_pre[k] <= g, for 0 <= g < S
__device__ __forceinline__ int find_segment(const int *seg_pre, int nseg, int g)
{
    int k = 0;
    if (nseg > 32) {                                                   // warp-uniform
        if (seg_pre[128] <= g) k = 128;
        if (seg_pre[k + 64] <= g) k += 64;
        if (seg_pre[k + 32] <= g) k += 32;
    }
    if (seg_pre[k + 16] <= g) k += 16;
    if (seg_pre[k + 8] <= g) k += 8;
    if (seg_pre[k + 4] <= g) k += 4;
    if (seg_pre[k + 2] <= g) k += 2;
    if (seg_pre[k + 1] <= g) k += 1;
    return k;
}

}  // namespace bem
