// Step a10 of DESIGN.md with SINGLE-PRECISION pair arithmetic (option "p2p_precision" = 1).
//
// The paper runs A^(sparse) X on the GPU "with single and double precision" and finds that
// "up to p_fmm = 12 the accuracy of the MVP practically is not affected by the precision of GPU computing"
// (Table 1: single 4e-7 vs double 4e-7 at p = 12; floor 5e-8 .. 2e-7 at p = 16, 20).
//
// What is single and what is not:
//  * positions are taken RELATIVE TO THE CENTRE OF THEIR OWN LEAF and divided by the leaf edge h in fp64, and
//    only then rounded to fp32 (sources once, at first use; targets when a pass stages them); the offset
//    between a source leaf and the target leaf is a small integer vector, added in fp32 -- the cancellation
//    in x - y happens between numbers of size <= 1.5, so the difference carries an absolute error ~1e-7 h
//    whatever the size of the cluster;
//  * strengths are scaled in fp64 (m/h, d/h^2: the sum is then in physical units) and rounded to fp32 by the
//    lift kernel;
//  * per pair: 12 FP32 instructions + MUFU.RSQ (7 + MUFU without dipoles);
//  * a lane adds the pairs of at most F_FLUSH rounds (2 F_FLUSH pairs per target) in fp32; these partial sums
//    are then converted to fp64 and summed over the lanes by a transposed butterfly, and everything across
//    lanes, warps and rounds is fp64 in a fixed order (bit-reproducible).
//
// The FP32 pipes are idle while the FP64 pipe runs the translations (DMMA) and P2M, so this kernel is a
// PERSISTENT grid of a few CTAs per SM (dynamic leaf counter) that bem_apply launches right after the lift,
// beside the whole far-field pass.
#include "common.cuh"
#include "morton.cuh"
#include "segments.cuh"
#include <algorithm>

namespace bem {

constexpr int F_THREADS = 128;
#ifndef F_MINB
#define F_MINB 6                    // CTAs per SM the register allocation allows (80 registers)
#endif
#ifndef F_SPL_N
#define F_SPL_N 1
#endif
constexpr int F_SPL = F_SPL_N;       // sources per lane and round: one shared-memory target read feeds F_SPL pairs
constexpr int F_WARPS = F_THREADS / 32;
constexpr int F_NT = 32;             // targets per pass (fp32 accumulators per lane)
constexpr int F_FLUSH = 8;           // rounds between two flushes of the fp32 partial sums

// SELF: a source may coincide with a target (V1: j = i, "i != j"; point clouds) -> adds nothing
template <bool DIP, bool SELF>
__device__ __forceinline__ float pair_f32(float acc, const float4 t, float sx, float sy, float sz, float m, float ax, float ay, float az)
{
    const float dx = t.x - sx, dy = t.y - sy, dz = t.z - sz;
    const float r2 = fmaf(dx, dx, fmaf(dy, dy, dz * dz));
    float inv;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(r2));
    if (SELF) inv = r2 > 0.0f ? inv : 0.0f;
    if (!DIP) return fmaf(inv, m, acc);
    const float dd = fmaf(ax, dx, fmaf(ay, dy, az * dz));
    return fmaf(inv, fmaf(-dd, inv * inv, m), acc);      // m/r - (d.dx)/r^3
}

// a shared-memory target.  volatile: the targets do not change inside the round loop, and the compiler would
// otherwise hoist all of them (64 registers) out of it.
template <int OFF>
__device__ __forceinline__ float4 lds_target(unsigned base)
{
    float4 t;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];" : "=f"(t.x), "=f"(t.y), "=f"(t.z), "=f"(t.w) : "r"(base), "n"(OFF));
    return t;
}
template <bool DIP, bool SELF, int T>
__device__ __forceinline__ void target_f32(float (&facc)[F_NT], unsigned tg_base, const float4 (&sp)[F_SPL], const float4 (&ss)[F_SPL])
{
    const float4 X = lds_target<16 * T>(tg_base);
#pragma unroll
    for (int j = 0; j < F_SPL; ++j) facc[T] = pair_f32<DIP, SELF>(facc[T], X, sp[j].x, sp[j].y, sp[j].z, ss[j].x, ss[j].y, ss[j].z, ss[j].w);
}

// fp32 source records (setup / first use): position relative to the centre of the source's own leaf, in leaf edges
__global__ void build_src_f32(const double4 *__restrict__ spos, const int32_t *__restrict__ leaf_of, const uint64_t *__restrict__ skey,
                              int64_t ns, double cx0, double cy0, double cz0, double h, float4 *__restrict__ out)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    uint32_t ix, iy, iz;
    morton_decode(skey[leaf_of[s]], &ix, &iy, &iz);
    const double4 p = spos[s];
    const double ih = 1.0 / h;
    out[s] = make_float4((float)((p.x - (cx0 + (ix + 0.5) * h)) * ih), (float)((p.y - (cy0 + (iy + 0.5) * h)) * ih),
                         (float)((p.z - (cz0 + (iz + 0.5) * h)) * ih), 0.0f);
}

// NTT targets (4, 8, 16, 24 or 32; straight-line code: NTT independent chains) against the F_SPL sources of the lane
template <bool DIP, bool SELF, int NTT>
__device__ __forceinline__ void round_f32(float (&facc)[F_NT], unsigned tg_base, const float4 (&sp)[F_SPL], const float4 (&ss)[F_SPL])
{
    target_f32<DIP, SELF, 0>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 1>(facc, tg_base, sp, ss);
    target_f32<DIP, SELF, 2>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 3>(facc, tg_base, sp, ss);
    if (NTT > 4) {
        target_f32<DIP, SELF, 4>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 5>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 6>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 7>(facc, tg_base, sp, ss);
    }
    if (NTT > 8) {
        target_f32<DIP, SELF, 8>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 9>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 10>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 11>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 12>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 13>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 14>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 15>(facc, tg_base, sp, ss);
    }
    if (NTT > 16) {
        target_f32<DIP, SELF, 16>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 17>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 18>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 19>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 20>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 21>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 22>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 23>(facc, tg_base, sp, ss);
    }
    if (NTT > 24) {
        target_f32<DIP, SELF, 24>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 25>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 26>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 27>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 28>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 29>(facc, tg_base, sp, ss);
        target_f32<DIP, SELF, 30>(facc, tg_base, sp, ss); target_f32<DIP, SELF, 31>(facc, tg_base, sp, ss);
    }
}

template <bool DIP, bool SELF>
__global__ void __launch_bounds__(F_THREADS, F_MINB)
p2p_leaf_kernel_f32(const double *__restrict__ tgt, const int32_t *__restrict__ tbegin, const uint64_t *__restrict__ tkey,
                    const int32_t *__restrict__ nbr, const int32_t *__restrict__ xptr, const int32_t *__restrict__ xsrc,
                    const int32_t *__restrict__ sbegin, const uint64_t *__restrict__ skey,
                    const float4 *__restrict__ spos, const float4 *__restrict__ sstr,
                    double cx0, double cy0, double cz0, double h, int leaf0, int nleaf, int *__restrict__ counter,
                    double *__restrict__ y)
{
    __shared__ float4 tg[F_NT];
    __shared__ double red[F_WARPS][F_NT];
    __shared__ int seg_off[SEG_MAX];                                   // (ox + 4) | (oy + 4) << 4 | (oz + 4) << 8
    __shared__ int seg_s0[SEG_MAX], seg_pre[SEG_MAX + 1], seg_n;
    __shared__ int cur_leaf;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const double inv_h = 1.0 / h;
    const unsigned tg_base = (unsigned)__cvta_generic_to_shared(tg);

    for (;;) {
        __syncthreads();                                               // everything of the previous leaf is consumed
        if (threadIdx.x == 0) cur_leaf = leaf0 + atomicAdd(counter, 1);
        __syncthreads();
        const int leaf = cur_leaf;
        if (leaf >= nleaf) return;
        const int t0 = tbegin[leaf], nt = tbegin[leaf + 1] - t0;
        uint32_t ix, iy, iz;
        morton_decode(tkey[leaf], &ix, &iy, &iz);
        const double cx = cx0 + (ix + 0.5) * h, cy = cy0 + (iy + 0.5) * h, cz = cz0 + (iz + 0.5) * h;
        if (warp == 0)
            build_segments(lane, leaf, nbr, xptr, xsrc, sbegin, seg_s0, seg_pre, &seg_n, [&](int k, int b) {
                int off = 0x444;                                       // source leaf - target leaf, in leaf edges (|.| <= 3)
                if (b >= 0) {
                    uint32_t jx, jy, jz;
                    morton_decode(skey[b], &jx, &jy, &jz);
                    off = ((int)jx - (int)ix + 4) | ((int)jy - (int)iy + 4) << 4 | ((int)jz - (int)iz + 4) << 8;
                }
                seg_off[k] = off;
            });
        __syncthreads();
        const int S = seg_pre[SEG_MAX];
        const int rounds = (S + F_THREADS * F_SPL - 1) / (F_THREADS * F_SPL);

        // source g of the concatenated neighbour list, moved into the frame of the target leaf
        // (g only grows from one round to the next: the segment index k of a lane's source moves forward)
        // (the offset of the segment is returned, not added: an add here would wait for the load it prefetches)
        auto load_source = [&](int g, int &k, float4 &p, float4 &q, int &o) {
            if (g < S) {
                while (seg_pre[k + 1] <= g) ++k;                       // last k with seg_pre[k] <= g
                const int idx = seg_s0[k] + (g - seg_pre[k]);
                o = seg_off[k];
                p = spos[idx];
                q = sstr[idx];
            } else {                                                   // far away, zero strength: adds exactly 0
                o = 0x444;
                p = make_float4(1e5f, 0.0f, 0.0f, 0.0f);
                q = make_float4(0.0f, 0.0f, 0.0f, 0.0f);
            }
        };

        for (int c0 = 0; c0 < nt; c0 += F_NT) {
            const int ntc = min(F_NT, nt - c0);
            __syncthreads();                                           // tg / red of the previous group are free
            if (threadIdx.x < F_NT) {
                float4 v = make_float4(0.0f, 0.0f, -1e5f, 0.0f);      // padding target: far from every source
                if (threadIdx.x < ntc) {
                    const int64_t t = t0 + c0 + threadIdx.x;
                    v = make_float4((float)((tgt[3 * t] - cx) * inv_h), (float)((tgt[3 * t + 1] - cy) * inv_h),
                                    (float)((tgt[3 * t + 2] - cz) * inv_h), 0.0f);
                }
                tg[threadIdx.x] = v;
            }
            __syncthreads();
            float facc[F_NT];
#pragma unroll
            for (int t = 0; t < F_NT; ++t) facc[t] = 0.0f;
            double dsum = 0.0;                                         // lane L: running fp64 sum of target L over the warp's lanes
            float4 sp[F_SPL], ss[F_SPL], pn[F_SPL], qn[F_SPL];
            int on[F_SPL];
            int seg[F_SPL];
#pragma unroll
            for (int j = 0; j < F_SPL; ++j) { seg[j] = 0; load_source(j * F_THREADS + threadIdx.x, seg[j], pn[j], qn[j], on[j]); }
#pragma unroll 1
            for (int r = 0; r < rounds; ++r) {
#pragma unroll
                for (int j = 0; j < F_SPL; ++j) {
                    sp[j] = make_float4(pn[j].x + (float)((on[j] & 15) - 4), pn[j].y + (float)((on[j] >> 4 & 15) - 4), pn[j].z + (float)((on[j] >> 8) - 4), 0.0f);
                    ss[j] = qn[j];
                }
                if (r + 1 < rounds) {                                  // prefetch the next round
#pragma unroll
                    for (int j = 0; j < F_SPL; ++j) load_source(((r + 1) * F_SPL + j) * F_THREADS + threadIdx.x, seg[j], pn[j], qn[j], on[j]);
                }
                if (ntc > 24) round_f32<DIP, SELF, 32>(facc, tg_base, sp, ss);          // warp-uniform
                else if (ntc > 16) round_f32<DIP, SELF, 24>(facc, tg_base, sp, ss);
                else if (ntc > 8) round_f32<DIP, SELF, 16>(facc, tg_base, sp, ss);
                else if (ntc > 4) round_f32<DIP, SELF, 8>(facc, tg_base, sp, ss);
                else round_f32<DIP, SELF, 4>(facc, tg_base, sp, ss);
                if ((r % F_FLUSH) == F_FLUSH - 1 || r == rounds - 1) {
                    // fp32 partial sums -> fp64, transposed butterfly: afterwards d[0] of lane L = sum over the lanes of facc[L]
                    double d[F_NT / 2];
#pragma unroll
                    for (int i = 0; i < F_NT / 2; ++i) {               // first step (lane distance 16) fused with the conversion
                        const bool up = (lane & 16) != 0;
                        const double send = (double)(up ? facc[i] : facc[i + 16]);
                        const double keep = (double)(up ? facc[i + 16] : facc[i]);
                        d[i] = keep + __shfl_xor_sync(0xffffffffu, send, 16);
                    }
#pragma unroll
                    for (int off = F_NT / 4; off >= 1; off >>= 1) {
                        const bool up = (lane & off) != 0;
#pragma unroll
                        for (int i = 0; i < off; ++i) {
                            const double send = up ? d[i] : d[i + off];
                            const double keep = up ? d[i + off] : d[i];
                            d[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
                        }
                    }
                    dsum += d[0];
#pragma unroll
                    for (int t = 0; t < F_NT; ++t) facc[t] = 0.0f;
                }
            }
            red[warp][lane] = dsum;
            __syncthreads();
            if (threadIdx.x < ntc) {
                double sum = red[0][threadIdx.x];
#pragma unroll
                for (int w = 1; w < F_WARPS; ++w) sum += red[w][threadIdx.x];
                y[t0 + c0 + threadIdx.x] = sum;
            }
        }
    }
}

// fp32 source records are built at the first apply that needs them (bem_setup frees them)
void ensure_p2p_f32(bem_ctx *c)
{
    if (c->src_pos_f.p && c->src_pos_f.n == (size_t)c->ns) return;
    const int lmax = c->sb.lmax;
    const double h = c->cube_side / (double)(1u << lmax);
    c->src_pos_f.alloc(c->ns);
    c->src_str_f.alloc(c->ns);
    build_src_f32<<<cdiv(c->ns, 256), 256, 0, c->stream>>>(c->src_pos.get(), c->sb.leaf_of.get(), c->sb.bkey[lmax].get(), c->ns,
                                                           c->cube_min[0], c->cube_min[1], c->cube_min[2], h, c->src_pos_f.get());
    KERNEL_CHECK();
}

// ctas_per_sm: size of the persistent grid (the kernel shares every SM with the FP64 kernels of the far field)
// leaves [leaf0, leaf1) of the target tree; part = 0 or 1 selects the leaf counter (two parts may be in flight at once)
void launch_p2p_leaves_f32(bem_ctx *c, cudaStream_t stream, int ctas_per_sm, int leaf0, int leaf1, int part)
{
    const int lmax = c->tb.lmax;
    const int nleaf = leaf1;
    if (leaf1 <= leaf0) return;
    const double h = c->cube_side / (double)(1u << lmax);
    const int grid = std::max(1, std::min(leaf1 - leaf0, ctas_per_sm * c->n_sm));
    CUDA_TRY(cudaMemsetAsync(c->p2p_counter.get() + part, 0, sizeof(int), stream));
    const bool self = c->quadrature != 0;
    static std::vector<char> attr_done;
    once_per_device(attr_done, c->device, [&]() {
        // same shared-memory carve-out as the row sums it runs beside (common.cuh): an SM only holds CTAs of one carve-out
        CUDA_TRY(cudaFuncSetAttribute(p2p_leaf_kernel_f32<true, true>, cudaFuncAttributePreferredSharedMemoryCarveout, CORUN_CARVEOUT));
        CUDA_TRY(cudaFuncSetAttribute(p2p_leaf_kernel_f32<true, false>, cudaFuncAttributePreferredSharedMemoryCarveout, CORUN_CARVEOUT));
        CUDA_TRY(cudaFuncSetAttribute(p2p_leaf_kernel_f32<false, true>, cudaFuncAttributePreferredSharedMemoryCarveout, CORUN_CARVEOUT));
        CUDA_TRY(cudaFuncSetAttribute(p2p_leaf_kernel_f32<false, false>, cudaFuncAttributePreferredSharedMemoryCarveout, CORUN_CARVEOUT));
    });
#define BEM_F32_ARGS c->tgt_pos.get(), c->tb.begin.get(), c->tb.bkey[lmax].get(), c->nbr.get(), c->xdir_ptr.p, c->xdir_src.p, c->sb.begin.get(), \
                     c->sb.bkey[lmax].get(), c->src_pos_f.get(), c->src_str_f.get(), c->cube_min[0], c->cube_min[1], \
                     c->cube_min[2], h, leaf0, nleaf, c->p2p_counter.get() + part, c->ypart.get() + c->N
    if (c->has_dipole) {
        if (self) p2p_leaf_kernel_f32<true, true><<<grid, F_THREADS, 0, stream>>>(BEM_F32_ARGS);
        else p2p_leaf_kernel_f32<true, false><<<grid, F_THREADS, 0, stream>>>(BEM_F32_ARGS);
    } else {
        if (self) p2p_leaf_kernel_f32<false, true><<<grid, F_THREADS, 0, stream>>>(BEM_F32_ARGS);
        else p2p_leaf_kernel_f32<false, false><<<grid, F_THREADS, 0, stream>>>(BEM_F32_ARGS);
    }
#undef BEM_F32_ARGS
    KERNEL_CHECK();
}

}  // namespace bem
