// Steps a4 (lift), a10 / a10' (P2P near field and direct-sum mode) and
// a11 + a12 (correction SpMV, combine, un-permute) of DESIGN.md.
//
// Point engine: Phi(x) = sum_s [ m_s / |x - y_s| - d_s.(x - y_s)/|x - y_s|^3 ],  y = Phi/(4 pi)
// (Eq. 13, with monopole strengths q.w and dipole strengths phi.N.w).
// This is the paper's A^(sparse) X, the part it runs on the GPU,
// and, over all pairs, its brute-force product.
#include "common.cuh"

namespace bem {

constexpr double INV_4PI = 0.079577471545947667884441881686257;

// ------------------------------------------------------------------ lift (a4)
// m = w (2/3 q[v0] + 1/6 q[v1] + 1/6 q[v2]),  d = w N (2/3 phi[v0] + 1/6 phi[v1] + 1/6 phi[v2])
// (P1 interpolation at the Gauss point; in V1 v0 = v1 = v2 = j, w = s_j, N = n_j: Eq. 17)
__global__ void lift_kernel(const double *__restrict__ q, const double *__restrict__ phi,
                            const double4 *__restrict__ lw, const int4 *__restrict__ lv, int64_t ns,
                            double4 *__restrict__ str)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    const int4 v = lv[s];
    const double4 w = lw[s];
    const double a = 2.0 / 3.0, b = 1.0 / 6.0;
    double qq = 0.0, ff = 0.0;
    if (q) qq = a * q[v.x] + b * q[v.y] + b * q[v.z];
    if (phi) ff = a * phi[v.x] + b * phi[v.y] + b * phi[v.z];
    str[s] = make_double4(w.x * qq, w.y * ff, w.z * ff, w.w * ff);
}

void launch_lift(bem_ctx *c, const double *q, const double *phi)
{
    lift_kernel<<<cdiv(c->ns, 256), 256, 0, c->stream>>>(q, phi, c->lift_w.get(), c->lift_vid.get(), c->ns, c->src_str.get());
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ pair kernel
// one (target, source) interaction; r2 == 0 (V1: source j = target i; "i != j") adds nothing
__device__ __forceinline__ double pair_term(double tx, double ty, double tz, const double4 &sp, const double4 &ss)
{
    const double dx = tx - sp.x, dy = ty - sp.y, dz = tz - sp.z;
    const double r2 = dx * dx + dy * dy + dz * dz;
    const double inv = r2 > 0.0 ? rsqrt(r2) : 0.0;
    const double dd = ss.y * dx + ss.z * dy + ss.w * dz;
    // m/r - (d.dx)/r^3 = inv * (m - dd * inv^2)
    return inv * (ss.x - dd * (inv * inv));
}

constexpr int P2P_THREADS = 128;
constexpr int P2P_TILE = 128;

// ------------------------------------------------------------------ direct mode (a10')
// grid = (target blocks, source splits); thread = one target; sources staged through shared memory
__global__ void __launch_bounds__(P2P_THREADS)
p2p_direct_kernel(const double *__restrict__ tgt, int64_t nt, const double4 *__restrict__ spos,
                  const double4 *__restrict__ sstr, int64_t ns, int64_t chunk, double *__restrict__ ypart)
{
    __shared__ double4 sp[P2P_TILE], ss[P2P_TILE];
    const int64_t t = (int64_t)blockIdx.x * P2P_THREADS + threadIdx.x;
    double tx = 0, ty = 0, tz = 0;
    if (t < nt) { tx = tgt[3 * t]; ty = tgt[3 * t + 1]; tz = tgt[3 * t + 2]; }
    const int64_t s0 = (int64_t)blockIdx.y * chunk, s1 = min(s0 + chunk, ns);
    double acc = 0.0;
    for (int64_t base = s0; base < s1; base += P2P_TILE) {
        const int n = (int)min((int64_t)P2P_TILE, s1 - base);
        __syncthreads();
        if (threadIdx.x < n) { sp[threadIdx.x] = spos[base + threadIdx.x]; ss[threadIdx.x] = sstr[base + threadIdx.x]; }
        __syncthreads();
#pragma unroll 4
        for (int j = 0; j < n; ++j) acc += pair_term(tx, ty, tz, sp[j], ss[j]);
    }
    if (t < nt) ypart[(int64_t)blockIdx.y * nt + t] = acc;
}

void launch_p2p_direct(bem_ctx *c)
{
    const int64_t chunk = (c->ns + c->nsplit - 1) / c->nsplit;
    dim3 grid(cdiv(c->N, P2P_THREADS), c->nsplit);
    p2p_direct_kernel<<<grid, P2P_THREADS, 0, c->stream>>>(c->tgt_pos.get(), c->N, c->src_pos.get(), c->src_str.get(),
                                                           c->ns, chunk, c->ypart.get());
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ FMM near field (a10)
// One CTA per target leaf.  The 128 threads are arranged as TT targets x SS source
// slices (TT * SS = 128, SS the largest power of two with TT >= targets in the leaf,
// at most 32): lanes of a warp hold different targets and read the same source from shared
// memory (a broadcast), slices are summed at the end in a fixed order -- no atomics,
// so two runs agree bit for bit.  y (engine order) already holds the far field (L2P).
__global__ void __launch_bounds__(P2P_THREADS)
p2p_leaf_kernel(const double *__restrict__ tgt, const int32_t *__restrict__ tbegin, const int32_t *__restrict__ nbr,
                const int32_t *__restrict__ sbegin, const double4 *__restrict__ spos, const double4 *__restrict__ sstr,
                double *__restrict__ y)
{
    __shared__ double4 sp[P2P_TILE], ss[P2P_TILE];
    __shared__ double red[P2P_THREADS];
    __shared__ int nb_s[27];
    const int leaf = blockIdx.x;
    const int t0 = tbegin[leaf], nt = tbegin[leaf + 1] - t0;
    if (threadIdx.x < 27) nb_s[threadIdx.x] = nbr[(int64_t)leaf * 27 + threadIdx.x];
    for (int c0 = 0; c0 < nt; c0 += P2P_THREADS) {
        const int ntc = min(nt - c0, P2P_THREADS);
        int SS = 1;
        while (SS < 32 && ntc * (SS * 2) <= P2P_THREADS) SS *= 2;
        const int TT = P2P_THREADS / SS;
        const int tl = threadIdx.x % TT, sl = threadIdx.x / TT;
        const bool active = tl < ntc;
        double tx = 0, ty = 0, tz = 0;
        if (active) { const int64_t t = t0 + c0 + tl; tx = tgt[3 * t]; ty = tgt[3 * t + 1]; tz = tgt[3 * t + 2]; }
        double acc = 0.0;
        __syncthreads();
        for (int k = 0; k < 27; ++k) {
            const int sbx = nb_s[k];
            if (sbx < 0) break;
            const int s0 = sbegin[sbx], s1 = sbegin[sbx + 1];
            for (int base = s0; base < s1; base += P2P_TILE) {
                const int n = min(P2P_TILE, s1 - base);
                __syncthreads();
                if (threadIdx.x < n) { sp[threadIdx.x] = spos[base + threadIdx.x]; ss[threadIdx.x] = sstr[base + threadIdx.x]; }
                __syncthreads();
                if (active)
                    for (int j = sl; j < n; j += SS) acc += pair_term(tx, ty, tz, sp[j], ss[j]);
            }
        }
        __syncthreads();
        red[threadIdx.x] = acc;
        __syncthreads();
        if (sl == 0 && active) {
            double sum = 0.0;
            for (int s = 0; s < SS; ++s) sum += red[s * TT + tl];
            y[t0 + c0 + tl] += sum;
        }
    }
}

void launch_p2p_leaves(bem_ctx *c)
{
    const int nleaf = c->tb.nbox[c->tb.lmax];
    p2p_leaf_kernel<<<nleaf, P2P_THREADS, 0, c->stream>>>(c->tgt_pos.get(), c->tb.begin.get(), c->nbr.get(), c->sb.begin.get(),
                                                          c->src_pos.get(), c->src_str.get(), c->ypart.get());
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ SpMV + combine (a11, a12)
// y_i = (1/4pi) sum_split ypart[split][map(i)] + sum_j ( C^S_ij q_j - C^D_ij phi_j ) [+ L_ii q_i - M_ii phi_i in V1]
// 8 lanes per row: consecutive lanes read consecutive (col, val) entries -- coalesced 4 B + 16 B loads.
constexpr int SPMV_LANES = 8;
__global__ void __launch_bounds__(256)
spmv_combine_kernel(const int64_t *__restrict__ rowptr, const int32_t *__restrict__ col, const double2 *__restrict__ val,
                    const double *__restrict__ q, const double *__restrict__ phi,
                    const double *__restrict__ ypart, int nsplit, const uint32_t *__restrict__ map,
                    const double *__restrict__ diagL, const double *__restrict__ diagM,
                    int64_t N, double *__restrict__ y)
{
    const int64_t gid = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    const int64_t i = gid / SPMV_LANES;
    const int lane = (int)(gid % SPMV_LANES);
    double acc = 0.0;
    if (i < N) {
        const int64_t b = rowptr[i], e = rowptr[i + 1];
        for (int64_t k = b + lane; k < e; k += SPMV_LANES) {
            const int j = col[k];
            const double2 v = val[k];
            if (q) acc += v.x * q[j];
            if (phi) acc -= v.y * phi[j];
        }
    }
#pragma unroll
    for (int d = SPMV_LANES / 2; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if (i < N && lane == 0) {
        const int64_t m = map ? map[i] : i;
        double far = 0.0;
        for (int s = 0; s < nsplit; ++s) far += ypart[(int64_t)s * N + m];
        double out = INV_4PI * far + acc;
        if (diagL) {
            if (q) out += diagL[i] * q[i];
            if (phi) out -= diagM[i] * phi[i];
        }
        y[i] = out;
    }
}

void launch_spmv_combine(bem_ctx *c, const double *q, const double *phi, double *y)
{
    const int64_t nthreads = c->N * SPMV_LANES;
    spmv_combine_kernel<<<cdiv(nthreads, 256), 256, 0, c->stream>>>(
        c->rowptr.get(), c->col.get(), c->val.get(), q, phi, c->ypart.get(), c->nsplit,
        c->mode == 0 ? c->tgt_inv.get() : nullptr,
        c->have_diag ? c->diagL.get() : nullptr, c->have_diag ? c->diagM.get() : nullptr, c->N, y);
    KERNEL_CHECK();
}

}  // namespace bem
