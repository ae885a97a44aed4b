// Steps a4 (lift), a10 / a10' (P2P near field and direct-sum mode) and
// a11 + a12 (correction SpMV, combine, un-permute) of DESIGN.md.
//
// Point engine: Phi(x) = sum_s [ m_s / |x - y_s| - d_s.(x - y_s)/|x - y_s|^3 ],  y = Phi/(4 pi)
// (Eq. 13, with monopole strengths q.w and dipole strengths phi.N.w).
// This is the paper's A^(sparse) X, the part it runs on the GPU,
// and, over all pairs, its brute-force product.
#include "common.cuh"
#include "segments.cuh"

namespace bem {

constexpr double INV_4PI = 0.079577471545947667884441881686257;

// ------------------------------------------------------------------ lift (a4)
// m = w (2/3 q[v0] + 1/6 q[v1] + 1/6 q[v2]),  d = w N (2/3 phi[v0] + 1/6 phi[v1] + 1/6 phi[v2])
// (P1 interpolation at the Gauss point; in V1 v0 = v1 = v2 = j, w = s_j, N = n_j: Eq. 17)
__global__ void lift_kernel(const double *__restrict__ q, const double *__restrict__ phi,
                            const double4 *__restrict__ lw, const int4 *__restrict__ lv, int64_t ns,
                            double4 *__restrict__ str, float4 *__restrict__ strf, double ih)
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
    // fp32 near field (p2p_f32.cu): strengths in leaf-edge units, m/h and d/h^2, rounded once
    if (strf) strf[s] = make_float4((float)(w.x * qq * ih), (float)(w.y * ff * ih * ih), (float)(w.z * ff * ih * ih), (float)(w.w * ff * ih * ih));
}

// point cloud (bem_create_points): source j carries the monopole q[j] and the dipole vector (dip[3j], dip[3j+1], dip[3j+2])
__global__ void lift_points_kernel(const double *__restrict__ q, const double *__restrict__ dip, const int4 *__restrict__ lv, int64_t ns,
                                   double4 *__restrict__ str, float4 *__restrict__ strf, double ih)
{
    const int64_t s = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= ns) return;
    const int64_t j = lv[s].x;
    const double m = q ? q[j] : 0.0;
    double dx = 0.0, dy = 0.0, dz = 0.0;
    if (dip) { dx = dip[3 * j]; dy = dip[3 * j + 1]; dz = dip[3 * j + 2]; }
    str[s] = make_double4(m, dx, dy, dz);
    if (strf) strf[s] = make_float4((float)(m * ih), (float)(dx * ih * ih), (float)(dy * ih * ih), (float)(dz * ih * ih));
}

void launch_lift(bem_ctx *c, const double *q, const double *phi)
{
    c->has_dipole = phi != nullptr;                 // the pair and P2M kernels skip the dipole terms otherwise
    const bool f32 = c->mode == 0 && c->p2p_precision == 1;
    const double ih = f32 ? (double)(1u << c->sb.lmax) / c->cube_side : 0.0;
    if (c->quadrature == 2) {
        lift_points_kernel<<<cdiv(c->ns, 256), 256, 0, c->stream>>>(q, phi, c->lift_vid.get(), c->ns, c->src_str.get(),
                                                                    f32 ? c->src_str_f.get() : nullptr, ih);
        KERNEL_CHECK();
        return;
    }
    lift_kernel<<<cdiv(c->ns, 256), 256, 0, c->stream>>>(q, phi, c->lift_w.get(), c->lift_vid.get(), c->ns, c->src_str.get(),
                                                         f32 ? c->src_str_f.get() : nullptr, ih);
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ pair kernel
// 1/sqrt(x) for x > 0 (0 for x == 0) to ~1 ulp: the hardware seed (MUFU.RSQ64H, relative error d ~ 2^-22)
// followed by ONE third-order step  y1 = y0 (1 + e/2 + 3 e^2/8),  e = 1 - x y0^2, whose residual is
// 5 e^3/16 ~ 2.5 d^3 < 1e-19 -- 5 FP64 instructions instead of the two Newton steps and the
// slow-path branch of the library rsqrt (P2P).
// SELF = false: the caller guarantees x > 0 (G3: a Gauss point never coincides with a vertex) and the test is left out
// ORD = 3: that step (direct-sum mode: 1e-12 against the oracle).  ORD = 2: the Newton step y1 = y0 (1 + e/2), which drops
// 3 e^2/8: MUFU.RSQ64H reads the high word of x only, so e is up to ~2e-6 and the dropped term a one-sided <= 4e-13 -- too
// much for the 1e-12 of direct mode, far below the truncation error of the FMM (1e-6 .. 1e-9), whose near field therefore
// runs 16 instead of 17 FP64 instructions per pair (option "p2p_exact" = 1 keeps ORD = 3 there too).
template <bool SELF, int ORD = 3>
__device__ __forceinline__ double rsqrt_pos(double x)
{
    double y0;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y0) : "d"(x));
    if (SELF) y0 = __double2hiint(x) > 0 ? y0 : 0.0;   // x >= 0 here; x == 0 (and subnormal x) -> 0, an integer test off the FP64 pipe
    const double e = fma(-x, y0 * y0, 1.0);
    if (ORD == 2) return fma(y0 * e, 0.5, y0);
    const double pe = fma(0.375, e, 0.5) * e;
    return fma(y0, pe, y0);
}

// one (target, source) interaction; r2 == 0 (V1: source j = target i; "i != j") adds nothing
// acc += that interaction (the last multiply and the accumulation are one FMA)
// DIP = false: monopole sources only (phi == NULL, every product of a GMRES iteration): 12 FP64 instructions instead of 17
template <bool DIP, bool SELF, int ORD = 3>
__device__ __forceinline__ double pair_acc(double acc, double tx, double ty, double tz, const double4 &sp, const double4 &ss)
{
    const double dx = tx - sp.x, dy = ty - sp.y, dz = tz - sp.z;
    const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
    const double inv = rsqrt_pos<SELF, ORD>(r2);
    if (!DIP) return fma(inv, ss.x, acc);
    const double dd = fma(ss.y, dx, fma(ss.z, dy, ss.w * dz));
    // m/r - (d.dx)/r^3 = inv * (m - dd * inv^2)
    return fma(inv, fma(-dd, inv * inv, ss.x), acc);
}

constexpr int P2P_THREADS = 128;
constexpr int P2P_TILE = 256;
constexpr int P2P_TPT = 4;            // direct mode: targets per thread

// ------------------------------------------------------------------ direct mode (a10')
// grid = (target blocks, source splits); thread = FOUR targets, so one shared-memory source read
// (4 x LDS.128, a broadcast) feeds four pairs -- measured with ncu, one target per thread is bound by
// the shared-memory pipe (88% LSU wavefronts at 48% FP64), not by FP64; sources staged in tiles of 256
template <bool DIP, bool SELF>
__global__ void __launch_bounds__(P2P_THREADS)
p2p_direct_kernel(const double *__restrict__ tgt, int64_t nt, const double4 *__restrict__ spos,
                  const double4 *__restrict__ sstr, int64_t ns, int64_t chunk, double *__restrict__ ypart)
{
    __shared__ double4 sp[P2P_TILE], ss[P2P_TILE];
    const int64_t tfirst = (int64_t)blockIdx.x * (P2P_TPT * P2P_THREADS) + threadIdx.x;
    double tx[P2P_TPT], ty[P2P_TPT], tz[P2P_TPT], acc[P2P_TPT];
#pragma unroll
    for (int k = 0; k < P2P_TPT; ++k) {
        const int64_t t = tfirst + (int64_t)k * P2P_THREADS;
        tx[k] = ty[k] = tz[k] = 0.0;
        acc[k] = 0.0;
        if (t < nt) { tx[k] = tgt[3 * t]; ty[k] = tgt[3 * t + 1]; tz[k] = tgt[3 * t + 2]; }
    }
    const int64_t s0 = (int64_t)blockIdx.y * chunk, s1 = min(s0 + chunk, ns);
    for (int64_t base = s0; base < s1; base += P2P_TILE) {
        const int n = (int)min((int64_t)P2P_TILE, s1 - base);
        __syncthreads();
        for (int i = threadIdx.x; i < n; i += P2P_THREADS) { sp[i] = spos[base + i]; ss[i] = sstr[base + i]; }
        __syncthreads();
#pragma unroll 2
        for (int j = 0; j < n; ++j) {
            const double4 p = sp[j], q = ss[j];
#pragma unroll
            for (int k = 0; k < P2P_TPT; ++k) acc[k] = pair_acc<DIP, SELF>(acc[k], tx[k], ty[k], tz[k], p, q);
        }
    }
#pragma unroll
    for (int k = 0; k < P2P_TPT; ++k) {
        const int64_t t = tfirst + (int64_t)k * P2P_THREADS;
        if (t < nt) ypart[(int64_t)blockIdx.y * nt + t] = acc[k];
    }
}

void launch_p2p_direct(bem_ctx *c)
{
    const int64_t chunk = (c->ns + c->nsplit - 1) / c->nsplit;
    dim3 grid(cdiv(c->N, P2P_TPT * P2P_THREADS), c->nsplit);
    const bool self = c->quadrature != 0;                       // V1 (j = i) and point clouds may have r = 0; G3 cannot
#define BEM_DIRECT(D, S) p2p_direct_kernel<D, S><<<grid, P2P_THREADS, 0, c->stream>>>(c->tgt_pos.get(), c->N, c->src_pos.get(), \
                                                                                      c->src_str.get(), c->ns, chunk, c->ypart.get())
    if (c->has_dipole) { if (self) BEM_DIRECT(true, true); else BEM_DIRECT(true, false); }
    else { if (self) BEM_DIRECT(false, true); else BEM_DIRECT(false, false); }
#undef BEM_DIRECT
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ FMM near field (a10)
// One CTA (4 warps) per target leaf.  The sources of its (up to 27) neighbouring source leaves are
// treated as ONE concatenated list of S sources; LANES HOLD SOURCES (one per lane and round, read
// straight from global memory into registers, 128 per CTA round) and loop over the targets of the
// leaf, 32 at a time, which are broadcast from shared memory (2 x LDS.128 per pair instead of 4, and
// with a warp-uniform address).  Every lane keeps 32 partial sums acc[t] in registers over all its
// rounds; one transposed butterfly (31 shuffle steps) at the end leaves the sum of acc[t] over the
// lanes in lane t, and the 4 warps are added through shared memory -- a fixed order, no atomics, so
// two runs agree bit for bit.  Work is ~ (targets) x ceil(S/128) x 128 pairs whatever the leaf sizes.
// The near field goes to its own slot of ypart (the far field, L2P, may still be running on the side stream).
constexpr int P2P_WARPS = P2P_THREADS / 32;
constexpr int P2P_NT = 16;           // targets per pass (register accumulators per lane); 8, 16 or 32

// (x, y, z) of a shared-memory point.  volatile: the targets do not change inside the round loop, and the
// compiler would otherwise hoist all 32 of them (96 doubles) out of it and spill them to local memory.
__device__ __forceinline__ void lds_point(unsigned addr, double &x, double &y, double &z)
{
    asm volatile("ld.shared.v2.f64 {%0, %1}, [%3];\n\tld.shared.f64 %2, [%3+16];" : "=d"(x), "=d"(y), "=d"(z) : "r"(addr));
}

template <bool DIP, bool SELF, int ORD>
__global__ void __launch_bounds__(P2P_THREADS, 5)
p2p_leaf_kernel(const double *__restrict__ tgt, const int32_t *__restrict__ tbegin, const int32_t *__restrict__ nbr,
                const int32_t *__restrict__ xptr, const int32_t *__restrict__ xsrc,
                const int32_t *__restrict__ sbegin, const double4 *__restrict__ spos, const double4 *__restrict__ sstr,
                double *__restrict__ y)
{
    __shared__ double4 tg[P2P_NT];
    __shared__ double red[P2P_WARPS][P2P_NT];
    __shared__ int seg_s0[SEG_MAX], seg_pre[SEG_MAX + 1], seg_n;
    const int leaf = blockIdx.x;
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int t0 = tbegin[leaf], nt = tbegin[leaf + 1] - t0;
    if (warp == 0) {
        if (nbr) build_segments(lane, leaf, nbr, xptr, xsrc, sbegin, seg_s0, seg_pre, &seg_n, [](int, int) {});
        else build_segments_csr(lane, leaf, xptr, reinterpret_cast<const int2 *>(xsrc), seg_s0, seg_pre, &seg_n);   // adaptive tree
    }
    __syncthreads();
    const int S = seg_pre[SEG_MAX];
    const int rounds = (S + P2P_THREADS - 1) / P2P_THREADS;
    const unsigned tg_base = (unsigned)__cvta_generic_to_shared(tg);

    // source g of the concatenated list; beyond the end a far-away point of zero strength (adds exactly 0)
    // (g only grows from one round to the next: the segment index k of the lane's source moves forward)
    auto load_source = [&](int g, int &k, double4 &p, double4 &q) {
        if (g < S) {
            while (seg_pre[k + 1] <= g) ++k;                           // last k with seg_pre[k] <= g
            const int idx = seg_s0[k] + (g - seg_pre[k]);
            p = spos[idx];
            q = sstr[idx];
        } else {
            p = make_double4(1e100, 0.0, 0.0, 0.0);
            q = make_double4(0.0, 0.0, 0.0, 0.0);
        }
    };

    for (int c0 = 0; c0 < nt; c0 += P2P_NT) {
        const int ntc = min(P2P_NT, nt - c0);
        __syncthreads();                                                // tg / red of the previous group are free
        if (threadIdx.x < P2P_NT) {
            double4 v = make_double4(0.0, 0.0, 0.0, 0.0);
            if (threadIdx.x < ntc) { const int64_t t = t0 + c0 + threadIdx.x; v = make_double4(tgt[3 * t], tgt[3 * t + 1], tgt[3 * t + 2], 0.0); }
            tg[threadIdx.x] = v;
        }
        __syncthreads();
        double acc[P2P_NT];
#pragma unroll
        for (int t = 0; t < P2P_NT; ++t) acc[t] = 0.0;
        double4 p, q, pn, qn;
        int seg = 0;
        load_source(threadIdx.x, seg, pn, qn);
#pragma unroll 1
        for (int r = 0; r < rounds; ++r) {
            p = pn; q = qn;
            if (r + 1 < rounds) load_source((r + 1) * P2P_THREADS + threadIdx.x, seg, pn, qn);   // prefetch the next round
#pragma unroll
            for (int tb = 0; tb < P2P_NT; tb += 8) {                    // 8 independent chains at a time
                if (tb + 8 <= ntc) {                                    // warp-uniform
#pragma unroll
                    for (int t = tb; t < tb + 8; ++t) {
                        double Tx, Ty, Tz;
                        lds_point(tg_base + 32u * t, Tx, Ty, Tz);
                        acc[t] = pair_acc<DIP, SELF, ORD>(acc[t], Tx, Ty, Tz, p, q);
                    }
                } else if (tb < ntc) {                                  // the last 1..7 targets: 4 + singles
                    if (tb + 4 <= ntc) {
#pragma unroll
                        for (int t = tb; t < tb + 4; ++t) {
                            double Tx, Ty, Tz;
                            lds_point(tg_base + 32u * t, Tx, Ty, Tz);
                            acc[t] = pair_acc<DIP, SELF, ORD>(acc[t], Tx, Ty, Tz, p, q);
                        }
#pragma unroll
                        for (int t = tb + 4; t < tb + 7; ++t) {
                            if (t < ntc) {
                                double Tx, Ty, Tz;
                                lds_point(tg_base + 32u * t, Tx, Ty, Tz);
                                acc[t] = pair_acc<DIP, SELF, ORD>(acc[t], Tx, Ty, Tz, p, q);
                            }
                        }
                    } else {
#pragma unroll
                        for (int t = tb; t < tb + 3; ++t) {
                            if (t < ntc) {
                                double Tx, Ty, Tz;
                                lds_point(tg_base + 32u * t, Tx, Ty, Tz);
                                acc[t] = pair_acc<DIP, SELF, ORD>(acc[t], Tx, Ty, Tz, p, q);
                            }
                        }
                    }
                }
            }
        }
        // transposed butterfly: afterwards acc[0] of lane L = sum over the 32 lanes of acc[L % P2P_NT]
#pragma unroll
        for (int off = 16; off >= P2P_NT; off >>= 1) {
#pragma unroll
            for (int i = 0; i < P2P_NT; ++i) acc[i] += __shfl_xor_sync(0xffffffffu, acc[i], off);
        }
#pragma unroll
        for (int off = P2P_NT / 2; off >= 1; off >>= 1) {
            const bool up = (lane & off) != 0;
#pragma unroll
            for (int i = 0; i < off; ++i) {
                const double send = up ? acc[i] : acc[i + off];
                const double keep = up ? acc[i + off] : acc[i];
                acc[i] = keep + __shfl_xor_sync(0xffffffffu, send, off);
            }
        }
        if (lane < P2P_NT) red[warp][lane] = acc[0];
        __syncthreads();
        if (threadIdx.x < ntc) {
            double sum = red[0][threadIdx.x];
#pragma unroll
            for (int w = 1; w < P2P_WARPS; ++w) sum += red[w][threadIdx.x];
            y[t0 + c0 + threadIdx.x] = sum;
        }
    }
}

void launch_p2p_leaves(bem_ctx *c)
{
    const int nleaf = c->adaptive ? c->ad.n_tleaf : c->tb.nbox[c->tb.lmax];
    static std::vector<char> attr_done;
    once_per_device(attr_done, c->device, [&]() {                                                      // same carve-out as the row sums it runs beside (common.cuh)
#define BEM_CARVE(D, S) CUDA_TRY(cudaFuncSetAttribute(p2p_leaf_kernel<D, S, 2>, cudaFuncAttributePreferredSharedMemoryCarveout, CORUN_CARVEOUT)); \
                        CUDA_TRY(cudaFuncSetAttribute(p2p_leaf_kernel<D, S, 3>, cudaFuncAttributePreferredSharedMemoryCarveout, CORUN_CARVEOUT))
        BEM_CARVE(true, true); BEM_CARVE(true, false); BEM_CARVE(false, true); BEM_CARVE(false, false);
#undef BEM_CARVE
    });
    const bool self = c->quadrature != 0;                       // V1 (j = i) and point clouds may have r = 0; G3 cannot
    // adaptive tree: target leaves in point order (ad.tleaf_begin), source ranges from the CSR (ad.near_ptr, ad.near_rng), nbr = null
    const int32_t *tbeg = c->adaptive ? c->ad.tleaf_begin.get() : c->tb.begin.get();
    const int32_t *nbr = c->adaptive ? nullptr : c->nbr.get();
    const int32_t *xp = c->adaptive ? c->ad.near_ptr.get() : c->xdir_ptr.p;
    const int32_t *xs = c->adaptive ? reinterpret_cast<const int32_t *>(c->ad.near_rng.get()) : c->xdir_src.p;
#define BEM_LEAF_O(D, S, O) p2p_leaf_kernel<D, S, O><<<nleaf, P2P_THREADS, 0, c->stream>>>(c->tgt_pos.get(), tbeg, nbr, xp, \
                           xs, c->sb.begin.get(), c->src_pos.get(), c->src_str.get(), c->ypart.get() + c->N)
#define BEM_LEAF(D, S) do { if (c->p2p_exact) BEM_LEAF_O(D, S, 3); else BEM_LEAF_O(D, S, 2); } while (0)
    if (c->has_dipole) { if (self) BEM_LEAF(true, true); else BEM_LEAF(true, false); }
    else { if (self) BEM_LEAF(false, true); else BEM_LEAF(false, false); }
#undef BEM_LEAF
#undef BEM_LEAF_O
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ SpMV + combine (a11, a12)
// y_i = (1/4pi) sum_split ypart[split][map(i)] + sum_j ( C^S_ij q_j - C^D_ij phi_j ) [+ L_ii q_i - M_ii phi_i in V1]
// 4 lanes per row: consecutive lanes read consecutive (col, val) entries -- coalesced 4 B + 16 B loads.
constexpr int SPMV_LANES = 4;          // measured on config 5 (16 entries per row): 1, 2, 4, 8, 16 lanes -> 0.29, 0.24, 0.24, 0.27, 0.47 ms
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
