// The steps either side of the solve in a time step (include/bem.h):
//   bem_surface_velocity   vertex areas and normals (Eq. 17) and the surface velocity
//                          v = n q + (n x v) x n with n x v from the contour integrals of phi (Eqs. 22-27)
//   bem_filter_*           the shape filter F = G (G* G)^-1 G* of bandwidth p_f (Eqs. 37-43), kept in
//                          the factored form  xhat = G (G^+ x)  (rank p_f^2 << N_d) and applied to all bubbles and all
//                          surface functions at once
#include "common.cuh"

#include <algorithm>
#include <cmath>

namespace bem {
bool is_device_ptr(const void *p);      // api.cu

// ------------------------------------------------------------------ vertex -> incident corners (fixed summation order)
__global__ void sv_corner_keys(const int32_t *F, int64_t n, uint64_t *keys)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) keys[i] = (uint64_t)F[i];
}
__global__ void sv_vertex_ranges(const uint64_t *keys, int64_t n, int64_t N, int32_t *begin)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    const int64_t lo = (i == 0) ? -1 : (int64_t)keys[i - 1];          // begin[v] = first i with keys[i] >= v
    const int64_t hi = (i == n) ? N : (int64_t)keys[i];
    for (int64_t v = lo + 1; v <= hi; ++v) begin[v] = (int32_t)i;
}

static void build_vertex_corners(bem_ctx *c)
{
    if (c->vc_begin.p && c->vc_begin.n == (size_t)c->N + 1) return;
    cudaStream_t s = c->stream;
    const int64_t nc = 3 * c->T;
    dvec<uint64_t> keys, keys_tmp;
    dvec<uint32_t> vals_tmp;
    keys.alloc(nc); keys_tmp.alloc(nc); vals_tmp.alloc(nc);
    c->vc_corner.alloc(nc);
    c->vc_begin.alloc(c->N + 1);
    sv_corner_keys<<<cdiv(nc, 256), 256, 0, s>>>(c->F.get(), nc, keys.get());
    KERNEL_CHECK();
    iota_u32(c->vc_corner.get(), nc, s);
    radix_sort_pairs(keys.get(), c->vc_corner.get(), keys_tmp.get(), vals_tmp.get(), nc, 0, 32, s);   // stable: corners of a vertex in mesh order
    sv_vertex_ranges<<<cdiv(nc + 1, 256), 256, 0, s>>>(keys.get(), nc, c->N, c->vc_begin.get());
    KERNEL_CHECK();
    CUDA_TRY(cudaStreamSynchronize(s));
}

// ------------------------------------------------------------------ Eq. 17 and Eqs. 22-27, one thread per vertex
__global__ void surface_velocity_kernel(const double *__restrict__ V, const int32_t *__restrict__ F, const int32_t *__restrict__ begin,
                                        const uint32_t *__restrict__ corner, const double *__restrict__ phi, const double *__restrict__ q,
                                        int64_t N, double *__restrict__ vel, double *__restrict__ nrm, double *__restrict__ area)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    double s3 = 0.0, mx = 0.0, my = 0.0, mz = 0.0, wx = 0.0, wy = 0.0, wz = 0.0;     // 3 s_j, m_j, sum (n x v)_k A_k
    for (int i = begin[j]; i < begin[j + 1]; ++i) {
        const int64_t k = corner[i] / 3;
        const int v1 = F[3 * k], v2 = F[3 * k + 1], v3 = F[3 * k + 2];
        const double x1 = V[3 * (int64_t)v1], y1 = V[3 * (int64_t)v1 + 1], z1 = V[3 * (int64_t)v1 + 2];
        const double x2 = V[3 * (int64_t)v2], y2 = V[3 * (int64_t)v2 + 1], z2 = V[3 * (int64_t)v2 + 2];
        const double x3 = V[3 * (int64_t)v3], y3 = V[3 * (int64_t)v3 + 1], z3 = V[3 * (int64_t)v3 + 2];
        const double ax = x2 - x1, ay = y2 - y1, az = z2 - z1, bx = x3 - x1, by = y3 - y1, bz = z3 - z1;
        const double cx = ay * bz - az * by, cy = az * bx - ax * bz, cz = ax * by - ay * bx;        // N_k 2 A_k
        s3 += 0.5 * sqrt(cx * cx + cy * cy + cz * cz);
        mx += 0.5 * cx; my += 0.5 * cy; mz += 0.5 * cz;
        if (phi) {
            const double f1 = phi[v1], f2 = phi[v2], f3 = phi[v3];                                  // Eq. 26 times A_k
            wx += 0.5 * ((x2 - x3) * f1 + (x3 - x1) * f2 + (x1 - x2) * f3);
            wy += 0.5 * ((y2 - y3) * f1 + (y3 - y1) * f2 + (y1 - y2) * f3);
            wz += 0.5 * ((z2 - z3) * f1 + (z3 - z1) * f2 + (z1 - z2) * f3);
        }
    }
    const double im = 1.0 / sqrt(mx * mx + my * my + mz * mz);
    const double nx = mx * im, ny = my * im, nz = mz * im;
    if (nrm) { nrm[3 * j] = nx; nrm[3 * j + 1] = ny; nrm[3 * j + 2] = nz; }
    if (area) area[j] = s3 / 3.0;
    if (vel) {
        const double ux = wx / s3, uy = wy / s3, uz = wz / s3;                                      // (n x v)_j, Eq. 27
        const double qq = q ? q[j] : 0.0;
        vel[3 * j] = nx * qq + (uy * nz - uz * ny);                                                 // Eq. 22
        vel[3 * j + 1] = ny * qq + (uz * nx - ux * nz);
        vel[3 * j + 2] = nz * qq + (ux * ny - uy * nx);
    }
}

// ------------------------------------------------------------------ Eqs. 28-29: mean curvature by the fitted paraboloid
// One thread per vertex.  The five neighbours are the first five distinct vertices met when walking the triangles of the
// vertex in mesh order, taking of each its two other vertices in cyclic order (reading R32).  Frame: z = n_j of
// Eq. 17, x and y any orthonormal pair (H = -B3 - B5 does not depend on it).  The 5 x 5 system of Eq. 28 is solved by
// Gaussian elimination with partial pivoting (the paper uses Cramer's rule: the same solution).
__global__ void surface_curvature_kernel(const double *__restrict__ V, const int32_t *__restrict__ F, const int32_t *__restrict__ begin,
                                         const uint32_t *__restrict__ corner, int64_t N, double *__restrict__ H)
{
    const int64_t j = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= N) return;
    double mx = 0.0, my = 0.0, mz = 0.0;
    int ring[5], nr = 0;
    for (int i = begin[j]; i < begin[j + 1]; ++i) {
        const uint32_t c = corner[i];
        const int64_t k = c / 3;
        const int a = (int)(c - 3 * k);
        const int v1 = F[3 * k], v2 = F[3 * k + 1], v3 = F[3 * k + 2];
        const double x1 = V[3 * (int64_t)v1], y1 = V[3 * (int64_t)v1 + 1], z1 = V[3 * (int64_t)v1 + 2];
        const double ax = V[3 * (int64_t)v2] - x1, ay = V[3 * (int64_t)v2 + 1] - y1, az = V[3 * (int64_t)v2 + 2] - z1;
        const double bx = V[3 * (int64_t)v3] - x1, by = V[3 * (int64_t)v3 + 1] - y1, bz = V[3 * (int64_t)v3 + 2] - z1;
        mx += 0.5 * (ay * bz - az * by); my += 0.5 * (az * bx - ax * bz); mz += 0.5 * (ax * by - ay * bx);
        const int cand[2] = {F[3 * k + (a + 1) % 3], F[3 * k + (a + 2) % 3]};
        for (int t = 0; t < 2; ++t) {
            bool seen = false;
            for (int r = 0; r < nr; ++r) seen = seen || ring[r] == cand[t];
            if (!seen && nr < 5) ring[nr++] = cand[t];
        }
    }
    const double nan = __longlong_as_double(0x7ff8000000000000ll);
    if (nr < 5) { H[j] = nan; return; }
    const double im = 1.0 / sqrt(mx * mx + my * my + mz * mz);
    const double zx = mx * im, zy = my * im, zz = mz * im;
    double ex, ey, ez;                                                 // e_x = normalised z x a, a = a coordinate axis away from z
    if (fabs(zx) < 0.9) { ex = 0.0; ey = zz; ez = -zy; } else { ex = -zz; ey = 0.0; ez = zx; }
    const double ie = 1.0 / sqrt(ex * ex + ey * ey + ez * ez);
    ex *= ie; ey *= ie; ez *= ie;
    const double fx = zy * ez - zz * ey, fy = zz * ex - zx * ez, fz = zx * ey - zy * ex;      // e_y = z x e_x
    double A[5][6];
    const double px = V[3 * j], py = V[3 * j + 1], pz = V[3 * j + 2];
    for (int l = 0; l < 5; ++l) {
        const double dx = V[3 * (int64_t)ring[l]] - px, dy = V[3 * (int64_t)ring[l] + 1] - py, dz = V[3 * (int64_t)ring[l] + 2] - pz;
        const double x = dx * ex + dy * ey + dz * ez, y = dx * fx + dy * fy + dz * fz, z = dx * zx + dy * zy + dz * zz;
        A[l][0] = x; A[l][1] = y; A[l][2] = x * x; A[l][3] = x * y; A[l][4] = y * y; A[l][5] = z;       // Eq. 28
    }
    for (int col = 0; col < 5; ++col) {
        int piv = col;
        for (int r = col + 1; r < 5; ++r) if (fabs(A[r][col]) > fabs(A[piv][col])) piv = r;
        if (A[piv][col] == 0.0) { H[j] = nan; return; }
        for (int cc = 0; cc < 6; ++cc) { const double t = A[col][cc]; A[col][cc] = A[piv][cc]; A[piv][cc] = t; }
        for (int r = col + 1; r < 5; ++r) {
            const double f = A[r][col] / A[col][col];
            for (int cc = col; cc < 6; ++cc) A[r][cc] -= f * A[col][cc];
        }
    }
    double B[5];
    for (int r = 4; r >= 0; --r) {
        double sum = A[r][5];
        for (int cc = r + 1; cc < 5; ++cc) sum -= A[r][cc] * B[cc];
        B[r] = sum / A[r][r];
    }
    H[j] = -B[2] - B[4];                                               // Eq. 29
}

// ------------------------------------------------------------------ bubble volumes (PAPER.md:108-115 gas law; "volume")
__global__ void bv_keys(const int32_t *F, const int32_t *bid, int64_t T, uint64_t *keys)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k < T) keys[k] = bid ? (uint64_t)bid[F[3 * k]] : 0ull;
}

// One warp per bubble.  V_m = sum_k (r_k1 - o).((r_k2 - o) x (r_k3 - o)) / 6 over the bubble's triangles -- the signed
// tetrahedra from a point o to every outward-oriented triangle of a closed surface; o = the first vertex of the bubble's
// first triangle, so that a bubble far from the origin loses no digits.  Lane l adds triangles l, l + 32, ... in mesh order,
// then a shuffle tree: the same bits on every call.
__global__ void bubble_volume_kernel(const double *__restrict__ V, const int32_t *__restrict__ F, const int32_t *__restrict__ begin,
                                     const uint32_t *__restrict__ tri, int nb, double *__restrict__ vol)
{
    const int b = (int)(((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
    if (b >= nb) return;
    const int i0 = begin[b], i1 = begin[b + 1];
    double acc = 0.0;
    if (i1 > i0) {
        const int64_t vo = F[3 * (int64_t)tri[i0]];
        const double ox = V[3 * vo], oy = V[3 * vo + 1], oz = V[3 * vo + 2];
        for (int i = i0 + lane; i < i1; i += 32) {
            const int64_t k = tri[i];
            const int64_t a = F[3 * k], bb = F[3 * k + 1], c = F[3 * k + 2];
            const double ax = V[3 * a] - ox, ay = V[3 * a + 1] - oy, az = V[3 * a + 2] - oz;
            const double bx = V[3 * bb] - ox, by = V[3 * bb + 1] - oy, bz = V[3 * bb + 2] - oz;
            const double cx = V[3 * c] - ox, cy = V[3 * c + 1] - oy, cz = V[3 * c + 2] - oz;
            acc += ax * (by * cz - bz * cy) + ay * (bz * cx - bx * cz) + az * (bx * cy - by * cx);
        }
    }
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if (lane == 0) vol[b] = acc / 6.0;
}

static void build_bubble_triangles(bem_ctx *c)
{
    if (c->bv_begin.p && c->bv_begin.n == (size_t)c->nbubbles + 1) return;
    cudaStream_t s = c->stream;
    const int64_t T = c->T;
    dvec<uint64_t> keys, keys_tmp;
    dvec<uint32_t> vals_tmp;
    keys.alloc(T); keys_tmp.alloc(T); vals_tmp.alloc(T);
    c->bv_tri.alloc(T);
    c->bv_begin.alloc(c->nbubbles + 1);
    bv_keys<<<cdiv(T, 256), 256, 0, s>>>(c->F.get(), c->bid.p, T, keys.get());
    KERNEL_CHECK();
    iota_u32(c->bv_tri.get(), T, s);
    if (c->nbubbles > 1) radix_sort_pairs(keys.get(), c->bv_tri.get(), keys_tmp.get(), vals_tmp.get(), T, 0, 32, s);   // stable
    sv_vertex_ranges<<<cdiv(T + 1, 256), 256, 0, s>>>(keys.get(), T, c->nbubbles, c->bv_begin.get());
    KERNEL_CHECK();
    CUDA_TRY(cudaStreamSynchronize(s));
}

// ------------------------------------------------------------------ shape filter
}  // namespace bem

struct bem_filter {
    int device = 0;
    int64_t nd = 0;
    int pf = 0, P = 0;
    bem::dvec<double> GT;       // [P x nd]   GT[j][i] = Y_j(theta_i, phi_i)        (Eq. 39, real orthonormal basis)
    bem::dvec<double> GpT;      // [nd x P]   GpT[i][j] = ((G^T G)^-1 G^T)[j][i]     (Eq. 40)
    bem::dvec<double> stage_in, stage_out;
    int use_dmma = 1;           // p_f <= 10: the two products on the FP64 tensor path (filter_apply_dmma); else plain FMA
    std::string err;
};

namespace bem {

// real orthonormal Y_n^m (Condon-Shortley phase) of one point: column n^2 (m = 0), n^2 + 2m - 1 (cos), n^2 + 2m (sin)
__global__ void filter_harmonics_kernel(const double *__restrict__ theta, const double *__restrict__ phi, int64_t nd, int pf, int P,
                                        double *__restrict__ GT)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nd) return;
    const double ct = cos(theta[i]), st = sin(theta[i]), ph = phi[i];
    double pmm = 0.28209479177387814347403972578039;                  // sqrt(1 / 4 pi)
    for (int m = 0; m < pf; ++m) {
        if (m > 0) pmm *= -sqrt((2.0 * m + 1.0) / (2.0 * m)) * st;
        const double cm = m == 0 ? 1.0 : 1.4142135623730950488 * cos(m * ph), sm = 1.4142135623730950488 * sin(m * ph);
        double p2 = 0.0, p1 = pmm;
        for (int n = m; n < pf; ++n) {
            double pn;
            if (n == m) pn = pmm;
            else {
                const double a = sqrt((4.0 * n * n - 1.0) / ((double)n * n - (double)m * m));
                const double b = sqrt((((double)n - 1.0) * (n - 1.0) - (double)m * m) / (4.0 * (n - 1.0) * (n - 1.0) - 1.0));
                pn = a * (ct * p1 - b * p2);
            }
            p2 = p1; p1 = pn;
            if (m == 0) GT[(size_t)(n * n) * nd + i] = pn;
            else { GT[(size_t)(n * n + 2 * m - 1) * nd + i] = pn * cm; GT[(size_t)(n * n + 2 * m) * nd + i] = pn * sm; }
        }
    }
}

// A = G^T G, one thread per entry (fixed order)
__global__ void filter_gram_kernel(const double *__restrict__ GT, int64_t nd, int P, double *__restrict__ A)
{
    const int a = blockIdx.x, b = blockIdx.y * blockDim.x + threadIdx.x;
    if (b >= P) return;
    const double *ra = GT + (size_t)a * nd, *rb = GT + (size_t)b * nd;
    double s = 0.0;
    for (int64_t i = 0; i < nd; ++i) s = fma(ra[i], rb[i], s);
    A[(size_t)a * P + b] = s;
}

// in-place Cholesky A = L L^T (lower triangle), one CTA; *ok = 0 if a pivot is not positive
__global__ void filter_cholesky_kernel(double *A, int P, int *ok)
{
    __shared__ double piv;
    for (int k = 0; k < P; ++k) {
        if (threadIdx.x == 0) {
            const double d = A[(size_t)k * P + k];
            if (!(d > 0.0)) *ok = 0;
            piv = sqrt(d > 0.0 ? d : 1.0);
            A[(size_t)k * P + k] = piv;
        }
        __syncthreads();
        for (int i = k + 1 + threadIdx.x; i < P; i += blockDim.x) A[(size_t)i * P + k] /= piv;
        __syncthreads();
        for (int i = k + 1 + threadIdx.x; i < P; i += blockDim.x) {
            const double lik = A[(size_t)i * P + k];
            for (int j = k + 1; j <= i; ++j) A[(size_t)i * P + j] -= lik * A[(size_t)j * P + k];
        }
        __syncthreads();
    }
}

// GpT[i][:] = (L L^T)^-1 G[i][:], one thread per mesh point
__global__ void filter_solve_kernel(const double *__restrict__ L, const double *__restrict__ GT, int64_t nd, int P, double *__restrict__ GpT)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nd) return;
    double *z = GpT + (size_t)i * P;
    for (int j = 0; j < P; ++j) {                                      // L w = g
        double s = GT[(size_t)j * nd + i];
        for (int k = 0; k < j; ++k) s -= L[(size_t)j * P + k] * z[k];
        z[j] = s / L[(size_t)j * P + j];
    }
    for (int j = P - 1; j >= 0; --j) {                                 // L^T z = w
        double s = z[j];
        for (int k = j + 1; k < P; ++k) s -= L[(size_t)k * P + j] * z[k];
        z[j] = s / L[(size_t)j * P + j];
    }
}

// xhat[c][:] = G (G^+ x[c][:]) for FC columns per CTA: x rows staged in shared memory, the P coefficients of every
// column in shared memory, G^T and G^+T streamed from L2 (coalesced over the thread index in both passes)
constexpr int FILTER_THREADS = 256;
__global__ void __launch_bounds__(FILTER_THREADS)
filter_apply_kernel(const double *__restrict__ x, int64_t ncols, int64_t nd, int P, int fc, const double *__restrict__ GT,
                    const double *__restrict__ GpT, double *__restrict__ xhat)
{
    extern __shared__ double fsm[];
    double *xs = fsm;                        // [fc][nd]
    double *cs = fsm + (size_t)fc * nd;      // [fc][P]
    const int64_t c0 = (int64_t)blockIdx.x * fc;
    const int nc = (int)min((int64_t)fc, ncols - c0);
    for (int64_t e = threadIdx.x; e < (int64_t)nc * nd; e += FILTER_THREADS) xs[e] = x[c0 * nd + e];
    __syncthreads();
    // coefficients C[c][j] = sum_i G^+[j][i] x[c][i]: thread (j, g) sums the points i = g (mod groups); the partial
    // sums of the groups are added in a fixed order
    const int groups = max(1, FILTER_THREADS / P);
    double *part = cs + (size_t)fc * P;      // [groups][fc][P]
    {
        const int j = threadIdx.x % P, g = threadIdx.x / P;
        if (g < groups) {
            double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            for (int64_t i = g; i < nd; i += groups) {
                const double gp = GpT[(size_t)i * P + j];
#pragma unroll
                for (int c = 0; c < 8; ++c) if (c < nc) acc[c] = fma(xs[(size_t)c * nd + i], gp, acc[c]);
            }
#pragma unroll
            for (int c = 0; c < 8; ++c) if (c < nc) part[((size_t)g * fc + c) * P + j] = acc[c];
        }
    }
    __syncthreads();
    for (int e = threadIdx.x; e < nc * P; e += FILTER_THREADS) {
        double sum = 0.0;
        for (int g = 0; g < groups; ++g) sum += part[(size_t)g * fc * P + e];
        cs[e] = sum;
    }
    __syncthreads();
    for (int64_t i = threadIdx.x; i < nd; i += FILTER_THREADS) {       // xhat[c][i] = sum_j G[i][j] C[c][j]
        double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
        for (int j = 0; j < P; ++j) {
            const double g = GT[(size_t)j * nd + i];
#pragma unroll
            for (int c = 0; c < 8; ++c) if (c < nc) acc[c] = fma(cs[(size_t)c * P + j], g, acc[c]);
        }
#pragma unroll
        for (int c = 0; c < 8; ++c) if (c < nc) xhat[(c0 + c) * nd + i] = acc[c];
    }
}


// ------------------------------------------------------------------ the same two products on the FP64 tensor path
// xhat = (x G^+T) G^T as two skinny GEMMs of mma.sync.m8n8k4.f64 (DMMA): a warp owns 16 columns of the batch (16 rows of the
// M dimension, two 8-row A fragments, so every B fragment feeds two DMMAs), a CTA two warps.
//   pass 1  C[16 x P]   = x[16 x N_d] . G^+T[N_d x P]     A from global memory (every x entry is read once), B = G^+T through L1
//   pass 2  xhat[16 x N_d] = C[16 x P] . G^T[P x N_d]     A = C through shared memory (accumulator layout -> A layout), B = G^T
// Fragment layouts of m8n8k4: A (8 x 4, row): lane l holds A[l / 4][l % 4]; B (4 x 8, col): lane l holds B[l % 4][l / 4];
// C (8 x 8): lane l holds C[l / 4][2 (l % 4)] and C[l / 4][2 (l % 4) + 1].  A warp reads all its rows of x before it
// writes them, so xhat may be x.
constexpr int FD_WARPS = 2, FD_ROWS = 16, FD_MAXNT = 32;      // P <= 256 -> at most 32 n-tiles in pass 1
__device__ __forceinline__ void fd_dmma(double &c0, double &c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n" : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int NT1>        // n-tiles of pass 1 = ceil(P / 8), a compile-time bound so that the accumulators stay in registers
__global__ void __launch_bounds__(FD_WARPS * 32)
filter_apply_dmma(const double *__restrict__ x, int64_t ncols, int nd, int P, const double *__restrict__ GT,
                  const double *__restrict__ GpT, double *__restrict__ xhat)
{
    extern __shared__ double fds[];                            // [FD_WARPS][16][cstride]
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int lr = lane >> 2, lk = lane & 3;
    const int cstride = 8 * NT1 + 4;                           // = 4 mod 8: conflict-free A-fragment reads of pass 2
    double *Cs = fds + (size_t)warp * FD_ROWS * cstride;
    const int64_t row0 = ((int64_t)blockIdx.x * FD_WARPS + warp) * FD_ROWS;
    const int64_t ra = row0 + lr, rb = row0 + 8 + lr;
    const bool va = ra < ncols, vb = rb < ncols;
    const double *xa = x + (va ? ra : 0) * nd, *xb = x + (vb ? rb : 0) * nd;

    // pass 1
    double acc[NT1][4];
#pragma unroll
    for (int t = 0; t < NT1; ++t) acc[t][0] = acc[t][1] = acc[t][2] = acc[t][3] = 0.0;
    for (int k0 = 0; k0 < nd; k0 += 4) {
        const int k = k0 + lk;
        const bool kv = k < nd;
        const double a0 = (va && kv) ? __ldg(xa + k) : 0.0, a1 = (vb && kv) ? __ldg(xb + k) : 0.0;
        const double *brow = GpT + (size_t)(kv ? k : 0) * P;
#pragma unroll
        for (int t = 0; t < NT1; ++t) {
            const int n = 8 * t + lr;
            const double b = (kv && n < P) ? __ldg(brow + n) : 0.0;
            fd_dmma(acc[t][0], acc[t][1], a0, b);
            fd_dmma(acc[t][2], acc[t][3], a1, b);
        }
    }
#pragma unroll
    for (int t = 0; t < NT1; ++t) {
        Cs[lr * cstride + 8 * t + 2 * lk] = acc[t][0];
        Cs[lr * cstride + 8 * t + 2 * lk + 1] = acc[t][1];
        Cs[(8 + lr) * cstride + 8 * t + 2 * lk] = acc[t][2];
        Cs[(8 + lr) * cstride + 8 * t + 2 * lk + 1] = acc[t][3];
    }
    __syncwarp();
    // pass 2: the A fragments of all k-steps (2 NT1 of them) stay in registers; columns n >= P of C are zero by construction
    double a0[2 * NT1], a1[2 * NT1];
#pragma unroll
    for (int ks = 0; ks < 2 * NT1; ++ks) {
        a0[ks] = Cs[lr * cstride + 4 * ks + lk];
        a1[ks] = Cs[(8 + lr) * cstride + 4 * ks + lk];
    }
    double *ya = xhat + (va ? ra : 0) * nd, *yb = xhat + (vb ? rb : 0) * nd;
    for (int n0 = 0; n0 < nd; n0 += 8) {
        double c0 = 0.0, c1 = 0.0, c2 = 0.0, c3 = 0.0;
        const int n = n0 + lr;
#pragma unroll
        for (int ks = 0; ks < 2 * NT1; ++ks) {
            const int k = 4 * ks + lk;
            const double b = (k < P && n < nd) ? __ldg(GT + (size_t)k * nd + n) : 0.0;
            fd_dmma(c0, c1, a0[ks], b);
            fd_dmma(c2, c3, a1[ks], b);
        }
        const int col = n0 + 2 * lk;
        if (va) { if (col < nd) ya[col] = c0; if (col + 1 < nd) ya[col + 1] = c1; }
        if (vb) { if (col < nd) yb[col] = c2; if (col + 1 < nd) yb[col + 1] = c3; }
    }
}

template <int NT1>
static void launch_filter_dmma(const double *x, int64_t ncols, int nd, int P, const double *GT, const double *GpT, double *xhat, cudaStream_t s)
{
    const size_t smem = (size_t)FD_WARPS * FD_ROWS * (8 * NT1 + 4) * sizeof(double);
    CUDA_TRY(cudaFuncSetAttribute(filter_apply_dmma<NT1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    filter_apply_dmma<NT1><<<cdiv(ncols, FD_WARPS * FD_ROWS), FD_WARPS * 32, smem, s>>>(x, ncols, nd, P, GT, GpT, xhat);
    KERNEL_CHECK();
}

}  // namespace bem

using namespace bem;

extern "C" {

bem_status bem_surface_velocity(bem_ctx *c, const double *phi, const double *q, double *v, double *normals_out, double *areas_out)
{
    if (!c || (!v && !normals_out && !areas_out)) return BEM_ERR_INVALID_ARG;
    if (c->quadrature == 2 || c->T == 0) { c->err = "bem_surface_velocity: the context holds a point cloud, not a mesh"; return BEM_ERR_INVALID_ARG; }
    if (v && !phi) { c->err = "bem_surface_velocity: phi is required for the velocity"; return BEM_ERR_INVALID_ARG; }
    try {
        CUDA_TRY(cudaSetDevice(c->device));
        build_vertex_corners(c);
        const int64_t N = c->N;
        cudaStream_t s = c->stream;
        dvec<double> dphi, dq, dv, dn, da;
        auto in = [&](const double *h, dvec<double> &d) -> const double * {
            if (!h || is_device_ptr(h)) return h;
            d.alloc(N);
            CUDA_TRY(cudaMemcpyAsync(d.get(), h, N * sizeof(double), cudaMemcpyHostToDevice, s));
            return d.get();
        };
        auto out = [&](double *h, dvec<double> &d, int64_t n) -> double * {
            if (!h || is_device_ptr(h)) return h;
            d.alloc(n);
            return d.get();
        };
        const double *pphi = in(phi, dphi), *pq = in(q, dq);
        double *pv = out(v, dv, 3 * N), *pn = out(normals_out, dn, 3 * N), *pa = out(areas_out, da, N);
        surface_velocity_kernel<<<cdiv(N, 128), 128, 0, s>>>(c->V.get(), c->F.get(), c->vc_begin.get(), c->vc_corner.get(), pphi, pq, N, pv, pn, pa);
        KERNEL_CHECK();
        bool sync = false;
        if (pv != v) { CUDA_TRY(cudaMemcpyAsync(v, pv, 3 * N * sizeof(double), cudaMemcpyDeviceToHost, s)); sync = true; }
        if (pn != normals_out) { CUDA_TRY(cudaMemcpyAsync(normals_out, pn, 3 * N * sizeof(double), cudaMemcpyDeviceToHost, s)); sync = true; }
        if (pa != areas_out) { CUDA_TRY(cudaMemcpyAsync(areas_out, pa, N * sizeof(double), cudaMemcpyDeviceToHost, s)); sync = true; }
        if (sync || dphi.p || dq.p) CUDA_TRY(cudaStreamSynchronize(s));
        return BEM_OK;
    } catch (const Error &e) {
        c->err = e.what();
        cudaGetLastError();
        return e.status;
    } catch (const std::bad_alloc &) {
        return BEM_ERR_OOM;
    } catch (const std::exception &) {
        cudaGetLastError();
        return BEM_ERR_CUDA;                                  // nothing may cross the extern "C" boundary
    } catch (...) {
        return BEM_ERR_CUDA;
    }
}

bem_status bem_surface_curvature(bem_ctx *c, double *H)
{
    if (!c || !H) return BEM_ERR_INVALID_ARG;
    if (c->quadrature == 2 || c->T == 0) { c->err = "bem_surface_curvature: the context holds a point cloud, not a mesh"; return BEM_ERR_INVALID_ARG; }
    try {
        CUDA_TRY(cudaSetDevice(c->device));
        build_vertex_corners(c);
        const int64_t N = c->N;
        dvec<double> dh;
        double *ph = H;
        if (!is_device_ptr(H)) { dh.alloc(N); ph = dh.get(); }
        surface_curvature_kernel<<<cdiv(N, 128), 128, 0, c->stream>>>(c->V.get(), c->F.get(), c->vc_begin.get(), c->vc_corner.get(), N, ph);
        KERNEL_CHECK();
        if (ph != H) {
            CUDA_TRY(cudaMemcpyAsync(H, ph, N * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            CUDA_TRY(cudaStreamSynchronize(c->stream));
        }
        return BEM_OK;
    } catch (const Error &e) {
        c->err = e.what();
        cudaGetLastError();
        return e.status;
    } catch (const std::bad_alloc &) {
        return BEM_ERR_OOM;
    } catch (const std::exception &) {
        cudaGetLastError();
        return BEM_ERR_CUDA;                                  // nothing may cross the extern "C" boundary
    } catch (...) {
        return BEM_ERR_CUDA;
    }
}

bem_status bem_bubble_volume(bem_ctx *c, double *vol_out, int64_t n_bubbles)
{
    if (!c || !vol_out) return BEM_ERR_INVALID_ARG;
    if (c->quadrature >= 2 || c->T == 0) { c->err = "bem_bubble_volume: the context holds no mesh"; return BEM_ERR_INVALID_ARG; }
    if (n_bubbles != c->nbubbles) {
        c->err = "bem_bubble_volume: n_bubbles must be the number of bubbles of the mesh (largest bubble id + 1; 1 without ids): " + std::to_string(c->nbubbles);
        return BEM_ERR_INVALID_ARG;
    }
    try {
        CUDA_TRY(cudaSetDevice(c->device));
        build_bubble_triangles(c);
        const int nb = c->nbubbles;
        dvec<double> dv;
        double *pv = vol_out;
        if (!is_device_ptr(vol_out)) { dv.alloc(nb); pv = dv.get(); }
        bubble_volume_kernel<<<cdiv((int64_t)nb * 32, 128), 128, 0, c->stream>>>(c->V.get(), c->F.get(), c->bv_begin.get(), c->bv_tri.get(), nb, pv);
        KERNEL_CHECK();
        if (pv != vol_out) {
            CUDA_TRY(cudaMemcpyAsync(vol_out, pv, nb * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
            CUDA_TRY(cudaStreamSynchronize(c->stream));
        }
        return BEM_OK;
    } catch (const Error &e) {
        c->err = e.what();
        cudaGetLastError();
        return e.status;
    } catch (const std::bad_alloc &) {
        return BEM_ERR_OOM;
    } catch (const std::exception &) {
        cudaGetLastError();
        return BEM_ERR_CUDA;                                  // nothing may cross the extern "C" boundary
    } catch (...) {
        return BEM_ERR_CUDA;
    }
}

bem_status bem_filter_create(const double *theta, const double *phi, int64_t n_d, int p_f, bem_filter **out)
{
    if (!out) return BEM_ERR_INVALID_ARG;
    *out = nullptr;
    if (!theta || !phi || n_d < 4 || p_f < 1 || p_f > 16 || (int64_t)p_f * p_f >= n_d) return BEM_ERR_INVALID_ARG;   // p_f < sqrt(N_d)
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) { cudaGetLastError(); return BEM_ERR_CUDA; }
    bem_filter *f = new (std::nothrow) bem_filter();
    if (!f) return BEM_ERR_OOM;
    cudaGetDevice(&f->device);
    f->nd = n_d; f->pf = p_f; f->P = p_f * p_f;
    try {
        const int P = f->P;
        dvec<double> th, ph, A;
        dvec<int> ok;
        th.alloc(n_d); ph.alloc(n_d); A.alloc((size_t)P * P); ok.alloc(1);
        CUDA_TRY(cudaMemcpy(th.get(), theta, n_d * sizeof(double), cudaMemcpyDefault));
        CUDA_TRY(cudaMemcpy(ph.get(), phi, n_d * sizeof(double), cudaMemcpyDefault));
        f->GT.alloc((size_t)P * n_d);
        f->GpT.alloc((size_t)n_d * P);
        filter_harmonics_kernel<<<cdiv(n_d, 128), 128>>>(th.get(), ph.get(), n_d, p_f, P, f->GT.get());
        KERNEL_CHECK();
        filter_gram_kernel<<<dim3(P, cdiv(P, 64)), 64>>>(f->GT.get(), n_d, P, A.get());
        KERNEL_CHECK();
        const int one = 1;
        CUDA_TRY(cudaMemcpy(ok.get(), &one, sizeof(int), cudaMemcpyHostToDevice));
        filter_cholesky_kernel<<<1, 256>>>(A.get(), P, ok.get());
        KERNEL_CHECK();
        filter_solve_kernel<<<cdiv(n_d, 64), 64>>>(A.get(), f->GT.get(), n_d, P, f->GpT.get());
        KERNEL_CHECK();
        int h_ok = 0;
        CUDA_TRY(cudaMemcpy(&h_ok, ok.get(), sizeof(int), cudaMemcpyDeviceToHost));
        if (!h_ok) { delete f; return BEM_ERR_BAD_MESH; }            // the angles do not resolve the band: G^T G is singular
    } catch (const Error &e) {
        cudaGetLastError();
        const bem_status st = e.status;
        delete f;
        return st;
    } catch (...) {                                              // nothing may cross the extern "C" boundary
        cudaGetLastError();
        delete f;
        return BEM_ERR_CUDA;
    }
    *out = f;
    return BEM_OK;
}

bem_status bem_filter_apply(bem_filter *f, const double *x, int64_t n_cols, double *xhat, void *cuda_stream)
{
    if (!f || !x || !xhat || n_cols < 0) return BEM_ERR_INVALID_ARG;
    if (n_cols == 0) return BEM_OK;
    try {
        CUDA_TRY(cudaSetDevice(f->device));
        cudaStream_t s = (cudaStream_t)cuda_stream;
        const size_t n = (size_t)n_cols * f->nd;
        const bool hx = !is_device_ptr(x), hy = !is_device_ptr(xhat);
        const double *dx = x;
        double *dy = xhat;
        if (hx) { if (f->stage_in.n < n) f->stage_in.alloc(n); CUDA_TRY(cudaMemcpyAsync(f->stage_in.get(), x, n * sizeof(double), cudaMemcpyHostToDevice, s)); dx = f->stage_in.get(); }
        if (hy) { if (f->stage_out.n < n) f->stage_out.alloc(n); dy = f->stage_out.get(); }
        const int nt1 = (f->P + 7) / 8;
        // tensor path: p_f <= 10 (the accumulators of pass 1 fit the registers) and a batch that fills the machine (a warp
        // owns 16 columns; measured: 108 columns of N_d = 2562 take 1.16 ms there against 0.47 ms on the FMA kernel)
        if (f->use_dmma && nt1 <= 13 && f->nd < (1 << 30) && n_cols >= 2048) {
            const int nd = (int)f->nd;
            if (nt1 <= 2) launch_filter_dmma<2>(dx, n_cols, nd, f->P, f->GT.get(), f->GpT.get(), dy, s);
            else if (nt1 <= 5) launch_filter_dmma<5>(dx, n_cols, nd, f->P, f->GT.get(), f->GpT.get(), dy, s);
            else if (nt1 <= 8) launch_filter_dmma<8>(dx, n_cols, nd, f->P, f->GT.get(), f->GpT.get(), dy, s);
            else if (nt1 <= 11) launch_filter_dmma<11>(dx, n_cols, nd, f->P, f->GT.get(), f->GpT.get(), dy, s);
            else launch_filter_dmma<13>(dx, n_cols, nd, f->P, f->GT.get(), f->GpT.get(), dy, s);
            if (hy) CUDA_TRY(cudaMemcpyAsync(xhat, dy, n * sizeof(double), cudaMemcpyDeviceToHost, s));
            if (hx || hy) CUDA_TRY(cudaStreamSynchronize(s));
            return BEM_OK;
        }
        int fc = 8;
        const int groups = std::max(1, FILTER_THREADS / f->P);
        auto bytes = [&](int k) { return ((size_t)k * (f->nd + (size_t)(1 + groups) * f->P)) * sizeof(double); };
        while (fc > 1 && bytes(fc) > 160 * 1024) fc >>= 1;
        const size_t smem = bytes(fc);
        if (smem > 200 * 1024) { f->err = "bem_filter_apply: N_d too large for the shared-memory staging"; return BEM_ERR_INVALID_ARG; }
        CUDA_TRY(cudaFuncSetAttribute(filter_apply_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
        filter_apply_kernel<<<cdiv(n_cols, fc), FILTER_THREADS, smem, s>>>(dx, n_cols, f->nd, f->P, fc, f->GT.get(), f->GpT.get(), dy);
        KERNEL_CHECK();
        if (hy) CUDA_TRY(cudaMemcpyAsync(xhat, dy, n * sizeof(double), cudaMemcpyDeviceToHost, s));
        if (hx || hy) CUDA_TRY(cudaStreamSynchronize(s));
        return BEM_OK;
    } catch (const Error &e) {
        f->err = e.what();
        cudaGetLastError();
        return e.status;
    } catch (const std::bad_alloc &) {
        return BEM_ERR_OOM;
    } catch (const std::exception &) {
        cudaGetLastError();
        return BEM_ERR_CUDA;                                  // nothing may cross the extern "C" boundary
    } catch (...) {
        return BEM_ERR_CUDA;
    }
}

const char *bem_filter_last_error(const bem_filter *f) { return f ? f->err.c_str() : "null filter"; }

void bem_filter_destroy(bem_filter *f)
{
    if (!f) return;
    cudaSetDevice(f->device);
    delete f;
}

}  // extern "C"
