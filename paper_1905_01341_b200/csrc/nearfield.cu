// Step a3: the near-field correction matrix of PAPER.md:432 --
// "the difference of the BEM matrices computed using high and low order
// quadratures ... sparse".  High order = the exact integral of (linear shape
// function x kernel) over a flat triangle, evaluated with closed-form
// edge-log / solid-angle expressions (the analytic route PAPER.md:177 points
// to); low order = the 3-point Gauss value the P2P kernel adds.  Near set of
// vertex i: triangles incident to i, and triangles with
// |r_i - c_k| <= eta * max_a |r_ka - c_k|  (reading R4).
#include "common.cuh"
#include "geom.cuh"

namespace bem {

constexpr double INV_4PI = 0.079577471545947667884441881686257;

// ------------------------------------------------------------------ exact integrals
// W^S_a = int_T lambda_a(y) / (4 pi |x-y|) dS,  W^D_a = int_T lambda_a(y) N.(x-y)/(4 pi |x-y|^3) dS
// for x not on the triangle.  With h = N.(x - r0), rho = x - h N (projection on the plane) and
// lambda_a(y) = lambda_a(rho) + g_a.(y - rho),  g_a = N x (edge opposite a)/(2A):
//   W^S_a = [ lambda_a(rho) I1 + g_a.Iv ]/4pi,   W^D_a = [ sign(h) lambda_a(rho) B + h g_a.Jv ]/4pi,
//   I1 = int 1/R = sum_e ( t_e f_e - |h| beta_e ),            B = |h| int 1/R^3 = sum_e beta_e,
//   Iv = int (y-rho)/R = 1/2 sum_e m_e ( R0_e^2 f_e + s+ R+ - s- R- ),   Jv = int (y-rho)/R^3 = - sum_e m_e f_e,
// per edge e (p- -> p+, unit tangent s, outward in-plane normal m = s x N): t = (p- - rho).m,
// s+- = (p+- - rho).s, R+- = |x - p+-|, R0^2 = t^2 + h^2, f = ln[(R+ + s+)/(R- + s-)],
// beta = atan(t s+/(R0^2 + |h| R+)) - atan(t s-/(R0^2 + |h| R-)).
__device__ void tri_weights_regular(const double r[3][3], const double x[3], double WS[3], double WD[3])
{
    double e1[3], e2[3], n[3];
    for (int d = 0; d < 3; ++d) { e1[d] = r[1][d] - r[0][d]; e2[d] = r[2][d] - r[0][d]; }
    n[0] = e1[1] * e2[2] - e1[2] * e2[1];
    n[1] = e1[2] * e2[0] - e1[0] * e2[2];
    n[2] = e1[0] * e2[1] - e1[1] * e2[0];
    const double twoA = sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
    for (int d = 0; d < 3; ++d) n[d] /= twoA;
    const double h = n[0] * (x[0] - r[0][0]) + n[1] * (x[1] - r[0][1]) + n[2] * (x[2] - r[0][2]);
    const double ah = fabs(h);
    double rho[3];
    for (int d = 0; d < 3; ++d) rho[d] = x[d] - h * n[d];
    double I1 = 0.0, B = 0.0, Iv[3] = {0, 0, 0}, Jv[3] = {0, 0, 0};
    for (int e = 0; e < 3; ++e) {
        const double *pm = r[(e + 1) % 3], *pp = r[(e + 2) % 3];
        double s[3], m[3];
        for (int d = 0; d < 3; ++d) s[d] = pp[d] - pm[d];
        const double len = sqrt(s[0] * s[0] + s[1] * s[1] + s[2] * s[2]);
        for (int d = 0; d < 3; ++d) s[d] /= len;
        m[0] = s[1] * n[2] - s[2] * n[1];
        m[1] = s[2] * n[0] - s[0] * n[2];
        m[2] = s[0] * n[1] - s[1] * n[0];
        double t = 0, sm = 0, sp = 0, Rm = 0, Rp = 0;
        for (int d = 0; d < 3; ++d) {
            const double am = pm[d] - rho[d], ap = pp[d] - rho[d];
            t += am * m[d];
            sm += am * s[d];
            sp += ap * s[d];
            Rm += (x[d] - pm[d]) * (x[d] - pm[d]);
            Rp += (x[d] - pp[d]) * (x[d] - pp[d]);
        }
        Rm = sqrt(Rm);
        Rp = sqrt(Rp);
        const double R02 = t * t + h * h;
        // the two forms are equal; pick the one without cancellation
        const double f = (sm + sp >= 0.0) ? log((Rp + sp) / (Rm + sm)) : log((Rm - sm) / (Rp - sp));
        const double beta = atan2(t * sp, R02 + ah * Rp) - atan2(t * sm, R02 + ah * Rm);
        I1 += t * f - ah * beta;
        B += beta;
        const double iv = 0.5 * (R02 * f + sp * Rp - sm * Rm);
        for (int d = 0; d < 3; ++d) { Iv[d] += m[d] * iv; Jv[d] -= m[d] * f; }
    }
    const double sg = h > 0.0 ? 1.0 : (h < 0.0 ? -1.0 : 0.0);
    for (int a = 0; a < 3; ++a) {
        const double *pm = r[(a + 1) % 3], *pp = r[(a + 2) % 3];
        double ed[3], g[3];
        for (int d = 0; d < 3; ++d) ed[d] = pp[d] - pm[d];
        g[0] = (n[1] * ed[2] - n[2] * ed[1]) / twoA;
        g[1] = (n[2] * ed[0] - n[0] * ed[2]) / twoA;
        g[2] = (n[0] * ed[1] - n[1] * ed[0]) / twoA;
        double lam = 0, gI = 0, gJ = 0;
        for (int d = 0; d < 3; ++d) { lam += g[d] * (rho[d] - pm[d]); gI += g[d] * Iv[d]; gJ += g[d] * Jv[d]; }
        WS[a] = INV_4PI * (lam * I1 + gI);
        WD[a] = INV_4PI * (sg * lam * B + h * gJ);
    }
}

// x = vertex a0 of the triangle.  W^D = 0 (x lies in the plane).  Duffy collapse
// y = x + u[(1-v) a + v b], a, b = edge vectors from x, c = b - a, l = |c|:
//   W^S_{a0} = (2A/4pi) 1/2 I0, W^S_{a0+1} = (2A/4pi) 1/2 (I0 - I1), W^S_{a0+2} = (2A/4pi) 1/2 I1,
//   I0 = int_0^1 dv/|a + v c| = ln[(|b| l + b.c)/(|a| l + a.c)]/l,  I1 = int_0^1 v dv/|a + v c| = (|b|-|a|)/l^2 - (a.c/l^2) I0.
__device__ void tri_weights_incident(const double r[3][3], int a0, double WS[3], double WD[3])
{
    const double *x = r[a0], *ra = r[(a0 + 1) % 3], *rb = r[(a0 + 2) % 3];
    double a[3], b[3], c[3];
    for (int d = 0; d < 3; ++d) { a[d] = ra[d] - x[d]; b[d] = rb[d] - x[d]; c[d] = b[d] - a[d]; }
    const double na = sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]);
    const double nb = sqrt(b[0] * b[0] + b[1] * b[1] + b[2] * b[2]);
    const double l2 = c[0] * c[0] + c[1] * c[1] + c[2] * c[2];
    const double l = sqrt(l2);
    const double ac = a[0] * c[0] + a[1] * c[1] + a[2] * c[2];
    const double bc = b[0] * c[0] + b[1] * c[1] + b[2] * c[2];
    const double cx = a[1] * b[2] - a[2] * b[1], cy = a[2] * b[0] - a[0] * b[2], cz = a[0] * b[1] - a[1] * b[0];
    const double fourA2 = cx * cx + cy * cy + cz * cz;        // (2A)^2 = |a x c|^2 = |b x c|^2
    // (|v| l + v.c)(|v| l - v.c) = |v x c|^2 = (2A)^2: use the product form when v.c < 0
    const double num = bc >= 0.0 ? nb * l + bc : fourA2 / (nb * l - bc);
    const double den = ac >= 0.0 ? na * l + ac : fourA2 / (na * l - ac);
    const double I0 = log(num / den) / l;
    const double I1 = (nb - na) / l2 - (ac / l2) * I0;
    const double f = 0.5 * sqrt(fourA2) * INV_4PI;
    WS[a0] = f * I0;
    WS[(a0 + 1) % 3] = f * (I0 - I1);
    WS[(a0 + 2) % 3] = f * I1;
    WD[0] = WD[1] = WD[2] = 0.0;
}

// ------------------------------------------------------------------ near-set search
// centroid and d2 with every operation rounded separately (the near test is a
// comparison in fp64 of a fixed expression; reading R4)
__device__ __forceinline__ double dot3_rn(const double *a, const double *b)
{
    return __dadd_rn(__dadd_rn(__dmul_rn(a[0], b[0]), __dmul_rn(a[1], b[1])), __dmul_rn(a[2], b[2]));
}
__global__ void tri_centroids(const double *V, const int32_t *F, int64_t T, double *cen, double *d2)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= T) return;
    const double *r[3] = {V + 3 * (int64_t)F[3 * k], V + 3 * (int64_t)F[3 * k + 1], V + 3 * (int64_t)F[3 * k + 2]};
    double c[3];
    for (int d = 0; d < 3; ++d) c[d] = __ddiv_rn(__dadd_rn(__dadd_rn(r[0][d], r[1][d]), r[2][d]), 3.0);
    double m = 0.0;
    for (int a = 0; a < 3; ++a) {
        double v[3];
        for (int d = 0; d < 3; ++d) v[d] = __dadd_rn(r[a][d], -c[d]);
        const double q = dot3_rn(v, v);
        if (q > m) m = q;
    }
    for (int d = 0; d < 3; ++d) cen[3 * k + d] = c[d];
    d2[k] = m;
}

struct Grid { double mn[3]; double h; int n[3]; };

__device__ __forceinline__ int grid_cell(const Grid &g, double x, int d)
{
    int c = (int)floor((x - g.mn[d]) / g.h);
    return c < 0 ? 0 : (c >= g.n[d] ? g.n[d] - 1 : c);
}
__global__ void tri_cells(const double *cen, int64_t T, Grid g, uint64_t *keys)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= T) return;
    const int cx = grid_cell(g, cen[3 * k], 0), cy = grid_cell(g, cen[3 * k + 1], 1), cz = grid_cell(g, cen[3 * k + 2], 2);
    keys[k] = (uint64_t)cx + (uint64_t)g.n[0] * ((uint64_t)cy + (uint64_t)g.n[1] * (uint64_t)cz);
}
__device__ __forceinline__ int64_t lower_bound_u64(const uint64_t *a, int64_t n, uint64_t v)
{
    int64_t lo = 0, hi = n;
    while (lo < hi) { const int64_t mid = (lo + hi) >> 1; if (a[mid] < v) lo = mid + 1; else hi = mid; }
    return lo;
}

// pass 0: count the near triangles of vertex i; pass 1: write them at near[ptr[i]..]
// X: the N collocation / evaluation points.  self: they are the vertices of the mesh (a triangle is near its own vertices
// whatever the distance); an evaluator's points lie off the surface and have no incident triangle.
__global__ void near_search(const double *X, const int32_t *F, const double *cen, const double *d2, int64_t N, int64_t T,
                            Grid g, const uint64_t *cell_sorted, const uint32_t *tri_sorted, double eta2, bool self,
                            int32_t *count, const int64_t *ptr, int32_t *near)
{
    const double *V = X;
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const double x[3] = {V[3 * i], V[3 * i + 1], V[3 * i + 2]};
    const int cx = grid_cell(g, x[0], 0), cy = grid_cell(g, x[1], 1), cz = grid_cell(g, x[2], 2);
    int cnt = 0;
    int64_t w = ptr ? ptr[i] : 0;
    for (int z = max(cz - 1, 0); z <= min(cz + 1, g.n[2] - 1); ++z)
        for (int y = max(cy - 1, 0); y <= min(cy + 1, g.n[1] - 1); ++y) {
            const uint64_t rowid = (uint64_t)g.n[0] * ((uint64_t)y + (uint64_t)g.n[1] * (uint64_t)z);
            const uint64_t lo = rowid + (uint64_t)max(cx - 1, 0), hi = rowid + (uint64_t)min(cx + 1, g.n[0] - 1);
            const int64_t b = lower_bound_u64(cell_sorted, T, lo), e = lower_bound_u64(cell_sorted, T, hi + 1);
            for (int64_t j = b; j < e; ++j) {
                const int64_t k = tri_sorted[j];
                const bool inc = self && ((F[3 * k] == i) || (F[3 * k + 1] == i) || (F[3 * k + 2] == i));
                double dc[3];
                for (int d = 0; d < 3; ++d) dc[d] = __dadd_rn(x[d], -cen[3 * k + d]);
                if (inc || dot3_rn(dc, dc) <= __dmul_rn(eta2, d2[k])) {
                    if (near) near[w++] = (int32_t)k;
                    ++cnt;
                }
            }
        }
    if (count) count[i] = cnt;
}

// number of distinct column vertices among the near triangles of row i
__global__ void csr_count(const int32_t *F, const int64_t *nptr, const int32_t *near, int64_t N, int32_t *count)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int64_t b = nptr[i], e = nptr[i + 1];
    int cnt = 0;
    for (int64_t j = b; j < e; ++j)
        for (int a = 0; a < 3; ++a) {
            const int v = F[3 * (int64_t)near[j] + a];
            bool seen = false;
            for (int64_t j2 = b; j2 <= j && !seen; ++j2)
                for (int a2 = 0; a2 < (j2 == j ? a : 3); ++a2)
                    if (F[3 * (int64_t)near[j2] + a2] == v) { seen = true; break; }
            if (!seen) ++cnt;
        }
    count[i] = cnt;
}

// fill row i: columns in order of first appearance, values = sum over near triangles of
// (exact - Gauss) weights of the matching local vertex
__global__ void csr_fill(const double *X, bool self, const double *V, const int32_t *F, const double *A, const double *Nrm,
                         const int64_t *nptr, const int32_t *near, int64_t N,
                         const int64_t *rowptr, int32_t *col, double2 *val, double *diagS)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= N) return;
    const int64_t b = nptr[i], e = nptr[i + 1];
    const int64_t r0 = rowptr[i];
    int ncol = 0;
    double sii = 0.0;                                            // S_ii = exact integral of vertex i's own hat function
    const double x[3] = {X[3 * i], X[3 * i + 1], X[3 * i + 2]};
    for (int64_t j = b; j < e; ++j) {
        const int64_t k = near[j];
        const int v[3] = {F[3 * k], F[3 * k + 1], F[3 * k + 2]};
        double r[3][3];
        for (int a = 0; a < 3; ++a)
            for (int d = 0; d < 3; ++d) r[a][d] = V[3 * (int64_t)v[a] + d];
        int inc = -1;
        for (int a = 0; a < 3; ++a)
            if (self && v[a] == i) inc = a;
        double WS[3], WD[3];
        if (inc >= 0) { tri_weights_incident(r, inc, WS, WD); sii += WS[inc]; }
        else tri_weights_regular(r, x, WS, WD);
        // minus the 3-point Gauss value (what lift + P2P add for this triangle)
        const double w = A[k] / 3.0;
        const double nx = Nrm[3 * k], ny = Nrm[3 * k + 1], nz = Nrm[3 * k + 2];
        for (int gi = 0; gi < 3; ++gi) {
            double y[3];
            gauss_point(V, v[0], v[1], v[2], gi, y);
            const double dx = x[0] - y[0], dy = x[1] - y[1], dz = x[2] - y[2];
            const double r2 = dx * dx + dy * dy + dz * dz;
            const double inv = 1.0 / sqrt(r2);
            const double kS = INV_4PI * w * inv;
            const double kD = INV_4PI * w * (nx * dx + ny * dy + nz * dz) * inv * inv * inv;
            for (int a = 0; a < 3; ++a) {
                const double lam = (a == gi) ? (2.0 / 3.0) : (1.0 / 6.0);
                WS[a] -= lam * kS;
                WD[a] -= lam * kD;
            }
        }
        for (int a = 0; a < 3; ++a) {
            int c = -1;
            for (int t = 0; t < ncol; ++t)
                if (col[r0 + t] == v[a]) { c = t; break; }
            if (c < 0) { c = ncol++; col[r0 + c] = v[a]; val[r0 + c] = make_double2(0.0, 0.0); }
            double2 cur = val[r0 + c];
            cur.x += WS[a];
            cur.y += WD[a];
            val[r0 + c] = cur;
        }
    }
    if (diagS) diagS[i] = sii;
}

void build_correction(bem_ctx *c)
{
    cudaStream_t s = c->stream;
    const bem_ctx *mc = mesh_of(c);                                  // an evaluator corrects against its parent's mesh
    const bool self = mc == c;
    const int64_t N = c->N, T = mc->T;
    dvec<double> cen, d2;
    cen.alloc(3 * T);
    d2.alloc(T);
    tri_centroids<<<cdiv(T, 256), 256, 0, s>>>(mc->V.get(), mc->F.get(), T, cen.get(), d2.get());
    KERNEL_CHECK();
    const double d2max = reduce_max(d2.get(), T, s);
    dvec<double> bb;
    bb.alloc(6);
    bbox3(mc->V.get(), mc->N, bb.get(), s);
    double hb[6];
    d2h_sync(hb, bb.get(), sizeof hb, s);
    Grid g;
    double ext = 0;
    for (int d = 0; d < 3; ++d) { g.mn[d] = hb[d]; ext = std::max(ext, hb[3 + d] - hb[d]); }
    double h = c->eta * sqrt(d2max) * (1.0 + 1e-9);
    if (!(h > ext / 256.0)) h = ext / 256.0;
    if (!(h > 0)) h = 1.0;
    g.h = h;
    for (int d = 0; d < 3; ++d) {
        const double nd = floor((hb[3 + d] - hb[d]) / h) + 1.0;
        g.n[d] = (int)std::min(nd, 258.0);
    }
    dvec<uint64_t> keys, keys_tmp;
    dvec<uint32_t> tri, tri_tmp;
    keys.alloc(T); keys_tmp.alloc(T); tri.alloc(T); tri_tmp.alloc(T);
    tri_cells<<<cdiv(T, 256), 256, 0, s>>>(cen.get(), T, g, keys.get());
    KERNEL_CHECK();
    iota_u32(tri.get(), T, s);
    radix_sort_pairs(keys.get(), tri.get(), keys_tmp.get(), tri_tmp.get(), T, 0, 32, s);

    const double eta2 = c->eta * c->eta;
    dvec<int32_t> cnt;
    dvec<int64_t> nptr;
    cnt.alloc(N);
    nptr.alloc(N + 1);
    near_search<<<cdiv(N, 128), 128, 0, s>>>(c->V.get(), mc->F.get(), cen.get(), d2.get(), N, T, g, keys.get(), tri.get(), eta2, self,
                                             cnt.get(), nullptr, nullptr);
    KERNEL_CHECK();
    scan_exclusive_i64(cnt.get(), nptr.get(), N, s);
    int64_t nnear = 0;
    d2h_sync(&nnear, nptr.get() + N, sizeof(int64_t), s);
    c->near_tris = nnear;
    dvec<int32_t> near;
    near.alloc(nnear);
    near_search<<<cdiv(N, 128), 128, 0, s>>>(c->V.get(), mc->F.get(), cen.get(), d2.get(), N, T, g, keys.get(), tri.get(), eta2, self,
                                             nullptr, nptr.get(), near.get());
    KERNEL_CHECK();
    csr_count<<<cdiv(N, 128), 128, 0, s>>>(mc->F.get(), nptr.get(), near.get(), N, cnt.get());
    KERNEL_CHECK();
    c->rowptr.alloc(N + 1);
    scan_exclusive_i64(cnt.get(), c->rowptr.get(), N, s);
    d2h_sync(&c->nnz, c->rowptr.get() + N, sizeof(int64_t), s);
    c->col.alloc(c->nnz);
    c->val.alloc(c->nnz);
    if (self) c->diagS.alloc(N);
    csr_fill<<<cdiv(N, 128), 128, 0, s>>>(c->V.get(), self, mc->V.get(), mc->F.get(), mc->triA.get(), mc->triN.get(), nptr.get(), near.get(), N,
                                          c->rowptr.get(), c->col.get(), c->val.get(), self ? c->diagS.get() : nullptr);
    KERNEL_CHECK();
    CUDA_TRY(cudaStreamSynchronize(s));
}

// V1 has no off-diagonal correction: an empty CSR (the diagonal is kept separately)
void build_empty_correction(bem_ctx *c)
{
    c->rowptr.alloc(c->N + 1);
    c->rowptr.zero(c->stream);
    c->col.alloc(1);
    c->val.alloc(1);
    c->nnz = 0;
    c->near_tris = 0;
}

}  // namespace bem
