// Step a0: mesh validation, triangle geometry, quadrature sources.
//   area A_k, unit normal N_k out of the bubble;
//   G3: three Gauss points per triangle, barycentric (2/3,1/6,1/6) permutations,
//       weight A_k/3 (reading R2);
//   V1: one source per vertex, s_j = 1/3 sum_{k ni j} A_k, n_j = m_j/|m_j|,
//       m_j = sum_{k ni j} N_k A_k (Eq. 17).
#include "common.cuh"
#include "geom.cuh"

namespace bem {

// ------------------------------------------------------------------ validation
// flags: bit0 index out of range, bit1 zero area / non-finite, bit2 triangle spans two bubbles
__global__ void check_triangles(const double *V, const int32_t *F, const int32_t *bid, int64_t N, int64_t T,
                                int *flags, uint64_t *edge_keys)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= T) return;
    int v[3];
    bool ok = true;
    for (int a = 0; a < 3; ++a) {
        v[a] = F[3 * k + a];
        if (v[a] < 0 || v[a] >= N) ok = false;
    }
    if (!ok) {
        atomicOr(flags, 1);
        for (int a = 0; a < 3; ++a) edge_keys[3 * k + a] = ~0ull;
        return;
    }
    double A, Nrm[3];
    tri_area_normal(V, v[0], v[1], v[2], &A, Nrm);
    if (!(A > 0.0) || !isfinite(A)) atomicOr(flags, 2);
    if (bid && (bid[v[0]] != bid[v[1]] || bid[v[0]] != bid[v[2]])) atomicOr(flags, 4);
    if (v[0] == v[1] || v[1] == v[2] || v[0] == v[2]) atomicOr(flags, 2);
    // directed edges (u -> w): key = (min << 32 | max) * 2 + (u > w)
    for (int a = 0; a < 3; ++a) {
        const uint64_t u = (uint64_t)v[a], w = (uint64_t)v[(a + 1) % 3];
        const uint64_t lo = u < w ? u : w, hi = u < w ? w : u;
        edge_keys[3 * k + a] = ((lo << 31 | hi) << 1) | (u > w ? 1ull : 0ull);
    }
}

// after sorting: keys must come in pairs (2e, 2e+1) with distinct e -- every undirected edge is
// used exactly once in each direction <=> closed, consistently oriented manifold
__global__ void check_edges(const uint64_t *keys, int64_t n, int *flags)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (2 * i + 1 >= n) return;
    const uint64_t a = keys[2 * i], b = keys[2 * i + 1];
    bool ok = ((a & 1ull) == 0) && (b == a + 1);
    if (2 * i + 2 < n && (keys[2 * i + 2] >> 1) == (a >> 1)) ok = false;
    if (!ok) atomicOr(flags, 8);
}

// signed volume per bubble: sum_k r0.(r1 x r2)/6 ; only its sign is used
__global__ void bubble_volumes(const double *V, const int32_t *F, const int32_t *bid, int64_t T, double *vol)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= T) return;
    const int a = F[3 * k], b = F[3 * k + 1], c = F[3 * k + 2];
    const double *r0 = V + 3 * (int64_t)a, *r1 = V + 3 * (int64_t)b, *r2 = V + 3 * (int64_t)c;
    // relative to r0 of the bubble's first... use triangle's own offset-free form about r0 of vertex a:
    // volume is translation invariant for a closed surface, so any common origin works; use the origin.
    const double cx = r1[1] * r2[2] - r1[2] * r2[1];
    const double cy = r1[2] * r2[0] - r1[0] * r2[2];
    const double cz = r1[0] * r2[1] - r1[1] * r2[0];
    atomicAdd(&vol[bid ? bid[a] : 0], (r0[0] * cx + r0[1] * cy + r0[2] * cz) / 6.0);
}
__global__ void check_volumes(const double *vol, int nb, int *flags)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < nb && !(vol[b] > 0.0)) atomicOr(flags, 16);
}
__global__ void max_i32(const int32_t *v, int64_t n, int *out)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { if (v[i] < 0) atomicOr(out + 1, 1); atomicMax(out, v[i]); }
}

void validate_mesh(bem_ctx *c)
{
    cudaStream_t s = c->stream;
    if (c->T % 2 != 0) throw Error(BEM_ERR_BAD_MESH, "odd number of triangles: surface cannot be closed");
    dvec<int> flags;
    flags.alloc(4);
    flags.zero(s);
    c->nbubbles = 1;
    if (c->bid.p) {
        max_i32<<<cdiv(c->N, 256), 256, 0, s>>>(c->bid.get(), c->N, flags.get() + 1);
        KERNEL_CHECK();
        int h[2];
        CUDA_TRY(cudaMemcpyAsync(h, flags.get() + 1, 2 * sizeof(int), cudaMemcpyDeviceToHost, s));
        CUDA_TRY(cudaStreamSynchronize(s));
        if (h[1]) throw Error(BEM_ERR_BAD_MESH, "negative bubble id");
        c->nbubbles = h[0] + 1;
    }
    const int64_t ne = 3 * c->T;
    dvec<uint64_t> keys, keys_tmp;
    dvec<uint32_t> vals, vals_tmp;
    keys.alloc(ne); keys_tmp.alloc(ne); vals.alloc(ne); vals_tmp.alloc(ne);
    check_triangles<<<cdiv(c->T, 256), 256, 0, s>>>(c->V.get(), c->F.get(), c->bid.p, c->N, c->T, flags.get(), keys.get());
    KERNEL_CHECK();
    int hf = 0;
    CUDA_TRY(cudaMemcpyAsync(&hf, flags.get(), sizeof(int), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    if (hf & 1) throw Error(BEM_ERR_BAD_MESH, "triangle vertex index out of range");
    if (hf & 2) throw Error(BEM_ERR_BAD_MESH, "zero-area or degenerate triangle");
    if (hf & 4) throw Error(BEM_ERR_BAD_MESH, "a triangle joins vertices of two bubbles");
    iota_u32(vals.get(), ne, s);
    radix_sort_pairs(keys.get(), vals.get(), keys_tmp.get(), vals_tmp.get(), ne, 0, 64, s);
    check_edges<<<cdiv(ne / 2 + 1, 256), 256, 0, s>>>(keys.get(), ne, flags.get());
    KERNEL_CHECK();
    dvec<double> vol;
    vol.alloc(c->nbubbles);
    vol.zero(s);
    bubble_volumes<<<cdiv(c->T, 256), 256, 0, s>>>(c->V.get(), c->F.get(), c->bid.p, c->T, vol.get());
    KERNEL_CHECK();
    check_volumes<<<cdiv(c->nbubbles, 256), 256, 0, s>>>(vol.get(), c->nbubbles, flags.get());
    KERNEL_CHECK();
    CUDA_TRY(cudaMemcpyAsync(&hf, flags.get(), sizeof(int), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    if (hf & 8) throw Error(BEM_ERR_BAD_MESH, "surface is not a closed, consistently oriented manifold (unmatched edge)");
    if (hf & 16) throw Error(BEM_ERR_BAD_MESH, "a bubble has non-positive signed volume: triangles must be counter-clockwise seen from the liquid");
}

// ------------------------------------------------------------------ geometry
__global__ void tri_geometry_kernel(const double *V, const int32_t *F, int64_t T, double *A, double *Nrm)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= T) return;
    double a, n[3];
    tri_area_normal(V, F[3 * k], F[3 * k + 1], F[3 * k + 2], &a, n);
    A[k] = a;
    Nrm[3 * k] = n[0]; Nrm[3 * k + 1] = n[1]; Nrm[3 * k + 2] = n[2];
}

void compute_geometry(bem_ctx *c)
{
    c->triA.alloc(c->T);
    c->triN.alloc(3 * c->T);
    tri_geometry_kernel<<<cdiv(c->T, 256), 256, 0, c->stream>>>(c->V.get(), c->F.get(), c->T, c->triA.get(), c->triN.get());
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ sources
// G3 source s = order[e] (e = engine position); original id g = 3k + gi
__global__ void build_sources_g3(const double *V, const int32_t *F, const double *A, const double *Nrm,
                                 const uint32_t *order, int64_t ns, double4 *pos, double4 *lw, int4 *lv)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= ns) return;
    const int64_t g = order ? order[e] : e;
    const int64_t k = g / 3;
    const int gi = (int)(g - 3 * k);
    const int v0 = F[3 * k + gi], v1 = F[3 * k + (gi + 1) % 3], v2 = F[3 * k + (gi + 2) % 3];
    double y[3];
    gauss_point(V, F[3 * k], F[3 * k + 1], F[3 * k + 2], gi, y);
    const double w = A[k] / 3.0;
    pos[e] = make_double4(y[0], y[1], y[2], 0.0);
    lw[e] = make_double4(w, w * Nrm[3 * k], w * Nrm[3 * k + 1], w * Nrm[3 * k + 2]);
    lv[e] = make_int4(v0, v1, v2, 0);
}

// (vertex, corner) incidence sorted by vertex gives a fixed summation order for s_j, m_j
__global__ void corner_keys(const int32_t *F, int64_t T, uint64_t *keys)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < 3 * T) keys[i] = (uint64_t)F[i];
}
__global__ void vertex_ranges(const uint64_t *keys, int64_t n, int64_t N, int32_t *begin)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    // begin[v] = first i with keys[i] >= v
    const int64_t lo = (i == 0) ? -1 : (int64_t)keys[i - 1];
    const int64_t hi = (i == n) ? N : (int64_t)keys[i];
    for (int64_t v = lo + 1; v <= hi; ++v) begin[v] = (int32_t)i;
}
__global__ void build_sources_v1(const double *V, const double *A, const double *Nrm, const uint32_t *corner,
                                 const int32_t *begin, const uint32_t *order, int64_t N,
                                 double4 *pos, double4 *lw, int4 *lv)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= N) return;
    const int64_t j = order ? order[e] : e;
    double s = 0, m[3] = {0, 0, 0};
    for (int i = begin[j]; i < begin[j + 1]; ++i) {
        const int64_t k = corner[i] / 3;
        s += A[k] / 3.0;
        for (int d = 0; d < 3; ++d) m[d] += Nrm[3 * k + d] * A[k];
    }
    const double nn = sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
    pos[e] = make_double4(V[3 * j], V[3 * j + 1], V[3 * j + 2], 0.0);
    lw[e] = make_double4(s, s * (m[0] / nn), s * (m[1] / nn), s * (m[2] / nn));
    lv[e] = make_int4((int)j, (int)j, (int)j, 0);
}

// point cloud: unit weight, no normal; strength j is the j-th entry of q
__global__ void build_sources_points(const double *P, const uint32_t *order, int64_t n, double4 *pos, double4 *lw, int4 *lv)
{
    const int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n) return;
    const int64_t j = order ? order[e] : e;
    pos[e] = make_double4(P[3 * j], P[3 * j + 1], P[3 * j + 2], 0.0);
    lw[e] = make_double4(1.0, 0.0, 0.0, 0.0);
    lv[e] = make_int4((int)j, (int)j, (int)j, 0);
}

// Build src_pos / lift_w / lift_vid in engine order (order == nullptr: natural order).
void build_sources(bem_ctx *c, const uint32_t *order)
{
    cudaStream_t s = c->stream;
    const bem_ctx *mc = mesh_of(c);
    c->ns = (c->quadrature == 0 || c->quadrature == 3) ? 3 * mc->T : (c->quadrature == 2 ? c->np : c->N);
    c->src_pos.alloc(c->ns);
    c->lift_w.alloc(c->ns);
    c->lift_vid.alloc(c->ns);
    c->src_str.alloc(c->ns);
    if (c->quadrature == 0 || c->quadrature == 3) {
        build_sources_g3<<<cdiv(c->ns, 256), 256, 0, s>>>(mc->V.get(), mc->F.get(), mc->triA.get(), mc->triN.get(), order,
                                                          c->ns, c->src_pos.get(), c->lift_w.get(), c->lift_vid.get());
        KERNEL_CHECK();
    } else if (c->quadrature == 2) {
        build_sources_points<<<cdiv(c->ns, 256), 256, 0, s>>>(c->P.get(), order, c->ns, c->src_pos.get(), c->lift_w.get(), c->lift_vid.get());
        KERNEL_CHECK();
    } else {
        const int64_t nc = 3 * c->T;
        dvec<uint64_t> keys, keys_tmp;
        dvec<uint32_t> vals, vals_tmp;
        dvec<int32_t> begin;
        keys.alloc(nc); keys_tmp.alloc(nc); vals.alloc(nc); vals_tmp.alloc(nc); begin.alloc(c->N + 1);
        corner_keys<<<cdiv(nc, 256), 256, 0, s>>>(c->F.get(), c->T, keys.get());
        KERNEL_CHECK();
        iota_u32(vals.get(), nc, s);
        radix_sort_pairs(keys.get(), vals.get(), keys_tmp.get(), vals_tmp.get(), nc, 0, 32, s);
        vertex_ranges<<<cdiv(nc + 1, 256), 256, 0, s>>>(keys.get(), nc, c->N, begin.get());
        KERNEL_CHECK();
        build_sources_v1<<<cdiv(c->N, 256), 256, 0, s>>>(c->V.get(), c->triA.get(), c->triN.get(), vals.get(), begin.get(),
                                                         order, c->N, c->src_pos.get(), c->lift_w.get(), c->lift_vid.get());
        KERNEL_CHECK();
        CUDA_TRY(cudaStreamSynchronize(s));
    }
}

// Gauss-point / vertex positions of all sources in natural order, AoS xyz (input of the Morton keys)
__global__ void source_points_g3(const double *V, const int32_t *F, int64_t T, double *xyz)
{
    const int64_t g = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= 3 * T) return;
    const int64_t k = g / 3;
    double y[3];
    gauss_point(V, F[3 * k], F[3 * k + 1], F[3 * k + 2], (int)(g - 3 * k), y);
    xyz[3 * g] = y[0]; xyz[3 * g + 1] = y[1]; xyz[3 * g + 2] = y[2];
}
void source_points(bem_ctx *c, dvec<double> &xyz)
{
    if (c->quadrature == 0 || c->quadrature == 3) {
        const bem_ctx *mc = mesh_of(c);
        xyz.alloc(9 * mc->T);
        source_points_g3<<<cdiv(3 * mc->T, 256), 256, 0, c->stream>>>(mc->V.get(), mc->F.get(), mc->T, xyz.get());
        KERNEL_CHECK();
    } else if (c->quadrature == 2) {
        xyz.alloc(3 * c->np);
        CUDA_TRY(cudaMemcpyAsync(xyz.get(), c->P.get(), 3 * c->np * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    } else {
        xyz.alloc(3 * c->N);
        CUDA_TRY(cudaMemcpyAsync(xyz.get(), c->V.get(), 3 * c->N * sizeof(double), cudaMemcpyDeviceToDevice, c->stream));
    }
}

}  // namespace bem
