// Steps a1 + a2: octree from 63-bit Morton keys, neighbour and
// interaction lists, all on the device.  PAPER.md:440: "the computational domain
// is scaled to a unit cube and recursively subdivided by an octree to level
// l_max ... 8^l boxes, empty boxes are skipped ... source and receiver data
// structures ... neighbor finding ... interaction lists (e.g., via
// bit-interleaving followed by a sorting algorithm)".
#include "common.cuh"
#include "morton.cuh"
#include "lists.cuh"

namespace bem {

// ------------------------------------------------------------------ keys
__global__ void morton_keys(const double *xyz, int64_t n, double mnx, double mny, double mnz, double inv_side, uint64_t *keys)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    keys[i] = morton_encode(cell21((xyz[3 * i] - mnx) * inv_side), cell21((xyz[3 * i + 1] - mny) * inv_side),
                            cell21((xyz[3 * i + 2] - mnz) * inv_side));
}

// hist[l] = number of adjacent sorted keys that first differ at level l (1..21)
__global__ void split_levels(const uint64_t *keys, int64_t n, int *hist)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x + 1;
    if (i >= n) return;
    const uint64_t x = keys[i] ^ keys[i - 1];
    if (x == 0) return;
    const int b = 63 - __clzll((long long)x);    // highest differing bit, 0..62
    atomicAdd(&hist[21 - b / 3], 1);
}

// ------------------------------------------------------------------ unique prefixes
__global__ void prefix_flags(const uint64_t *keys, int64_t n, int shift, int32_t *flags)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    flags[i] = (i == 0 || (keys[i] >> shift) != (keys[i - 1] >> shift)) ? 1 : 0;
}
// ids = inclusive count - 1; for the first element of every group write its key prefix and position
__global__ void prefix_fill(const uint64_t *keys, int64_t n, int shift, const int32_t *flags, const int32_t *excl,
                            uint64_t *ukey, int32_t *ubegin, int32_t *group_of)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i > n) return;
    if (i == n) { ubegin[excl[n]] = (int32_t)n; return; }
    const int32_t id = excl[i] + flags[i] - 1;
    if (group_of) group_of[i] = id;
    if (flags[i]) { ukey[id] = keys[i] >> shift; ubegin[id] = (int32_t)i; }
}

static int unique_level(const uint64_t *keys, int64_t n, int shift, dvec<uint64_t> &ukey, dvec<int32_t> &ubegin,
                        int32_t *group_of, int expect, cudaStream_t s)
{
    dvec<int32_t> flags, excl;
    flags.alloc(n);
    excl.alloc(n + 1);
    prefix_flags<<<cdiv(n, 256), 256, 0, s>>>(keys, n, shift, flags.get());
    KERNEL_CHECK();
    scan_exclusive_i32(flags.get(), excl.get(), n, s);
    int total = 0;
    d2h_sync(&total, excl.get() + n, sizeof(int), s);
    if (expect >= 0 && total != expect) throw Error(BEM_ERR_CUDA, "octree: box count mismatch between histogram and scan");
    ukey.alloc(total);
    ubegin.alloc(total + 1);
    prefix_fill<<<cdiv(n + 1, 256), 256, 0, s>>>(keys, n, shift, flags.get(), excl.get(), ukey.get(), ubegin.get(), group_of);
    KERNEL_CHECK();
    CUDA_TRY(cudaStreamSynchronize(s));
    return total;
}

// sort the points of one set and count its boxes on every level
void boxset_sort(BoxSet &bs, const double *xyz, int64_t n, const double cube_min[3], double cube_side, int counts[22], cudaStream_t s)
{
    bs.npts = n;
    bs.key_sorted.alloc(n);
    bs.perm.alloc(n);
    dvec<uint64_t> ktmp;
    dvec<uint32_t> vtmp;
    ktmp.alloc(n);
    vtmp.alloc(n);
    morton_keys<<<cdiv(n, 256), 256, 0, s>>>(xyz, n, cube_min[0], cube_min[1], cube_min[2], 1.0 / cube_side, bs.key_sorted.get());
    KERNEL_CHECK();
    iota_u32(bs.perm.get(), n, s);
    radix_sort_pairs(bs.key_sorted.get(), bs.perm.get(), ktmp.get(), vtmp.get(), n, 0, 64, s);
    dvec<int> hist;
    hist.alloc(24);
    hist.zero(s);
    if (n > 1) {
        split_levels<<<cdiv(n - 1, 256), 256, 0, s>>>(bs.key_sorted.get(), n, hist.get());
        KERNEL_CHECK();
    }
    int h[24];
    CUDA_TRY(cudaMemcpyAsync(h, hist.get(), sizeof h, cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    int acc = 1;
    counts[0] = 1;
    for (int l = 1; l <= 21; ++l) { acc += h[l]; counts[l] = acc; }
}

// box tables of levels 0..lmax from the sorted keys
void boxset_build(BoxSet &bs, int lmax, const int counts[22], cudaStream_t s)
{
    bs.lmax = lmax;
    const int64_t n = bs.npts;
    bs.leaf_of.alloc(n);
    bs.nbox[lmax] = unique_level(bs.key_sorted.get(), n, 3 * (21 - lmax), bs.bkey[lmax], bs.begin, bs.leaf_of.get(), counts[lmax], s);
    for (int l = lmax - 1; l >= 0; --l) {
        const int nc = bs.nbox[l + 1];
        bs.parent[l + 1].alloc(nc);
        bs.nbox[l] = unique_level(bs.bkey[l + 1].get(), nc, 3, bs.bkey[l], bs.child[l], bs.parent[l + 1].get(), counts[l], s);
    }
    bs.base[0] = bs.base[1] = bs.base[2] = 0;
    for (int l = 2; l <= lmax; ++l) bs.base[l + 1] = bs.base[l] + bs.nbox[l];
}

// ------------------------------------------------------------------ lists
// source leaves adjacent to (or equal to) each target leaf, in fixed (dz, dy, dx) order, -1 padded
__global__ void neighbour_lists(const uint64_t *tkey, int ntb, const uint64_t *skey, int nsb, int level, int32_t *nbr,
                                const int32_t *tbegin, const int32_t *sbegin, unsigned long long *pair_count)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntb) return;
    uint32_t ix, iy, iz;
    morton_decode(tkey[t], &ix, &iy, &iz);
    const int lim = 1 << level;
    int cnt = 0;
    unsigned long long ns = 0;
    for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
                const int x = (int)ix + dx, y = (int)iy + dy, z = (int)iz + dz;
                if (x < 0 || y < 0 || z < 0 || x >= lim || y >= lim || z >= lim) continue;
                const int b = find_box(skey, nsb, morton_encode(x, y, z));
                if (b >= 0) { nbr[(int64_t)t * 27 + cnt++] = b; ns += (unsigned long long)(sbegin[b + 1] - sbegin[b]); }
            }
    for (int k = cnt; k < 27; ++k) nbr[(int64_t)t * 27 + k] = -1;
    atomicAdd(pair_count, ns * (unsigned long long)(tbegin[t + 1] - tbegin[t]));
}

// pairs the near-field kernel EXECUTES: it pads the concatenated source list of a target leaf (neighbours + direct far
// boxes) to whole rounds of `round` sources (p2p.cu), so a leaf costs nt x ceil(S / round) x round pairs
__global__ void executed_pairs(const int32_t *tbegin, const int32_t *nbr, const int32_t *xptr, const int32_t *xsrc,
                               const int32_t *sbegin, int ntl, int round, unsigned long long *out)
{
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntl) return;
    long long S = 0;
    for (int k = 0; k < 27; ++k) { const int b = nbr[(int64_t)t * 27 + k]; if (b >= 0) S += sbegin[b + 1] - sbegin[b]; }
    if (xptr) for (int k = xptr[t]; k < xptr[t + 1]; ++k) { const int b = xsrc[k]; S += sbegin[b + 1] - sbegin[b]; }
    const long long nt = tbegin[t + 1] - tbegin[t];
    atomicAdd(out, (unsigned long long)(nt * ((S + round - 1) / round) * round));
}

// L2L: one pair per target box: its parent's local expansion through the matrix of its octant
__global__ void l2l_pairs(const uint64_t *tkey, const int32_t *tparent, int nt, int tbase_parent, int32_t *src, int32_t *mat, int32_t *ptr)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j > nt) return;
    ptr[j] = j;
    if (j == nt) return;
    src[j] = tbase_parent + tparent[j];
    mat[j] = MAT_L2L + (int)(tkey[j] & 7ull);
}

__global__ void m2m_pairs(const uint64_t *ckey, int nc, int cbase, int32_t *src, int32_t *mat)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nc) return;
    src[j] = cbase + j;
    mat[j] = MAT_M2M + (int)(ckey[j] & 7ull);
}

__global__ void mat_keys(const int32_t *mat, int64_t n, uint64_t *keys, int *hist)
{
    const int64_t k = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    keys[k] = (uint64_t)mat[k];
    atomicAdd(&hist[mat[k]], 1);
}
__global__ void stage_finish(const uint32_t *order, const int32_t *src, int64_t n, int32_t *src_sorted, int32_t *krow)
{
    const int64_t r = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (r >= n) return;
    const uint32_t k = order[r];
    src_sorted[r] = src[k];
    krow[r] = (int32_t)k;
}

constexpr int GEMM_TM = 64;   // rows per GEMM tile (translate.cu uses the same constant)


// from target-major (src, mat) pairs to a Stage: rows sorted by matrix, tiles, inverse positions
void finish_stage(bem_ctx *c, Stage &st, dvec<int32_t> &src, dvec<int32_t> &mat, cudaStream_t s)
{
    const int64_t n = st.npairs;
    st.src_sorted.alloc(n);
    st.krow.alloc(n);
    std::vector<int> h(N_MATS, 0);
    if (n > 0) {
        dvec<uint64_t> keys, ktmp;
        dvec<uint32_t> order, otmp;
        dvec<int> hist;
        keys.alloc(n); ktmp.alloc(n); order.alloc(n); otmp.alloc(n);
        hist.alloc(N_MATS);
        hist.zero(s);
        mat_keys<<<cdiv(n, 256), 256, 0, s>>>(mat.get(), n, keys.get(), hist.get());
        KERNEL_CHECK();
        iota_u32(order.get(), n, s);
        radix_sort_pairs(keys.get(), order.get(), ktmp.get(), otmp.get(), n, 0, 16, s);
        stage_finish<<<cdiv(n, 256), 256, 0, s>>>(order.get(), src.get(), n, st.src_sorted.get(), st.krow.get());
        KERNEL_CHECK();
        CUDA_TRY(cudaMemcpyAsync(h.data(), hist.get(), N_MATS * sizeof(int), cudaMemcpyDeviceToHost, s));
        CUDA_TRY(cudaStreamSynchronize(s));
    }
    std::vector<Tile> tiles;
    int row = 0;
    for (int m = 0; m < MAT_L2L; ++m) c->m2l_hist[m] += h[m];           // pairs per M2L matrix (statistics, api.cu)
    for (int m = 0; m < N_MATS; ++m) {
        for (int r = 0; r < h[m]; r += GEMM_TM) {
            Tile t;
            t.mat = m;
            t.row0 = row + r;
            t.nrows = std::min(GEMM_TM, h[m] - r);
            t.flags = ((m >= MAT_L2L && m < MAT_M2M) ? 1 : 0) | (m < MAT_L2L ? 2 : 0);
            tiles.push_back(t);
        }
        row += h[m];
    }
    st.tile_mat_host.clear();
    for (const Tile &t : tiles) st.tile_mat_host.push_back(t.mat);
    st.mat_t = std::move(mat);
    st.ntiles = (int)tiles.size();
    st.ntiles_split = 0;
    for (const Tile &t : tiles) st.ntiles_split += (t.flags & 2) ? 1 : 0;
    st.tiles.alloc(tiles.size());
    if (!tiles.empty()) {
        CUDA_TRY(cudaMemcpyAsync(st.tiles.get(), tiles.data(), tiles.size() * sizeof(Tile), cudaMemcpyHostToDevice, s));
        CUDA_TRY(cudaStreamSynchronize(s));                              // `tiles` is a local
    }
}

void build_lists(bem_ctx *c)
{
    cudaStream_t s = c->stream;
    BoxSet &sb = c->sb, &tb = c->tb;
    const int lmax = tb.lmax;
    // near field
    const int ntl = tb.nbox[lmax];
    c->nbr.alloc((size_t)ntl * 27);
    dvec<unsigned long long> pc;
    pc.alloc(1);
    pc.zero(s);
    neighbour_lists<<<cdiv(ntl, 128), 128, 0, s>>>(tb.bkey[lmax].get(), ntl, sb.bkey[lmax].get(), sb.nbox[lmax], lmax, c->nbr.get(),
                                                   tb.begin.get(), sb.begin.get(), pc.get());
    KERNEL_CHECK();
    unsigned long long hp = 0;
    d2h_sync(&hp, pc.get(), sizeof hp, s);
    c->p2p_pairs = (int64_t)hp;
    c->xdir_pairs = 0;
    c->xdir_ptr.free();
    c->xdir_src.free();

    // M2L stages, levels 2..lmax
    c->m2l.clear();
    c->m2l.resize(lmax + 1);
    c->m2l_pairs = 0;
    for (int m = 0; m < MAT_L2L; ++m) c->m2l_hist[m] = 0;
    int64_t max_pairs = 0;
    for (int l = 2; l <= lmax; ++l) {
        Stage &st = c->m2l[l];
        const int nt = tb.nbox[l];
        st.ntgt = nt;
        st.out_base = tb.base[l];
        st.out_is_local = true;
        dvec<int32_t> cnt, xcnt;
        cnt.alloc(nt);
        st.ptr.alloc(nt + 1);
        const int64_t dmax = l == lmax ? c->direct_max_eff : 0;
        if (dmax > 0) { xcnt.alloc(nt); c->xdir_ptr.alloc(nt + 1); pc.zero(s); }
        interaction_lists<<<cdiv(nt, 128), 128, 0, s>>>(tb.bkey[l].get(), nt, l, sb.bkey[l - 1].get(), sb.nbox[l - 1], sb.child[l - 1].get(),
                                                        sb.bkey[l].get(), l > 2 ? tb.parent[l].get() : nullptr, sb.base[l],
                                                        l > 2 ? tb.base[l - 1] : 0, cnt.get(), nullptr, nullptr, nullptr,
                                                        tb.begin.get(), sb.begin.get(), dmax, dmax > 0 ? xcnt.get() : nullptr, nullptr, nullptr, pc.get(), AdaptiveFlags());
        KERNEL_CHECK();
        if (dmax > 0) {
            scan_exclusive_i32(xcnt.get(), c->xdir_ptr.get(), nt, s);
            int xt = 0;
            d2h_sync(&xt, c->xdir_ptr.get() + nt, sizeof(int), s);
            unsigned long long xp = 0;
            d2h_sync(&xp, pc.get(), sizeof xp, s);
            c->xdir_pairs = xt;
            c->p2p_pairs += (int64_t)xp;
            c->xdir_src.alloc(xt);
        }
        scan_exclusive_i32(cnt.get(), st.ptr.get(), nt, s);
        int total = 0;
        d2h_sync(&total, st.ptr.get() + nt, sizeof(int), s);
        st.npairs = total;
        dvec<int32_t> src, mat;
        src.alloc(total);
        mat.alloc(total);
        interaction_lists<<<cdiv(nt, 128), 128, 0, s>>>(tb.bkey[l].get(), nt, l, sb.bkey[l - 1].get(), sb.nbox[l - 1], sb.child[l - 1].get(),
                                                        sb.bkey[l].get(), l > 2 ? tb.parent[l].get() : nullptr, sb.base[l],
                                                        l > 2 ? tb.base[l - 1] : 0, nullptr, st.ptr.get(), src.get(), mat.get(),
                                                        tb.begin.get(), sb.begin.get(), dmax, nullptr, dmax > 0 ? c->xdir_ptr.get() : nullptr,
                                                        dmax > 0 ? c->xdir_src.get() : nullptr, pc.get(), AdaptiveFlags());
        KERNEL_CHECK();
        finish_stage(c, st, src, mat, s);
        c->m2l_pairs += total;
        st.scratch_off = max_pairs;                           // regions of the levels one after the other
        max_pairs += total;
    }
    {
        pc.zero(s);
        executed_pairs<<<cdiv(ntl, 128), 128, 0, s>>>(tb.begin.get(), c->nbr.get(), c->xdir_ptr.p, c->xdir_src.p, sb.begin.get(), ntl, 128, pc.get());
        KERNEL_CHECK();
        unsigned long long ex = 0;
        d2h_sync(&ex, pc.get(), sizeof ex, s);
        c->p2p_pairs_exec = (int64_t)ex;
    }
    // M2M stages: parents on level l = lmax-1 .. 2
    c->m2m.clear();
    c->m2m.resize(lmax + 1);
    for (int l = lmax - 1; l >= 2; --l) {
        Stage &st = c->m2m[l];
        const int nc = sb.nbox[l + 1];
        st.ntgt = sb.nbox[l];
        st.out_base = sb.base[l];
        st.out_is_local = false;
        st.npairs = nc;
        st.ptr.alloc(st.ntgt + 1);
        CUDA_TRY(cudaMemcpyAsync(st.ptr.get(), sb.child[l].get(), (st.ntgt + 1) * sizeof(int32_t), cudaMemcpyDeviceToDevice, s));
        dvec<int32_t> src, mat;
        src.alloc(nc);
        mat.alloc(nc);
        m2m_pairs<<<cdiv(nc, 256), 256, 0, s>>>(sb.bkey[l + 1].get(), nc, sb.base[l + 1], src.get(), mat.get());
        KERNEL_CHECK();
        finish_stage(c, st, src, mat, s);
        st.scratch_off = 0;                                   // M2M runs before any M2L tile: aliases the first region
        max_pairs = std::max<int64_t>(max_pairs, nc);
    }
    // L2L stages: children on level l = 3 .. lmax (run after every M2L row has been summed: alias the first region)
    c->l2l.clear();
    c->l2l.resize(lmax + 1);
    for (int l = 3; l <= lmax; ++l) {
        Stage &st = c->l2l[l];
        const int nt = tb.nbox[l];
        st.ntgt = nt;
        st.out_base = tb.base[l];
        st.out_is_local = true;
        st.accumulate = true;
        st.npairs = nt;
        st.ptr.alloc(nt + 1);
        dvec<int32_t> src, mat;
        src.alloc(nt);
        mat.alloc(nt);
        l2l_pairs<<<cdiv(nt + 1, 256), 256, 0, s>>>(tb.bkey[l].get(), tb.parent[l].get(), nt, tb.base[l - 1], src.get(), mat.get(), st.ptr.get());
        KERNEL_CHECK();
        finish_stage(c, st, src, mat, s);
        st.scratch_off = 0;
        max_pairs = std::max<int64_t>(max_pairs, nt);
    }
}

}  // namespace bem
