// Adaptive octree (option "tree" = 1, reading R9 stage 2; PAPER.md:440 gives the uniform tree, BASELINE.json
// asks config 3 to "stress the adaptive octree" and config 2 for "leaf <= 64 points").
//
// Rule.  A geometric box is SUBDIVIDED iff it holds more than leaf_size sources or lies above level lmin (the depth the
// uniform rule gives for the same leaf_size, option "tree_min_level": the adaptive tree is never coarser than the uniform
// one, it only refines the boxes that are denser than the mean); the deepest level never is.  A box EXISTS iff its parent is subdivided; a LEAF is an existing box that is not subdivided.  Source and
// target trees follow the same rule (the source count of the geometric box), so they are subdivided alike.
//
// Lists of a target leaf t of level lt, walking its ancestors a_2 .. a_lt = t (every source point is met exactly once):
//   V  at every level l: existing source boxes of level l that are children of the neighbours of parent(a_l) and do not
//      touch a_l -> M2L (the uniform machinery, restricted to existing boxes; tree.cu interaction_lists);
//   U  source boxes of level lt that touch t, leaf or not: ALL their sources are summed directly (a finer source leaf that
//      does not touch t -- the classical W list -- is summed directly too: exact, and a few points by construction);
//   X  source LEAVES of a coarser level l < lt that touch a_l: summed directly with t (they have no children to translate).
// The direct ranges of a target leaf form one CSR row (near_ptr, near_rng) that the pair kernel reads as its segment list.
// Upward: P2M on the source leaves of every level, M2M from the existing children.  Downward: L2L to the existing
// children, L2P at the target leaf of every point.
#include "common.cuh"
#include "morton.cuh"
#include "segments.cuh"
#include "lists.cuh"
#include <algorithm>

namespace bem {

void finish_stage(bem_ctx *c, Stage &st, dvec<int32_t> &src, dvec<int32_t> &mat, cudaStream_t s);     // tree.cu
// first point of every box of a level from the level below: pbeg[j] = pbeg_child[child[j]], j = 0 .. n (n + 1 entries)
__global__ void parent_ranges(const int32_t *child, const int32_t *pbeg_child, int n, int32_t *pbeg)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j <= n) pbeg[j] = pbeg_child[child[j]];
}

__global__ void src_flags(int level, int lcap, int lmin, int n, const int32_t *pbeg, const int32_t *parent, const uint8_t *ex_par,
                          const uint8_t *sub_par, int leaf_size, uint8_t *ex, uint8_t *sub, int *any_ex, int *want_deeper)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n) return;
    const bool e = level <= 2 ? true : (ex_par[parent[b]] && sub_par[parent[b]]);
    const int cnt = pbeg[b + 1] - pbeg[b];
    ex[b] = e;
    sub[b] = e && level < lcap && (level < lmin || cnt > leaf_size);
    if (e) *any_ex = 1;
    if (e && level == lcap && cnt > leaf_size) *want_deeper = 1;   // the probe depth cut a box that the rule would subdivide
}

// a target box is subdivided iff the geometric box is: the flag of the source box with the same key (no source box: not)
__global__ void tgt_flags(int level, int lcap, int lmin, int n, const uint64_t *tkey, const int32_t *parent, const uint8_t *ex_par,
                          const uint8_t *sub_par, const uint64_t *skey, int nsb, const uint8_t *s_sub, uint8_t *ex, uint8_t *sub)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= n) return;
    const bool e = level <= 2 ? true : (ex_par[parent[b]] && sub_par[parent[b]]);
    bool s = false;
    if (e && level < lcap) {
        if (level < lmin) s = true;
        else { const int i = find_box(skey, nsb, tkey[b]); s = i >= 0 && s_sub[i]; }
    }
    ex[b] = e;
    sub[b] = s;
}

__global__ void flag_leaves(const uint8_t *ex, const uint8_t *sub, int n, int32_t *f)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n) f[b] = (ex[b] && !sub[b]) ? 1 : 0;
}
__global__ void flag_bytes(const uint8_t *ex, int n, int32_t *f)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n) f[b] = ex[b] ? 1 : 0;
}
__global__ void scatter_ids(const int32_t *f, const int32_t *pos, int n, int32_t *out)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n && f[b]) out[pos[b]] = b;
}

// existing children of level l + 1 -> their parents: target-major pairs (children of a parent are contiguous)
__global__ void m2m_pairs_adaptive(const uint64_t *ckey, const int32_t *f, const int32_t *pos, int nc, int cbase, int32_t *src, int32_t *mat)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j >= nc || !f[j]) return;
    src[pos[j]] = cbase + j;
    mat[pos[j]] = MAT_M2M + (int)(ckey[j] & 7ull);
}
__global__ void m2m_ptr_adaptive(const int32_t *child, const int32_t *pos, int np, int32_t *ptr)
{
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p <= np) ptr[p] = pos[child[p]];                     // pos has nc + 1 entries (the total at the end)
}
// one L2L pair per EXISTING target box of the level
__global__ void l2l_pairs_adaptive(const uint64_t *tkey, const int32_t *tparent, const int32_t *f, const int32_t *pos, int nt,
                                   int tbase_parent, int32_t *src, int32_t *mat, int32_t *ptr)
{
    const int j = blockIdx.x * blockDim.x + threadIdx.x;
    if (j > nt) return;
    ptr[j] = pos[j];
    if (j == nt || !f[j]) return;
    src[pos[j]] = tbase_parent + tparent[j];
    mat[pos[j]] = MAT_L2L + (int)(tkey[j] & 7ull);
}

struct LevelTables {                                           // device pointers of every level, passed by value
    const uint64_t *skey[MAX_LEVEL + 1], *tkey[MAX_LEVEL + 1];
    const int32_t *tparent[MAX_LEVEL + 1], *s_pbeg[MAX_LEVEL + 1], *t_pbeg[MAX_LEVEL + 1];
    const uint8_t *s_ex[MAX_LEVEL + 1], *s_sub[MAX_LEVEL + 1], *t_ex[MAX_LEVEL + 1], *t_sub[MAX_LEVEL + 1];
    const int32_t *x_ptr[MAX_LEVEL + 1], *x_src[MAX_LEVEL + 1];
    int nsb[MAX_LEVEL + 1], tbase[MAX_LEVEL + 2];
    int lmax;
};

// the leaf of every target point: climb from its box of the deepest level to the one box that exists and is not subdivided
__global__ void point_leaves(const int32_t *leaf_of, int64_t n, LevelTables L, int32_t *pt_gbox)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= n) return;
    int b = leaf_of[t], g = -1;
    for (int l = L.lmax; l >= 2; --l) {
        if (L.t_ex[l][b] && !L.t_sub[l][b]) { g = L.tbase[l] + b; break; }
        b = L.tparent[l][b];
    }
    pt_gbox[t] = g;
}
__global__ void leaf_starts(const int32_t *pt_gbox, int64_t n, int32_t *f)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t < n) f[t] = (t == 0 || pt_gbox[t] != pt_gbox[t - 1]) ? 1 : 0;
}
__global__ void leaf_fill(const int32_t *pt_gbox, const int32_t *f, const int32_t *pos, int64_t n, int32_t *begin, int32_t *gbox)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t > n) return;
    if (t == n) { begin[pos[n]] = (int32_t)n; return; }
    if (f[t]) { begin[pos[t]] = (int32_t)t; gbox[pos[t]] = pt_gbox[t]; }
}
__global__ void all_box_tables(const uint64_t *tkey, int n, int base, int level, uint64_t *key_all, uint8_t *lev_all)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b < n) { key_all[base + b] = tkey[b]; lev_all[base + b] = (uint8_t)level; }
}

// direct source ranges of every target leaf (count pass: rng == nullptr).  Order: the coarser levels first, then the own
// level, then the far leaves summed directly -- a fixed order, so the sums are bit-reproducible.
__global__ void near_lists(const int32_t *tleaf_gbox, const int32_t *tleaf_begin, int nleaf, LevelTables L,
                           int32_t *count, const int32_t *ptr, int2 *rng, unsigned long long *pairs, unsigned long long *pairs_exec,
                           unsigned long long *pairs_wx)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nleaf) return;
    const int g = tleaf_gbox[i];
    int lt = 2;
    while (lt < L.lmax && g >= L.tbase[lt + 1]) ++lt;
    const int b = g - L.tbase[lt];
    uint32_t ix, iy, iz;
    morton_decode(L.tkey[lt][b], &ix, &iy, &iz);
    int cnt = 0;
    int w = ptr ? ptr[i] : 0;
    long long S = 0;
    long long SX = 0;       // statistics (BEM_S_P2P_PAIRS_WX): sources of the ranges an FMM with M2P / P2L would not sum directly
    for (int l = 2; l <= lt; ++l) {
        const int sh = lt - l;
        const int ax = (int)(ix >> sh), ay = (int)(iy >> sh), az = (int)(iz >> sh);     // the ancestor of level l
        const int lim = 1 << l;
        for (int dz = -1; dz <= 1; ++dz)
            for (int dy = -1; dy <= 1; ++dy)
                for (int dx = -1; dx <= 1; ++dx) {
                    const int x = ax + dx, y = ay + dy, z = az + dz;
                    if (x < 0 || y < 0 || z < 0 || x >= lim || y >= lim || z >= lim) continue;
                    const int sbx = find_box(L.skey[l], L.nsb[l], morton_encode(x, y, z));
                    if (sbx < 0 || !L.s_ex[l][sbx]) continue;
                    if (l < lt && L.s_sub[l][sbx]) continue;                            // its children are met one level down
                    const int s0 = L.s_pbeg[l][sbx], n = L.s_pbeg[l][sbx + 1] - s0;
                    if (rng) rng[w++] = make_int2(s0, n);
                    ++cnt;
                    S += n;
                    if (!count) continue;
                    if (l < lt) {
                        // X list: a coarser source leaf next to the ancestor that does not touch the leaf itself (P2L would serve)
                        const int lox = x << sh, loy = y << sh, loz = z << sh, ext = (1 << sh);
                        const bool touch = (int)ix >= lox - 1 && (int)ix <= lox + ext && (int)iy >= loy - 1 && (int)iy <= loy + ext &&
                                           (int)iz >= loz - 1 && (int)iz <= loz + ext;
                        if (!touch) SX += n;
                    } else if (L.s_sub[l][sbx]) {
                        // W list: children of a subdivided neighbour that do not touch the leaf (M2P would serve)
                        for (int ch = 0; ch < 8; ++ch) {
                            const int cx = 2 * x + (ch & 1), cy = 2 * y + ((ch >> 1) & 1), cz = 2 * z + (ch >> 2);
                            const int cb = find_box(L.skey[l + 1], L.nsb[l + 1], morton_encode(cx, cy, cz));
                            if (cb < 0) continue;
                            const bool touch = cx >= 2 * (int)ix - 1 && cx <= 2 * (int)ix + 2 && cy >= 2 * (int)iy - 1 && cy <= 2 * (int)iy + 2 &&
                                               cz >= 2 * (int)iz - 1 && cz <= 2 * (int)iz + 2;
                            if (!touch) SX += L.s_pbeg[l + 1][cb + 1] - L.s_pbeg[l + 1][cb];
                        }
                    }
                }
    }
    if (L.x_ptr[lt]) {                                                                  // far leaves of the own level summed directly
        for (int k = L.x_ptr[lt][b]; k < L.x_ptr[lt][b + 1]; ++k) {
            const int sbx = L.x_src[lt][k];
            const int s0 = L.s_pbeg[lt][sbx], n = L.s_pbeg[lt][sbx + 1] - s0;
            if (rng) rng[w++] = make_int2(s0, n);
            ++cnt;
            S += n;
        }
    }
    if (count) {
        count[i] = cnt;
        const long long nt = tleaf_begin[i + 1] - tleaf_begin[i];
        atomicAdd(pairs, (unsigned long long)(nt * S));
        atomicAdd(pairs_exec, (unsigned long long)(nt * ((S + 127) / 128) * 128));
        atomicAdd(pairs_wx, (unsigned long long)(nt * SX));
    }
}

__global__ void max_i32(const int32_t *v, int n, int *out)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) atomicMax(out, v[i]);
}

// ------------------------------------------------------------------ host side
static void build_ranges(BoxSet &bs, dvec<int32_t> *pbeg, cudaStream_t s)
{
    const int lmax = bs.lmax;
    pbeg[lmax].alloc(bs.nbox[lmax] + 1);
    CUDA_TRY(cudaMemcpyAsync(pbeg[lmax].get(), bs.begin.get(), (bs.nbox[lmax] + 1) * sizeof(int32_t), cudaMemcpyDeviceToDevice, s));
    for (int l = lmax - 1; l >= 0; --l) {
        pbeg[l].alloc(bs.nbox[l] + 1);
        parent_ranges<<<cdiv(bs.nbox[l] + 1, 256), 256, 0, s>>>(bs.child[l].get(), pbeg[l + 1].get(), bs.nbox[l], pbeg[l].get());
        KERNEL_CHECK();
    }
}

// source flags of levels 0 .. sb.lmax; returns the deepest level on which a box exists (*want_deeper: the rule would
// subdivide a box of the deepest level built)
int adaptive_source_flags(bem_ctx *c, bool *want_deeper)
{
    cudaStream_t s = c->stream;
    BoxSet &sb = c->sb;
    Adaptive &ad = c->ad;
    const int lcap = sb.lmax;
    build_ranges(sb, ad.s_pbeg, s);
    dvec<int> any;
    any.alloc(MAX_LEVEL + 2);
    any.zero(s);
    for (int l = 0; l <= lcap; ++l) {
        const int n = sb.nbox[l];
        ad.s_ex[l].alloc(n);
        ad.s_sub[l].alloc(n);
        src_flags<<<cdiv(n, 256), 256, 0, s>>>(l, lcap, ad.lmin, n, ad.s_pbeg[l].get(), l > 0 ? sb.parent[l].get() : nullptr,
                                               l > 0 ? ad.s_ex[l - 1].get() : nullptr, l > 0 ? ad.s_sub[l - 1].get() : nullptr,
                                               c->leaf_size, ad.s_ex[l].get(), ad.s_sub[l].get(), any.get() + l, any.get() + MAX_LEVEL + 1);
        KERNEL_CHECK();
    }
    int h[MAX_LEVEL + 2];
    d2h_sync(h, any.get(), sizeof h, s);
    if (want_deeper) *want_deeper = h[MAX_LEVEL + 1] != 0;
    int deepest = 2;
    for (int l = 2; l <= lcap; ++l) if (h[l]) deepest = l;
    return deepest;
}

// ids of the flagged entries, in order; returns their number
static int compact_flags(const int32_t *flags, int n, dvec<int32_t> &pos, dvec<int32_t> *ids, cudaStream_t s)
{
    pos.alloc(n + 1);
    scan_exclusive_i32(flags, pos.get(), n, s);
    int total = 0;
    d2h_sync(&total, pos.get() + n, sizeof(int), s);
    if (ids) {
        ids->alloc(total);
        if (n > 0) { scatter_ids<<<cdiv(n, 256), 256, 0, s>>>(flags, pos.get(), n, ids->get()); KERNEL_CHECK(); }
    }
    return total;
}

void build_adaptive(bem_ctx *c)
{
    cudaStream_t s = c->stream;
    BoxSet &sb = c->sb, &tb = c->tb;
    Adaptive &ad = c->ad;
    const int lmax = sb.lmax;
    // flags (the source flags were computed for this depth by adaptive_source_flags)
    build_ranges(tb, ad.t_pbeg, s);
    for (int l = 0; l <= lmax; ++l) {
        const int n = tb.nbox[l];
        ad.t_ex[l].alloc(n);
        ad.t_sub[l].alloc(n);
        tgt_flags<<<cdiv(n, 256), 256, 0, s>>>(l, lmax, ad.lmin, n, tb.bkey[l].get(), l > 0 ? tb.parent[l].get() : nullptr,
                                               l > 0 ? ad.t_ex[l - 1].get() : nullptr, l > 0 ? ad.t_sub[l - 1].get() : nullptr,
                                               sb.bkey[l].get(), sb.nbox[l], ad.s_sub[l].get(), ad.t_ex[l].get(), ad.t_sub[l].get());
        KERNEL_CHECK();
    }
    // source leaves of every level (P2M)
    ad.n_src_leaves = 0;
    for (int l = 2; l <= lmax; ++l) {
        const int n = sb.nbox[l];
        dvec<int32_t> f, pos;
        f.alloc(n);
        flag_leaves<<<cdiv(n, 256), 256, 0, s>>>(ad.s_ex[l].get(), ad.s_sub[l].get(), n, f.get());
        KERNEL_CHECK();
        ad.n_sleaf[l] = compact_flags(f.get(), n, pos, &ad.sleaf[l], s);
        ad.n_src_leaves += ad.n_sleaf[l];
    }
    // global tables of the target boxes, leaf of every target point, target leaves in point order
    const int ntot = tb.total();
    ad.tkey_all.alloc(ntot);
    ad.tlev_all.alloc(ntot);
    LevelTables L;
    memset(&L, 0, sizeof L);
    L.lmax = lmax;
    for (int l = 0; l <= lmax; ++l) {
        L.skey[l] = sb.bkey[l].get(); L.tkey[l] = tb.bkey[l].get();
        L.tparent[l] = l > 0 ? tb.parent[l].get() : nullptr;
        L.s_pbeg[l] = ad.s_pbeg[l].get(); L.t_pbeg[l] = ad.t_pbeg[l].get();
        L.s_ex[l] = ad.s_ex[l].get(); L.s_sub[l] = ad.s_sub[l].get(); L.t_ex[l] = ad.t_ex[l].get(); L.t_sub[l] = ad.t_sub[l].get();
        L.nsb[l] = sb.nbox[l];
        L.tbase[l] = tb.base[l];
    }
    L.tbase[lmax + 1] = tb.base[lmax + 1];
    for (int l = 2; l <= lmax; ++l) {
        all_box_tables<<<cdiv(tb.nbox[l], 256), 256, 0, s>>>(tb.bkey[l].get(), tb.nbox[l], tb.base[l], l, ad.tkey_all.get(), ad.tlev_all.get());
        KERNEL_CHECK();
    }
    const int64_t N = c->N;
    ad.pt_gbox.alloc(N);
    point_leaves<<<cdiv(N, 256), 256, 0, s>>>(tb.leaf_of.get(), N, L, ad.pt_gbox.get());
    KERNEL_CHECK();
    {
        dvec<int32_t> f, pos;
        f.alloc(N);
        leaf_starts<<<cdiv(N, 256), 256, 0, s>>>(ad.pt_gbox.get(), N, f.get());
        KERNEL_CHECK();
        ad.n_tleaf = compact_flags(f.get(), (int)N, pos, nullptr, s);
        ad.tleaf_begin.alloc(ad.n_tleaf + 1);
        ad.tleaf_gbox.alloc(ad.n_tleaf);
        leaf_fill<<<cdiv(N + 1, 256), 256, 0, s>>>(ad.pt_gbox.get(), f.get(), pos.get(), N, ad.tleaf_begin.get(), ad.tleaf_gbox.get());
        KERNEL_CHECK();
    }

    dvec<unsigned long long> pc;
    pc.alloc(3);
    // M2L stages of the existing boxes, levels 2 .. lmax; far pairs between two sparse leaves go to the direct lists
    c->m2l.clear();
    c->m2l.resize(lmax + 1);
    c->m2l_pairs = 0;
    for (int m = 0; m < MAT_L2L; ++m) c->m2l_hist[m] = 0;
    int64_t max_pairs = 0;
    unsigned long long xpairs_total = 0;
    for (int l = 2; l <= lmax; ++l) {
        Stage &st = c->m2l[l];
        const int nt = tb.nbox[l];
        st.ntgt = nt;
        st.out_base = tb.base[l];
        st.out_is_local = true;
        {
            dvec<int32_t> f, pos;
            f.alloc(nt);
            flag_bytes<<<cdiv(nt, 256), 256, 0, s>>>(ad.t_ex[l].get(), nt, f.get());
            KERNEL_CHECK();
            st.n_list = compact_flags(f.get(), nt, pos, &st.tgt_list, s);
        }
        dvec<int32_t> cnt, xcnt;
        cnt.alloc(nt);
        st.ptr.alloc(nt + 1);
        const int64_t dmax = c->direct_max_eff;
        AdaptiveFlags af;
        af.t_ex = ad.t_ex[l].get(); af.t_sub = ad.t_sub[l].get(); af.s_sub = ad.s_sub[l].get();
        af.s_ex_parent = ad.s_ex[l - 1].get(); af.s_sub_parent = ad.s_sub[l - 1].get();
        if (dmax > 0) { xcnt.alloc(nt); ad.x_ptr[l].alloc(nt + 1); pc.zero(s); }
        else { ad.x_ptr[l].free(); ad.x_src[l].free(); }
        interaction_lists<<<cdiv(nt, 128), 128, 0, s>>>(tb.bkey[l].get(), nt, l, sb.bkey[l - 1].get(), sb.nbox[l - 1], sb.child[l - 1].get(),
                                                        sb.bkey[l].get(), l > 2 ? tb.parent[l].get() : nullptr, sb.base[l],
                                                        l > 2 ? tb.base[l - 1] : 0, cnt.get(), nullptr, nullptr, nullptr,
                                                        ad.t_pbeg[l].get(), ad.s_pbeg[l].get(), dmax, dmax > 0 ? xcnt.get() : nullptr, nullptr, nullptr,
                                                        pc.get(), af);
        KERNEL_CHECK();
        if (dmax > 0) {
            scan_exclusive_i32(xcnt.get(), ad.x_ptr[l].get(), nt, s);
            int xt = 0;
            d2h_sync(&xt, ad.x_ptr[l].get() + nt, sizeof(int), s);
            ad.x_src[l].alloc(xt);
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
                                                        ad.t_pbeg[l].get(), ad.s_pbeg[l].get(), dmax, nullptr, dmax > 0 ? ad.x_ptr[l].get() : nullptr,
                                                        dmax > 0 ? ad.x_src[l].get() : nullptr, pc.get(), af);
        KERNEL_CHECK();
        finish_stage(c, st, src, mat, s);
        c->m2l_pairs += total;
        st.scratch_off = max_pairs;
        max_pairs += total;
    }
    (void)xpairs_total;
    // M2M: existing children of level l + 1 -> parents of level l (a parent without children keeps what P2M wrote)
    c->m2m.clear();
    c->m2m.resize(lmax + 1);
    for (int l = lmax - 1; l >= 2; --l) {
        Stage &st = c->m2m[l];
        const int nc = sb.nbox[l + 1];
        st.ntgt = sb.nbox[l];
        st.out_base = sb.base[l];
        st.out_is_local = false;
        st.keep_empty = true;
        {
            dvec<int32_t> f, pos;
            f.alloc(st.ntgt);
            flag_bytes<<<cdiv(st.ntgt, 256), 256, 0, s>>>(ad.s_sub[l].get(), st.ntgt, f.get());      // parents that have children
            KERNEL_CHECK();
            st.n_list = compact_flags(f.get(), st.ntgt, pos, &st.tgt_list, s);
        }
        dvec<int32_t> f, pos;
        f.alloc(nc);
        flag_bytes<<<cdiv(nc, 256), 256, 0, s>>>(ad.s_ex[l + 1].get(), nc, f.get());
        KERNEL_CHECK();
        const int total = compact_flags(f.get(), nc, pos, nullptr, s);
        st.npairs = total;
        st.ptr.alloc(st.ntgt + 1);
        m2m_ptr_adaptive<<<cdiv(st.ntgt + 1, 256), 256, 0, s>>>(sb.child[l].get(), pos.get(), st.ntgt, st.ptr.get());
        KERNEL_CHECK();
        dvec<int32_t> src, mat;
        src.alloc(total);
        mat.alloc(total);
        m2m_pairs_adaptive<<<cdiv(nc, 256), 256, 0, s>>>(sb.bkey[l + 1].get(), f.get(), pos.get(), nc, sb.base[l + 1], src.get(), mat.get());
        KERNEL_CHECK();
        finish_stage(c, st, src, mat, s);
        st.scratch_off = 0;
        max_pairs = std::max<int64_t>(max_pairs, total);
    }
    // L2L: parents of level l - 1 -> existing children of level l
    c->l2l.clear();
    c->l2l.resize(lmax + 1);
    for (int l = 3; l <= lmax; ++l) {
        Stage &st = c->l2l[l];
        const int nt = tb.nbox[l];
        st.ntgt = nt;
        st.out_base = tb.base[l];
        st.out_is_local = true;
        st.accumulate = true;
        dvec<int32_t> f, pos;
        f.alloc(nt);
        flag_bytes<<<cdiv(nt, 256), 256, 0, s>>>(ad.t_ex[l].get(), nt, f.get());
        KERNEL_CHECK();
        const int total = compact_flags(f.get(), nt, pos, &st.tgt_list, s);
        st.n_list = total;
        st.npairs = total;
        st.ptr.alloc(nt + 1);
        dvec<int32_t> src, mat;
        src.alloc(total);
        mat.alloc(total);
        l2l_pairs_adaptive<<<cdiv(nt + 1, 256), 256, 0, s>>>(tb.bkey[l].get(), tb.parent[l].get(), f.get(), pos.get(), nt, tb.base[l - 1],
                                                             src.get(), mat.get(), st.ptr.get());
        KERNEL_CHECK();
        finish_stage(c, st, src, mat, s);
        st.scratch_off = 0;
        max_pairs = std::max<int64_t>(max_pairs, total);
    }

    // direct source ranges of the target leaves
    for (int l = 0; l <= lmax; ++l) { L.x_ptr[l] = ad.x_ptr[l].p; L.x_src[l] = ad.x_src[l].p; }
    dvec<int32_t> cnt;
    cnt.alloc(ad.n_tleaf);
    pc.zero(s);
    near_lists<<<cdiv(ad.n_tleaf, 128), 128, 0, s>>>(ad.tleaf_gbox.get(), ad.tleaf_begin.get(), ad.n_tleaf, L, cnt.get(), nullptr, nullptr,
                                                     pc.get(), pc.get() + 1, pc.get() + 2);
    KERNEL_CHECK();
    ad.near_ptr.alloc(ad.n_tleaf + 1);
    scan_exclusive_i32(cnt.get(), ad.near_ptr.get(), ad.n_tleaf, s);
    int nseg = 0;
    d2h_sync(&nseg, ad.near_ptr.get() + ad.n_tleaf, sizeof(int), s);
    unsigned long long hp[3];
    d2h_sync(hp, pc.get(), sizeof hp, s);
    c->p2p_pairs = (int64_t)hp[0];
    c->p2p_pairs_exec = (int64_t)hp[1];
    c->p2p_pairs_wx = (int64_t)hp[2];
    dvec<int> mx;
    mx.alloc(1);
    mx.zero(s);
    max_i32<<<cdiv(ad.n_tleaf, 256), 256, 0, s>>>(cnt.get(), ad.n_tleaf, mx.get());
    KERNEL_CHECK();
    int longest = 0;
    d2h_sync(&longest, mx.get(), sizeof(int), s);
    const int limit = std::min(c->seg_limit, (int)SEG_MAX);
    ad.row_overflow = longest > limit;                             // bem_setup tries once more without the direct far pairs (api.cu)
    if (longest > limit)
        throw Error(BEM_ERR_INVALID_ARG, "adaptive tree: a target leaf has " + std::to_string(longest) + " direct source ranges, more than the " +
                                         std::to_string(limit) + " the pair kernel's table holds (raise leaf_size or lower direct_pairs)");
    ad.near_rng.alloc(nseg);
    near_lists<<<cdiv(ad.n_tleaf, 128), 128, 0, s>>>(ad.tleaf_gbox.get(), ad.tleaf_begin.get(), ad.n_tleaf, L, nullptr, ad.near_ptr.get(),
                                                     ad.near_rng.get(), pc.get(), pc.get() + 1, pc.get() + 2);
    KERNEL_CHECK();
    CUDA_TRY(cudaStreamSynchronize(s));
}

}  // namespace bem
