// The interaction-list kernel shared by the uniform tree (tree.cu) and the adaptive tree (adaptive.cu).
#pragma once
#include "common.cuh"
#include "morton.cuh"

namespace bem {

// Interaction (V) list of target box t at `level`: source boxes that are children of the
// parent's neighbours and not adjacent to t.
// count pass (src == nullptr) or fill pass.
static __global__ void interaction_lists(const uint64_t *tkey, int ntb, int level,
                                  const uint64_t *skey_parent, int nsb_parent, const int32_t *schild_parent,
                                  const uint64_t *skey, const int32_t *tparent, int sbase, int tbase_parent,
                                  int32_t *count, const int32_t *ptr, int32_t *src, int32_t *mat,
                                  const int32_t *tbegin, const int32_t *sbegin, int64_t direct_max,
                                  int32_t *xcount, const int32_t *xptr, int32_t *xsrc, unsigned long long *xpairs,
                                  const AdaptiveFlags af)
{
    // adaptive tree (adaptive.cu): only EXISTING boxes take part -- a target box exists iff its parent is subdivided, and the
    // children of a source box of the parent level exist iff that box is subdivided (a source LEAF of the parent level that
    // touches the parent is summed directly instead); a pair goes to the direct list only between two leaves
    const int t = blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= ntb) return;
    if (af.t_ex && !af.t_ex[t]) { if (count) count[t] = 0; if (xcount) xcount[t] = 0; return; }
    const bool t_leaf = !af.t_sub || !af.t_sub[t];
    uint32_t ix, iy, iz;
    morton_decode(tkey[t], &ix, &iy, &iz);
    const int px = ix >> 1, py = iy >> 1, pz = iz >> 1;
    const int lim = 1 << (level - 1);
    int cnt = 0;
    int w = ptr ? ptr[t] : 0;
    // leaf level, direct_max > 0: a pair whose boxes hold nt x ns <= direct_max point pairs costs less summed directly
    // than translated (one M2L = 4 nre^2 flop whatever the boxes hold): it goes to the near field (list xsrc) instead
    const int64_t ntp = direct_max > 0 ? tbegin[t + 1] - tbegin[t] : 0;
    int xc = 0, xw = xptr ? xptr[t] : 0;
    unsigned long long xp = 0;
    for (int dz = -1; dz <= 1; ++dz)
        for (int dy = -1; dy <= 1; ++dy)
            for (int dx = -1; dx <= 1; ++dx) {
                const int x = px + dx, y = py + dy, z = pz + dz;
                if (x < 0 || y < 0 || z < 0 || x >= lim || y >= lim || z >= lim) continue;
                const int pb = find_box(skey_parent, nsb_parent, morton_encode(x, y, z));
                if (pb < 0) continue;
                if (af.s_ex_parent && !(af.s_ex_parent[pb] && af.s_sub_parent[pb])) continue;
                for (int c = schild_parent[pb]; c < schild_parent[pb + 1]; ++c) {
                    uint32_t cx, cy, cz;
                    morton_decode(skey[c], &cx, &cy, &cz);
                    const int ox = (int)ix - (int)cx, oy = (int)iy - (int)cy, oz = (int)iz - (int)cz;   // target - source
                    if (max(max(abs(ox), abs(oy)), abs(oz)) < 2) continue;                           // adjacent: near field
                    if (direct_max > 0 && t_leaf && (!af.s_sub || !af.s_sub[c])) {
                        const int64_t nsp = sbegin[c + 1] - sbegin[c];
                        if (ntp * nsp <= direct_max) {
                            if (xsrc) xsrc[xw++] = c;
                            ++xc;
                            xp += (unsigned long long)(ntp * nsp);
                            continue;
                        }
                    }
                    if (src) { src[w] = sbase + c; mat[w] = MAT_M2L + (ox + 3) + 7 * (oy + 3) + 49 * (oz + 3); ++w; }
                    ++cnt;
                }
            }
    if (count) count[t] = cnt;
    if (xcount) { xcount[t] = xc; if (xp) atomicAdd(xpairs, xp); }
}

}  // namespace bem
