// Flat-triangle geometry shared by the setup kernels (step a0).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bem {

// A = |e1 x e2|/2,  N = (e1 x e2)/|e1 x e2|,  e1 = r1-r0, e2 = r2-r0
__device__ __forceinline__ void tri_area_normal(const double *V, int v0, int v1, int v2, double *A, double *N)
{
    const double *r0 = V + 3 * (int64_t)v0, *r1 = V + 3 * (int64_t)v1, *r2 = V + 3 * (int64_t)v2;
    const double e1x = r1[0] - r0[0], e1y = r1[1] - r0[1], e1z = r1[2] - r0[2];
    const double e2x = r2[0] - r0[0], e2y = r2[1] - r0[1], e2z = r2[2] - r0[2];
    const double cx = e1y * e2z - e1z * e2y, cy = e1z * e2x - e1x * e2z, cz = e1x * e2y - e1y * e2x;
    const double nn = sqrt(cx * cx + cy * cy + cz * cz);
    *A = 0.5 * nn;
    N[0] = cx / nn; N[1] = cy / nn; N[2] = cz / nn;
}

// Gauss point gi of the triangle (v0,v1,v2): barycentric weight 2/3 on vertex gi, 1/6 on the others.
// Every product and sum is rounded separately (no FMA contraction), in the order
// (l0 r0 + l1 r1) + l2 r2, so that the point is the IEEE value of that expression
// on any machine -- the P2P kernel and the correction matrix must see bit-identical points.
__device__ __forceinline__ void gauss_point(const double *V, int v0, int v1, int v2, int gi, double *y)
{
    const double *r0 = V + 3 * (int64_t)v0, *r1 = V + 3 * (int64_t)v1, *r2 = V + 3 * (int64_t)v2;
    const double big = 2.0 / 3.0, small = 1.0 / 6.0;
    const double l0 = gi == 0 ? big : small, l1 = gi == 1 ? big : small, l2 = gi == 2 ? big : small;
#pragma unroll
    for (int d = 0; d < 3; ++d)
        y[d] = __dadd_rn(__dadd_rn(__dmul_rn(l0, r0[d]), __dmul_rn(l1, r1[d])), __dmul_rn(l2, r2[d]));
}

}  // namespace bem
