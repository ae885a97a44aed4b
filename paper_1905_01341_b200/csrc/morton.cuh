// 63-bit Morton keys: 21 bits per axis, bit-interleaved x (bit 0), y (bit 1), z (bit 2)
// ("bit-interleaving"; reading R11).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace bem {

__host__ __device__ __forceinline__ uint64_t spread3(uint64_t x)
{
    x &= 0x1fffffull;
    x = (x | x << 32) & 0x1f00000000ffffull;
    x = (x | x << 16) & 0x1f0000ff0000ffull;
    x = (x | x << 8) & 0x100f00f00f00f00full;
    x = (x | x << 4) & 0x10c30c30c30c30c3ull;
    x = (x | x << 2) & 0x1249249249249249ull;
    return x;
}
__host__ __device__ __forceinline__ uint32_t compact3(uint64_t x)
{
    x &= 0x1249249249249249ull;
    x = (x ^ (x >> 2)) & 0x10c30c30c30c30c3ull;
    x = (x ^ (x >> 4)) & 0x100f00f00f00f00full;
    x = (x ^ (x >> 8)) & 0x1f0000ff0000ffull;
    x = (x ^ (x >> 16)) & 0x1f00000000ffffull;
    x = (x ^ (x >> 32)) & 0x1fffffull;
    return (uint32_t)x;
}
__host__ __device__ __forceinline__ uint64_t morton_encode(uint32_t ix, uint32_t iy, uint32_t iz)
{
    return spread3(ix) | (spread3(iy) << 1) | (spread3(iz) << 2);
}
__host__ __device__ __forceinline__ void morton_decode(uint64_t k, uint32_t *ix, uint32_t *iy, uint32_t *iz)
{
    *ix = compact3(k); *iy = compact3(k >> 1); *iz = compact3(k >> 2);
}
// unit-cube coordinate u in [0,1] -> cell index min(floor(u 2^21), 2^21 - 1)
__host__ __device__ __forceinline__ uint32_t cell21(double u)
{
    double v = floor(u * 2097152.0);
    if (!(v > 0.0)) v = 0.0;
    if (v > 2097151.0) v = 2097151.0;
    return (uint32_t)v;
}

// index of key k in the ascending array keys[0..n), or -1
__device__ __forceinline__ int find_box(const uint64_t *keys, int n, uint64_t k)
{
    int lo = 0, hi = n;
    while (lo < hi) { const int mid = (lo + hi) >> 1; if (keys[mid] < k) lo = mid + 1; else hi = mid; }
    return (lo < n && keys[lo] == k) ? lo : -1;
}

}  // namespace bem
