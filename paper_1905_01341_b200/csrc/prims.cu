// Device primitives used by bem_setup: exclusive scan, stable LSD radix sort of
// (u64 key, u32 value) pairs, bounding box, max.  The paper builds its octree by
// "bit-interleaving followed by a sorting algorithm" on the CPU, with a serial
// sort; here all of it runs on the device.
#include "common.cuh"

namespace bem {

std::atomic<size_t> g_device_bytes{0};

// ------------------------------------------------------------------ scan
constexpr int SCAN_THREADS = 256;
constexpr int SCAN_ITEMS = 8;
constexpr int SCAN_TILE = SCAN_THREADS * SCAN_ITEMS;

template <class TO>
__device__ __forceinline__ TO block_exclusive_scan(TO v, TO *total, TO *smem /* [SCAN_THREADS/32] */)
{
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    TO x = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        TO y = __shfl_up_sync(0xffffffffu, x, d);
        if (lane >= d) x += y;
    }
    if (lane == 31) smem[warp] = x;
    __syncthreads();
    TO woff = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < SCAN_THREADS / 32; ++w) {
        TO s = smem[w];
        if (w < warp) woff += s;
        tot += s;
    }
    __syncthreads();
    *total = tot;
    return woff + x - v;
}

template <class TI, class TO>
__global__ void scan_tile_sums(const TI *in, TO *sums, int64_t n)
{
    __shared__ TO sm[SCAN_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    TO v = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k)
        if (base + k < n) v += (TO)in[base + k];
    TO tot;
    block_exclusive_scan<TO>(v, &tot, sm);
    if (threadIdx.x == 0) sums[blockIdx.x] = tot;
}

template <class TI, class TO>
__global__ void scan_tile_apply(const TI *in, const TO *offs, TO *out, int64_t n, int write_total)
{
    __shared__ TO sm[SCAN_THREADS / 32];
    const int64_t base = (int64_t)blockIdx.x * SCAN_TILE + (int64_t)threadIdx.x * SCAN_ITEMS;
    TO item[SCAN_ITEMS];
    TO v = 0;
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        item[k] = (base + k < n) ? (TO)in[base + k] : (TO)0;
        v += item[k];
    }
    TO tot;
    TO ex = block_exclusive_scan<TO>(v, &tot, sm) + offs[blockIdx.x];
#pragma unroll
    for (int k = 0; k < SCAN_ITEMS; ++k) {
        if (base + k < n) out[base + k] = ex;
        ex += item[k];
    }
    // the grand total goes to out[n]
    if (write_total && base <= n - 1 && n - 1 < base + SCAN_ITEMS) out[n] = ex;
}

template <class TI, class TO>
static void scan_impl(const TI *in, TO *out, int64_t n, cudaStream_t s, int write_total)
{
    if (n <= 0) {
        if (write_total) CUDA_TRY(cudaMemsetAsync(out, 0, sizeof(TO), s));
        return;
    }
    const int nb = cdiv(n, SCAN_TILE);
    dvec<TO> sums, offs;
    sums.alloc(nb);
    offs.alloc(nb + 1);
    scan_tile_sums<TI, TO><<<nb, SCAN_THREADS, 0, s>>>(in, sums.get(), n);
    KERNEL_CHECK();
    if (nb > 1) scan_impl<TO, TO>(sums.get(), offs.get(), nb, s, 0);
    else CUDA_TRY(cudaMemsetAsync(offs.get(), 0, sizeof(TO), s));
    scan_tile_apply<TI, TO><<<nb, SCAN_THREADS, 0, s>>>(in, offs.get(), out, n, write_total);
    KERNEL_CHECK();
    CUDA_TRY(cudaStreamSynchronize(s));   // temporaries are freed on return
}

void scan_exclusive_i32(const int32_t *in, int32_t *out, int64_t n, cudaStream_t s) { scan_impl<int32_t, int32_t>(in, out, n, s, 1); }
void scan_exclusive_i64(const int32_t *in, int64_t *out, int64_t n, cudaStream_t s) { scan_impl<int32_t, int64_t>(in, out, n, s, 1); }

// ------------------------------------------------------------------ radix sort
// One pass sorts on an 8-bit digit.  The input is cut into tiles of SORT_TILE
// consecutive elements, one warp per tile.  (1) per-tile digit histograms,
// (2) exclusive scan of the histogram table laid out digit-major, so that entry
// (digit, tile) becomes the first output slot of that tile's elements with that
// digit, (3) each warp walks its tile in order, 32 elements per round, and ranks
// equal digits inside a round with __match_any_sync -- stable by construction.
constexpr int SORT_WARPS = 8;
constexpr int SORT_ROUNDS = 64;
constexpr int SORT_TILE = 32 * SORT_ROUNDS;

__global__ void sort_hist(const uint64_t *keys, int64_t n, int shift, int ntiles, int32_t *table)
{
    __shared__ int h[SORT_WARPS][256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x * SORT_WARPS + warp;
    for (int d = lane; d < 256; d += 32) h[warp][d] = 0;
    __syncwarp();
    if (tile < ntiles) {
        const int64_t t0 = (int64_t)tile * SORT_TILE;
        const int64_t t1 = min(t0 + (int64_t)SORT_TILE, n);
        for (int64_t i = t0 + lane; i < t1; i += 32) atomicAdd(&h[warp][(keys[i] >> shift) & 255u], 1);
        __syncwarp();
        for (int d = lane; d < 256; d += 32) table[(int64_t)d * ntiles + tile] = h[warp][d];
    }
}

__global__ void sort_scatter(const uint64_t *keys, const uint32_t *vals, uint64_t *keys_out, uint32_t *vals_out,
                             int64_t n, int shift, int ntiles, const int32_t *table_scanned)
{
    __shared__ int off[SORT_WARPS][256];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int tile = blockIdx.x * SORT_WARPS + warp;
    if (tile >= ntiles) return;
    for (int d = lane; d < 256; d += 32) off[warp][d] = table_scanned[(int64_t)d * ntiles + tile];
    __syncwarp();
    const int64_t t0 = (int64_t)tile * SORT_TILE;
    const int64_t t1 = min(t0 + (int64_t)SORT_TILE, n);
    for (int64_t r0 = t0; r0 < t1; r0 += 32) {
        const int64_t i = r0 + lane;
        const bool valid = i < t1;
        uint64_t k = 0;
        uint32_t v = 0;
        if (valid) { k = keys[i]; v = vals[i]; }
        const unsigned digit = valid ? (unsigned)((k >> shift) & 255u) : (256u + lane);
        const unsigned peers = __match_any_sync(0xffffffffu, digit);
        const int rank = __popc(peers & ((1u << lane) - 1u));
        int base = 0;
        if (valid) base = off[warp][digit];
        __syncwarp();
        if (valid && rank == 0) off[warp][digit] = base + __popc(peers);
        __syncwarp();
        if (valid) { keys_out[base + rank] = k; vals_out[base + rank] = v; }
    }
}

void radix_sort_pairs(uint64_t *keys, uint32_t *vals, uint64_t *keys_tmp, uint32_t *vals_tmp,
                      int64_t n, int begin_bit, int end_bit, cudaStream_t s)
{
    if (n <= 1) return;
    const int ntiles = cdiv(n, SORT_TILE);
    const int nblocks = cdiv(ntiles, SORT_WARPS);
    dvec<int32_t> table, scanned;
    table.alloc((size_t)256 * ntiles);
    scanned.alloc((size_t)256 * ntiles + 1);
    uint64_t *kin = keys, *kout = keys_tmp;
    uint32_t *vin = vals, *vout = vals_tmp;
    int npass = 0;
    for (int shift = begin_bit; shift < end_bit; shift += 8) {
        sort_hist<<<nblocks, SORT_WARPS * 32, 0, s>>>(kin, n, shift, ntiles, table.get());
        KERNEL_CHECK();
        scan_exclusive_i32(table.get(), scanned.get(), (int64_t)256 * ntiles, s);
        sort_scatter<<<nblocks, SORT_WARPS * 32, 0, s>>>(kin, vin, kout, vout, n, shift, ntiles, scanned.get());
        KERNEL_CHECK();
        std::swap(kin, kout);
        std::swap(vin, vout);
        ++npass;
    }
    if (npass & 1) {   // result sits in the tmp arrays
        CUDA_TRY(cudaMemcpyAsync(keys, keys_tmp, n * sizeof(uint64_t), cudaMemcpyDeviceToDevice, s));
        CUDA_TRY(cudaMemcpyAsync(vals, vals_tmp, n * sizeof(uint32_t), cudaMemcpyDeviceToDevice, s));
    }
    CUDA_TRY(cudaStreamSynchronize(s));
}

__global__ void iota_kernel(uint32_t *v, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) v[i] = (uint32_t)i;
}
void iota_u32(uint32_t *v, int64_t n, cudaStream_t s)
{
    if (n <= 0) return;
    iota_kernel<<<cdiv(n, 256), 256, 0, s>>>(v, n);
    KERNEL_CHECK();
}

// ------------------------------------------------------------------ reductions
__global__ void bbox_partial(const double *xyz, int64_t n, double *part /* [grid*6] */)
{
    double mn[3] = {1e300, 1e300, 1e300}, mx[3] = {-1e300, -1e300, -1e300};
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x)
        for (int d = 0; d < 3; ++d) {
            const double v = xyz[3 * i + d];
            mn[d] = fmin(mn[d], v);
            mx[d] = fmax(mx[d], v);
        }
    __shared__ double sm[256][6];
    for (int d = 0; d < 3; ++d) { sm[threadIdx.x][d] = mn[d]; sm[threadIdx.x][3 + d] = mx[d]; }
    __syncthreads();
    for (int st = blockDim.x / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st)
            for (int d = 0; d < 3; ++d) {
                sm[threadIdx.x][d] = fmin(sm[threadIdx.x][d], sm[threadIdx.x + st][d]);
                sm[threadIdx.x][3 + d] = fmax(sm[threadIdx.x][3 + d], sm[threadIdx.x + st][3 + d]);
            }
        __syncthreads();
    }
    if (threadIdx.x < 6) part[blockIdx.x * 6 + threadIdx.x] = sm[0][threadIdx.x];
}
__global__ void bbox_final(const double *part, int nparts, double *out6)
{
    if (threadIdx.x < 6) {
        const int d = threadIdx.x;
        double v = part[d];
        for (int b = 1; b < nparts; ++b) v = d < 3 ? fmin(v, part[b * 6 + d]) : fmax(v, part[b * 6 + d]);
        out6[d] = v;
    }
}
void bbox3(const double *xyz, int64_t n, double *out6, cudaStream_t s)
{
    const int nb = (int)std::min<int64_t>(512, cdiv(n, 256));
    dvec<double> part;
    part.alloc((size_t)nb * 6);
    bbox_partial<<<nb, 256, 0, s>>>(xyz, n, part.get());
    KERNEL_CHECK();
    bbox_final<<<1, 32, 0, s>>>(part.get(), nb, out6);
    KERNEL_CHECK();
    CUDA_TRY(cudaStreamSynchronize(s));
}

__global__ void max_partial(const double *v, int64_t n, double *part)
{
    double m = -1e300;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) m = fmax(m, v[i]);
    __shared__ double sm[256];
    sm[threadIdx.x] = m;
    __syncthreads();
    for (int st = blockDim.x / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st) sm[threadIdx.x] = fmax(sm[threadIdx.x], sm[threadIdx.x + st]);
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = sm[0];
}
double reduce_max(const double *v, int64_t n, cudaStream_t s)
{
    const int nb = (int)std::min<int64_t>(512, cdiv(n, 256));
    dvec<double> part;
    part.alloc(nb);
    max_partial<<<nb, 256, 0, s>>>(v, n, part.get());
    KERNEL_CHECK();
    std::vector<double> h(nb);
    CUDA_TRY(cudaMemcpyAsync(h.data(), part.get(), nb * sizeof(double), cudaMemcpyDeviceToHost, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    double m = h[0];
    for (double x : h) m = std::max(m, x);
    return m;
}

}  // namespace bem
