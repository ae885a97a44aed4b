// bem_direct_sum_static: the all-pairs sum of the two Laplace kernels (Eq. 13, in point form) for callers
// that must not allocate device memory.
//
// Who that is.  Every other entry of this library calls cudaMalloc somewhere (bem_create, bem_setup, the staging of
// bem_apply, the Krylov basis of bem_solve).  Some hosts cannot afford that at the time they want a potential:
//   * a time-stepping code that sized its own arenas at start-up and left the device full -- a cudaMalloc then fails, or
//     succeeds only by luck of what the pool happens to have returned to the driver;
//   * a process that shares the GPU under a fixed memory budget (an MPS client limit, a MIG slice handed out by a
//     scheduler): memory taken behind the owner's back is memory another tenant was promised;
//   * a latency-bound loop: cudaMalloc and cudaFree synchronise the whole device, so one call stalls every other stream
//     of the process in the middle of a step.
// For them the partial sums of the direct kernel -- the only scratch the all-pairs path needs (p2p.cu keeps them in
// bem_ctx::ypart, allocated by bem_setup) -- live in a file-scope __device__ array below.  The price: the array is part of
// the library image, so EVERY GPU that loads libbem_b200.so carries its 8 MiB until the process exits, used or not, and
// its size is a compile-time maximum (BEM_DIRECT_STATIC_MAX_TARGETS targets per call).
//
// The kernels here are this file's own (direct-sum arithmetic restated, not shared with p2p.cu): sources are read
// straight from the caller's [n x 3] arrays, so no packed copy of them is needed either.
#include "common.cuh"

#include <algorithm>
#include <mutex>

namespace {

constexpr int DS_THREADS = 128;
constexpr int DS_TPT = 4;                  // targets per thread: one shared-memory source read feeds four pairs
constexpr int DS_TILE = 256;               // sources staged per round
constexpr int DS_MAX_SPLIT = 16;           // source chunks per target block (fills the SMs when there are few targets)
constexpr int64_t DS_MAX_TARGETS = BEM_DIRECT_STATIC_MAX_TARGETS;
constexpr int DS_MAX_DEVICES = 64;

// The scratch: partial sums [split][target], split < DS_MAX_SPLIT.  In HOST code this name is only a handle for
// cudaGetSymbolAddress -- it is not a device address and must never be handed to a kernel as one.
static __device__ __align__(256) double g_ds_partials[DS_MAX_SPLIT * DS_MAX_TARGETS];

// per device: the address of g_ds_partials on that device, looked up once (set-up, under the mutex)
std::mutex g_ds_mutex;
double *g_ds_ptr[DS_MAX_DEVICES] = {nullptr};

thread_local std::string g_ds_error = "no error";

// chunk `blockIdx.y` of the sources against 512 targets; partial sums to part[blockIdx.y * nt + t]
template <bool DIP>
__global__ void __launch_bounds__(DS_THREADS)
ds_partial_kernel(const double *__restrict__ tgt, int64_t nt, const double *__restrict__ src, const double *__restrict__ q,
                  const double *__restrict__ dip, int64_t ns, int64_t chunk, double *__restrict__ part)
{
    __shared__ double sxyz[3 * DS_TILE], sm[DS_TILE], sd[DIP ? 3 * DS_TILE : 1];
    const int64_t tfirst = (int64_t)blockIdx.x * (DS_TPT * DS_THREADS) + threadIdx.x;
    double tx[DS_TPT], ty[DS_TPT], tz[DS_TPT], acc[DS_TPT];
#pragma unroll
    for (int k = 0; k < DS_TPT; ++k) {
        const int64_t t = tfirst + (int64_t)k * DS_THREADS;
        tx[k] = ty[k] = tz[k] = 0.0;
        acc[k] = 0.0;
        if (t < nt) { tx[k] = tgt[3 * t]; ty[k] = tgt[3 * t + 1]; tz[k] = tgt[3 * t + 2]; }
    }
    const int64_t s0 = (int64_t)blockIdx.y * chunk, s1 = min(s0 + chunk, ns);
    for (int64_t base = s0; base < s1; base += DS_TILE) {
        const int n = (int)min((int64_t)DS_TILE, s1 - base);
        __syncthreads();
        for (int i = threadIdx.x; i < 3 * n; i += DS_THREADS) {
            sxyz[i] = src[3 * base + i];
            if (DIP) sd[i] = dip[3 * base + i];
        }
        for (int i = threadIdx.x; i < n; i += DS_THREADS) sm[i] = q ? q[base + i] : 0.0;
        __syncthreads();
#pragma unroll 2
        for (int j = 0; j < n; ++j) {
            const double px = sxyz[3 * j], py = sxyz[3 * j + 1], pz = sxyz[3 * j + 2], m = sm[j];
            double ex = 0.0, ey = 0.0, ez = 0.0;
            if (DIP) { ex = sd[3 * j]; ey = sd[3 * j + 1]; ez = sd[3 * j + 2]; }
#pragma unroll
            for (int k = 0; k < DS_TPT; ++k) {
                const double dx = tx[k] - px, dy = ty[k] - py, dz = tz[k] - pz;
                const double r2 = fma(dx, dx, fma(dy, dy, dz * dz));
                const double inv = r2 > 0.0 ? rsqrt(r2) : 0.0;          // a source on the target adds nothing (x_i != y_j)
                if (DIP) {
                    const double dd = fma(ex, dx, fma(ey, dy, ez * dz));
                    acc[k] = fma(inv, fma(-dd, inv * inv, m), acc[k]);  // m/r - d.(x - y)/r^3
                } else {
                    acc[k] = fma(inv, m, acc[k]);
                }
            }
        }
    }
#pragma unroll
    for (int k = 0; k < DS_TPT; ++k) {
        const int64_t t = tfirst + (int64_t)k * DS_THREADS;
        if (t < nt) part[(int64_t)blockIdx.y * nt + t] = acc[k];
    }
}

// y[t] = (1/4 pi) sum of the chunks in chunk order: the same bits on every call
__global__ void ds_combine_kernel(const double *__restrict__ part, int nsplit, int64_t nt, double *__restrict__ y)
{
    const int64_t t = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (t >= nt) return;
    double s = 0.0;
    for (int k = 0; k < nsplit; ++k) s += part[(int64_t)k * nt + t];
    y[t] = s * 0.07957747154594767;     // 1 / (4 pi)
}

// must be a device (or managed) pointer of device `dev`; host memory would need a staging buffer, i.e. an allocation
void require_device_ptr(const void *p, const char *name, int dev)
{
    cudaPointerAttributes a;
    const cudaError_t e = cudaPointerGetAttributes(&a, p);
    if (e != cudaSuccess) { cudaGetLastError(); throw bem::Error(BEM_ERR_INVALID_ARG, std::string("bem_direct_sum_static: cannot classify pointer ") + name); }
    if (a.type != cudaMemoryTypeDevice && a.type != cudaMemoryTypeManaged)
        throw bem::Error(BEM_ERR_INVALID_ARG, std::string("bem_direct_sum_static: ") + name +
                                              " is not device memory (this entry copies nothing: staging a host array would need an allocation)");
    if (a.type == cudaMemoryTypeDevice && a.device != dev)
        throw bem::Error(BEM_ERR_INVALID_ARG, std::string("bem_direct_sum_static: ") + name +
                                              " lives on another device than the current one (cudaSetDevice to the owner of the buffers first)");
}

// set-up, once per device, with that device current: the device address of the scratch array
double *scratch_of_current_device(int dev)
{
    std::lock_guard<std::mutex> lock(g_ds_mutex);
    if (!g_ds_ptr[dev]) {
        double *p = nullptr;
        CUDA_TRY(cudaGetSymbolAddress((void **)&p, g_ds_partials));
        if (!p) throw bem::Error(BEM_ERR_CUDA, "bem_direct_sum_static: cudaGetSymbolAddress returned a null address");
        g_ds_ptr[dev] = p;
    }
    return g_ds_ptr[dev];
}

}  // namespace

extern "C" bem_status bem_direct_sum_static(const double *sources, int64_t n_sources, const double *q, const double *d,
                                            const double *targets, int64_t n_targets, double *y, void *cuda_stream)
{
    try {
        if (n_targets < 0 || n_sources < 0) throw bem::Error(BEM_ERR_INVALID_ARG, "bem_direct_sum_static: negative size");
        if (n_targets > DS_MAX_TARGETS) {
            char buf[256];
            snprintf(buf, sizeof buf, "bem_direct_sum_static: n_targets = %lld exceeds BEM_DIRECT_STATIC_MAX_TARGETS = %lld, the size the "
                                      "built-in scratch was compiled for (split the targets into several calls, or use bem_create_points)",
                     (long long)n_targets, (long long)DS_MAX_TARGETS);
            throw bem::Error(BEM_ERR_INVALID_ARG, buf);
        }
        if (n_sources > (int64_t)0x7fffffff) throw bem::Error(BEM_ERR_INVALID_ARG, "bem_direct_sum_static: n_sources exceeds 2^31 - 1");
        if (n_targets == 0) return BEM_OK;
        if (!targets || !y) throw bem::Error(BEM_ERR_INVALID_ARG, "bem_direct_sum_static: targets and y must not be NULL");
        if (n_sources > 0 && !sources) throw bem::Error(BEM_ERR_INVALID_ARG, "bem_direct_sum_static: sources is NULL");
        int dev = 0;
        CUDA_TRY(cudaGetDevice(&dev));
        if (dev < 0 || dev >= DS_MAX_DEVICES) throw bem::Error(BEM_ERR_INVALID_ARG, "bem_direct_sum_static: device index out of range");
        require_device_ptr(targets, "targets", dev);
        require_device_ptr(y, "y", dev);
        if (n_sources > 0) require_device_ptr(sources, "sources", dev);
        if (q && n_sources > 0) require_device_ptr(q, "q", dev);
        if (d && n_sources > 0) require_device_ptr(d, "d", dev);
        cudaStream_t s = (cudaStream_t)cuda_stream;
        if (n_sources == 0 || (!q && !d)) {                    // no source carries a strength
            CUDA_TRY(cudaMemsetAsync(y, 0, (size_t)n_targets * sizeof(double), s));
            return BEM_OK;
        }
        double *part = scratch_of_current_device(dev);         // first call on this device: the set-up
        const int tblocks = bem::cdiv(n_targets, DS_TPT * DS_THREADS);
        int nsplit = bem::cdiv(2 * 148, tblocks);
        nsplit = std::min(nsplit, bem::cdiv(n_sources, DS_TILE));
        nsplit = std::max(1, std::min(nsplit, DS_MAX_SPLIT));
        const int64_t chunk = (n_sources + nsplit - 1) / nsplit;
        const dim3 grid(tblocks, nsplit);
        // every slot (split < nsplit, target < n_targets) is overwritten below before the combine kernel reads it: what an
        // earlier call left in the array is never seen, and nothing has to be cleared
        if (d) ds_partial_kernel<true><<<grid, DS_THREADS, 0, s>>>(targets, n_targets, sources, q, d, n_sources, chunk, part);
        else ds_partial_kernel<false><<<grid, DS_THREADS, 0, s>>>(targets, n_targets, sources, q, nullptr, n_sources, chunk, part);
        KERNEL_CHECK();
        ds_combine_kernel<<<bem::cdiv(n_targets, 256), 256, 0, s>>>(part, nsplit, n_targets, y);
        KERNEL_CHECK();
        return BEM_OK;
    } catch (const bem::Error &e) {
        g_ds_error = e.what();
        return e.status;
    } catch (const std::exception &e) {
        g_ds_error = e.what();
        return BEM_ERR_CUDA;
    } catch (...) {
        g_ds_error = "bem_direct_sum_static: unknown error";
        return BEM_ERR_CUDA;
    }
}

extern "C" const char *bem_direct_sum_static_last_error(void) { return g_ds_error.c_str(); }
