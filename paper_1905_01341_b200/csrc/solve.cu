// Step a13: bem_solve = unpreconditioned GMRES around bem_apply
// (section 3.8: "unpreconditioned GMRES"; Eqs. 15-16,
// PAPER.md:160-171:  L q = b,  b = -1/2 phi + M phi  with the diagonal rule of
// PAPER.md:204 folded into c_i, reading R6).
// Vector work runs on the device with fixed-order reductions.  Orthogonalisation is
// classical Gram-Schmidt applied twice (CGS2, as stable as modified Gram-Schmidt): all
// k+1 inner products of a pass come from ONE batched kernel and one host read, and the
// update w -= V h is one kernel -- the k-th iteration costs 2 syncs instead of k+1.  The
// (k+1) x k Hessenberg least-squares problem is updated on the host with Givens rotations.
#include "common.cuh"

#include <cmath>

namespace bem {
void apply_device(bem_ctx *c, const double *q, const double *phi, double *y);
bool is_device_ptr(const void *p);

constexpr int DOT_BLOCKS = 592, DOT_THREADS = 256;

__global__ void __launch_bounds__(DOT_THREADS)
dot_partial(const double *__restrict__ a, const double *__restrict__ b, int64_t n, double *__restrict__ part)
{
    double s = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) s = fma(a[i], b[i], s);
    __shared__ double sm[DOT_THREADS];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int st = DOT_THREADS / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st) sm[threadIdx.x] += sm[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[blockIdx.x] = sm[0];
}
__global__ void __launch_bounds__(DOT_THREADS)
dot_final(const double *__restrict__ part, int nparts, double *__restrict__ out)
{
    __shared__ double sm[DOT_THREADS];
    double s = 0.0;
    for (int i = threadIdx.x; i < nparts; i += DOT_THREADS) s += part[i];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int st = DOT_THREADS / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st) sm[threadIdx.x] += sm[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) *out = sm[0];
}
// y += a x
__global__ void axpy_kernel(double a, const double *__restrict__ x, double *__restrict__ y, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) y[i] = fma(a, x[i], y[i]);
}
// y = a x
__global__ void scale_kernel(double a, const double *__restrict__ x, double *__restrict__ y, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) y[i] = a * x[i];
}
// b = -c .* phi - y     (y = bem_apply(0, phi) = -D phi)
__global__ void rhs_kernel(const double *__restrict__ cf, const double *__restrict__ phi, const double *__restrict__ y,
                           double *__restrict__ b, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) b[i] = -cf[i] * phi[i] - y[i];
}
// y = x ./ d ;  y += x ./ d
__global__ void divide_kernel(const double *__restrict__ x, const double *__restrict__ d, double *__restrict__ y, int64_t n, int accumulate)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) y[i] = accumulate ? y[i] + x[i] / d[i] : x[i] / d[i];
}
// r = b - w
__global__ void sub_kernel(const double *__restrict__ b, const double *__restrict__ w, double *__restrict__ r, int64_t n)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) r[i] = b[i] - w[i];
}

// part[j * gridDim.x + bx] = partial <w, V_j> of block bx  (grid = (MD_BLOCKS, nvec))
constexpr int MD_BLOCKS = 148;
__global__ void __launch_bounds__(DOT_THREADS)
multi_dot_partial(const double *__restrict__ w, const double *__restrict__ V, int64_t n, double *__restrict__ part)
{
    const double *v = V + (size_t)blockIdx.y * n;
    double s = 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (int64_t)gridDim.x * blockDim.x) s = fma(w[i], v[i], s);
    __shared__ double sm[DOT_THREADS];
    sm[threadIdx.x] = s;
    __syncthreads();
    for (int st = DOT_THREADS / 2; st > 0; st >>= 1) {
        if (threadIdx.x < st) sm[threadIdx.x] += sm[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) part[(size_t)blockIdx.y * gridDim.x + blockIdx.x] = sm[0];
}
// out[j] = sum_bx part[j][bx]   (one block of 32 threads per j; fixed order)
__global__ void multi_dot_final(const double *__restrict__ part, int nparts, double *__restrict__ out)
{
    double s = 0.0;
    for (int i = threadIdx.x; i < nparts; i += 32) s += part[(size_t)blockIdx.x * nparts + i];
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_xor_sync(0xffffffffu, s, d);
    if (threadIdx.x == 0) out[blockIdx.x] = s;
}
// w -= sum_j h[j] V_j
__global__ void multi_axpy(const double *__restrict__ h, const double *__restrict__ V, int nvec, int64_t n, double *__restrict__ w)
{
    const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    double acc = w[i];
    for (int j = 0; j < nvec; ++j) acc = fma(-__ldg(h + j), V[(size_t)j * n + i], acc);
    w[i] = acc;
}

struct Krylov {
    bem_ctx *c;
    int64_t n;
    dvec<double> part, out, mpart, mout;
    // h[0..nvec) = V^T w, then w -= V h
    void project_out(const double *V, int nvec, double *w, double *h_host)
    {
        if ((size_t)nvec * MD_BLOCKS > mpart.n) { mpart.alloc((size_t)2 * nvec * MD_BLOCKS); mout.alloc((size_t)2 * nvec); }
        multi_dot_partial<<<dim3(MD_BLOCKS, nvec), DOT_THREADS, 0, c->stream>>>(w, V, n, mpart.get());
        KERNEL_CHECK();
        multi_dot_final<<<nvec, 32, 0, c->stream>>>(mpart.get(), MD_BLOCKS, mout.get());
        KERNEL_CHECK();
        multi_axpy<<<cdiv(n, 256), 256, 0, c->stream>>>(mout.get(), V, nvec, n, w);
        KERNEL_CHECK();
        CUDA_TRY(cudaMemcpyAsync(h_host, mout.get(), nvec * sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
    }
    double dot(const double *a, const double *b)
    {
        dot_partial<<<DOT_BLOCKS, DOT_THREADS, 0, c->stream>>>(a, b, n, part.get());
        KERNEL_CHECK();
        dot_final<<<1, DOT_THREADS, 0, c->stream>>>(part.get(), DOT_BLOCKS, out.get());
        KERNEL_CHECK();
        double h;
        CUDA_TRY(cudaMemcpyAsync(&h, out.get(), sizeof(double), cudaMemcpyDeviceToHost, c->stream));
        CUDA_TRY(cudaStreamSynchronize(c->stream));
        return h;
    }
    void axpy(double a, const double *x, double *y) { axpy_kernel<<<cdiv(n, 256), 256, 0, c->stream>>>(a, x, y, n); KERNEL_CHECK(); }
    void scale(double a, const double *x, double *y) { scale_kernel<<<cdiv(n, 256), 256, 0, c->stream>>>(a, x, y, n); KERNEL_CHECK(); }
};

bem_status solve_impl(bem_ctx *c, const double *phi_in, double *q_io, int use_x0, double tol, int max_iter,
                      int *iters_out, double *relres_out)
{
    cudaStream_t s = c->stream;
    const int64_t n = c->N;
    const size_t bytes = n * sizeof(double);
    dvec<double> phi, x, b, w, r;
    phi.alloc(n); x.alloc(n); b.alloc(n); w.alloc(n); r.alloc(n);
    CUDA_TRY(cudaMemcpyAsync(phi.get(), phi_in, bytes, cudaMemcpyDefault, s));
    if (use_x0) CUDA_TRY(cudaMemcpyAsync(x.get(), q_io, bytes, cudaMemcpyDefault, s));
    else x.zero(s);
    Krylov K{c, n};
    K.part.alloc(DOT_BLOCKS);
    K.out.alloc(1);

    struct TimingOff {                                           // the products of the solve are not timed; restored on every exit
        bem_ctx *c; int saved;
        explicit TimingOff(bem_ctx *cc) : c(cc), saved(cc->timing) { c->timing = 0; }
        ~TimingOff() { c->timing = saved; }
    } timing_off(c);
    // right-hand side (Eq. 16): b = -c phi + D phi
    apply_device(c, nullptr, phi.get(), w.get());
    rhs_kernel<<<cdiv(n, 256), 256, 0, s>>>(c->cfree.get(), phi.get(), w.get(), b.get(), n);
    KERNEL_CHECK();
    const double bnorm = std::sqrt(K.dot(b.get(), b.get()));
    int iters = 0;
    double relres = 0.0;
    bool converged = false;
    if (bnorm == 0.0) {
        x.zero(s);
        converged = true;
    } else {
        const int m = c->gmres_restart > 0 ? std::min(c->gmres_restart, std::max(max_iter, 1)) : std::max(max_iter, 1);
        // Krylov basis: grown by doubling (64 vectors first) instead of (max_iter + 1) vectors up front -- config 5 with
        // max_iter = 400 would reserve 8.2 GB for the 148-222 vectors it ends up using
        dvec<double> basis;
        int cap = std::min(m + 1, 64);
        basis.alloc((size_t)cap * n);
        auto grow = [&](int need) {
            if (need <= cap) return;
            int ncap = cap;
            while (ncap < need) ncap = std::min(m + 1, 2 * ncap);
            dvec<double> nb;
            nb.alloc((size_t)ncap * n);
            CUDA_TRY(cudaMemcpyAsync(nb.get(), basis.get(), (size_t)cap * n * sizeof(double), cudaMemcpyDeviceToDevice, s));
            CUDA_TRY(cudaStreamSynchronize(s));
            basis = std::move(nb);
            cap = ncap;
        };
        std::vector<double> H((size_t)(m + 1) * m, 0.0), cs(m), sn(m), g(m + 1), yv(m), hh(2 * (m + 1));
        auto Vk = [&](int k) { return basis.get() + (size_t)k * n; };
        bool x_is_zero = !use_x0;
        const double *dpre = nullptr;                       // option "precond": D = diag(S)
        if (c->precond == 1) dpre = c->have_diag ? c->diagL.get() : (c->diagS.p ? c->diagS.get() : nullptr);
        while (true) {
            if (x_is_zero) CUDA_TRY(cudaMemcpyAsync(r.get(), b.get(), bytes, cudaMemcpyDeviceToDevice, s));
            else {
                apply_device(c, x.get(), nullptr, w.get());
                sub_kernel<<<cdiv(n, 256), 256, 0, s>>>(b.get(), w.get(), r.get(), n);
                KERNEL_CHECK();
            }
            const double beta = std::sqrt(K.dot(r.get(), r.get()));
            relres = beta / bnorm;
            if (relres <= tol) { converged = true; break; }
            if (iters >= max_iter) break;
            K.scale(1.0 / beta, r.get(), Vk(0));
            std::fill(g.begin(), g.end(), 0.0);
            g[0] = beta;
            int k = 0;
            for (; k < m && iters < max_iter; ++k) {
                if (dpre) {                                 // right preconditioning: w = S (D^-1 v_k)
                    divide_kernel<<<cdiv(n, 256), 256, 0, s>>>(Vk(k), dpre, r.get(), n, 0);
                    KERNEL_CHECK();
                    apply_device(c, r.get(), nullptr, w.get());
                } else apply_device(c, Vk(k), nullptr, w.get());
                K.project_out(basis.get(), k + 1, w.get(), hh.data());          // CGS2: two passes of classical Gram-Schmidt
                K.project_out(basis.get(), k + 1, w.get(), hh.data() + (m + 1));
                for (int i = 0; i <= k; ++i) H[(size_t)i * m + k] = hh[i] + hh[m + 1 + i];
                const double hn = std::sqrt(K.dot(w.get(), w.get()));
                H[(size_t)(k + 1) * m + k] = hn;
                grow(k + 2);
                if (hn > 0.0) K.scale(1.0 / hn, w.get(), Vk(k + 1));
                for (int i = 0; i < k; ++i) {              // previous rotations
                    const double t = cs[i] * H[(size_t)i * m + k] + sn[i] * H[(size_t)(i + 1) * m + k];
                    H[(size_t)(i + 1) * m + k] = -sn[i] * H[(size_t)i * m + k] + cs[i] * H[(size_t)(i + 1) * m + k];
                    H[(size_t)i * m + k] = t;
                }
                const double a = H[(size_t)k * m + k], bb = H[(size_t)(k + 1) * m + k];
                const double d = std::hypot(a, bb);
                cs[k] = d > 0 ? a / d : 1.0;
                sn[k] = d > 0 ? bb / d : 0.0;
                H[(size_t)k * m + k] = d;
                H[(size_t)(k + 1) * m + k] = 0.0;
                g[k + 1] = -sn[k] * g[k];
                g[k] = cs[k] * g[k];
                ++iters;
                relres = std::fabs(g[k + 1]) / bnorm;
                if (relres <= tol || hn == 0.0) { ++k; break; }
            }
            // x += V y,  H(0:k,0:k) y = g(0:k)
            for (int i = k - 1; i >= 0; --i) {
                double t = g[i];
                for (int j = i + 1; j < k; ++j) t -= H[(size_t)i * m + j] * yv[j];
                yv[i] = t / H[(size_t)i * m + i];
            }
            if (dpre) {                                     // x += D^-1 (V y)
                r.zero(s);
                for (int i = 0; i < k; ++i) K.axpy(yv[i], Vk(i), r.get());
                divide_kernel<<<cdiv(n, 256), 256, 0, s>>>(r.get(), dpre, x.get(), n, 1);
                KERNEL_CHECK();
            } else
                for (int i = 0; i < k; ++i) K.axpy(yv[i], Vk(i), x.get());
            x_is_zero = false;
            if (relres <= tol || iters >= max_iter) {
                // true residual of the returned iterate (one more product, as Matlab's gmres does)
                apply_device(c, x.get(), nullptr, w.get());
                sub_kernel<<<cdiv(n, 256), 256, 0, s>>>(b.get(), w.get(), r.get(), n);
                KERNEL_CHECK();
                relres = std::sqrt(K.dot(r.get(), r.get())) / bnorm;
                converged = relres <= tol * (1.0 + 1e-6) || relres <= tol;
                if (converged || iters >= max_iter) break;
            }
        }
    }
    CUDA_TRY(cudaMemcpyAsync(q_io, x.get(), bytes, cudaMemcpyDefault, s));
    CUDA_TRY(cudaStreamSynchronize(s));
    if (iters_out) *iters_out = iters;
    if (relres_out) *relres_out = relres;
    return converged ? BEM_OK : BEM_ERR_NOT_CONVERGED;
}

}  // namespace bem

extern "C" bem_status bem_solve(bem_ctx *c, const double *phi, double *q, int use_q_as_x0, double tol, int max_iter,
                                int *iters_out, double *relres_out)
{
    if (!c || !phi || !q || !(tol > 0.0) || max_iter < 0) return BEM_ERR_INVALID_ARG;
    if (c->quadrature >= 2) { c->err = "bem_solve: not available for a point cloud or an evaluator"; return BEM_ERR_INVALID_ARG; }
    if (!c->ready || !c->have_cfree) { c->err = "bem_solve before bem_setup"; return BEM_ERR_NOT_SETUP; }
    try {
        cudaSetDevice(c->device);
        return bem::solve_impl(c, phi, q, use_q_as_x0, tol, max_iter, iters_out, relres_out);
    } catch (const bem::Error &e) {
        c->err = e.what();
        cudaGetLastError();
        return e.status;
    } catch (const std::bad_alloc &) {
        c->err = "bem_solve: out of host memory (Hessenberg of max_iter^2 entries: set option gmres_restart)";
        return BEM_ERR_OOM;
    } catch (const std::exception &e) {
        c->err = e.what();
        return BEM_ERR_CUDA;
    } catch (...) {
        c->err = "unknown error";
        return BEM_ERR_CUDA;
    }
}
