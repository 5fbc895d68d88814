// vec_kernels.cu — a8: the Davidson vector kernels ("Lánczos or
// Davidson": the Rayleigh–Ritz dots, the Ritz vector / residual combination, the diagonal
// preconditioner and Gram–Schmidt all run over ψ-sized FP64 vectors).
//
// All kernels run over the flat padded arena of a ψ layout (n doubles, n a multiple of 16, padding
// zero and preserved by every linear operation).  They are HBM-bound: 16-byte loads, grid-stride
// loops over a grid sized to the SM count, and — for the reductions — a two-stage, fixed-order
// scheme (per-thread strided sums → warp shuffle tree → per-CTA partial in scratch → one CTA sums
// the partials in index order), so results are bit-reproducible run to run.  No atomics.
#include "internal.h"

#include <mutex>

namespace dmrgk {

constexpr int VEC_THREADS = 256;
constexpr int VEC_MAX_BLOCKS = 1184;   // 148 SMs × 8 resident CTAs; fixed, so sums do not depend on the device

static inline int vec_grid(int64_t n2) {
    int64_t g = (n2 + VEC_THREADS - 1) / VEC_THREADS;
    if (g < 1) g = 1;
    if (g > VEC_MAX_BLOCKS) g = VEC_MAX_BLOCKS;
    return int(g);
}

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

// CTA-wide fixed-order sum of NV values per thread; result valid in thread 0.
template <int NV>
__device__ __forceinline__ void block_sum(double (&acc)[NV], double* sh /*[NV][8]*/) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int j = 0; j < NV; ++j) {
        acc[j] = warp_sum(acc[j]);
        if (lane == 0) sh[j * 8 + warp] = acc[j];
    }
    __syncthreads();
    if (threadIdx.x == 0) {
#pragma unroll
        for (int j = 0; j < NV; ++j) {
            double s = 0.0;
#pragma unroll
            for (int w = 0; w < VEC_THREADS / 32; ++w) s += sh[j * 8 + w];
            acc[j] = s;
        }
    }
}

// stage 1 of out[j] = Σ_i X[j·stride + i]·y[i]:  partial[block][j0 + j]
template <int NV>
__global__ void __launch_bounds__(VEC_THREADS)
multi_dot_stage1(int64_t n2, int nv, int j0, const double2* __restrict__ X, int64_t stride2,
                 const double2* __restrict__ y, double* __restrict__ partial, int nv_total) {
    __shared__ double sh[NV * 8];
    double acc[NV];
#pragma unroll
    for (int j = 0; j < NV; ++j) acc[j] = 0.0;
    for (int64_t i = int64_t(blockIdx.x) * VEC_THREADS + threadIdx.x; i < n2;
         i += int64_t(gridDim.x) * VEC_THREADS) {
        const double2 b = y[i];
#pragma unroll
        for (int j = 0; j < NV; ++j)
            if (j < nv) {
                const double2 a = __ldg(X + int64_t(j0 + j) * stride2 + i);
                acc[j] = fma(a.x, b.x, acc[j]);
                acc[j] = fma(a.y, b.y, acc[j]);
            }
    }
    block_sum<NV>(acc, sh);
    if (threadIdx.x == 0)
#pragma unroll
        for (int j = 0; j < NV; ++j)
            if (j < nv) partial[int64_t(blockIdx.x) * nv_total + j0 + j] = acc[j];
}

// stage 2: out[j] = Σ_b partial[b][j], b ascending per lane then a shuffle tree; one warp per j.
__global__ void __launch_bounds__(VEC_THREADS)
multi_dot_stage2(int nblocks, int nv, const double* __restrict__ partial, double* __restrict__ out) {
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    for (int j = warp; j < nv; j += VEC_THREADS / 32) {
        double s = 0.0;
        for (int b = lane; b < nblocks; b += 32) s += partial[int64_t(b) * nv + j];
        s = warp_sum(s);
        if (lane == 0) out[j] = s;
    }
}

// y = beta·y + alpha·Σ_j coef[j]·X_j   (beta = 0: y is not read)
__global__ void __launch_bounds__(VEC_THREADS)
multi_axpy_kernel(int64_t n2, int nv, const double2* __restrict__ X, int64_t stride2,
                  const double* __restrict__ coef, double alpha, double beta, double2* __restrict__ y) {
    __shared__ double c[64];
    for (int j = threadIdx.x; j < nv; j += VEC_THREADS) c[j] = alpha * coef[j];
    __syncthreads();
    for (int64_t i = int64_t(blockIdx.x) * VEC_THREADS + threadIdx.x; i < n2;
         i += int64_t(gridDim.x) * VEC_THREADS) {
        double2 s = make_double2(0.0, 0.0);
        if (beta != 0.0) {
            const double2 o = y[i];
            s.x = beta * o.x;
            s.y = beta * o.y;
        }
#pragma unroll 4
        for (int j = 0; j < nv; ++j) {
            const double2 a = __ldg(X + int64_t(j) * stride2 + i);
            s.x = fma(c[j], a.x, s.x);
            s.y = fma(c[j], a.y, s.y);
        }
        y[i] = s;
    }
}

__global__ void __launch_bounds__(VEC_THREADS)
axpby_kernel(int64_t n2, double alpha, const double2* __restrict__ x, double beta, double2* __restrict__ y) {
    for (int64_t i = int64_t(blockIdx.x) * VEC_THREADS + threadIdx.x; i < n2;
         i += int64_t(gridDim.x) * VEC_THREADS) {
        const double2 a = x[i];
        double2 s = make_double2(alpha * a.x, alpha * a.y);
        if (beta != 0.0) {
            const double2 o = y[i];
            s.x = fma(beta, o.x, s.x);
            s.y = fma(beta, o.y, s.y);
        }
        y[i] = s;
    }
}

// x = alpha·x in place (one pointer: the two-pointer kernels above promise __restrict__)
__global__ void __launch_bounds__(VEC_THREADS)
scal_kernel(int64_t n2, double alpha, double2* x) {
    for (int64_t i = int64_t(blockIdx.x) * VEC_THREADS + threadIdx.x; i < n2;
         i += int64_t(gridDim.x) * VEC_THREADS) {
        double2 v = x[i];
        v.x *= alpha;
        v.y *= alpha;
        x[i] = v;
    }
}

__global__ void __launch_bounds__(VEC_THREADS)
scal_dev_kernel(int64_t n2, const double* __restrict__ alpha_dev, int inv, int sqrt_first,
                const double2* x, double2* y) {      // y may alias x (in-place normalisation): no __restrict__
    double a = *alpha_dev;
    if (sqrt_first) a = sqrt(a);
    const double f = inv ? (a != 0.0 ? 1.0 / a : 0.0) : a;   // 1/0 → 0: a vanished vector stays a zero vector, never Inf/NaN
    for (int64_t i = int64_t(blockIdx.x) * VEC_THREADS + threadIdx.x; i < n2;
         i += int64_t(gridDim.x) * VEC_THREADS) {
        double2 v = x[i];
        v.x *= f;
        v.y *= f;
        y[i] = v;
    }
}

// r = Σ_j y_j (W_j − θ V_j); partial[block] = Σ r²   (y = coef[0..m), θ = coef[m])
__global__ void __launch_bounds__(VEC_THREADS)
residual_stage1(int64_t n2, int m, const double2* __restrict__ V, const double2* __restrict__ W,
                int64_t stride2, const double* __restrict__ coef, double2* __restrict__ r,
                double* __restrict__ partial) {
    __shared__ double c[64];
    __shared__ double sh[8];
    for (int j = threadIdx.x; j <= m; j += VEC_THREADS) c[j] = coef[j];
    __syncthreads();
    const double theta = c[m];
    double acc[1] = {0.0};
    for (int64_t i = int64_t(blockIdx.x) * VEC_THREADS + threadIdx.x; i < n2;
         i += int64_t(gridDim.x) * VEC_THREADS) {
        double2 wy = make_double2(0.0, 0.0), vy = make_double2(0.0, 0.0);
#pragma unroll 4
        for (int j = 0; j < m; ++j) {
            const double2 w = __ldg(W + int64_t(j) * stride2 + i);
            const double2 v = __ldg(V + int64_t(j) * stride2 + i);
            wy.x = fma(c[j], w.x, wy.x);
            wy.y = fma(c[j], w.y, wy.y);
            vy.x = fma(c[j], v.x, vy.x);
            vy.y = fma(c[j], v.y, vy.y);
        }
        double2 rr;
        rr.x = wy.x - theta * vy.x;
        rr.y = wy.y - theta * vy.y;
        r[i] = rr;
        acc[0] = fma(rr.x, rr.x, acc[0]);
        acc[0] = fma(rr.y, rr.y, acc[0]);
    }
    block_sum<1>(acc, sh);
    if (threadIdx.x == 0) partial[blockIdx.x] = acc[0];
}

// t = r / (θ − d), |θ − d| < 1e-10 → ±1e-10 (sign of the denominator, +0 → +)
__global__ void __launch_bounds__(VEC_THREADS)
precond_kernel(int64_t n, const double* __restrict__ r, const double* __restrict__ d,
               const double* __restrict__ theta_dev, double* __restrict__ t) {
    const double theta = *theta_dev;
    for (int64_t i = int64_t(blockIdx.x) * VEC_THREADS + threadIdx.x; i < n;
         i += int64_t(gridDim.x) * VEC_THREADS) {
        double den = theta - d[i];
        if (fabs(den) < 1e-10) den = (den < 0.0) ? -1e-10 : 1e-10;
        t[i] = r[i] / den;
    }
}

static int32_t check_vec(const char* who, dmrgk_ctx* ctx, int64_t n) {
    if (!ctx) return fail(DMRGK_EINVAL, "%s: ctx is NULL", who);
    if (n < 0 || (n & 15)) return fail(DMRGK_EINVAL, "%s: n = %lld must be a non-negative multiple of 16", who, (long long)n);
    return DMRGK_OK;
}

template <int NV>
static void launch_dot1(int grid, cudaStream_t st, int64_t n2, int nv, int j0, const double* X, int64_t stride,
                        const double* y, double* partial, int nv_total) {
    multi_dot_stage1<NV><<<grid, VEC_THREADS, 0, st>>>(n2, nv, j0, reinterpret_cast<const double2*>(X), stride / 2,
                                                       reinterpret_cast<const double2*>(y), partial, nv_total);
    count_launch();
}

}  // namespace dmrgk

using namespace dmrgk;

extern "C" {

int64_t dmrgk_vec_scratch_bytes(int32_t nv) {
    if (nv < 1) nv = 1;
    return round_up(int64_t(VEC_MAX_BLOCKS) * nv * 8, 128);
}

int32_t dmrgk_vec_multi_dot(dmrgk_ctx* ctx, int64_t n, int32_t nv, const double* X_dev, int64_t stride,
                            const double* y_dev, double* out_dev, void* scratch_dev, void* stream) {
    DMRGK_TRY(check_vec("vec_multi_dot", ctx, n));
    if (nv < 0) return fail(DMRGK_EINVAL, "vec_multi_dot: nv < 0");
    if (nv == 0) return DMRGK_OK;
    if (!X_dev || !y_dev || !out_dev || !scratch_dev) return fail(DMRGK_EINVAL, "vec_multi_dot: NULL pointer");
    if (stride & 1) return fail(DMRGK_EINVAL, "vec_multi_dot: stride must be even");
    if (!aligned128(X_dev) || !aligned128(y_dev) || (stride & 15))
        return fail(DMRGK_EALIGN, "vec_multi_dot: vectors must be 128-byte aligned (stride a multiple of 16)");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n2 = n / 2;
    const int grid = vec_grid(n2);
    double* partial = static_cast<double*>(scratch_dev);
    for (int j0 = 0; j0 < nv; j0 += 8) {
        const int c = std::min(8, nv - j0);
        if (c == 1) launch_dot1<1>(grid, st, n2, c, j0, X_dev, stride, y_dev, partial, nv);
        else if (c <= 4) launch_dot1<4>(grid, st, n2, c, j0, X_dev, stride, y_dev, partial, nv);
        else launch_dot1<8>(grid, st, n2, c, j0, X_dev, stride, y_dev, partial, nv);
        DMRGK_CUDA(cudaGetLastError());
    }
    multi_dot_stage2<<<1, VEC_THREADS, 0, st>>>(grid, nv, partial, out_dev);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

// ---- dmrgk_vec_multi_dot_noalloc: the same dots for callers that have no device memory to give ----
// dmrgk_vec_multi_dot needs a caller-allocated scratch buffer for its per-CTA partial sums.  Some users
// of this library cannot supply one: a sweep driver that has already handed the whole of HBM to the
// operator arenas and the staging ring (config 5 is sized to do exactly that), a C or Fortran host
// code that is given a fixed set of device buffers by its framework and owns no allocator, or a step
// running next to the side-stream operator copies, where a cudaMalloc / cudaFree would synchronise the
// device and stall that overlap.  For them the partial sums live in the array below, which is part
// of the library image: every GPU that loads libdmrgk.so holds these 592 KiB until the process exits.
//
//   * limit: nv ≤ DMRGK_NOALLOC_MAX_NV (64); n is not limited (the grid is capped at VEC_MAX_BLOCKS).
//   * nothing has to start at zero: stage 2 reads partial[b][j] only for b < grid, j < nv, and stage 1
//     of the same call has written every one of those, so the previous call's contents are never read.
//   * there is ONE array per GPU, shared by every call from every thread and stream: two calls whose
//     kernels can overlap on the GPU (different streams, no ordering between them) race on it.
//   * `vec_noalloc_partials` as written in HOST code is only the host-side stand-in of the symbol, not a
//     device address; the kernels get the address cudaGetSymbolAddress returns, fetched once per device
//     with that device current, by the first call on that device.  That first call therefore does a
//     little set-up work (it may load the module) and should be made before any stream capture begins.
constexpr int DMRGK_NOALLOC_MAX_NV = 64;
constexpr int DMRGK_NOALLOC_MAX_DEVICES = 64;
static __device__ __align__(256) double vec_noalloc_partials[size_t(VEC_MAX_BLOCKS) * DMRGK_NOALLOC_MAX_NV];

static std::mutex g_noalloc_mu;
static double* g_noalloc_ptr[DMRGK_NOALLOC_MAX_DEVICES] = {};   // device address of the array, per device

// Device address of vec_noalloc_partials on `device` (which must be current).  No allocation.
static int32_t noalloc_partials(int device, double** out) {
    std::lock_guard<std::mutex> lk(g_noalloc_mu);
    if (!g_noalloc_ptr[device]) {
        double* p = nullptr;
        DMRGK_CUDA(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), vec_noalloc_partials));
        if (!p) return fail(DMRGK_ECUDA, "vec_multi_dot_noalloc: cudaGetSymbolAddress returned NULL");
        g_noalloc_ptr[device] = p;
    }
    *out = g_noalloc_ptr[device];
    return DMRGK_OK;
}

int32_t dmrgk_vec_multi_dot_noalloc(dmrgk_ctx* ctx, int64_t n, int32_t nv, const double* X_dev, int64_t stride,
                                    const double* y_dev, double* out_dev, void* stream) {
    DMRGK_TRY(check_vec("vec_multi_dot_noalloc", ctx, n));
    if (nv < 0) return fail(DMRGK_EINVAL, "vec_multi_dot_noalloc: nv < 0");
    if (nv > DMRGK_NOALLOC_MAX_NV)
        return fail(DMRGK_EINVAL, "vec_multi_dot_noalloc: nv = %d exceeds the built-in scratch (at most %d vectors per "
                                  "call; use dmrgk_vec_multi_dot with your own scratch, or split the call)",
                    nv, DMRGK_NOALLOC_MAX_NV);
    if (ctx->device < 0 || ctx->device >= DMRGK_NOALLOC_MAX_DEVICES)
        return fail(DMRGK_EINVAL, "vec_multi_dot_noalloc: device %d outside [0, %d)", ctx->device, DMRGK_NOALLOC_MAX_DEVICES);
    if (nv == 0) return DMRGK_OK;
    if (!X_dev || !y_dev || !out_dev) return fail(DMRGK_EINVAL, "vec_multi_dot_noalloc: NULL pointer");
    if (stride & 1) return fail(DMRGK_EINVAL, "vec_multi_dot_noalloc: stride must be even");
    if (!aligned128(X_dev) || !aligned128(y_dev) || (stride & 15))
        return fail(DMRGK_EALIGN, "vec_multi_dot_noalloc: vectors must be 128-byte aligned (stride a multiple of 16)");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    double* partial = nullptr;
    DMRGK_TRY(noalloc_partials(ctx->device, &partial));
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n2 = n / 2;
    const int grid = vec_grid(n2);
    for (int j0 = 0; j0 < nv; j0 += 8) {
        const int c = std::min(8, nv - j0);
        if (c == 1) launch_dot1<1>(grid, st, n2, c, j0, X_dev, stride, y_dev, partial, nv);
        else if (c <= 4) launch_dot1<4>(grid, st, n2, c, j0, X_dev, stride, y_dev, partial, nv);
        else launch_dot1<8>(grid, st, n2, c, j0, X_dev, stride, y_dev, partial, nv);
        DMRGK_CUDA(cudaGetLastError());
    }
    multi_dot_stage2<<<1, VEC_THREADS, 0, st>>>(grid, nv, partial, out_dev);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t dmrgk_vec_multi_axpy(dmrgk_ctx* ctx, int64_t n, int32_t nv, const double* X_dev, int64_t stride,
                             const double* coef_dev, double alpha, double beta, double* y_dev, void* stream) {
    DMRGK_TRY(check_vec("vec_multi_axpy", ctx, n));
    if (nv < 0 || nv > 64) return fail(DMRGK_EINVAL, "vec_multi_axpy: nv = %d outside [0, 64]", nv);
    if (n == 0) return DMRGK_OK;
    if (!y_dev || (nv && (!X_dev || !coef_dev))) return fail(DMRGK_EINVAL, "vec_multi_axpy: NULL pointer");
    if ((nv && !aligned128(X_dev)) || !aligned128(y_dev) || (stride & 15))
        return fail(DMRGK_EALIGN, "vec_multi_axpy: vectors must be 128-byte aligned (stride a multiple of 16)");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    const int64_t n2 = n / 2;
    multi_axpy_kernel<<<vec_grid(n2), VEC_THREADS, 0, (cudaStream_t)stream>>>(
        n2, nv, reinterpret_cast<const double2*>(X_dev), stride / 2, coef_dev, alpha, beta,
        reinterpret_cast<double2*>(y_dev));
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t dmrgk_vec_axpby(dmrgk_ctx* ctx, int64_t n, double alpha, const double* x_dev, double beta,
                        double* y_dev, void* stream) {
    DMRGK_TRY(check_vec("vec_axpby", ctx, n));
    if (n == 0) return DMRGK_OK;
    if (!x_dev || !y_dev) return fail(DMRGK_EINVAL, "vec_axpby: NULL pointer");
    if (!aligned128(x_dev) || !aligned128(y_dev)) return fail(DMRGK_EALIGN, "vec_axpby: vectors must be 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    const int64_t n2 = n / 2;
    axpby_kernel<<<vec_grid(n2), VEC_THREADS, 0, (cudaStream_t)stream>>>(
        n2, alpha, reinterpret_cast<const double2*>(x_dev), beta, reinterpret_cast<double2*>(y_dev));
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t dmrgk_vec_scal_dev(dmrgk_ctx* ctx, int64_t n, const double* alpha_dev, int32_t mode,
                           const double* x_dev, double* y_dev, void* stream) {
    DMRGK_TRY(check_vec("vec_scal_dev", ctx, n));
    if (n == 0) return DMRGK_OK;
    if (!alpha_dev || !x_dev || !y_dev) return fail(DMRGK_EINVAL, "vec_scal_dev: NULL pointer");
    if (mode < 0 || mode > 3) return fail(DMRGK_EINVAL, "vec_scal_dev: mode must be 0..3");
    if (!aligned128(x_dev) || !aligned128(y_dev)) return fail(DMRGK_EALIGN, "vec_scal_dev: vectors must be 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    const int64_t n2 = n / 2;
    scal_dev_kernel<<<vec_grid(n2), VEC_THREADS, 0, (cudaStream_t)stream>>>(
        n2, alpha_dev, mode & 1, (mode >> 1) & 1, reinterpret_cast<const double2*>(x_dev),
        reinterpret_cast<double2*>(y_dev));
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t dmrgk_vec_residual(dmrgk_ctx* ctx, int64_t n, int32_t m, const double* V_dev, const double* W_dev,
                           int64_t stride, const double* coef_dev, double* r_dev, double* out_dev,
                           void* scratch_dev, void* stream) {
    DMRGK_TRY(check_vec("vec_residual", ctx, n));
    if (m < 1 || m > 63) return fail(DMRGK_EINVAL, "vec_residual: m = %d outside [1, 63]", m);
    if (!V_dev || !W_dev || !coef_dev || !r_dev || !out_dev || !scratch_dev)
        return fail(DMRGK_EINVAL, "vec_residual: NULL pointer");
    if (!aligned128(V_dev) || !aligned128(W_dev) || !aligned128(r_dev) || (stride & 15))
        return fail(DMRGK_EALIGN, "vec_residual: vectors must be 128-byte aligned (stride a multiple of 16)");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    cudaStream_t st = (cudaStream_t)stream;
    const int64_t n2 = n / 2;
    const int grid = vec_grid(n2);
    double* partial = static_cast<double*>(scratch_dev);
    residual_stage1<<<grid, VEC_THREADS, 0, st>>>(n2, m, reinterpret_cast<const double2*>(V_dev),
                                                  reinterpret_cast<const double2*>(W_dev), stride / 2, coef_dev,
                                                  reinterpret_cast<double2*>(r_dev), partial);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    multi_dot_stage2<<<1, VEC_THREADS, 0, st>>>(grid, 1, partial, out_dev);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t dmrgk_vec_precond(dmrgk_ctx* ctx, int64_t n, const double* r_dev, const double* diag_dev,
                          const double* theta_dev, double* t_dev, void* stream) {
    DMRGK_TRY(check_vec("vec_precond", ctx, n));
    if (n == 0) return DMRGK_OK;
    if (!r_dev || !diag_dev || !theta_dev || !t_dev) return fail(DMRGK_EINVAL, "vec_precond: NULL pointer");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    precond_kernel<<<vec_grid(n), VEC_THREADS, 0, (cudaStream_t)stream>>>(n, r_dev, diag_dev, theta_dev, t_dev);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

// ---- the BLAS-1 names of SURVEY §8(b) (dot, nrm2, axpy, scal), thin forms of the kernels above ----
__global__ void sqrt_inplace_kernel(double* x) { x[0] = sqrt(x[0]); }

int32_t dmrgk_vec_dot(dmrgk_ctx* ctx, int64_t n, const double* x_dev, const double* y_dev, double* out_dev,
                      void* scratch_dev, void* stream) {
    return dmrgk_vec_multi_dot(ctx, n, 1, x_dev, n, y_dev, out_dev, scratch_dev, stream);
}

int32_t dmrgk_vec_nrm2(dmrgk_ctx* ctx, int64_t n, const double* x_dev, double* out_dev, void* scratch_dev,
                       void* stream) {
    DMRGK_TRY(dmrgk_vec_multi_dot(ctx, n, 1, x_dev, n, x_dev, out_dev, scratch_dev, stream));
    if (n == 0) return DMRGK_OK;
    sqrt_inplace_kernel<<<1, 1, 0, (cudaStream_t)stream>>>(out_dev);
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

int32_t dmrgk_vec_axpy(dmrgk_ctx* ctx, int64_t n, double alpha, const double* x_dev, double* y_dev, void* stream) {
    return dmrgk_vec_axpby(ctx, n, alpha, x_dev, 1.0, y_dev, stream);
}

int32_t dmrgk_vec_scal(dmrgk_ctx* ctx, int64_t n, double alpha, double* x_dev, void* stream) {
    DMRGK_TRY(check_vec("vec_scal", ctx, n));
    if (n == 0) return DMRGK_OK;
    if (!x_dev) return fail(DMRGK_EINVAL, "vec_scal: NULL pointer");
    if (!aligned128(x_dev)) return fail(DMRGK_EALIGN, "vec_scal: vector must be 128-byte aligned");
    DMRGK_CUDA(cudaSetDevice(ctx->device));
    const int64_t n2 = n / 2;
    scal_kernel<<<vec_grid(n2), VEC_THREADS, 0, (cudaStream_t)stream>>>(n2, alpha, reinterpret_cast<double2*>(x_dev));
    count_launch();
    DMRGK_CUDA(cudaGetLastError());
    return DMRGK_OK;
}

}  // extern "C"
