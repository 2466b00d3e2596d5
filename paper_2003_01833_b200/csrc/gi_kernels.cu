// gi_kernels.cu -- the steps of Green Iteration that follow the convolution, on the device
// (arXiv 2003.01833 Algorithm 2 lines 4-7):
//
//   line 4  eps_new = eps_old - <V psi_old, psi_old - psi_new> / <psi_new, psi_new>        Eq. (27)
//   line 5  psi <- psi_new - sum_j <psi_new, phi_j> phi_j     (converged wavefunctions phi_j, j < i)
//   line 6  psi <- psi / sqrt(<psi, psi>)
//   line 7  residual = || psi - psi_old ||_2
//
// <a, b> = sum_i w_i a_i b_i (quadrature sum; reading R22).  All four steps are HBM-bound
// reductions / axpys over arrays of N doubles; the output of the convolution never leaves the device
// between two convolutions (188-1246 per SCF step).
//
// Three streaming kernels + one finishing block.  Every reduction is two-level with a FIXED grid and a
// fixed summation order (thread-strided partial sums, fixed-shape block tree, block partials summed by the
// consumer in the same fixed pattern) => bitwise reproducible, no atomics.  The consumer kernel's prologue finishes the
// producer's reduction, so no extra launch or host round trip sits between the steps.
#include <cuda_runtime.h>
#include <cmath>
#include <cstdint>
#include <mutex>
#include <string>

#include "../../include/bltc.h"
#include "gi_kernels.cuh"

namespace bltc {
namespace {

constexpr int kGiThreads = 256;
constexpr int kGiJT = 8;            // phi_j handled per pass of the dot-product kernel

// fixed-shape block reduction: warp shuffle tree, then warp 0 over the 8 warp sums
__device__ __forceinline__ double block_sum(double v, double* s_warp) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    __syncthreads();                                 // s_warp may still be read from the previous call
    if (lane == 0) s_warp[warp] = v;
    __syncthreads();
    double t = 0.0;
    if (warp == 0) {
        t = lane < kGiThreads / 32 ? s_warp[lane] : 0.0;
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) t += __shfl_down_sync(0xffffffffu, t, o);
    }
    return t;                                        // valid in thread 0
}

// sum over the producer's blocks of partial[b * stride + q] by ONE WARP in a fixed order: lane l adds the blocks
// l, l + 32, ... (independent loads, pipelined), then the fixed shuffle tree.  Valid in every lane.
// (A single thread walking 1184 block partials costs 1184 dependent L2 round trips: 0.3 ms; a block-wide tree
// per quantity costs two barriers each: 65 us for 22 quantities.)
__device__ __forceinline__ double warp_sum_block_partials(const double* __restrict__ partial, int nblk, int stride,
                                                          int q) {
    double s = 0.0;
    for (int b = threadIdx.x & 31; b < nblk; b += 32) s += partial[(size_t)b * stride + q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    return s;
}

// K1: partial[b][0] = sum w f (psi_old - psi_new), [1] = sum w psi_new^2, [2 + j] = sum w psi_new phi_j
__global__ void __launch_bounds__(kGiThreads)
gi_dots_kernel(const double* __restrict__ w, const double* __restrict__ psi_old, const double* __restrict__ f_old,
               const double* __restrict__ psi_new, const double* __restrict__ phi, int n_prev, int64_t n,
               double* __restrict__ partial) {
    __shared__ double s_warp[kGiThreads / 32];
    const int stride = 2 + n_prev;
    const int64_t i0 = (int64_t)blockIdx.x * kGiThreads + threadIdx.x, step = (int64_t)gridDim.x * kGiThreads;
    {
        double num = 0.0, nn = 0.0;
        for (int64_t i = i0; i < n; i += step) {
            const double wi = w[i], pn = psi_new[i];
            num = fma(wi * f_old[i], psi_old[i] - pn, num);
            nn = fma(wi * pn, pn, nn);
        }
        const double a = block_sum(num, s_warp);
        const double b = block_sum(nn, s_warp);
        if (threadIdx.x == 0) { partial[(size_t)blockIdx.x * stride] = a; partial[(size_t)blockIdx.x * stride + 1] = b; }
    }
    for (int j0 = 0; j0 < n_prev; j0 += kGiJT) {
        double c[kGiJT];
#pragma unroll
        for (int j = 0; j < kGiJT; ++j) c[j] = 0.0;
        for (int64_t i = i0; i < n; i += step) {
            const double wp = w[i] * psi_new[i];
#pragma unroll
            for (int j = 0; j < kGiJT; ++j)
                if (j0 + j < n_prev) c[j] = fma(wp, phi[(size_t)(j0 + j) * n + i], c[j]);
        }
#pragma unroll
        for (int j = 0; j < kGiJT; ++j) {
            if (j0 + j < n_prev) {                   // uniform across the block
                const double t = block_sum(c[j], s_warp);
                if (threadIdx.x == 0) partial[(size_t)blockIdx.x * stride + 2 + j0 + j] = t;
            }
        }
    }
}

// K2: finish K1's sums; block 0 writes eps_new, delta and the coefficients; psi <- psi_new - sum_j c_j phi_j
// (in place), partial2[b] = sum w psi^2
__global__ void __launch_bounds__(kGiThreads)
gi_deflate_kernel(const double* __restrict__ w, double* __restrict__ psi_new, const double* __restrict__ phi,
                  int n_prev, int64_t n, const double* __restrict__ partial, int nblk1, double eps_old,
                  double* __restrict__ result, double* __restrict__ partial2) {
    extern __shared__ double s_c[];                  // [2 + n_prev]
    __shared__ double s_warp[kGiThreads / 32];
    const int stride = 2 + n_prev;
    for (int q = threadIdx.x >> 5; q < stride; q += kGiThreads / 32) {     // one warp per quantity
        const double t = warp_sum_block_partials(partial, nblk1, stride, q);
        if ((threadIdx.x & 31) == 0) s_c[q] = t;
    }
    __syncthreads();
    if (blockIdx.x == 0) {
        if (threadIdx.x == 0) {
            const double delta = s_c[0] / s_c[1];    // Eq. (27)
            result[kGiEpsNew] = eps_old - delta;
            result[kGiDelta] = delta;
        }
        for (int j = threadIdx.x; j < n_prev; j += kGiThreads) result[kGiCoeff + j] = s_c[2 + j];
    }
    const int64_t i0 = (int64_t)blockIdx.x * kGiThreads + threadIdx.x, step = (int64_t)gridDim.x * kGiThreads;
    double nn = 0.0;
    for (int64_t i = i0; i < n; i += step) {
        double p = psi_new[i];
        for (int j = 0; j < n_prev; ++j) p = fma(-s_c[2 + j], phi[(size_t)j * n + i], p);
        if (n_prev) psi_new[i] = p;
        nn = fma(w[i] * p, p, nn);
    }
    const double t = block_sum(nn, s_warp);
    if (threadIdx.x == 0) partial2[blockIdx.x] = t;
}

// K3: finish the norm; psi <- psi / norm (in place); partial3[b] = sum w (psi - psi_old)^2
__global__ void __launch_bounds__(kGiThreads)
gi_normalize_kernel(const double* __restrict__ w, const double* __restrict__ psi_old, double* __restrict__ psi,
                    int64_t n, const double* __restrict__ partial2, int nblk2, double* __restrict__ result,
                    double* __restrict__ partial3) {
    __shared__ double s_norm;
    __shared__ double s_warp[kGiThreads / 32];
    if (threadIdx.x < 32) {
        const double t = warp_sum_block_partials(partial2, nblk2, 1, 0);
        if (threadIdx.x == 0) {
            s_norm = sqrt(t);
            if (blockIdx.x == 0) result[kGiNorm] = s_norm;
        }
    }
    __syncthreads();
    const double nrm = s_norm;
    const int64_t i0 = (int64_t)blockIdx.x * kGiThreads + threadIdx.x, step = (int64_t)gridDim.x * kGiThreads;
    double rr = 0.0;
    for (int64_t i = i0; i < n; i += step) {
        const double p = psi[i] / nrm;
        psi[i] = p;
        const double d = p - psi_old[i];
        rr = fma(w[i] * d, d, rr);
    }
    const double t = block_sum(rr, s_warp);
    if (threadIdx.x == 0) partial3[blockIdx.x] = t;
}

// K4: one warp finishes the residual
__global__ void gi_finish_kernel(const double* __restrict__ partial3, int nblk3, double* __restrict__ result) {
    const double t = warp_sum_block_partials(partial3, nblk3, 1, 0);
    if (threadIdx.x == 0) result[kGiResidual] = sqrt(t);
}

}  // namespace

int gi_grid_blocks(int64_t n, int sm_count) {
    const int64_t need = (n + kGiThreads - 1) / kGiThreads;
    const int64_t cap = (int64_t)(sm_count > 0 ? sm_count : 148) * 8;     // 8 resident CTAs of 256 threads per SM
    return (int)(need < 1 ? 1 : (need < cap ? need : cap));
}

cudaError_t launch_gi_update(const double* w, const double* psi_old, const double* f_old, double* psi_new,
                             const double* phi, int n_prev, int64_t n, double eps_old, double* result,
                             double* scratch, int nblk, cudaStream_t st) {
    const int stride = 2 + n_prev;
    double* partial = scratch;                       // [nblk][2 + n_prev]
    double* partial2 = partial + (size_t)nblk * stride;
    double* partial3 = partial2 + nblk;
    gi_dots_kernel<<<nblk, kGiThreads, 0, st>>>(w, psi_old, f_old, psi_new, phi, n_prev, n, partial);
    gi_deflate_kernel<<<nblk, kGiThreads, stride * sizeof(double), st>>>(w, psi_new, phi, n_prev, n, partial, nblk,
                                                                          eps_old, result, partial2);
    gi_normalize_kernel<<<nblk, kGiThreads, 0, st>>>(w, psi_old, psi_new, n, partial2, nblk, result, partial3);
    gi_finish_kernel<<<1, 32, 0, st>>>(partial3, nblk, result);
    return cudaGetLastError();
}

size_t gi_scratch_doubles(int n_prev, int nblk) { return (size_t)nblk * (2 + n_prev) + 2 * (size_t)nblk; }

}  // namespace bltc

// ---------------------------------------------------------------------------------------------------------------
// bltc_gi_update_noalloc (include/bltc.h): the same four kernels as bltc_gi_update, for callers that are not allowed
// to allocate device memory.  bltc_gi_update takes the block partial sums of its two-level reductions from the
// library's stream-ordered pool (cudaMallocFromPoolAsync); here they live in the fixed array below, which is part of
// the library image: the driver reserves it on every GPU that loads libbltc.so and keeps it until the process exits.
//
// Size: kGiNoallocMaxBlocks x (2 + kGiNoallocMaxPrev) doubles for the dot products + 2 x kGiNoallocMaxBlocks for the
// norm and the residual = 139,264 doubles = 1.06 MiB per GPU.
//
// Nothing in the array has to start at zero: each of the three reductions writes every slot it later reads (one slot
// per block and quantity, all blocks of the fixed grid), so what the previous call left behind is never read and no
// clearing pass is needed.  What the shared array does cost is concurrency: two calls in flight on the same GPU at
// the same time (two streams, two host threads, two graphs) write the same slots and corrupt each other's sums.
namespace {

constexpr int kGiNoallocMaxPrev = BLTC_GI_NOALLOC_MAX_PREV;
constexpr int kGiNoallocMaxBlocks = 2048;
constexpr size_t kGiNoallocDoubles =
    (size_t)kGiNoallocMaxBlocks * (2 + kGiNoallocMaxPrev) + 2 * (size_t)kGiNoallocMaxBlocks;

static __device__ __align__(256) double g_gi_noalloc_scratch[kGiNoallocDoubles];

constexpr int kMaxDevices = 64;

struct GiNoallocDevice {
    double* scratch = nullptr;       // DEVICE address of g_gi_noalloc_scratch on this GPU
    int nblk_cap = 0;                // SM count x 8, at most kGiNoallocMaxBlocks
};

// Per-GPU set-up, done by the first call on each device with that device current.  In host code the name
// g_gi_noalloc_scratch is only the handle the runtime registered for the symbol; the address a kernel can
// dereference differs per GPU and has to be asked for.  cudaGetSymbolAddress may initialise the context and load the
// module, which is why the first call on a device belongs before any stream capture.
cudaError_t gi_noalloc_device(GiNoallocDevice* out) {
    static std::mutex mu;
    static GiNoallocDevice table[kMaxDevices];
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!table[dev].scratch) {
        double* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_gi_noalloc_scratch);
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return e;
        const int cap = (sms > 0 ? sms : 148) * 8;
        table[dev].nblk_cap = cap < kGiNoallocMaxBlocks ? cap : kGiNoallocMaxBlocks;
        table[dev].scratch = ptr;
    }
    *out = table[dev];
    return cudaSuccess;
}

bool gi_noalloc_on_device(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return false; }
    return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

extern "C" int bltc_gi_update_noalloc(const double* w, const double* psi_old, const double* f_old, double* psi_new,
                                      const double* phi, int n_prev, int64_t N, double eps_old, double* result,
                                      bltc_stream stream) {
    using bltc::set_last_error;
    // argument and size checks first: they need no device, and a refused call must not touch the shared array
    if (!w || !psi_old || !f_old || !psi_new || !result) return set_last_error(BLTC_EINVAL, "NULL argument");
    if (N < 1 || N > 2000000000LL) return set_last_error(BLTC_EINVAL, "N must be in [1, 2e9]");
    if (n_prev < 0) return set_last_error(BLTC_EINVAL, "n_prev must be >= 0");
    if (n_prev > kGiNoallocMaxPrev)
        return set_last_error(BLTC_EINVAL,
                              ("bltc_gi_update_noalloc: n_prev = " + std::to_string(n_prev) +
                               " exceeds BLTC_GI_NOALLOC_MAX_PREV = " + std::to_string(kGiNoallocMaxPrev) +
                               ", the most the library's fixed scratch array holds; use bltc_gi_update").c_str());
    if (n_prev > 0 && !phi) return set_last_error(BLTC_EINVAL, "phi is NULL but n_prev > 0");
    if (!std::isfinite(eps_old)) return set_last_error(BLTC_EINVAL, "eps_old must be finite");
    // host buffers would need a staging copy on the device, i.e. an allocation: refused here
    if (!gi_noalloc_on_device(w) || !gi_noalloc_on_device(psi_old) || !gi_noalloc_on_device(f_old) ||
        !gi_noalloc_on_device(psi_new) || !gi_noalloc_on_device(result) || (n_prev > 0 && !gi_noalloc_on_device(phi)))
        return set_last_error(BLTC_EINVAL,
                              "bltc_gi_update_noalloc: every buffer must be device memory (staging a host buffer "
                              "would allocate); use bltc_gi_update for host buffers");
    GiNoallocDevice d;
    cudaError_t e = gi_noalloc_device(&d);
    if (e != cudaSuccess) {
        cudaGetLastError();
        return set_last_error(BLTC_ECUDA, (std::string("bltc_gi_update_noalloc set-up (cudaGetSymbolAddress): ") +
                                           cudaGetErrorString(e)).c_str());
    }
    // the grid of bltc_gi_update (gi_grid_blocks), so that both entry points sum in the same order
    const int64_t need = (N + bltc::kGiThreads - 1) / bltc::kGiThreads;
    const int nblk = (int)(need < d.nblk_cap ? need : d.nblk_cap);
    if (bltc::gi_scratch_doubles(n_prev, nblk) > kGiNoallocDoubles)       // cannot happen given the two caps above
        return set_last_error(BLTC_EINVAL, "bltc_gi_update_noalloc: scratch array too small");
    e = bltc::launch_gi_update(w, psi_old, f_old, psi_new, phi, n_prev, N, eps_old, result, d.scratch, nblk,
                               static_cast<cudaStream_t>(stream));
    if (e != cudaSuccess) {
        cudaGetLastError();
        return set_last_error(BLTC_ECUDA, (std::string("bltc_gi_update_noalloc launch: ") + cudaGetErrorString(e)).c_str());
    }
    return BLTC_OK;
}
