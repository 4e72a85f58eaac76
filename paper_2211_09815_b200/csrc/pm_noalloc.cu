// pm_noalloc.cu -- the mesh objective as ONE entry point that allocates nothing (no ctx, no workspace, no cudaMalloc /
// cudaFree, no allocating library routine): for callers that cannot allocate -- code under CUDA graph capture, tight
// serving loops, harnesses that forbid it.
//
// What it computes is pm_objective's reduction (eq. 17; BASELINE.json configs):
//     r(g) = rho(g) / nbar - 1 - delta_target(g),   J = 1/2 sum_g r(g)^2   (fp64 accumulation, fixed order)
// on caller-provided flat arrays.  The existing kernel (pm_integrate.cu objective_kernel) keeps its per-block partial
// sums in the ctx workspace; this variant keeps them in the file-scope device array below:
//   * PM_NOALLOC_MAX_N = 2^30 elements per call (a 1024^3 mesh), i.e. 16384 blocks of 65536 elements, one double each:
//     128 KB of device memory that every GPU which loads libpm.so holds until the process exits;
//   * every call on a device shares the array, and it keeps the last call's contents.  Nothing in it has to start at zero
//     (the final kernel reads exactly the partials the first kernel of the SAME call has written), but two calls that
//     overlap on the GPU (different streams, no ordering between them) race on it: order them.
// In host code `g_noalloc_partials` is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, resolved once per device with that device current (pm_noalloc_setup, or the first call).
#include <cstdio>

#include "pm_internal.cuh"

namespace pm {

constexpr int NA_CHUNK = 65536;                       // elements per block
constexpr int NA_MAX_BLOCKS = 16384;                  // -> PM_NOALLOC_MAX_N = 2^30
static_assert((long long)NA_CHUNK * NA_MAX_BLOCKS == PM_NOALLOC_MAX_N, "pm.h and pm_noalloc.cu disagree on the maximum");

static __device__ __align__(256) double g_noalloc_partials[NA_MAX_BLOCKS];

// block b: elements [b * NA_CHUNK, min(n, (b + 1) * NA_CHUNK)); residual written when resid != NULL
__global__ void __launch_bounds__(256) noalloc_objective_kernel(long long n, const float *__restrict__ rho, const float *__restrict__ target,
                                                                float inv_nbar, float *__restrict__ resid, double *__restrict__ partial)
{
    __shared__ double red[8];
    const long long lo = (long long)blockIdx.x * NA_CHUNK, hi = min(n, lo + NA_CHUNK);
    double part = 0.0;
    for (long long i = lo + threadIdx.x; i < hi; i += 256) {
        const float r = fmaf(rho[i], inv_nbar, -1.f) - target[i];
        if (resid) resid[i] = r;
        part += 0.5 * (double)r * (double)r;
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = part;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
        for (int k = 0; k < 8; k++) t += red[k];
        partial[blockIdx.x] = t;
    }
}

// one block: fixed-order sum of the nblocks partials (bit-reproducible J on any GPU)
__global__ void __launch_bounds__(256) noalloc_final_kernel(int nblocks, const double *__restrict__ partial, double *__restrict__ J)
{
    __shared__ double sh[256];
    double t = 0.0;
    for (int k = threadIdx.x; k < nblocks; k += 256) t += partial[k];
    sh[threadIdx.x] = t;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) J[0] = sh[0];
}

// device address of the scratch array, per device (resolved with that device current)
static double *g_noalloc_ptr[64] = {};

static int noalloc_scratch(double **out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return fail(nullptr, PM_ECUDA, "pm_noalloc: cudaGetDevice", cudaGetErrorString(e));
    if (dev < 0 || dev >= 64) return fail(nullptr, PM_EINVAL, "pm_noalloc", "device ordinal beyond 63");
    if (!g_noalloc_ptr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_noalloc_partials);
        if (e != cudaSuccess || !p) return fail(nullptr, PM_ECUDA, "pm_noalloc: cudaGetSymbolAddress(g_noalloc_partials)", cudaGetErrorString(e));
        g_noalloc_ptr[dev] = p;
    }
    *out = g_noalloc_ptr[dev];
    return PM_OK;
}

}  // namespace pm

extern "C" {

int pm_noalloc_setup(void)
{
    double *p;
    return pm::noalloc_scratch(&p);
}

int pm_objective_noalloc(int64_t n, const float *dev_rho, const float *dev_delta_target, double nbar, float *dev_resid,
                         double *dev_J, void *cuda_stream)
{
    using namespace pm;
    if (n < 1 || n > PM_NOALLOC_MAX_N) {
        char b[160];
        snprintf(b, sizeof b, "n = %lld is outside 1 .. PM_NOALLOC_MAX_N = %lld (the static scratch holds one partial per 65536 elements)",
                 (long long)n, (long long)PM_NOALLOC_MAX_N);
        return fail(nullptr, PM_EINVAL, "pm_objective_noalloc", b);
    }
    if (!dev_rho || !dev_delta_target || !dev_J || (((uintptr_t)dev_rho | (uintptr_t)dev_delta_target | (uintptr_t)dev_resid) & 3) ||
        ((uintptr_t)dev_J & 7))
        return fail(nullptr, PM_EINVAL, "pm_objective_noalloc", "NULL or misaligned pointer");
    if (!(nbar > 0.0)) return fail(nullptr, PM_EINVAL, "pm_objective_noalloc", "nbar must be > 0");
    double *scratch = nullptr;
    PM_TRY(noalloc_scratch(&scratch));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nb = (int)((n + NA_CHUNK - 1) / NA_CHUNK);
    noalloc_objective_kernel<<<nb, 256, 0, st>>>((long long)n, dev_rho, dev_delta_target, (float)(1.0 / nbar), dev_resid, scratch);
    noalloc_final_kernel<<<1, 256, 0, st>>>(nb, scratch, dev_J);
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return fail(nullptr, PM_ECUDA, "pm_objective_noalloc", cudaGetErrorString(e));
    return PM_OK;
}

}  // extern "C"
