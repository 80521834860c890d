// noalloc.cu — tigre_residual_noalloc: the SART / SIRT residual r = W .* (b - Ax) with ||b - Ax||_2^2 (eq. 2; the
// same arithmetic per element as tigre_residual / residual_kernel of elementwise.cu), for callers that cannot allocate:
// code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  tigre_residual takes its fp64
// accumulator from the stream-ordered pool (or the caller's workspace); this entry point takes its scratch from a
// FILE-SCOPE array in device memory instead and calls no cudaMalloc / cudaFree / cudaMallocAsync / allocating library routine,
// creates no stream or event, and does not synchronise.
//
// The scratch: one fp64 partial sum per CTA, NA_MAX_BLOCKS = 16384 of them = 128 KiB, held by every GPU that loads the
// library until the process exits.  A CTA owns NA_CHUNK = 16384 consecutive elements, so the largest call is
// TIGRE_RESIDUAL_NOALLOC_MAX_N = 2^28 elements (1 GiB per array; a C3 subset is 2.8e7); larger n is rejected with
// TIGRE_ERR_TOO_LARGE before anything is launched (split the call).
//
// Every call on a device shares the array and finds the previous call's partials in it.  Nothing has to start at zero: kernel 1
// OVERWRITES slot [blockIdx.x] of each of its ceil(n / NA_CHUNK) CTAs, kernel 2 (same stream, after it) reads exactly those slots
// and none beyond, in a fixed order (so *nrm2 is bitwise reproducible, unlike the atomics of tigre_residual).  Two calls that
// OVERLAP on the GPU (different streams, or graphs replayed concurrently) race on the array: their nrm2 is undefined (r is
// still right).  Calls on one stream, or ordered by events, are safe.
//
// In host code the array's NAME is a host-side stand-in, not a device address, so the address is taken once per device, with that
// device current, by cudaGetSymbolAddress (checked), and that pointer is what the kernels get.
#include <mutex>
#include "common.cuh"

namespace tg {
namespace {

constexpr int NA_THREADS = 256;
constexpr int NA_PER_THREAD = 64;
constexpr size_t NA_CHUNK = (size_t)NA_THREADS * NA_PER_THREAD;   // elements per CTA (a multiple of 4)
constexpr int NA_MAX_BLOCKS = 16384;
static_assert(NA_CHUNK * NA_MAX_BLOCKS == TIGRE_RESIDUAL_NOALLOC_MAX_N, "the header states the limit the scratch array gives");

static __device__ __align__(256) double g_na_partial[NA_MAX_BLOCKS];

__device__ __forceinline__ float na_elem(float b, float a, const float* __restrict__ W, size_t i, double& s) {
    float d = b - a;
    s += (double)d * d;
    if (W) d *= W[i];
    return d;
}

// kernel 1: r and one partial sum of squares per CTA.  VEC: all four arrays are 16-byte aligned.
template <bool VEC>
__global__ void __launch_bounds__(NA_THREADS)
na_residual_kernel(const float* __restrict__ b, const float* __restrict__ Ax, const float* __restrict__ W, float* __restrict__ r,
                   size_t n, double* __restrict__ partial) {
    const size_t lo = (size_t)blockIdx.x * NA_CHUNK, hi = lo + NA_CHUNK < n ? lo + NA_CHUNK : n;
    double s = 0.0;
    size_t tail = lo;
    if (VEC) {
        const size_t hi4 = lo + ((hi - lo) & ~(size_t)3);   // lo is a multiple of 4
        for (size_t i = lo + 4 * (size_t)threadIdx.x; i < hi4; i += 4 * NA_THREADS) {
            const float4 bb = __ldg(reinterpret_cast<const float4*>(b + i)), aa = __ldg(reinterpret_cast<const float4*>(Ax + i));
            float4 d = make_float4(bb.x - aa.x, bb.y - aa.y, bb.z - aa.z, bb.w - aa.w);
            s += (double)d.x * d.x + (double)d.y * d.y + (double)d.z * d.z + (double)d.w * d.w;
            if (W) {
                const float4 ww = __ldg(reinterpret_cast<const float4*>(W + i));
                d.x *= ww.x, d.y *= ww.y, d.z *= ww.z, d.w *= ww.w;
            }
            *reinterpret_cast<float4*>(r + i) = d;
        }
        tail = hi4;
    }
    for (size_t i = tail + threadIdx.x; i < hi; i += NA_THREADS) r[i] = na_elem(b[i], Ax[i], W, i, s);
    if (!partial) return;
    __shared__ double sh[NA_THREADS / 32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        double t = 0.0;
#pragma unroll
        for (int w = 0; w < NA_THREADS / 32; ++w) t += sh[w];
        partial[blockIdx.x] = t;   // overwritten, never accumulated: the last call's value in this slot does not matter
    }
}

// kernel 2: one CTA adds the nblocks partials of THIS call in a fixed order
__global__ void __launch_bounds__(NA_THREADS) na_final_kernel(const double* __restrict__ partial, int nblocks, double* __restrict__ nrm2) {
    __shared__ double sh[NA_THREADS];
    double s = 0.0;
    for (int i = threadIdx.x; i < nblocks; i += NA_THREADS) s += partial[i];
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int o = NA_THREADS / 2; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) *nrm2 = sh[0];
}

// ---- set-up: the device address of the scratch array, once per device
constexpr int NA_MAX_DEVICES = 64;
std::mutex g_na_mu;
double* g_na_ptr[NA_MAX_DEVICES] = {};   // [device ordinal]; nullptr = not asked yet

int na_scratch_of_current_device(double** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess) {
        (void)cudaGetLastError();
        return TIGRE_ERR_NO_DEVICE;
    }
    if (dev < 0 || dev >= NA_MAX_DEVICES) return TIGRE_ERR_ARG;
    std::lock_guard<std::mutex> lk(g_na_mu);
    if (!g_na_ptr[dev]) {
        // `dev` is the current device here, so this is the address of ITS copy of the array (every device that loads the
        // module has one).  g_na_partial itself, used in host code, is only the host-side handle of the symbol.
        double* p = nullptr;
        TG_CUDA(cudaGetSymbolAddress((void**)&p, g_na_partial));
        if (!p) return TIGRE_ERR_CUDA;
        g_na_ptr[dev] = p;
    }
    *out = g_na_ptr[dev];
    return TIGRE_OK;
}

}  // namespace
}  // namespace tg

using namespace tg;

extern "C" TIGRE_API int tigre_residual_noalloc(const float* b, const float* Ax, const float* W, float* r, size_t n, double* nrm2_dev,
                                                void* cuda_stream) {
    if (n > (size_t)TIGRE_RESIDUAL_NOALLOC_MAX_N) return TIGRE_ERR_TOO_LARGE;   // before anything is launched or written
    cudaStream_t st = (cudaStream_t)cuda_stream;
    double* scratch = nullptr;
    TG_TRY(na_scratch_of_current_device(&scratch));
    if (n == 0) {
        if (nrm2_dev) TG_CUDA(cudaMemsetAsync(nrm2_dev, 0, sizeof(double), st));   // an empty sum
        return TIGRE_OK;
    }
    if (!b || !Ax || !r) return TIGRE_ERR_ARG;
    const int nblocks = (int)((n + NA_CHUNK - 1) / NA_CHUNK);   // <= NA_MAX_BLOCKS by the check above
    const bool vec = ((((uintptr_t)b | (uintptr_t)Ax | (uintptr_t)r | (uintptr_t)W) & 15) == 0);
    double* partial = nrm2_dev ? scratch : nullptr;
    if (vec) na_residual_kernel<true><<<nblocks, NA_THREADS, 0, st>>>(b, Ax, W, r, n, partial);
    else na_residual_kernel<false><<<nblocks, NA_THREADS, 0, st>>>(b, Ax, W, r, n, partial);
    if (nrm2_dev) na_final_kernel<<<1, NA_THREADS, 0, st>>>(scratch, nblocks, nrm2_dev);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
