// peaks.cu — step-0 microbenchmarks ("shared memory 128 B/clk/SM, L1 gather 1
// wavefront/clk/SM and 18 944 thread-instr/clk are nominal and must be confirmed; L2 bandwidth is unknown until measured;
// pinned H2D / D2H to be measured").  The projector rooflines of bench.py rest on these rates, so they are measured on the
// device the bench runs on, by kernels of this library, each timed with CUDA events on the caller's stream (best of 5 after
// a warm-up).  tigre_microbench(kind, &value, stream):
//   TIGRE_PEAK_FFMA     fp32 multiply-adds issued per second, all SMs (thread-instructions / s of the plain-ALU issue slots)
//   TIGRE_PEAK_SMEM     bytes / s of conflict-free 128-bit shared-memory loads, all SMs
//   TIGRE_PEAK_L1_LINES distinct 128-byte lines / s served by L1 hits when every lane of a request reads its own line
//                       (a fully divergent gather: 32 lines per request), all SMs
//   TIGRE_PEAK_L2       bytes / s of 128-bit loads that miss L1 and hit L2 (48 MB working set, ld.global.cg)
//   TIGRE_PEAK_H2D / TIGRE_PEAK_D2H  bytes / s of one 1 GiB cudaMemcpyAsync from / to pinned host memory
//   TIGRE_PEAK_HBM_COPY bytes / s (read + write) of a 2 GiB device-to-device copy kernel (float4, grid-stride)
//   TIGRE_PEAK_SM_HZ    SM clock seen by clock64() against the global timer while the FFMA kernel runs
#include <algorithm>
#include <cstring>
#include "common.cuh"

namespace tg {
namespace {

constexpr int PK_THREADS = 256;

__global__ void __launch_bounds__(PK_THREADS) pk_ffma_kernel(float* out, int iters, float a, float b, unsigned long long* clk) {
    float x[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) x[j] = (float)(threadIdx.x + j);
    unsigned long long t0 = 0, c0 = 0;
    if (clk && threadIdx.x == 0 && blockIdx.x == 0) {
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t0));
        c0 = clock64();
    }
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u)
#pragma unroll
            for (int j = 0; j < 8; ++j) x[j] = fmaf(x[j], a, b);
    }
    if (clk && threadIdx.x == 0 && blockIdx.x == 0) {
        unsigned long long t1;
        const unsigned long long c1 = clock64();
        asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t1));
        clk[0] = c1 - c0, clk[1] = t1 - t0;
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += x[j];
    if (s == 12345.678f) out[0] = s;   // never true: keeps the chain alive
}

__global__ void __launch_bounds__(PK_THREADS) pk_smem_kernel(float* out, int iters) {
    __shared__ float4 sm[PK_THREADS * 4];
    for (int i = threadIdx.x; i < PK_THREADS * 4; i += PK_THREADS) sm[i] = make_float4((float)i, 1.f, 2.f, 3.f);
    __syncthreads();
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    int idx = threadIdx.x;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {   // four DISTINCT 16-byte words per thread and iteration (the array holds 4 per thread)
            const float4 v = sm[(idx + u * PK_THREADS) & (PK_THREADS * 4 - 1)];   // consecutive lanes, consecutive 16-byte words
            acc.x += v.x, acc.y += v.y, acc.z += v.z, acc.w += v.w;
        }
        idx = (idx + 32) & (PK_THREADS * 4 - 1);
    }
    if (acc.x + acc.y + acc.z + acc.w == 12345.678f) out[0] = acc.x;
}

// every lane reads its own 128-byte line of a per-warp 4 KB window (hot in L1 after the first touch)
__global__ void __launch_bounds__(PK_THREADS) pk_l1_kernel(const float* __restrict__ buf, float* out, int iters) {
    const int warp = (blockIdx.x * PK_THREADS + threadIdx.x) >> 5, lane = threadIdx.x & 31;
    const float* p = buf + (size_t)warp * 1024 + lane * 32;
    // the word each lane reads within ITS line depends on the value just loaded (the buffer holds zeros, which the compiler
    // cannot know): a loop-invariant address would be hoisted out of the loop.  64 resident warps per SM hide the chain.
    float acc = 0.f;
    int off = lane;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int u = 0; u < 8; ++u) {
            const float v = __ldca(p + (off & 31));
            off += 1 + __float_as_int(v);
            acc += v;
        }
    }
    if (acc == 12345.678f) out[0] = acc;
}

__global__ void __launch_bounds__(PK_THREADS) pk_l2_kernel(const float4* __restrict__ buf, size_t n4, float* out, int passes) {
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int p = 0; p < passes; ++p)
        for (size_t i = blockIdx.x * (size_t)PK_THREADS + threadIdx.x; i < n4; i += (size_t)gridDim.x * PK_THREADS) {
            const float4 v = __ldcg(buf + i);
            acc.x += v.x, acc.y += v.y, acc.z += v.z, acc.w += v.w;
        }
    if (acc.x + acc.y + acc.z + acc.w == 12345.678f) out[0] = acc.x;
}

__global__ void __launch_bounds__(PK_THREADS) pk_copy_kernel(const float4* __restrict__ in, float4* __restrict__ outp, size_t n4) {
    for (size_t i = blockIdx.x * (size_t)PK_THREADS + threadIdx.x; i < n4; i += (size_t)gridDim.x * PK_THREADS) outp[i] = in[i];
}

template <class F>
int best_ms(F&& run, cudaStream_t st, double& ms_out, int reps = 5) {
    cudaEvent_t a, b;
    TG_CUDA(cudaEventCreate(&a));
    TG_CUDA(cudaEventCreate(&b));
    double best = 1e300;
    int rc = TIGRE_OK;
    for (int r = 0; r <= reps && rc == TIGRE_OK; ++r) {   // r = 0 warms up
        cudaEventRecord(a, st);
        rc = run();
        cudaEventRecord(b, st);
        if (cudaEventSynchronize(b) != cudaSuccess) rc = TIGRE_ERR_CUDA;
        float t = 0.f;
        cudaEventElapsedTime(&t, a, b);
        if (r > 0) best = std::min(best, (double)t);
    }
    cudaEventDestroy(a);
    cudaEventDestroy(b);
    if (cudaGetLastError() != cudaSuccess) rc = TIGRE_ERR_CUDA;
    ms_out = best;
    return rc;
}

}  // namespace

int microbench(int kind, double* value, cudaStream_t st) {
    int dev = 0, sms = 148;
    TG_CUDA(cudaGetDevice(&dev));
    TG_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
    const int ctas = sms * (2048 / PK_THREADS);   // every SM full
    TempBuf scratch;
    TG_TRY(scratch.alloc(256, st));
    float* out = scratch.as<float>();
    double ms = 0.0;
    switch (kind) {
        case TIGRE_PEAK_FFMA:
        case TIGRE_PEAK_SM_HZ: {
            const int iters = 1 << 15;
            TempBuf clk;
            TG_TRY(clk.alloc(2 * sizeof(unsigned long long), st));
            TG_TRY(best_ms([&] { pk_ffma_kernel<<<ctas, PK_THREADS, 0, st>>>(out, iters, 0.999f, 0.001f, clk.as<unsigned long long>()); return TIGRE_OK; }, st, ms));
            if (kind == TIGRE_PEAK_SM_HZ) {
                unsigned long long h[2] = {0, 1};
                TG_CUDA(cudaMemcpyAsync(h, clk.p, sizeof h, cudaMemcpyDeviceToHost, st));
                TG_CUDA(cudaStreamSynchronize(st));
                *value = h[1] ? (double)h[0] / ((double)h[1] * 1e-9) : 0.0;
            } else {
                *value = (double)ctas * PK_THREADS * (double)iters * 32.0 / (ms * 1e-3);
            }
            return TIGRE_OK;
        }
        case TIGRE_PEAK_SMEM: {
            const int iters = 1 << 13;
            TG_TRY(best_ms([&] { pk_smem_kernel<<<ctas, PK_THREADS, 0, st>>>(out, iters); return TIGRE_OK; }, st, ms));
            *value = (double)ctas * PK_THREADS * (double)iters * 4.0 * 16.0 / (ms * 1e-3);
            return TIGRE_OK;
        }
        case TIGRE_PEAK_L1_LINES: {
            const int iters = 1 << 11;
            TempBuf buf;
            const size_t nwarps = (size_t)ctas * PK_THREADS / 32;
            TG_TRY(buf.alloc(nwarps * 4096, st));
            TG_CUDA(cudaMemsetAsync(buf.p, 0, nwarps * 4096, st));
            TG_TRY(best_ms([&] { pk_l1_kernel<<<ctas, PK_THREADS, 0, st>>>(buf.as<float>(), out, iters); return TIGRE_OK; }, st, ms));
            *value = (double)ctas * PK_THREADS * (double)iters * 8.0 / (ms * 1e-3);   // one line per lane-load
            return TIGRE_OK;
        }
        case TIGRE_PEAK_L2: {
            const size_t bytes = (size_t)48 << 20;
            const int passes = 64;
            TempBuf buf;
            TG_TRY(buf.alloc(bytes, st));
            TG_CUDA(cudaMemsetAsync(buf.p, 0, bytes, st));
            TG_TRY(best_ms([&] { pk_l2_kernel<<<ctas, PK_THREADS, 0, st>>>(buf.as<float4>(), bytes / 16, out, passes); return TIGRE_OK; }, st, ms));
            *value = (double)bytes * passes / (ms * 1e-3);
            return TIGRE_OK;
        }
        case TIGRE_PEAK_H2D:
        case TIGRE_PEAK_D2H: {
            const size_t bytes = (size_t)1 << 30;
            void* host = nullptr;
            TG_CUDA(cudaHostAlloc(&host, bytes, cudaHostAllocDefault));
            TempBuf buf;
            int rc = buf.alloc(bytes, st);
            if (rc == TIGRE_OK) {
                memset(host, 0, bytes);
                rc = best_ms([&] {
                    const cudaError_t e = kind == TIGRE_PEAK_H2D ? cudaMemcpyAsync(buf.p, host, bytes, cudaMemcpyHostToDevice, st)
                                                                 : cudaMemcpyAsync(host, buf.p, bytes, cudaMemcpyDeviceToHost, st);
                    return e == cudaSuccess ? TIGRE_OK : TIGRE_ERR_CUDA;
                }, st, ms, 3);
            }
            buf.release();
            cudaStreamSynchronize(st);
            cudaFreeHost(host);
            TG_TRY(rc);
            *value = (double)bytes / (ms * 1e-3);
            return TIGRE_OK;
        }
        case TIGRE_PEAK_HBM_COPY: {
            const size_t bytes = (size_t)2 << 30;
            TempBuf a, b;
            TG_TRY(a.alloc(bytes, st));
            TG_TRY(b.alloc(bytes, st));
            TG_CUDA(cudaMemsetAsync(a.p, 0, bytes, st));
            TG_TRY(best_ms([&] { pk_copy_kernel<<<ctas, PK_THREADS, 0, st>>>(a.as<float4>(), b.as<float4>(), bytes / 16); return TIGRE_OK; }, st, ms));
            *value = 2.0 * (double)bytes / (ms * 1e-3);
            return TIGRE_OK;
        }
    }
    return TIGRE_ERR_ARG;
}

}  // namespace tg
