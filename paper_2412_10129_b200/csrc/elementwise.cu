// elementwise.cu — the HBM-bound half of the Kaczmarz family (eq. 6 at 135):
// residual r = W.*(b - Ax), update x = max(0, x + lambda V.*g), weight inversion, the CGLS
// vector recurrences.  (The FDK pre-filter lives in fdk.cu.)
// Grid-stride kernels, float4 where alignment allows, grids sized as a multiple of the SM count.
// Reductions: fp32 products accumulated in fp64 per thread, block tree, one fp64 atomic per block.
#include <cmath>
#include "common.cuh"

namespace tg {

static int ew_blocks(size_t n, int per_thread = 4) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    size_t want = (n + (size_t)256 * per_thread - 1) / ((size_t)256 * per_thread);
    size_t cap = (size_t)sms * 8;
    if (want < 1) want = 1;
    return (int)(want < cap ? want : cap);
}

__device__ __forceinline__ double block_sum(double v) {
    __shared__ double sh[32];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    if (l == 0) sh[w] = v;
    __syncthreads();
    v = (threadIdx.x < (blockDim.x >> 5)) ? sh[threadIdx.x] : 0.0;
    if (w == 0) {
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;
}

// r[j][i] = W[j][i] * (b[view_idx[j]][i] - Ax[j][i]);  nrm2 += sum (b - Ax)^2
__global__ void __launch_bounds__(256)
residual_kernel(const float* __restrict__ b, const int32_t* __restrict__ view_idx, const float* __restrict__ Ax,
                const float* __restrict__ W, float* __restrict__ r, size_t per_view, int nViews,
                double* __restrict__ nrm2) {
    const size_t n4 = per_view >> 2;  // per_view % 4 == 0 guaranteed by the launcher (else scalar path)
    double s = 0.0;
    const size_t total = n4 * nViews;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(i / n4);
        const size_t k = i - (size_t)j * n4;
        const size_t src = (size_t)(view_idx ? view_idx[j] : j) * n4 + k;
        const float4 bb = __ldg(reinterpret_cast<const float4*>(b) + src);
        const float4 aa = __ldg(reinterpret_cast<const float4*>(Ax) + i);
        float4 d = make_float4(bb.x - aa.x, bb.y - aa.y, bb.z - aa.z, bb.w - aa.w);
        s += (double)d.x * d.x + (double)d.y * d.y + (double)d.z * d.z + (double)d.w * d.w;
        if (W) {   // W is laid out like Ax / r (view-list order)
            const float4 ww = __ldg(reinterpret_cast<const float4*>(W) + i);
            d.x *= ww.x, d.y *= ww.y, d.z *= ww.z, d.w *= ww.w;
        }
        reinterpret_cast<float4*>(r)[i] = d;
    }
    if (nrm2) {
        s = block_sum(s);
        if (threadIdx.x == 0) atomicAdd(nrm2, s);
    }
}
__global__ void __launch_bounds__(256)
residual_kernel_scalar(const float* __restrict__ b, const int32_t* __restrict__ view_idx, const float* __restrict__ Ax,
                       const float* __restrict__ W, float* __restrict__ r, size_t per_view, int nViews,
                       double* __restrict__ nrm2) {
    double s = 0.0;
    const size_t total = per_view * nViews;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const int j = (int)(i / per_view);
        const size_t src = (size_t)(view_idx ? view_idx[j] : j) * per_view + (i - (size_t)j * per_view);
        float d = b[src] - Ax[i];
        s += (double)d * d;
        if (W) d *= W[i];
        r[i] = d;
    }
    if (nrm2) {
        s = block_sum(s);
        if (threadIdx.x == 0) atomicAdd(nrm2, s);
    }
}

int launch_residual(const float* b, const int32_t* view_idx, const float* Ax, const float* W, float* r,
                    size_t per_view, int nViews, double* d_nrm2, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    const size_t total = per_view * nViews;
    if (total == 0) return TIGRE_OK;
    const bool al = ((per_view & 3) == 0) && ((((uintptr_t)b | (uintptr_t)Ax | (uintptr_t)r | (uintptr_t)W) & 15) == 0);
    if (al) residual_kernel<<<ew_blocks(total / 4), 256, 0, st>>>(b, view_idx, Ax, W, r, per_view, nViews, d_nrm2);
    else residual_kernel_scalar<<<ew_blocks(total), 256, 0, st>>>(b, view_idx, Ax, W, r, per_view, nViews, d_nrm2);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

__global__ void __launch_bounds__(256)
update_kernel(float* __restrict__ x, const float* __restrict__ g, const float* __restrict__ V, float lambda, int nonneg,
              size_t n, int vec) {
    if (vec) {
        const size_t n4 = n >> 2;
        for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
            float4 xx = reinterpret_cast<float4*>(x)[i];
            const float4 gg = __ldg(reinterpret_cast<const float4*>(g) + i);
            float4 vv = make_float4(1.f, 1.f, 1.f, 1.f);
            if (V) vv = __ldg(reinterpret_cast<const float4*>(V) + i);
            xx.x = fmaf(lambda * vv.x, gg.x, xx.x), xx.y = fmaf(lambda * vv.y, gg.y, xx.y);
            xx.z = fmaf(lambda * vv.z, gg.z, xx.z), xx.w = fmaf(lambda * vv.w, gg.w, xx.w);
            if (nonneg) xx.x = fmaxf(xx.x, 0.f), xx.y = fmaxf(xx.y, 0.f), xx.z = fmaxf(xx.z, 0.f), xx.w = fmaxf(xx.w, 0.f);
            reinterpret_cast<float4*>(x)[i] = xx;
        }
        // tail
        for (size_t i = (n4 << 2) + blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
            float xx = fmaf(lambda * (V ? V[i] : 1.f), g[i], x[i]);
            x[i] = nonneg ? fmaxf(xx, 0.f) : xx;
        }
    } else {
        for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
            float xx = fmaf(lambda * (V ? V[i] : 1.f), g[i], x[i]);
            x[i] = nonneg ? fmaxf(xx, 0.f) : xx;
        }
    }
}
int launch_update(float* x, const float* g, const float* V, float lambda, int nonneg, size_t n, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    if (n == 0) return TIGRE_OK;
    const int vec = ((((uintptr_t)x | (uintptr_t)g | (uintptr_t)V) & 15) == 0) ? 1 : 0;
    update_kernel<<<ew_blocks(n / 4 + 1), 256, 0, st>>>(x, g, V, lambda, nonneg, n, vec);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

// x <- max(0, x + lambda V g) (as update_kernel) AND xT[z][x][y] <- the new x: the Siddon / interpolated Ax kernels read an
// (x,y)-transposed copy for x-dominant rays; writing it here saves re-reading the volume in a separate transpose pass.
__global__ void __launch_bounds__(256)
update_t_kernel(float* __restrict__ x, float* __restrict__ xT, const float* __restrict__ g, const float* __restrict__ V,
                float lambda, int nonneg, int nx, int ny) {
    __shared__ float tile[32][33];
    const size_t slice = (size_t)nx * ny * blockIdx.z;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int ix = x0 + threadIdx.x, iy = y0 + j;
        if (ix < nx && iy < ny) {
            const size_t i = slice + (size_t)iy * nx + ix;
            float v = fmaf(lambda * (V ? __ldg(V + i) : 1.f), __ldg(g + i), x[i]);
            if (nonneg) v = fmaxf(v, 0.f);
            x[i] = v;
            tile[j][threadIdx.x] = v;
        }
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int iy = y0 + threadIdx.x, ix = x0 + j;
        if (ix < nx && iy < ny) xT[slice + (size_t)ix * ny + iy] = tile[threadIdx.x][j];
    }
}
int launch_update_t(float* x, float* xT, const float* g, const float* V, float lambda, int nonneg, int nx, int ny, int nz,
                    cudaStream_t st) {
    dim3 tb(32, 8), grid((nx + 31) / 32, (ny + 31) / 32, nz);
    if (grid.y > 65535 || grid.z > 65535) return TIGRE_ERR_ARG;
    ProfScope ps(PK_EW, st);
    update_t_kernel<<<grid, tb, 0, st>>>(x, xT, g, V, lambda, nonneg, nx, ny);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

__global__ void __launch_bounds__(256) invert_kernel(float* __restrict__ w, size_t n, float eps, const float* __restrict__ d_max, float rel) {
    const float e = d_max ? rel * (*d_max) : eps;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float v = w[i];
        w[i] = v > e ? 1.0f / v : 0.f;
    }
}
__global__ void __launch_bounds__(256) max_kernel(const float* __restrict__ v, size_t n, float* __restrict__ out) {
    float m = 0.f;   // column sums are non-negative
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) m = fmaxf(m, v[i]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_down_sync(0xffffffffu, m, o));
    if ((threadIdx.x & 31) == 0) atomicMax(reinterpret_cast<int*>(out), __float_as_int(m));   // valid for m >= 0
}
int launch_invert_rows(float* w, size_t n, float eps, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    if (n == 0) return TIGRE_OK;
    invert_kernel<<<ew_blocks(n), 256, 0, st>>>(w, n, eps, nullptr, 0.f);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
int launch_invert_cols(float* v, size_t n, float rel_eps, cudaStream_t st) {
    ProfScope ps(PK_EW, st, 2);
    if (n == 0) return TIGRE_OK;
    TempBuf mx;
    TG_TRY(mx.alloc(sizeof(float), st));
    TG_CUDA(cudaMemsetAsync(mx.p, 0, sizeof(float), st));
    max_kernel<<<ew_blocks(n), 256, 0, st>>>(v, n, mx.as<float>());
    invert_kernel<<<ew_blocks(n), 256, 0, st>>>(v, n, 0.f, mx.as<float>(), rel_eps);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

// MLEM / OSEM (eq. 5; reading P33): q[j][i] = b[view_idx[j]][i] / Ax[j][i] where Ax > 0, else 0 (in place over Ax is fine)
__global__ void __launch_bounds__(256) ratio_kernel(const float* __restrict__ b, const int32_t* __restrict__ view_idx,
                                                    const float* __restrict__ Ax, float* __restrict__ q, size_t per_view, size_t total) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t j = i / per_view;
        const size_t src = (size_t)(view_idx ? view_idx[j] : (int32_t)j) * per_view + (i - j * per_view);
        const float p = Ax[i];
        q[i] = p > 0.f ? __ldg(b + src) / p : 0.f;
    }
}
int launch_ratio(const float* b, const int32_t* view_idx, const float* Ax, float* q, size_t per_view, int nViews, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    const size_t total = per_view * nViews;
    if (total == 0) return TIGRE_OK;
    ratio_kernel<<<ew_blocks(total), 256, 0, st>>>(b, view_idx, Ax, q, per_view, total);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
// x <- x * V * g   (the multiplicative update of eq. 5; V = 1/(A^T 1))
__global__ void __launch_bounds__(256) mul_update_kernel(float* __restrict__ x, const float* __restrict__ g, const float* __restrict__ V,
                                                         size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        x[i] = x[i] * __ldg(V + i) * __ldg(g + i);
}
int launch_mul_update(float* x, const float* g, const float* V, size_t n, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    if (n == 0) return TIGRE_OK;
    mul_update_kernel<<<ew_blocks(n), 256, 0, st>>>(x, g, V, n);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

// W[j][iv][iu] *= colw[j][iu]   (data-redundancy weighting of the row weights, reading P17)
__global__ void __launch_bounds__(256) scale_columns_kernel(float* __restrict__ W, const float* __restrict__ colw, int nu, size_t per,
                                                            size_t total) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t j = i / per;
        const int iu = (int)((i - j * per) % (size_t)nu);
        W[i] *= __ldg(colw + j * nu + iu);
    }
}
int launch_scale_columns(float* W, const float* colw, int nViews, int nv, int nu, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    const size_t per = (size_t)nv * nu, total = per * nViews;
    if (total == 0) return TIGRE_OK;
    scale_columns_kernel<<<ew_blocks(total), 256, 0, st>>>(W, colw, nu, per, total);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
__global__ void __launch_bounds__(256) dot_kernel(const float* __restrict__ a, const float* __restrict__ b, size_t n, double* __restrict__ out) {
    double s = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        s += (double)a[i] * (double)b[i];
    s = block_sum(s);
    if (threadIdx.x == 0) atomicAdd(out, s);
}
int launch_dot(const float* a, const float* b, size_t n, double* d_out, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    TG_CUDA(cudaMemsetAsync(d_out, 0, sizeof(double), st));
    if (n == 0) return TIGRE_OK;
    dot_kernel<<<ew_blocks(n), 256, 0, st>>>(a, b, n, d_out);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
// ASD-POCS step statistics (reading P23): out[0] += ||a - b||^2, out[1] += <a - b, b - c>, out[2] += ||b - c||^2
__global__ void __launch_bounds__(256) diff_stats_kernel(const float* __restrict__ a, const float* __restrict__ b,
                                                         const float* __restrict__ c, size_t n, double* __restrict__ out) {
    double s0 = 0.0, s1 = 0.0, s2 = 0.0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float bb = b[i];
        const double u = (double)(a[i] - bb), v = (double)(bb - c[i]);
        s0 += u * u, s1 += u * v, s2 += v * v;
    }
    s0 = block_sum(s0);
    __syncthreads();
    s1 = block_sum(s1);
    __syncthreads();
    s2 = block_sum(s2);
    if (threadIdx.x == 0) atomicAdd(out, s0), atomicAdd(out + 1, s1), atomicAdd(out + 2, s2);
}
int launch_diff_stats(const float* a, const float* b, const float* c, size_t n, double* d_out3, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    TG_CUDA(cudaMemsetAsync(d_out3, 0, 3 * sizeof(double), st));
    if (n == 0) return TIGRE_OK;
    diff_stats_kernel<<<ew_blocks(n), 256, 0, st>>>(a, b, c, n, d_out3);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
__global__ void __launch_bounds__(256) axpy_kernel(float* __restrict__ y, const float* __restrict__ x, const double* num, const double* den, float sign, size_t n) {
    const float a = sign * (float)(*num / *den);
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) y[i] = fmaf(a, x[i], y[i]);
}
int launch_axpy(float* y, const float* x, const double* d_num, const double* d_den, float sign, size_t n, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    if (n == 0) return TIGRE_OK;
    axpy_kernel<<<ew_blocks(n), 256, 0, st>>>(y, x, d_num, d_den, sign, n);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
__global__ void __launch_bounds__(256) xpby_kernel(float* __restrict__ p, const float* __restrict__ s, const double* num, const double* den, size_t n) {
    const float bta = (float)(*num / *den);
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = fmaf(bta, p[i], s[i]);
}
int launch_xpby(float* p, const float* s, const double* d_num, const double* d_den, size_t n, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    if (n == 0) return TIGRE_OK;
    xpby_kernel<<<ew_blocks(n), 256, 0, st>>>(p, s, d_num, d_den, n);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
__global__ void __launch_bounds__(256) scale_kernel(float* __restrict__ x, float a, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) x[i] *= a;
}
int launch_scale(float* x, float a, size_t n, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    if (n == 0) return TIGRE_OK;
    scale_kernel<<<ew_blocks(n), 256, 0, st>>>(x, a, n);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

__global__ void __launch_bounds__(256) fill_kernel(float* __restrict__ x, float a, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) x[i] = a;
}
int launch_fill(float* x, float a, size_t n, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    if (n == 0) return TIGRE_OK;
    fill_kernel<<<ew_blocks(n), 256, 0, st>>>(x, a, n);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
int launch_max(const float* v, size_t n, float* d_max, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    if (n == 0) return TIGRE_OK;
    max_kernel<<<ew_blocks(n), 256, 0, st>>>(v, n, d_max);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

__global__ void __launch_bounds__(256) count_reduce_kernel(const uint32_t* __restrict__ c, size_t n, unsigned long long* __restrict__ out) {
    unsigned long long s = 0;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) s += c[i];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) atomicAdd(out, s);
}
int launch_count_reduce(const uint32_t* c, size_t n, unsigned long long* d_total, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    TG_CUDA(cudaMemsetAsync(d_total, 0, sizeof(unsigned long long), st));
    if (n == 0) return TIGRE_OK;
    count_reduce_kernel<<<ew_blocks(n), 256, 0, st>>>(c, n, d_total);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg
