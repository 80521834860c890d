// tv.cu — total-variation / adaptive-weighted TV term, its gradient and the gradient-descent minimiser
// (section 2.2.3 eqs. 7-8; readings P20-P22 of DESIGN.md).
//
//   AwTV(x) = sum_p sqrt( w_x dx^2 + w_y dy^2 + w_z dz^2 + eps ),  d_a = x[p] - x[p - e_a],  w_a = exp(-(d_a/delta)^2)
// over the voxels p that have all their backward neighbours; TV is delta = infinity (w = 1).  With
//   T_p = sqrt(.),  a_a(p) = dT_p/dd_a = d_a w_a (1 - d_a^2/delta^2) / T_p
// the gradient is  g[p] = a_x(p) + a_y(p) + a_z(p) - a_x(p+e_x) - a_y(p+e_y) - a_z(p+e_z).
//
// A stencil, HBM-bound by its bytes (read x once, write g once = 8 B per voxel) — and close to the SFU limit in
// the adaptive case (3 exp + 1 rsqrt per voxel), which is why the a_a are computed ONCE per voxel into shared
// memory (tile plus a one-voxel forward halo) instead of once per use: a CTA stages the x tile with its halo,
// forms T and the three a_a for (TX+1)(TY+1)(TZ+1) voxels, then writes TX*TY*TZ gradients.  The same pass
// returns sum T (the value) and sum g^2 (the minimiser's normalisation) in fp64.
#include <algorithm>
#include <cmath>
#include "common.cuh"

namespace tg {

namespace {

constexpr int TV_TX = 32, TV_TY = 8, TV_TZ = 8;
constexpr int XS_X = TV_TX + 2, XS_Y = TV_TY + 2, XS_Z = TV_TZ + 2;   // x tile with a halo of one on both sides
constexpr int AS_X = TV_TX + 1, AS_Y = TV_TY + 1, AS_Z = TV_TZ + 1;   // a tile with a forward halo of one

__device__ __forceinline__ float ex2_fast(float x) {
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float rsqrt_fast(float x) {
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

__device__ __forceinline__ double block_sum256(double v, double* sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int t = threadIdx.y * blockDim.x + threadIdx.x;
    if ((t & 31) == 0) sh[t >> 5] = v;
    __syncthreads();
    v = t < 8 ? sh[t] : 0.0;
    if (t < 32) {
#pragma unroll
        for (int o = 4; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;
}

// AW: adaptive weights (finite delta).  nl2 = -log2(e)/delta^2, id2 = 1/delta^2.
template <bool AW>
__global__ void __launch_bounds__(TV_TX* TV_TY)
tv_gradient_kernel(const float* __restrict__ x, int nx, int ny, int nz, float nl2, float id2, float eps,
                   float* __restrict__ g, double* __restrict__ d_val, double* __restrict__ d_gg) {
    __shared__ float xs[XS_Z][XS_Y][XS_X];
    __shared__ float ax[AS_Z][AS_Y][AS_X], ay[AS_Z][AS_Y][AS_X], az[AS_Z][AS_Y][AS_X];
    __shared__ double red[8];
    const int x0 = blockIdx.x * TV_TX, y0 = blockIdx.y * TV_TY, z0 = blockIdx.z * TV_TZ;
    const int tid = threadIdx.y * TV_TX + threadIdx.x;
    // ---- 1. the x tile, halo of one voxel on every side (zero outside the volume: never used there)
    for (int i = tid; i < XS_Z * XS_Y * XS_X; i += TV_TX * TV_TY) {
        const int lx = i % XS_X, ly = (i / XS_X) % XS_Y, lz = i / (XS_X * XS_Y);
        const int gx = x0 + lx - 1, gy = y0 + ly - 1, gz = z0 + lz - 1;
        float v = 0.f;
        if ((unsigned)gx < (unsigned)nx && (unsigned)gy < (unsigned)ny && (unsigned)gz < (unsigned)nz)
            v = __ldg(x + ((size_t)gz * ny + gy) * nx + gx);
        xs[lz][ly][lx] = v;
    }
    __syncthreads();
    // ---- 2. T and the three derivatives a_a for the tile and its forward halo
    const bool hx = nx > 1, hy = ny > 1, hz = nz > 1;   // an axis of length 1 drops out (P20)
    double val = 0.0;
    for (int i = tid; i < AS_Z * AS_Y * AS_X; i += TV_TX * TV_TY) {
        const int lx = i % AS_X, ly = (i / AS_X) % AS_Y, lz = i / (AS_X * AS_Y);
        const int gx = x0 + lx, gy = y0 + ly, gz = z0 + lz;
        float fx = 0.f, fy = 0.f, fz = 0.f;
        // summation domain: inside the volume, index >= 1 along every axis that exists
        if (gx < nx && gy < ny && gz < nz && (!hx || gx >= 1) && (!hy || gy >= 1) && (!hz || gz >= 1)) {
            const float c = xs[lz + 1][ly + 1][lx + 1];
            const float dx = hx ? c - xs[lz + 1][ly + 1][lx] : 0.f;
            const float dy = hy ? c - xs[lz + 1][ly][lx + 1] : 0.f;
            const float dz = hz ? c - xs[lz][ly + 1][lx + 1] : 0.f;
            const float qx = dx * dx, qy = dy * dy, qz = dz * dz;
            float wx = 1.f, wy = 1.f, wz = 1.f;
            if (AW) wx = ex2_fast(qx * nl2), wy = ex2_fast(qy * nl2), wz = ex2_fast(qz * nl2);
            const float q = fmaf(wx, qx, fmaf(wy, qy, fmaf(wz, qz, eps)));
            const float it = q > 0.f ? rsqrt_fast(q) : 0.f;
            if (AW) wx *= fmaf(-qx, id2, 1.f), wy *= fmaf(-qy, id2, 1.f), wz *= fmaf(-qz, id2, 1.f);
            fx = dx * wx * it, fy = dy * wy * it, fz = dz * wz * it;
            if (lx < TV_TX && ly < TV_TY && lz < TV_TZ) val += (double)(q * it);   // T_p of the tile's own voxels
        }
        ax[lz][ly][lx] = fx, ay[lz][ly][lx] = fy, az[lz][ly][lx] = fz;
    }
    __syncthreads();
    // ---- 3. gradients of the tile's own voxels
    double gg = 0.0;
    if (g) {
        const int lx = threadIdx.x, ly = threadIdx.y;
        const int gx = x0 + lx, gy = y0 + ly;
        if (gx < nx && gy < ny) {
#pragma unroll
            for (int lz = 0; lz < TV_TZ; ++lz) {
                const int gz = z0 + lz;
                if (gz < nz) {
                    const float v = ax[lz][ly][lx] + ay[lz][ly][lx] + az[lz][ly][lx] - ax[lz][ly][lx + 1] - ay[lz][ly + 1][lx] -
                                    az[lz + 1][ly][lx];
                    g[((size_t)gz * ny + gy) * nx + gx] = v;
                    gg += (double)v * v;
                }
            }
        }
    }
    if (d_val) {
        val = block_sum256(val, red);
        if (tid == 0) atomicAdd(d_val, val);
        __syncthreads();
    }
    if (d_gg && g) {
        gg = block_sum256(gg, red);
        if (tid == 0) atomicAdd(d_gg, gg);
    }
}

// x <- x - alpha * g / sqrt(gg)   (P22; nothing happens when the gradient vanishes)
__global__ void __launch_bounds__(256) tv_step_kernel(float* __restrict__ x, const float* __restrict__ g, float alpha,
                                                      const double* __restrict__ d_gg, size_t n) {
    const double gg = *d_gg;
    if (!(gg > 0.0)) return;
    const float s = alpha * (float)(1.0 / sqrt(gg));
    const size_t n4 = n >> 2;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        float4 a = reinterpret_cast<float4*>(x)[i];
        const float4 b = __ldg(reinterpret_cast<const float4*>(g) + i);
        a.x = fmaf(-s, b.x, a.x), a.y = fmaf(-s, b.y, a.y), a.z = fmaf(-s, b.z, a.z), a.w = fmaf(-s, b.w, a.w);
        reinterpret_cast<float4*>(x)[i] = a;
    }
    for (size_t i = (n4 << 2) + blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
        x[i] = fmaf(-s, g[i], x[i]);
}

}  // namespace

// value and/or gradient of AwTV (delta <= 0 or infinite: TV).  g, d_val, d_gg may each be NULL; the two
// accumulators must be zeroed by the caller.
int launch_tv_gradient(const float* x, int nx, int ny, int nz, float delta, float eps, float* g, double* d_val, double* d_gg,
                       cudaStream_t st) {
    if (nx <= 0 || ny <= 0 || nz <= 0) return TIGRE_ERR_ARG;
    dim3 block(TV_TX, TV_TY), grid((nx + TV_TX - 1) / TV_TX, (ny + TV_TY - 1) / TV_TY, (nz + TV_TZ - 1) / TV_TZ);
    if (grid.y > 65535 || grid.z > 65535) return TIGRE_ERR_ARG;
    ProfScope ps(PK_EW, st);
    const bool aw = delta > 0.f && std::isfinite(delta);
    if (aw) {
        const float id2 = 1.0f / (delta * delta);
        tv_gradient_kernel<true><<<grid, block, 0, st>>>(x, nx, ny, nz, -1.4426950408889634f * id2, id2, eps, g, d_val, d_gg);
    } else {
        tv_gradient_kernel<false><<<grid, block, 0, st>>>(x, nx, ny, nz, 0.f, 0.f, eps, g, d_val, d_gg);
    }
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

int launch_tv_step(float* x, const float* g, float alpha, const double* d_gg, size_t n, cudaStream_t st) {
    if (n == 0) return TIGRE_OK;
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const size_t want = (n / 4 + 255) / 256 + 1;
    const int blocks = (int)std::min<size_t>(want, (size_t)sms * 8);
    ProfScope ps(PK_EW, st);
    if ((reinterpret_cast<uintptr_t>(x) & 15) || (reinterpret_cast<uintptr_t>(g) & 15)) return TIGRE_ERR_ARG;
    tv_step_kernel<<<blocks, 256, 0, st>>>(x, g, alpha, d_gg, n);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg
