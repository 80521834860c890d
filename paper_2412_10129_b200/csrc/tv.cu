// tv.cu — total-variation / adaptive-weighted TV term, its gradient and the gradient-descent minimiser
// (section 2.2.3 eqs. 7-8; readings P20-P22 of DESIGN.md).
//
//   AwTV(x) = sum_p sqrt( w_x dx^2 + w_y dy^2 + w_z dz^2 + eps ),  d_a = x[p] - x[p - e_a],  w_a = exp(-(d_a/delta)^2)
// over the voxels p that have all their backward neighbours; TV is delta = infinity (w = 1).  With
//   T_p = sqrt(.),  a_a(p) = dT_p/dd_a = d_a w_a (1 - d_a^2/delta^2) / T_p
// the gradient is  g[p] = a_x(p) + a_y(p) + a_z(p) - a_x(p+e_x) - a_y(p+e_y) - a_z(p+e_z).
//
// A stencil, HBM-bound by its bytes (read x once, write g once = 8 B per voxel) and, in the adaptive case, close
// to the SFU limit (3 exp + 1 rsqrt per voxel): so T and the a_a are computed ONCE per voxel and handed to the
// three neighbours that need them (shuffle, shared memory, the next plane) instead of once per use.  The same
// pass returns sum T (the value) and sum g^2 (the minimiser's normalisation) in fp64.
#include <algorithm>
#include <cmath>
#include "common.cuh"

namespace tg {

namespace {

constexpr int TV_BX = 32, TV_BY = 16;   // threads per CTA; it owns (BX-1) x (BY-1) columns, the last column / row is halo
constexpr int TV_ZCHUNK = 64;           // planes per CTA along z
#define TV_PF 4                         // planes of x loaded ahead of the one being worked on

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

__device__ __forceinline__ double block_sum512(double v, double* sh) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    const int t = threadIdx.y * blockDim.x + threadIdx.x;
    if ((t & 31) == 0) sh[t >> 5] = v;
    __syncthreads();
    v = t < (int)(blockDim.x * blockDim.y) >> 5 ? sh[t] : 0.0;
    if (t < 32) {
#pragma unroll
        for (int o = 8; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    }
    return v;
}

// AW: adaptive weights (finite delta).  nl2 = -log2(e)/delta^2, id2 = 1/delta^2.
// Streaming along z: a CTA of 32 x 16 threads owns 31 x 15 columns of voxels and walks TV_ZCHUNK planes; a thread
// forms T and the three a_a of ITS voxel once per plane (x[p - e_z] is the previous plane's value, kept in a
// register; x[p - e_x], x[p - e_y] are L1 hits), gets a_x(p + e_x) from the next lane (shuffle), a_y(p + e_y) from
// the next row (shared memory, double buffered: one barrier per plane) and a_z(p + e_z) one plane later, which is
// when the gradient of the previous plane is written.
template <bool AW>
__global__ void __launch_bounds__(TV_BX* TV_BY)
tv_gradient_kernel(const float* __restrict__ x, int nx, int ny, int nz, float nl2, float id2, float eps,
                   float* __restrict__ g, double* __restrict__ d_val, double* __restrict__ d_gg) {
    __shared__ float say[2][TV_BY][TV_BX];
    __shared__ double red[16];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int gx = blockIdx.x * (TV_BX - 1) + tx, gy = blockIdx.y * (TV_BY - 1) + ty;
    const int zs = blockIdx.z * TV_ZCHUNK, ze = min(zs + TV_ZCHUNK, nz);
    const bool hx = nx > 1, hy = ny > 1, hz = nz > 1;   // an axis of length 1 drops out (P20)
    const bool inside = gx < nx && gy < ny;
    const bool owner = inside && tx < TV_BX - 1 && ty < TV_BY - 1;
    const bool dom_xy = inside && (!hx || gx >= 1) && (!hy || gy >= 1);
    const size_t plane = (size_t)nx * ny;
    size_t idx = ((size_t)zs * ny + gy) * nx + gx;
    const float* px = x + idx;                 // this thread's voxel in the current plane
    float* pg = g ? g + idx : nullptr;
    float xprev = (inside && hz && zs >= 1) ? __ldg(px - plane) : 0.f;
    float Sprev = 0.f;
    // partial sums in fp32 over 16 planes at a time, then into fp64 (fp64 arithmetic per voxel would dominate the
    // instruction count: the fp64 pipe of this part is narrow)
    float vacc = 0.f, gacc = 0.f;
    double val = 0.0, gg = 0.0;
    int buf = 0;
    const bool ldx = hx && gx >= 1, ldy = hy && gy >= 1;
    // the z walk is a chain of dependent iterations: without loads in flight ahead of it a thread has 4 bytes
    // outstanding and the SM far too few to cover the HBM latency, so x[p] of the next TV_PF planes sits in a register queue
    const int zlast = min(ze, nz - 1);        // last plane this CTA reads
    float cq[TV_PF];
#pragma unroll
    for (int i = 0; i < TV_PF; ++i) cq[i] = (inside && zs + i <= zlast) ? __ldg(px + (size_t)i * plane) : 0.f;
#pragma unroll 4
    for (int z = zs; z <= ze; ++z) {          // plane ze is visited for its a_z only (nothing beyond the volume)
        float c = 0.f, fx = 0.f, fy = 0.f, fz = 0.f, T = 0.f;
        const float cnow = cq[0];
#pragma unroll
        for (int i = 0; i + 1 < TV_PF; ++i) cq[i] = cq[i + 1];
        cq[TV_PF - 1] = (inside && z + TV_PF <= zlast) ? __ldg(px + (size_t)TV_PF * plane) : 0.f;
        if (inside && z < nz) {
            c = cnow;
            if (dom_xy && (!hz || z >= 1)) {   // summation domain: index >= 1 along every axis that exists
                const float dx = ldx ? c - __ldg(px - 1) : 0.f;
                const float dy = ldy ? c - __ldg(px - nx) : 0.f;
                const float dz = hz ? c - xprev : 0.f;
                const float qx = dx * dx, qy = dy * dy, qz = dz * dz;
                float wx = 1.f, wy = 1.f, wz = 1.f;
                if (AW) wx = ex2_fast(qx * nl2), wy = ex2_fast(qy * nl2), wz = ex2_fast(qz * nl2);
                const float q = fmaf(wx, qx, fmaf(wy, qy, fmaf(wz, qz, eps)));
                const float it = q > 0.f ? rsqrt_fast(q) : 0.f;
                if (AW) wx *= fmaf(-qx, id2, 1.f), wy *= fmaf(-qy, id2, 1.f), wz *= fmaf(-qz, id2, 1.f);
                fx = dx * wx * it, fy = dy * wy * it, fz = dz * wz * it;
                T = q * it;
            }
        }
        const float fxn = __shfl_down_sync(0xffffffffu, fx, 1);      // a_x(p + e_x); lane 31 is halo, never an owner
        say[buf][ty][tx] = fy;
        __syncthreads();
        const float fyn = ty + 1 < TV_BY ? say[buf][ty + 1][tx] : 0.f;   // a_y(p + e_y)
        buf ^= 1;
        if (owner) {
            if (z > zs && pg) {                 // the previous plane is complete now: its a_z(p + e_z) is this fz
                const float v = Sprev - fz;
                pg[-(ptrdiff_t)plane] = v;
                gacc = fmaf(v, v, gacc);
            }
            if (z < ze) vacc += T;
        }
        if (((z - zs) & 15) == 15) val += (double)vacc, gg += (double)gacc, vacc = 0.f, gacc = 0.f;
        Sprev = fx + fy + fz - fxn - fyn;
        xprev = c;
        px += plane;
        if (pg) pg += plane;
    }
    val += (double)vacc, gg += (double)gacc;
    if (d_val) {
        val = block_sum512(val, red);
        if (tx == 0 && ty == 0) atomicAdd(d_val, val);
        __syncthreads();
    }
    if (d_gg && g) {
        gg = block_sum512(gg, red);
        if (tx == 0 && ty == 0) atomicAdd(d_gg, gg);
    }
}

// The same streaming walk with FOUR voxels along x per thread (rows of nx % 4 == 0 floats, 16-byte aligned): the scalar
// kernel above spends ~100 thread-instructions per voxel on addresses, predicates, the barrier and the exchange, which
// makes it issue-bound at a quarter of the HBM rate; here one float4 load / store / shared-memory exchange and one
// shuffle serve four voxels, a_x(p + e_x) of three of them is the thread's own register, and the domain tests are a
// per-voxel threshold under the rsqrt (thr = 0 on the summation domain, +inf outside: it = 0 there).
// CTA = 32 x 16 threads = 31 x 4 columns by 15 rows of owned voxels (last lane / row are halo).
constexpr int V4_BY = 12;
constexpr int V4_PF = 4;
#ifndef V4_UNROLL
#define V4_UNROLL 1
#endif
constexpr int V4_UNR = V4_UNROLL;

template <bool AW>
__device__ __forceinline__ void tv_voxel(float dx, float dy, float dz, float thr, float nl2, float id2, float eps, float& fx,
                                         float& fy, float& fz, float& T) {
    const float qx = dx * dx, qy = dy * dy, qz = dz * dz;
    float wx = 1.f, wy = 1.f, wz = 1.f;
    if (AW) wx = ex2_fast(qx * nl2), wy = ex2_fast(qy * nl2), wz = ex2_fast(qz * nl2);
    const float q = AW ? fmaf(wx, qx, fmaf(wy, qy, fmaf(wz, qz, eps))) : fmaf(dx, dx, fmaf(dy, dy, fmaf(dz, dz, eps)));
    const float it = q > thr ? rsqrt_fast(q) : 0.f;
    if (AW) wx *= fmaf(-qx, id2, 1.f), wy *= fmaf(-qy, id2, 1.f), wz *= fmaf(-qz, id2, 1.f);
    if (AW) fx = dx * wx * it, fy = dy * wy * it, fz = dz * wz * it;
    else fx = dx * it, fy = dy * it, fz = dz * it;
    T = q * it;
}

__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }

template <bool AW>
__global__ void __launch_bounds__(32 * V4_BY, 2)
tv_gradient_v4_kernel(const float* __restrict__ x, int nx, int ny, int nz, float nl2, float id2, float eps,
                      float* __restrict__ g, double* __restrict__ d_val, double* __restrict__ d_gg) {
    __shared__ float4 say[2][V4_BY][32];
    __shared__ double red[16];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int gx = blockIdx.x * (31 * 4) + tx * 4, gy = blockIdx.y * (V4_BY - 1) + ty;
    const int zs = blockIdx.z * TV_ZCHUNK, ze = min(zs + TV_ZCHUNK, nz);
    const bool inside = gx < nx && gy < ny;
    const bool owner = inside && tx < 31 && ty < V4_BY - 1;
    const float inf = __int_as_float(0x7f800000);
    const float thr_a = (inside && gy >= 1 && gx >= 1) ? 0.f : inf;   // voxel 0 of the four
    const float thr_b = (inside && gy >= 1) ? 0.f : inf;              // voxels 1..3
    const bool ldy = inside && gy >= 1, ldl = inside && tx == 0 && gx >= 1;
    const size_t plane = (size_t)nx * ny;
    const size_t idx = ((size_t)zs * ny + gy) * nx + gx;
    const float* px = x + idx;
    float* pg = g ? g + idx : nullptr;
    const int zlast = min(ze, nz - 1);        // last plane this CTA reads
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    float4 xprev = (inside && zs >= 1) ? ld4(px - plane) : zero4;
    float4 cq[V4_PF];
#pragma unroll
    for (int i = 0; i < V4_PF; ++i) cq[i] = (inside && zs + i <= zlast) ? ld4(px + (size_t)i * plane) : zero4;
    float4 uq = (ldy && zs <= zlast) ? ld4(px - nx) : zero4;          // row above, this plane
    float lq = (ldl && zs <= zlast) ? __ldg(px - 1) : 0.f;            // left neighbour of lane 0's first voxel
    float4 Sprev = zero4;
    float vacc = 0.f, gacc = 0.f;
    double val = 0.0, gg = 0.0;
    int buf = 0;
#pragma unroll(V4_UNR)
    for (int z = zs; z <= ze; ++z) {
        const float4 c = cq[0], u = uq;
        const float lft = lq;
#pragma unroll
        for (int i = 0; i + 1 < V4_PF; ++i) cq[i] = cq[i + 1];
        cq[V4_PF - 1] = (inside && z + V4_PF <= zlast) ? ld4(px + (size_t)V4_PF * plane) : zero4;
        uq = (ldy && z + 1 <= zlast) ? ld4(px + plane - nx) : zero4;
        lq = (ldl && z + 1 <= zlast) ? __ldg(px + plane - 1) : 0.f;
        const bool zin = z >= 1 && z < nz;
        const float ta = zin ? thr_a : inf, tb = zin ? thr_b : inf;
        float l = __shfl_up_sync(0xffffffffu, c.w, 1);
        if (tx == 0) l = lft;
        float4 fx, fy, fz, T;
        tv_voxel<AW>(c.x - l, c.x - u.x, c.x - xprev.x, ta, nl2, id2, eps, fx.x, fy.x, fz.x, T.x);
        tv_voxel<AW>(c.y - c.x, c.y - u.y, c.y - xprev.y, tb, nl2, id2, eps, fx.y, fy.y, fz.y, T.y);
        tv_voxel<AW>(c.z - c.y, c.z - u.z, c.z - xprev.z, tb, nl2, id2, eps, fx.z, fy.z, fz.z, T.z);
        tv_voxel<AW>(c.w - c.z, c.w - u.w, c.w - xprev.w, tb, nl2, id2, eps, fx.w, fy.w, fz.w, T.w);
        const float fxr = __shfl_down_sync(0xffffffffu, fx.x, 1);     // a_x of the next lane's first voxel
        say[buf][ty][tx] = fy;
        __syncthreads();
        const float4 fyn = ty + 1 < V4_BY ? say[buf][ty + 1][tx] : zero4;
        buf ^= 1;
        if (owner) {
            if (z > zs && pg) {
                float4 v;
                v.x = Sprev.x - fz.x, v.y = Sprev.y - fz.y, v.z = Sprev.z - fz.z, v.w = Sprev.w - fz.w;
                *reinterpret_cast<float4*>(pg - plane) = v;
                gacc = fmaf(v.x, v.x, fmaf(v.y, v.y, fmaf(v.z, v.z, fmaf(v.w, v.w, gacc))));
            }
            if (z < ze) vacc += (T.x + T.y) + (T.z + T.w);
        }
        if (((z - zs) & 15) == 15) val += (double)vacc, gg += (double)gacc, vacc = 0.f, gacc = 0.f;
        Sprev.x = fx.x + fy.x + fz.x - fx.y - fyn.x;
        Sprev.y = fx.y + fy.y + fz.y - fx.z - fyn.y;
        Sprev.z = fx.z + fy.z + fz.z - fx.w - fyn.z;
        Sprev.w = fx.w + fy.w + fz.w - fxr - fyn.w;
        xprev = c;
        px += plane;
        if (pg) pg += plane;
    }
    val += (double)vacc, gg += (double)gacc;
    if (d_val) {
        val = block_sum512(val, red);
        if (tx == 0 && ty == 0) atomicAdd(d_val, val);
        __syncthreads();
    }
    if (d_gg && g) {
        gg = block_sum512(gg, red);
        if (tx == 0 && ty == 0) atomicAdd(d_gg, gg);
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

bool g_tv_scalar = false;   // test hook (tigre_set_tv_path): force the one-voxel-per-thread kernel

// value and/or gradient of AwTV (delta <= 0 or infinite: TV).  g, d_val, d_gg may each be NULL; the two
// accumulators must be zeroed by the caller.
int launch_tv_gradient(const float* x, int nx, int ny, int nz, float delta, float eps, float* g, double* d_val, double* d_gg,
                       cudaStream_t st) {
    if (nx <= 0 || ny <= 0 || nz <= 0) return TIGRE_ERR_ARG;
    dim3 block(TV_BX, TV_BY), grid((nx + TV_BX - 2) / (TV_BX - 1), (ny + TV_BY - 2) / (TV_BY - 1), (nz + TV_ZCHUNK - 1) / TV_ZCHUNK);
    if (grid.y > 65535 || grid.z > 65535) return TIGRE_ERR_ARG;
    ProfScope ps(PK_EW, st);
    const bool aw = delta > 0.f && std::isfinite(delta);
    const bool vec4 = (nx & 3) == 0 && ny > 1 && nz > 1 && !(reinterpret_cast<uintptr_t>(x) & 15) &&
                      !(reinterpret_cast<uintptr_t>(g) & 15) && !g_tv_scalar;
    if (vec4) {
        dim3 b4(32, V4_BY), g4((nx + 123) / 124, (ny + V4_BY - 2) / (V4_BY - 1), grid.z);
        if (g4.y > 65535) return TIGRE_ERR_ARG;
        const float id2 = aw ? 1.0f / (delta * delta) : 0.f;
        if (aw) tv_gradient_v4_kernel<true><<<g4, b4, 0, st>>>(x, nx, ny, nz, -1.4426950408889634f * id2, id2, eps, g, d_val, d_gg);
        else tv_gradient_v4_kernel<false><<<g4, b4, 0, st>>>(x, nx, ny, nz, 0.f, 0.f, eps, g, d_val, d_gg);
    } else if (aw) {
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

extern "C" int tigre_set_tv_path(int path) {
    if (path < 0 || path > 1) return TIGRE_ERR_ARG;
    tg::g_tv_scalar = path == 1;
    return TIGRE_OK;
}
