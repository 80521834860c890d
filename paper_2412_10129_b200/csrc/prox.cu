// prox.cu — TV proximal operator for FISTA (readings P24, P25).
//
//   prox(f) = argmin_u 1/2 ||u - f||^2 + lam TV(u)   by the dual projection iteration
//   d = div p - f/lam;   G = grad d;   p <- (p + tau G) / (1 + tau |G|);   u = f - lam div p
// grad = forward differences (zero at the upper border of every axis), div = -grad^T (backward differences of p, p = 0
// outside; p at an upper border never leaves 0, so it needs no special case).
//
// HBM-bound: the dual field p is three volumes (separate arrays: unit-stride along x for each component).  One
// iteration = two passes: `div` reads p (12 B) and f (4 B) and writes d (4 B); `update` reads d (4 B) and p (12 B) and
// writes p (12 B) = 48 B per voxel; the shifted reads (i - 1, i - nx, i - nx*ny, i + ...) are L1 / L2 hits.  The two
// passes cannot be one without recomputing d four times per voxel (the update at i needs d at i and its three
// forward neighbours, each of which needs p at four places).  Four voxels along x per thread when rows are 16-byte
// aligned.
#include <algorithm>
#include <cmath>
#include "common.cuh"

namespace tg {

namespace {

template <int V>
struct Vec;
template <>
struct Vec<1> {
    float v[1];
    __device__ __forceinline__ static Vec ld(const float* p) { return Vec{{__ldg(p)}}; }
    __device__ __forceinline__ void st(float* p) const { *p = v[0]; }
};
template <>
struct Vec<4> {
    float v[4];
    __device__ __forceinline__ static Vec ld(const float* p) {
        const float4 t = __ldg(reinterpret_cast<const float4*>(p));
        return Vec{{t.x, t.y, t.z, t.w}};
    }
    __device__ __forceinline__ void st(float* p) const { *reinterpret_cast<float4*>(p) = make_float4(v[0], v[1], v[2], v[3]); }
};

// thread t handles voxels [V*t, V*t + V) of the flattened volume; rows are multiples of V, so they share iy, iz
__device__ __forceinline__ bool locate(size_t i, int nx, int ny, int& ix, int& iy, int& iz) {
    const size_t row = i / (unsigned)nx;
    ix = (int)(i - row * (unsigned)nx);
    iz = (int)(row / (unsigned)ny);
    iy = (int)(row - (size_t)iz * (unsigned)ny);
    return true;
}

// out = div p - f * s_f      (FINAL = false: d, s_f = 1/lam)
// out = f - lam * div p      (FINAL = true:  u)
template <int V, bool FINAL>
__global__ void __launch_bounds__(256)
prox_div_kernel(const float* __restrict__ px, const float* __restrict__ py, const float* __restrict__ pz,
                const float* __restrict__ f, float s, float* __restrict__ out, int nx, int ny, int nz, size_t nvec) {
    const size_t plane = (size_t)nx * ny;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < nvec; t += (size_t)gridDim.x * blockDim.x) {
        const size_t i = t * V;
        int ix, iy, iz;
        locate(i, nx, ny, ix, iy, iz);
        const Vec<V> a = Vec<V>::ld(px + i), b = Vec<V>::ld(py + i), c = Vec<V>::ld(pz + i), ff = Vec<V>::ld(f + i);
        Vec<V> bm, cm, o;
        if (iy >= 1) bm = Vec<V>::ld(py + i - nx);
        if (iz >= 1) cm = Vec<V>::ld(pz + i - plane);
        float left = ix >= 1 ? __ldg(px + i - 1) : 0.f;
#pragma unroll
        for (int j = 0; j < V; ++j) {
            float dv = a.v[j] - left;
            left = a.v[j];
            dv += b.v[j] - (iy >= 1 ? bm.v[j] : 0.f);
            dv += c.v[j] - (iz >= 1 ? cm.v[j] : 0.f);
            o.v[j] = FINAL ? fmaf(-s, dv, ff.v[j]) : fmaf(-s, ff.v[j], dv);
        }
        o.st(out + i);
    }
}

// p <- (p + tau G) / (1 + tau |G|),  G = forward differences of d
template <int V>
__global__ void __launch_bounds__(256)
prox_update_kernel(float* __restrict__ px, float* __restrict__ py, float* __restrict__ pz, const float* __restrict__ d,
                   float tau, int nx, int ny, int nz, size_t nvec) {
    const size_t plane = (size_t)nx * ny;
    for (size_t t = blockIdx.x * (size_t)blockDim.x + threadIdx.x; t < nvec; t += (size_t)gridDim.x * blockDim.x) {
        const size_t i = t * V;
        int ix, iy, iz;
        locate(i, nx, ny, ix, iy, iz);
        const Vec<V> dc = Vec<V>::ld(d + i);
        Vec<V> dy, dz;
        const bool hy = iy + 1 < ny, hz = iz + 1 < nz;
        if (hy) dy = Vec<V>::ld(d + i + nx);
        if (hz) dz = Vec<V>::ld(d + i + plane);
        const bool hx_last = ix + V < nx;                  // the last voxel of this thread has a right neighbour
        const float right = hx_last ? __ldg(d + i + V) : 0.f;
        Vec<V> a = Vec<V>::ld(px + i), b = Vec<V>::ld(py + i), c = Vec<V>::ld(pz + i);
#pragma unroll
        for (int j = 0; j < V; ++j) {
            const float nxt = j + 1 < V ? dc.v[j + 1 < V ? j + 1 : j] : right;
            const float gx = (j + 1 < V || hx_last) ? nxt - dc.v[j] : 0.f;
            const float gy = hy ? dy.v[j] - dc.v[j] : 0.f;
            const float gz = hz ? dz.v[j] - dc.v[j] : 0.f;
            const float nrm = sqrtf(fmaf(gx, gx, fmaf(gy, gy, gz * gz)));
            const float sc = __fdividef(1.f, fmaf(tau, nrm, 1.f));
            a.v[j] = fmaf(tau, gx, a.v[j]) * sc;
            b.v[j] = fmaf(tau, gy, b.v[j]) * sc;
            c.v[j] = fmaf(tau, gz, c.v[j]) * sc;
        }
        a.st(px + i), b.st(py + i), c.st(pz + i);
    }
}

// FISTA momentum (P25): y = xn + c (xn - x);  x = xn
__global__ void __launch_bounds__(256) momentum_kernel(float* __restrict__ y, float* __restrict__ x, const float* __restrict__ xn,
                                                       float c, size_t n) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        const float a = xn[i];
        y[i] = fmaf(c, a - x[i], a);
        x[i] = a;
    }
}

int blocks_for(size_t n) {
    int dev = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    const size_t want = (n + 255) / 256;
    return (int)std::max<size_t>(1, std::min<size_t>(want, (size_t)sms * 16));
}

bool vec4_ok(int nx, const void* a, const void* b, const void* c, const void* d, const void* e) {
    return (nx & 3) == 0 && (((uintptr_t)a | (uintptr_t)b | (uintptr_t)c | (uintptr_t)d | (uintptr_t)e) & 15) == 0;
}

}  // namespace

// d = div p - f/lam  (final = false)   or   u = f - lam div p  (final = true)
int launch_prox_div(const float* px, const float* py, const float* pz, const float* f, float lam, bool final, float* out, int nx,
                    int ny, int nz, cudaStream_t st) {
    const size_t n = (size_t)nx * ny * nz;
    if (n == 0) return TIGRE_OK;
    ProfScope ps(PK_EW, st);
    const float s = final ? lam : 1.0f / lam;
    if (vec4_ok(nx, px, py, pz, f, out)) {
        if (final) prox_div_kernel<4, true><<<blocks_for(n / 4), 256, 0, st>>>(px, py, pz, f, s, out, nx, ny, nz, n / 4);
        else prox_div_kernel<4, false><<<blocks_for(n / 4), 256, 0, st>>>(px, py, pz, f, s, out, nx, ny, nz, n / 4);
    } else {
        if (final) prox_div_kernel<1, true><<<blocks_for(n), 256, 0, st>>>(px, py, pz, f, s, out, nx, ny, nz, n);
        else prox_div_kernel<1, false><<<blocks_for(n), 256, 0, st>>>(px, py, pz, f, s, out, nx, ny, nz, n);
    }
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

int launch_prox_update(float* px, float* py, float* pz, const float* d, float tau, int nx, int ny, int nz, cudaStream_t st) {
    const size_t n = (size_t)nx * ny * nz;
    if (n == 0) return TIGRE_OK;
    ProfScope ps(PK_EW, st);
    if (vec4_ok(nx, px, py, pz, d, d)) prox_update_kernel<4><<<blocks_for(n / 4), 256, 0, st>>>(px, py, pz, d, tau, nx, ny, nz, n / 4);
    else prox_update_kernel<1><<<blocks_for(n), 256, 0, st>>>(px, py, pz, d, tau, nx, ny, nz, n);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

int launch_momentum(float* y, float* x, const float* xn, float c, size_t n, cudaStream_t st) {
    if (n == 0) return TIGRE_OK;
    ProfScope ps(PK_EW, st);
    momentum_kernel<<<blocks_for(n), 256, 0, st>>>(y, x, xn, c, n);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg
