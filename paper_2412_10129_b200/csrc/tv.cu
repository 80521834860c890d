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
#include <cuda.h>
#include <algorithm>
#include <cmath>
#include <mutex>
#include "common.cuh"
#include "tma.cuh"

namespace tg {

namespace {

constexpr int TV_BX = 32, TV_BY = 16;   // threads per CTA; it owns (BX-1) x (BY-1) columns, the last column / row is halo
#ifndef TVZ
#define TVZ 64
#endif
constexpr int TV_ZCHUNK = TVZ;           // planes per CTA along z
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
        for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
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
    __shared__ double red[32];
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

// The same streaming walk with FOUR voxels along x per thread and the planes of x staged into shared memory by TMA
// (rows of nx % 4 == 0 floats, 16-byte aligned).  History of this kernel on 512^3 (profiles/r1_tv.md): the scalar kernel
// above spends ~100 thread-instructions per voxel on addresses, predicates, the barrier and the exchange (issue-bound,
// 1.7 TB/s); four voxels per thread with register prefetch queues cut that to ~40, but then the walk waits, at every
// plane's barrier, for the slowest load (3.3 TB/s).  Here one elected thread issues ONE cp.async.bulk.tensor per plane:
// the tile's rows with a 4-float apron on both sides and the row above ((TM_BY + 1) x 136 floats; TMA's zero fill is
// the outside of the volume) into a ring of TM_D planes, so TM_D planes per CTA are in flight with no registers held,
// and x[p - e_x], x[p - e_y] are shared-memory reads of the same tile.  Domain tests are a per-voxel threshold under
// the rsqrt (thr = 0 on the summation domain, +inf outside: it = 0 there).
// CTA = TM_BY row warps (a tile of 128 x TM_BY voxels, its last row halo: its a_y feeds the row above) + one edge warp
// (lane r forms a_x of the voxel just right of the tile in row r, which the last lane of that row subtracts; lane 0 is
// also the TMA producer).
#ifndef TMBY
#define TMBY 15
#define TMD 6
#endif
constexpr int TM_BY = TMBY;
constexpr int TM_D = TMD;
constexpr int TM_W = 136;                       // floats per staged row: 4 apron + 128 + 4 apron
constexpr int TM_PLANE = (TM_BY + 1) * TM_W;    // floats per staged plane

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

__device__ __forceinline__ void cta_sync() { asm volatile("bar.sync 0;" ::: "memory"); }   // same barrier from two code paths
__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
static_assert((TM_BY + 1) % 4 == 0, "a staged plane must be a multiple of 128 bytes (TMA destination alignment)");
constexpr size_t TM_SMEM = (size_t)TM_D * TM_PLANE * 4 + 2 * TM_BY * 32 * 16 + 64 * 4 + TM_D * 8;

struct TmRow {   // a row-warp thread's walk state
    float4 xprev, Sprev;
    float* pg;
    float vacc, gacc;
    double val, gg;
};

// One plane of a row-warp thread.  EDGE = false: 1 <= i <= nplanes - 2, i.e. the plane exists (1 <= z < nz, z < ze) and the
// previous plane has been visited: nothing is tested.
template <bool AW, bool EDGE>
__device__ __forceinline__ void tm_plane(TmRow& w, int i, int zs, int ze, int nz, int nreal, int& s, uint32_t& parity, uint64_t* full,
                                         const float* ring, float4* say, const float* sedge, int oc, int ou, int tx, int ty,
                                         float thr_a, float thr_b, bool owner, bool hasg, size_t plane, float nl2, float id2,
                                         float eps) {
    const float inf = __int_as_float(0x7f800000);
    const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
    const int z = zs + i;
    float4 c = zero4, u = zero4;
    float l = 0.f;
    if (!EDGE || i < nreal) {
        mbar_wait(full + s, parity);
        const float* T = ring + s * TM_PLANE;
        c = *reinterpret_cast<const float4*>(T + oc);
        u = *reinterpret_cast<const float4*>(T + ou);
        l = __shfl_up_sync(0xffffffffu, c.w, 1);
        if (tx == 0) l = T[oc - 1];
    }
    float ta = thr_a, tb = thr_b;
    if (EDGE && !(z >= 1 && z < nz)) ta = inf, tb = inf;
    float4 fx, fy, fz, T4;
    tv_voxel<AW>(c.x - l, c.x - u.x, c.x - w.xprev.x, ta, nl2, id2, eps, fx.x, fy.x, fz.x, T4.x);
    tv_voxel<AW>(c.y - c.x, c.y - u.y, c.y - w.xprev.y, tb, nl2, id2, eps, fx.y, fy.y, fz.y, T4.y);
    tv_voxel<AW>(c.z - c.y, c.z - u.z, c.z - w.xprev.z, tb, nl2, id2, eps, fx.z, fy.z, fz.z, T4.z);
    tv_voxel<AW>(c.w - c.z, c.w - u.w, c.w - w.xprev.w, tb, nl2, id2, eps, fx.w, fy.w, fz.w, T4.w);
    float fxr = __shfl_down_sync(0xffffffffu, fx.x, 1);       // a_x of the next lane's first voxel
    float4* sb = say + (i & 1) * (TM_BY * 32);
    sb[ty * 32 + tx] = fy;
    cta_sync();
    float4 fyn = zero4;
    if (ty + 1 < TM_BY) fyn = sb[(ty + 1) * 32 + tx];         // a_y(p + e_y)
    if (tx == 31) fxr = sedge[(i & 1) * 32 + ty];             // the last lane's neighbour is the edge warp's voxel
    if (owner) {
        if ((!EDGE || i > 0) && hasg) {       // the previous plane is complete now: its a_z(p + e_z) is this fz
            float4 v;
            v.x = w.Sprev.x - fz.x, v.y = w.Sprev.y - fz.y, v.z = w.Sprev.z - fz.z, v.w = w.Sprev.w - fz.w;
            *reinterpret_cast<float4*>(w.pg - plane) = v;
            w.gacc = fmaf(v.x, v.x, fmaf(v.y, v.y, fmaf(v.z, v.z, fmaf(v.w, v.w, w.gacc))));
        }
        if (!EDGE || z < ze) w.vacc += (T4.x + T4.y) + (T4.z + T4.w);
    }
    // partial sums in fp32 over 16 planes at a time, then into fp64
    if ((i & 15) == 15) w.val += (double)w.vacc, w.gg += (double)w.gacc, w.vacc = 0.f, w.gacc = 0.f;
    w.Sprev.x = fx.x + fy.x + fz.x - fx.y - fyn.x;
    w.Sprev.y = fx.y + fy.y + fz.y - fx.z - fyn.y;
    w.Sprev.z = fx.z + fy.z + fz.z - fx.w - fyn.z;
    w.Sprev.w = fx.w + fy.w + fz.w - fxr - fyn.w;
    w.xprev = c;
    w.pg += plane;
    if (++s == TM_D) s = 0, parity ^= 1;
}

template <bool AW>
__global__ void __launch_bounds__(32 * (TM_BY + 1), 2)
tv_gradient_tma_kernel(const __grid_constant__ CUtensorMap tmap, const float* __restrict__ x, int nx, int ny, int nz, float nl2,
                       float id2, float eps, float* __restrict__ g, double* __restrict__ d_val, double* __restrict__ d_gg) {
    extern __shared__ __align__(128) unsigned char tv_smem[];
    float* ring = reinterpret_cast<float*>(tv_smem);                 // [TM_D][TM_BY + 1][TM_W]
    float4* say = reinterpret_cast<float4*>(ring + TM_D * TM_PLANE);  // [2][TM_BY][32]   a_y of the plane, for the row above
    float* sedge = reinterpret_cast<float*>(say + 2 * TM_BY * 32);    // [2][32]          a_x right of the tile, per row
    uint64_t* full = reinterpret_cast<uint64_t*>(sedge + 64);         // [TM_D]
    __shared__ double red[32];
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int gx0 = blockIdx.x * 128, gy0 = blockIdx.y * (TM_BY - 1);
    const int zs = blockIdx.z * TV_ZCHUNK, ze = min(zs + TV_ZCHUNK, nz);
    const int nplanes = ze - zs + 1;          // planes zs..ze are visited; plane ze for its a_z only (plane nz does not exist)
    const int nreal = min(ze, nz - 1) - zs + 1;   // planes that are loaded
    const size_t plane = (size_t)nx * ny;
    const float inf = __int_as_float(0x7f800000);
    const bool producer = ty == TM_BY && tx == 0;
    if (producer) {
        for (int s = 0; s < TM_D; ++s) mbar_init(full + s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (producer) {
        for (int i = 0; i < TM_D && i < nreal; ++i) {
            mbar_arrive_expect_tx(full + i, TM_PLANE * 4);
            tma_load_3d(ring + i * TM_PLANE, &tmap, gx0 - 4, gy0 - 1, zs + i, full + i);
        }
    }
    double val = 0.0, gg = 0.0;
    int s = 0;
    uint32_t parity = 0;
    if (ty == TM_BY) {
        // ---- edge warp: one voxel per row and plane, the column right of the tile; lane 0 refills the ring
        const int ex = gx0 + 128, ey = gy0 + tx;
        const bool on = tx < TM_BY && ex < nx && ey < ny && ey >= 1;
        const int rr = min(tx, TM_BY - 1);
        float xprev = zs >= 1 ? __ldg(x + ((size_t)(zs - 1) * ny + min(ey, ny - 1)) * nx + min(ex, nx - 1)) : 0.f;
        for (int i = 0; i < nplanes; ++i) {
            const int z = zs + i;
            float c = 0.f, l = 0.f, u = 0.f;
            if (i < nreal) {
                mbar_wait(full + s, parity);
                const float* T = ring + s * TM_PLANE;
                c = T[(rr + 1) * TM_W + 132], l = T[(rr + 1) * TM_W + 131], u = T[rr * TM_W + 132];
            }
            const float thr = (on && z >= 1 && z < nz) ? 0.f : inf;
            float fx, fy, fz, Tq;
            tv_voxel<AW>(c - l, c - u, c - xprev, thr, nl2, id2, eps, fx, fy, fz, Tq);
            sedge[(i & 1) * 32 + tx] = fx;
            cta_sync();
            // every thread has read plane i: its slot takes plane i + TM_D
            if (producer && i + TM_D < nreal) {
                mbar_arrive_expect_tx(full + s, TM_PLANE * 4);
                tma_load_3d(ring + s * TM_PLANE, &tmap, gx0 - 4, gy0 - 1, z + TM_D, full + s);
            }
            xprev = c;
            if (++s == TM_D) s = 0, parity ^= 1;
        }
    } else {
        const int gx = gx0 + 4 * tx, gy = gy0 + ty;
        const bool inside = gx < nx && gy < ny;
        const bool owner = inside && ty < TM_BY - 1;
        const bool hasg = g != nullptr;
        const float thr_a = (inside && gy >= 1 && gx >= 1) ? 0.f : inf;   // voxel 0 of the four
        const float thr_b = (inside && gy >= 1) ? 0.f : inf;              // voxels 1..3
        // threads outside the volume address a clamped column (never stored to; their terms are switched off by thr)
        const size_t idx = ((size_t)zs * ny + min(gy, ny - 1)) * nx + min(gx, nx - 4);
        const float4 zero4 = make_float4(0.f, 0.f, 0.f, 0.f);
        float4 xprev = zs >= 1 ? ld4(x + idx - plane) : zero4;
        float* pg = g + idx;                  // never dereferenced when g is NULL
        float4 Sprev = zero4;
        float vacc = 0.f, gacc = 0.f;
        const int oc = (ty + 1) * TM_W + 4 + 4 * tx, ou = ty * TM_W + 4 + 4 * tx;
        TmRow w{xprev, Sprev, pg, vacc, gacc, val, gg};
        // first and last plane of the chunk carry the tests (z = 0, z = nz, nothing to write yet, no T to count);
        // the planes between are interior to the volume and run without them
        tm_plane<AW, true>(w, 0, zs, ze, nz, nreal, s, parity, full, ring, say, sedge, oc, ou, tx, ty, thr_a, thr_b, owner, hasg,
                           plane, nl2, id2, eps);
        for (int i = 1; i < nplanes - 1; ++i)
            tm_plane<AW, false>(w, i, zs, ze, nz, nreal, s, parity, full, ring, say, sedge, oc, ou, tx, ty, thr_a, thr_b, owner, hasg,
                                plane, nl2, id2, eps);
        tm_plane<AW, true>(w, nplanes - 1, zs, ze, nz, nreal, s, parity, full, ring, say, sedge, oc, ou, tx, ty, thr_a, thr_b, owner,
                           hasg, plane, nl2, id2, eps);
        vacc = w.vacc, gacc = w.gacc, val = w.val, gg = w.gg;
        val += (double)vacc, gg += (double)gacc;
    }
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

namespace {
typedef TensorMapEncodeTiledFn TvEncodeFn;
inline TvEncodeFn tv_encode_fn() { return tensor_map_encoder(); }
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
    TvEncodeFn enc = tv_encode_fn();
    const bool vec4 = (nx & 3) == 0 && ny > 1 && nz > 1 && !(reinterpret_cast<uintptr_t>(x) & 15) &&
                      !(reinterpret_cast<uintptr_t>(g) & 15) && !g_tv_scalar && enc;
    if (vec4) {
        CUtensorMap map;
        const cuuint64_t gdim[3] = {(cuuint64_t)nx, (cuuint64_t)ny, (cuuint64_t)nz};
        const cuuint64_t gstr[2] = {(cuuint64_t)nx * sizeof(float), (cuuint64_t)nx * ny * sizeof(float)};
        const cuuint32_t box[3] = {(cuuint32_t)TM_W, (cuuint32_t)(TM_BY + 1), 1};
        const cuuint32_t estr[3] = {1, 1, 1};
        if (enc(&map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(x), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
            return TIGRE_ERR_ARG;
        static std::once_flag once;
        std::call_once(once, [] {
            cudaFuncSetAttribute(tv_gradient_tma_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TM_SMEM);
            cudaFuncSetAttribute(tv_gradient_tma_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)TM_SMEM);
        });
        dim3 b4(32, TM_BY + 1), g4((nx + 127) / 128, (ny + TM_BY - 2) / (TM_BY - 1), grid.z);
        if (g4.y > 65535) return TIGRE_ERR_ARG;
        const float id2 = aw ? 1.0f / (delta * delta) : 0.f;
        if (aw) tv_gradient_tma_kernel<true><<<g4, b4, TM_SMEM, st>>>(map, x, nx, ny, nz, -1.4426950408889634f * id2, id2, eps, g, d_val, d_gg);
        else tv_gradient_tma_kernel<false><<<g4, b4, TM_SMEM, st>>>(map, x, nx, ny, nz, 0.f, 0.f, eps, g, d_val, d_gg);
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
