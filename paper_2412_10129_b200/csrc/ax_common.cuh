// ax_common.cuh — declarations shared by the ray-driven kernels (ax.cu: gathers through L1 / L2; ax_tma.cu: the interpolated
// projector with boxes of the volume staged into shared memory by TMA).
#pragma once
#include <cmath>
#include "common.cuh"

namespace tg {

// Launch configuration, overridable with -D for sweeps (measured on C3 / C2 / C4):
//   AXMB   CTAs per SM of the Siddon kernel: 9 (56 registers); 5-6 / 7 / 8 / 10 / 12 / 16 give 986 / 1093 / 1139 / 1149 / 1130 / 1071
//          against 1165 G samples/s
//          (before the voted groups below); with them 8 / 9 / 10 give 1364 / 1359 / 1337 at AXG 4 and 7 / 8 / 9 give 1327 / 1347 / 1397 at AXG 6
//   AXG    slabs per warp-voted group of the Siddon march (see the kernel): 6; 2 / 3 / 4 / 8 gave 1224 / 1252 / 1293 / 1245 before the
//          second load of a slab was predicated, 4 / 5 / 6 / 7 / 8 give 1359 / 1346 / 1397 / 1342 / 1361 G samples/s with it (C3)
//   AXIMB  CTAs per SM of the interpolated kernel: 8 (64 registers); 9 the same, 10 and 12 spill and lose 9-12 %
//   AXI_ROWS  rows of the volume per lockstep step of the interpolated kernel: 8; 2 / 3 / 4 / 6 / 12 / 16 / 32 give 318 / 323 / 342 / 342 /
//          345 / 347 / 318 against 352 G samples/s on C2 (C3-sized: 405 / 411 / 443 / 452 / 465 / 464 / 455 against 459)
//   AXTV   detector rows per CTA (tile = 32 x AXTV pixels): 4; 1, 2 and 8 lose 0.3-4 % (with the voted groups: 2 rows x 18 CTAs 1390, 8 rows x 4 / 5 CTAs 1331 / 1339 against 1397)
//   AXTU   detector columns per CTA (a multiple of 32; one warp = 32 consecutive pixels of a row): 32 x 4 rows; 64 x 2 / 64 x 4 (4 CTAs) /
//          128 x 1 / 64 x 1 (18 CTAs) give 1347 / 1288 / 1325 / 1328 against 1352 G samples/s (C3, one launch through tigre_Ax):
//          sharing L1 lines between the two warps of a row does not pay (ax.cu only: ax_tma.cu wants 32)
#ifndef AXIMB
#define AXIMB 8
#endif
#ifndef AXMB
#define AXMB 9
#endif
#ifndef AXG
#define AXG 6
#endif

struct AxP {
    int nx, ny, nz, nu, nv;
    float hx, hy, hz;     // voxel pitch, mm
    double hxd, hyd, hzd;
    double delta;         // interpolated step, mm
    int nUt, nVt;         // tiles per view
    int iv0, iv1;         // detector rows computed: [iv0, iv1)
    int zs0, zs1;         // interpolated mode: z-slices present in `vol` (which points at slice zs0)
    int accumulate;
};

#ifndef AXTV
#define AXTV 4
#endif
#ifndef AXTU
#define AXTU 32
#endif
constexpr int AX_TU = AXTU, AX_TV = AXTV;   // AX_TU: a multiple of 32 (a warp is 32 consecutive pixels of one detector row)
constexpr int AXI_ROWS = 8;

// a[i] += v without a return value, on GLOBAL memory, said so explicitly: through a generic pointer (the scatter kernels pick
// vol or volT at run time) atomicAdd compiles to a generic ATOM with a shared-memory CAS fall-back path behind a branch
// (ncu: 24 long-scoreboard stall cycles per issue, issue slots 29 % busy on C3) instead of one RED.E.ADD.F32
__device__ __forceinline__ void red_add_global(float* a, float v) {
    asm volatile("red.global.add.f32 [%0], %1;" ::"l"(__cvta_generic_to_global(a)), "f"(v) : "memory");
}

__device__ __forceinline__ double sel3(int k, double a, double b, double c) { return k == 0 ? a : (k == 1 ? b : c); }

// tile order: u-tile fastest, then view, then v-band slowest: all views of one detector-row band
// run together, so the z-slab of the volume they gather from stays resident in L2.
__device__ __forceinline__ bool ax_decode(const AxP& p, int nViews, int& view, int& iu, int& iv) {
    long long t = blockIdx.x;
    int ut = (int)(t % p.nUt);
    t /= p.nUt;
    view = (int)(t % nViews);
    int vt = (int)(t / nViews);
    iu = ut * AX_TU + threadIdx.x;
    iv = p.iv0 + vt * AX_TV + threadIdx.y;
    return iu < p.nu && iv < p.iv1;
}


// ------------------------------------------------------------------------------------------
// Interpolated mode.  Per-ray state produced by the fp64 set-up; all coordinates are centre-index
// coordinates relative to the volume centre, c = (xi - 1/2) - n/2, in the (possibly swapped) axes X, Y, z.
struct InterpRay {
    float x0, y0, z0, sx, sy, sz;   // position at l_in and step per sample
    int k0, kA, kB, Kuse;           // samples [k0,Kuse); [kA,kB) need no bounds checks
    bool useT;
};

// The fp64 per-ray set-up of the interpolated projector (reading P9): entry point, step, sample ranges.  forceT: -1 = each ray
// picks the layout it runs across (x-dominant rays read the transposed copy), 0 / 1 = the caller's choice for all rays
// (the TMA kernel stages ONE layout per CTA).  cnt = K of reading P9 (the metric's sample count).
template <bool UNIT, bool COUNT>
__device__ __forceinline__ void interp_setup(const RayView& rv, const AxP& p, int iu, int iv, int forceT, InterpRay& r, uint32_t& cnt) {
    // fp64 set-up in voxel-index coordinates (voxel centres at integer + 1/2)
    double S[3], d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        S[k] = rv.S[k] + iu * rv.dSU[k] + iv * rv.dSV[k];   // parallel beam: every ray has its own start (P29)
        d[k] = rv.P0[k] + iu * rv.dU[k] + iv * rv.dV[k] - S[k];
    }
    const double h[3] = {p.hxd, p.hyd, p.hzd};
    const int n[3] = {p.nx, p.ny, p.nz};
    const double Lmm = sqrt(d[0] * h[0] * d[0] * h[0] + d[1] * h[1] * d[1] * h[1] + d[2] * h[2] * d[2] * h[2]);
    cnt = 0;
    r.x0 = r.y0 = r.z0 = r.sx = r.sy = r.sz = 0.f;
    r.k0 = r.kA = r.kB = r.Kuse = 0;
    // Rays that run mostly along x read the (x,y)-transposed copy of the volume with the roles of x and y
    // swapped (trilinear interpolation is symmetric under the swap): neighbouring lanes, which then differ
    // mostly in y, touch neighbouring addresses.
    r.useT = UNIT ? false : (forceT < 0 ? fabs(d[0]) > fabs(d[1]) : forceT != 0);
    const int nX = r.useT ? p.ny : p.nx, nY = r.useT ? p.nx : p.ny;
    const int hx = nX >> 1, hy = nY >> 1, hz = p.nz >> 1;
    if (Lmm > 0.0) {
        // slab clip against B+ = box grown by half a voxel, in mm along the ray
        double lin = 0.0, lout = Lmm;
        bool miss = false;
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            const double w = d[k] / Lmm;      // index units per mm
            if (w != 0.0) {
                const double t1 = (-0.5 - S[k]) / w, t2 = ((double)n[k] + 0.5 - S[k]) / w;
                lin = fmax(lin, fmin(t1, t2)), lout = fmin(lout, fmax(t1, t2));
            } else if (S[k] < -0.5 || S[k] > (double)n[k] + 0.5) miss = true;
        }
        if (!miss && lout > lin) {
            const long long K = (long long)ceil((lout - lin) / p.delta);
            cnt = (uint32_t)K;
            if (!COUNT) {
                const int X = r.useT ? 1 : 0, Y = r.useT ? 0 : 1;
                const double dX = sel3(X, d[0], d[1], d[2]), dY = sel3(Y, d[0], d[1], d[2]);
                const double SX = sel3(X, S[0], S[1], S[2]), SY = sel3(Y, S[0], S[1], S[2]);
                r.x0 = (float)(SX + lin * dX / Lmm - 0.5 - hx);
                r.y0 = (float)(SY + lin * dY / Lmm - 0.5 - hy);
                r.z0 = (float)(S[2] + lin * d[2] / Lmm - 0.5 - hz);
                r.sx = (float)(p.delta * dX / Lmm), r.sy = (float)(p.delta * dY / Lmm), r.sz = (float)(p.delta * d[2] / Lmm);
                // samples beyond the detector end of the segment are dropped (l_k > |p-S|)
                const long long Kmax = (long long)floor((Lmm - lin) / p.delta - 0.5) + 1;
                r.Kuse = (int)min(K, max(Kmax, 0LL));
                if (p.zs0 > 0 || p.zs1 < p.nz) {
                    // only a z-slab of the volume is present: skip the samples none of whose taps can lie in
                    // it (conservative by one sample and 0.01 voxel; taps are bounds-checked anyway)
                    const float za = (float)(p.zs0 - hz) - 1.01f, zb = (float)(p.zs1 - hz) + 0.01f;
                    if (fabsf(r.sz) > 1e-9f) {
                        const float ka = (za - r.z0) / r.sz - 0.5f, kb = (zb - r.z0) / r.sz - 0.5f;
                        const float klo = fminf(fmaxf(fminf(ka, kb), -1.f), (float)r.Kuse + 1.f);
                        const float khi = fminf(fmaxf(fmaxf(ka, kb), -1.f), (float)r.Kuse + 1.f);
                        r.k0 = max((int)floorf(klo) - 1, 0);
                        r.Kuse = min((int)ceilf(khi) + 2, r.Kuse);
                    } else if (r.z0 < za - 1.f || r.z0 > zb + 1.f) {
                        r.Kuse = 0;
                    }
                    r.k0 = min(r.k0, r.Kuse);
                }
                // interior samples [kA, kB): all eight taps inside the (slab of the) volume with 0.01 voxel and
                // one sample to spare, so they need no bounds checks
                r.kA = r.kB = r.Kuse;
                if (!UNIT) {
                    float tlo = (float)r.k0, thi = (float)r.Kuse;   // in units of t = k + 1/2
                    const float lo3[3] = {(float)(-hx) + 0.01f, (float)(-hy) + 0.01f, (float)(p.zs0 - hz) + 0.01f};
                    const float hi3[3] = {(float)(nX - 1 - hx) - 0.01f, (float)(nY - 1 - hy) - 0.01f, (float)(p.zs1 - 1 - hz) - 0.01f};
                    const float c3[3] = {r.x0, r.y0, r.z0}, s3[3] = {r.sx, r.sy, r.sz};
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        if (fabsf(s3[q]) > 1e-7f) {
                            const float t1 = (lo3[q] - c3[q]) / s3[q], t2 = (hi3[q] - c3[q]) / s3[q];
                            tlo = fmaxf(tlo, fminf(t1, t2)), thi = fminf(thi, fmaxf(t1, t2));
                        } else if (c3[q] < lo3[q] || c3[q] > hi3[q]) {
                            thi = tlo - 4.f;
                        }
                    }
                    r.kA = min(max((int)ceilf(tlo - 0.5f) + 1, r.k0), r.Kuse);
                    r.kB = min(max((int)floorf(thi - 0.5f), r.kA), r.Kuse);
                }
            }
        }
    }
}

}  // namespace tg
