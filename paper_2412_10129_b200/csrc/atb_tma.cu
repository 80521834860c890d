// atb_tma.cu — voxel-driven backprojection with the detector footprints staged into shared memory by
// TMA (BASELINE.json north_star: "each batch's detector footprint is staged into shared memory by TMA,
// and accumulation stays in registers"; DESIGN.md O-C for what is computed).
//
// A CTA owns a tile of 32 x 12 x 32 voxels: 4 x 3 consumer warps, each 8 (x) x 4 (y) columns of voxels, every
// thread the 32 voxels along z of one column, their sums in registers over all views (thin slabs: 4 x 4 warps,
// 16 voxels along z).  One extra PRODUCER
// warp walks the views ahead of the consumers: for each view it projects the 8 corner voxels of the tile (the
// projective map is quasi-linear, so they bound the footprint), and issues ONE cp.async.bulk.tensor load of
// the BU x BV pixel box around it into a ring of shared-memory stages (mbarrier full/empty pairs), together
// with the view's table entry.  TMA zero-fills whatever lies outside the detector, which IS the zero border
// of the bilinear interpolation, so the consumers read their four taps from shared memory with no bounds
// checks.  A view whose footprint does not fit the box (extreme magnification / tilt) is flagged and its
// taps are gathered through L1/L2 instead.
//
// Views whose detector columns are parallel to the volume's z axis (every circular-orbit view without
// detector tilt: rowU.z = rowW.z = rowG.z = 0) take a cheaper inner loop: the magnification, the
// column pair, its fraction and the u-part of the weight are constant along the thread's z-run.
#include <cuda.h>
#include <cmath>
#include <cstdlib>
#include <mutex>
#include <type_traits>
#include "atb_common.cuh"
#include "tma.cuh"

namespace tg {

namespace {

constexpr int TMA_STAGES_MAX = 8;

struct StageInfo {   // written by the producer before it arms the stage's full barrier
    int c0, c1;      // absolute detector index of the box origin (u, v)
    int fits;
    int lin;         // tilted view: over this tile's z-runs 1/W is linear and the weight quadratic in k to 2e-7 (see the general branch)
    float4 rU, rV, rW, rG, cst;   // the view's table entry: consumers read it here (shared-memory latency, broadcast)
};

}  // namespace

extern int g_atb_path;   // atb.cu
int* g_atb_box_meta = nullptr;   // tigre_Atb_boxes (api.cu): host int[8] to fill, and the device buffer for the boxes
int32_t* g_atb_boxes = nullptr;

// BU (box width, pixels) is a template parameter so that the second tap row is an immediate offset; the
// launcher picks the smallest of 48, 80, ... 240 (all = 16 mod 32: with the 8 x 4 lane layout below, the taps
// of one warp span < 16 columns of at most a few adjacent rows, and rows 16 banks apart do not collide).
// FUSE: the OS-SART update in the epilogue (AtbP::fuse).  A template flag, not a branch on p.fuse: the branch alone cost the plain
// kernel's tilted-view loop 4 % (C4 999 -> 962 GUPS: a different register allocation in the loops above it).
template <int MODE, int WX, int WY, int ZR, int BU, bool FUSE = false>
__global__ void __launch_bounds__(32 * (WX * WY + 1), 2)
atb_tma_kernel(const __grid_constant__ CUtensorMap tmap, const float* __restrict__ proj, const VoxView* __restrict__ views,
               int nViews, AtbP p, int BV, int nStages, float* __restrict__ vol, int4* __restrict__ boxes) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int stageElems = (BU * BV + 31) & ~31;   // 128-byte multiple
    float* tiles = reinterpret_cast<float*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(tiles + (size_t)nStages * stageElems);
    uint64_t* empty = full + TMA_STAGES_MAX;
    StageInfo* info = reinterpret_cast<StageInfo*>(empty + TMA_STAGES_MAX);

    constexpr int BX = 8 * WX, BY = 4 * WY, NW = WX * WY;   // tile = WX x WY consumer warps of 8 x 4 voxel columns
    const int lane = threadIdx.x, warp = threadIdx.y;
    const int x0 = blockIdx.x * BX, y0 = blockIdx.y * BY, zb = blockIdx.z * ZR;   // zb relative to p.z0
    if (lane == 0 && warp == 0) {
        for (int s = 0; s < nStages; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, NW);
        }
        mbar_fence_init();
    }
    __syncthreads();

    if (warp == NW) {
        // ------------------------------------------------------------ producer warp
        const int c = lane & 7;   // corner of the tile's box of voxel centres
        const float cxf = (float)(x0 + ((c & 1) ? BX - 1 : 0)) - p.cx;
        const float cyf = (float)(y0 + ((c & 2) ? BY - 1 : 0)) - p.cy;
        const float czf = (float)(p.z0 + zb + ((c & 4) ? ZR - 1 : 0)) - p.cz;
        int s = 0;
        uint32_t ph = 1;   // parity of the "stage is free" phase the producer waits for (first pass: free by construction)
        for (int a = 0; a < nViews; ++a) {
            const float4* vp = reinterpret_cast<const float4*>(views + a);
            const float4 rU = __ldg(vp), rV = __ldg(vp + 1), rW = __ldg(vp + 2), rG = __ldg(vp + 3), cst = __ldg(vp + 4);
            const float U = fmaf(rU.x, cxf, fmaf(rU.y, cyf, fmaf(rU.z, czf, rU.w)));
            const float V = fmaf(rV.x, cxf, fmaf(rV.y, cyf, fmaf(rV.z, czf, rV.w)));
            const float W = fmaf(rW.x, cxf, fmaf(rW.y, cyf, fmaf(rW.z, czf, rW.w)));
            const float t = rcp_fast(W);
            float ulo = U * t, vlo = V * t, uhi = ulo, vhi = vlo;
            // smallest depth of the tile's corners (W, and the FDK weight's G): what the bounds of the general branch divide by
            float dmin = MODE == TIGRE_ATB_FDK ? fminf(W, fmaf(rG.x, cxf, fmaf(rG.y, cyf, fmaf(rG.z, czf, rG.w)))) : W;
#pragma unroll
            for (int o = 4; o > 0; o >>= 1) {
                ulo = fminf(ulo, __shfl_xor_sync(0xffffffffu, ulo, o)), uhi = fmaxf(uhi, __shfl_xor_sync(0xffffffffu, uhi, o));
                vlo = fminf(vlo, __shfl_xor_sync(0xffffffffu, vlo, o)), vhi = fmaxf(vhi, __shfl_xor_sync(0xffffffffu, vhi, o));
                dmin = fminf(dmin, __shfl_xor_sync(0xffffffffu, dmin, o));
            }
            if (lane == 0) {
                // box origin one pixel below the smallest tap; taps reach floor(max)+1, one more of slack for
                // the consumers' own rounding: extent floor(max) - floor(min) + 4 must fit
                const bool finite = fabsf(ulo) < 1.0e6f && fabsf(uhi) < 1.0e6f && fabsf(vlo) < 1.0e6f && fabsf(vhi) < 1.0e6f;
                int fits = 0, c0 = 0, c1 = 0;
                if (finite) {
                    // TMA wants the box to start on a 16-byte boundary of the row: round u down to a multiple of 4
                    const int u0 = (((int)floorf(ulo) - 1 + p.hu) & ~3) - p.hu, v0 = (int)floorf(vlo) - 1;
                    fits = ((int)floorf(uhi) + 3 - u0 <= BU) && ((int)floorf(vhi) + 3 - v0 <= BV);
                    c0 = u0 + p.hu, c1 = v0 + p.hv;
                }
                if (a >= nStages) mbar_wait(empty + s, ph);
                info[s].c0 = c0, info[s].c1 = c1, info[s].fits = fits;
                {
                    // General (tilted) views: along a z-run of ZR voxels W(k) = W0 + k rW.z and the matched weight is km N(k) / W(k)^3 with
                    // N = |(sx W, du Eu, dv Ev)| the norm of a vector linear in k (slope b, |b|^2 = qC below); FDK: 1 / G(k)^2.  With
                    // rho = max(|rW.z| / Wmin, |b| / (sx Wmin), |rG.z| / Gmin) the third logarithmic derivative of the weight is below
                    // 60 rho^3, so the quadratic through its values at k = 0, h, 2h (h = (ZR-1)/2) is off by < 0.064 * 60 (rho h)^3, and
                    // 1/W expanded to first order about the middle of the run by (|rW.z| h / W)^2.  Both below 2e-7 / 1e-8: the consumers
                    // take one reciprocal and three exact weights per run instead of a reciprocal and a square root per voxel.
                    const float dEu = fmaf(-cst.z, rW.z, rU.z), dEv = fmaf(-cst.w, rW.z, rV.z);
                    const float b2 = MODE == TIGRE_ATB_FDK ? 0.f : fmaf(p.du2 * dEu, dEu, fmaf(p.dv2 * dEv, dEv, cst.y * rW.z * rW.z));
                    const float h = 0.5f * (float)(ZR - 1), inv = dmin > 0.f ? 1.0f / dmin : 3.0e38f;
                    const float rhoW = fabsf(rW.z) * inv;
                    const float rho = fmaxf(fmaxf(rhoW, fabsf(rG.z) * inv), MODE == TIGRE_ATB_FDK ? 0.f : sqrtf(b2 / fmaxf(cst.y, 1e-30f)) * inv);
                    const float e = rho * h, eW = rhoW * h;
                    // z-aligned views (the branch below with one reciprocal per run): the matched weight is wk sqrt(q(k)) = wk |a + b k| with
                    // |b| = dv |rV.z| t and |a + b k| >= sx; the third derivative of such a norm N is below 1.155 |b|^3 / N^2, so the quadratic
                    // through sqrt(q) at k = 0, h, 2h is off by < 0.064 * 1.155 (rhoZ h)^3 relative (bit 1 of the flag)
                    const float rhoZ = MODE == TIGRE_ATB_FDK ? 0.f : sqrtf(p.dv2 / fmaxf(cst.y, 1e-30f)) * fabsf(rV.z) * inv;
                    const float eZ = rhoZ * h;
                    info[s].lin = ((3.84f * e * e * e < 2.0e-7f && eW * eW < 1.0e-8f) ? 1 : 0) | ((0.074f * eZ * eZ * eZ < 1.0e-7f) ? 2 : 0);
                }
                if (boxes)   // tigre_Atb_boxes (reading P19(b)): the staged box of this (tile, view), absolute detector indices
                    boxes[((size_t)(blockIdx.z * gridDim.y + blockIdx.y) * gridDim.x + blockIdx.x) * nViews + a] = make_int4(c0, c1, fits, 0);
                info[s].rU = rU, info[s].rV = rV, info[s].rW = rW, info[s].rG = rG, info[s].cst = cst;
                if (fits) {
                    mbar_arrive_expect_tx(full + s, (uint32_t)(BU * BV * sizeof(float)));
                    tma_load_3d(tiles + (size_t)s * stageElems, &tmap, c0, c1 - p.row0, a, full + s);
                } else {
                    mbar_arrive(full + s);
                }
            }
            __syncwarp();
            if (++s == nStages) s = 0, ph ^= 1;
        }
        return;
    }

    // ---------------------------------------------------------------- consumer warps
    // a warp owns 8 (x) x 4 (y) columns of voxels: a compact detector footprint (few shared-memory bank
    // conflicts) and still 32-byte store segments
    const int ix = x0 + (warp % WX) * 8 + (lane & 7), iy = y0 + (warp / WX) * 4 + (lane >> 3);
    const bool active = ix < p.nx && iy < p.ny;
    const float cxf = (float)ix - p.cx, cyf = (float)iy - p.cy, czf = (float)(p.z0 + zb) - p.cz;
    float acc[ZR];
#pragma unroll
    for (int k = 0; k < ZR; ++k) acc[k] = 0.f;
    const size_t per = (size_t)p.nu * p.nrows;
    const uint32_t tiles_s = smem_u32(tiles);
    int s = 0;
    uint32_t ph = 0;
    for (int a = 0; a < nViews; ++a) {
        mbar_wait(full + s, ph);
        const int c0 = info[s].c0, c1 = info[s].c1, fits = info[s].fits;
        const float4 rU = info[s].rU, rV = info[s].rV, rW = info[s].rW, cst = info[s].cst;
        // the depth row G only enters the FDK weight
        const float4 rG = MODE == TIGRE_ATB_FDK ? info[s].rG : make_float4(0.f, 0.f, 0.f, 1.f);
        const float U0 = fmaf(rU.x, cxf, fmaf(rU.y, cyf, fmaf(rU.z, czf, rU.w)));
        const float V0 = fmaf(rV.x, cxf, fmaf(rV.y, cyf, fmaf(rV.z, czf, rV.w)));
        const float W0 = fmaf(rW.x, cxf, fmaf(rW.y, cyf, fmaf(rW.z, czf, rW.w)));
        const float G0 = fmaf(rG.x, cxf, fmaf(rG.y, cyf, fmaf(rG.z, czf, rG.w)));
        if (!fits) {
            // footprint larger than the staged box: gather this view through L1/L2 (bounds-checked, clamped)
            if (active) {
                const float* pa = proj + (size_t)a * per;
#pragma unroll
                for (int k = 0; k < ZR; ++k) {
                    const float kf = (float)k;
                    const TapW tw = voxel_view<MODE, true>(fmaf(kf, rU.z, U0), fmaf(kf, rV.z, V0), fmaf(kf, rW.z, W0),
                                                           fmaf(kf, rG.z, G0), cst, p);
                    acc[k] = fmaf(tw.w, bilinear_global(pa, tw.iu, tw.iv, tw.au, tw.av, p), acc[k]);
                }
            }
        } else if (!active) {
            // voxels outside the volume (ragged tile): nothing to add, but the warp still releases the stage
        } else if (rU.z == 0.f && rW.z == 0.f && rG.z == 0.f) {
            // detector columns parallel to z: per view and thread, one reciprocal, one column pair; the weight
            // w = wk * sqrt(q(k)) with q quadratic in k (matched) or w = wk (FDK); wk is folded into the
            // u-interpolation weights
            const float t = rcp_fast(W0);
            const float fu = U0 * t;
            int iu;
            const float flu = floor_magic(fu, iu);
            const float au = fu - flu;
            const float fv0 = V0 * t, dfv = rV.z * t;
            float wk, qA = 0.f, qB = 0.f, qC = 0.f;
            if (MODE == TIGRE_ATB_FDK) {
                const float ig = rcp_fast(G0);
                wk = ig * ig;
            } else {
                const float eu = fu - cst.z, ev0 = fv0 - cst.w;
                wk = (cst.x * t) * t;
                qA = fmaf(p.dv2 * ev0, ev0, fmaf(p.du2 * eu, eu, cst.y));
                qB = 2.f * p.dv2 * ev0 * dfv, qC = p.dv2 * dfv * dfv;
            }
            // where the producer's bound holds the square root itself is replaced by the quadratic through its values at k = 0, h, 2h
            // (three MUFU.SQRT per run instead of one per voxel; the Horner form below then yields sqrt(q) directly)
            const bool surrogate = MODE != TIGRE_ATB_FDK && (info[s].lin & 2) && p.lin_ok;
            if (surrogate) {
                constexpr float H = 0.5f * (float)(ZR - 1);
                const float s0 = sqrt_fast(qA), s1 = sqrt_fast(fmaf(fmaf(qC, H, qB), H, qA)), s2 = sqrt_fast(fmaf(fmaf(qC, 2.f * H, qB), 2.f * H, qA));
                qA = s0;
                qC = ((s2 - s1) - (s1 - s0)) * (0.5f / (H * H));
                qB = fmaf(-qC, H, (s1 - s0) * (1.0f / H));
            }
            const float wa = wk * (1.f - au), wb = wk * au;
            // byte address (shared window) of the tap column in row 0 of the stage, minus the magic-number
            // bias of floor_magic times the row pitch (mod 2^32): the row address is then ONE integer
            // multiply-add of the raw bits of (fv - 1/2) + 1.5*2^23
            uint32_t col = tiles_s + (uint32_t)(s * stageElems + (iu + p.hu - c0) + (p.hv - c1) * BU) * 4u -
                           (uint32_t)p.magic * (uint32_t)(BU * 4);   // p.magic = 0x4B400000, opaque to the compiler
                                                                      // (as a literal it is re-added before every load)
            asm volatile("" : "+r"(col));   // ... and so is the sum: nvcc factors it back into (bits - magic) * pitch, an IADD3 per update
            // (the loop is instantiated twice so that the choice is a branch around it, not a predicated MUFU in it)
            auto zrun = [&](auto sur_tag) {
            constexpr bool SUR = decltype(sur_tag)::value;
#pragma unroll
            for (int k = 0; k < ZR; ++k) {
                const float fv = fmaf((float)k, dfv, fv0);
                // row index and fraction: FRND.FLOOR on the conversion pipe (idle since the square root left this loop) and two adds; the
                // magic-number floor of atb_common.cuh takes four adds on the FMA / ALU pipes (C3 1210 -> 1230 GUPS, C2 FDK 1112 -> 1140)
                const float fl = floorf(fv);
                const float av = fv - fl;
                const float tm = fl + 12582912.0f;   // exact: the integer in the low mantissa bits
                const uint32_t q = col + __float_as_uint(tm) * (uint32_t)(BU * 4);
                float p00, p10, p01, p11;
                asm volatile(
                    "ld.shared.f32 %0, [%4];\n\t"
                    "ld.shared.f32 %1, [%4+4];\n\t"
                    "ld.shared.f32 %2, [%4+%5];\n\t"
                    "ld.shared.f32 %3, [%4+%6];"
                    : "=f"(p00), "=f"(p10), "=f"(p01), "=f"(p11)
                    : "r"(q), "n"(BU * 4), "n"(BU * 4 + 4));
                const float r0 = fmaf(p10, wb, p00 * wa), r1 = fmaf(p11, wb, p01 * wa);
                const float val = fmaf(av, r1 - r0, r0);
                if (MODE == TIGRE_ATB_FDK) {
                    acc[k] += val;
                } else {
                    const float kf = (float)k;
                    const float qk = fmaf(fmaf(qC, kf, qB), kf, qA);
                    acc[k] = fmaf(SUR ? qk : sqrt_fast(qk), val, acc[k]);
                }
            }
            };
            if (surrogate) zrun(std::true_type{});
            else zrun(std::false_type{});
        } else if ((info[s].lin & 1) && p.lin_ok) {
            // general view whose z-runs are short against the depth (the producer's bound): 1/W to first order about the middle of
            // the run (one reciprocal, Newton-refined), the weight as the quadratic through its exact values at k = 0, h, 2h
            constexpr float H = 0.5f * (float)(ZR - 1);
            const float Wm = fmaf(H, rW.z, W0);
            float tm_ = rcp_fast(Wm);
            tm_ = tm_ * fmaf(-Wm, tm_, 2.0f);
            const float dt = -rW.z * tm_ * tm_, t0 = fmaf(-H, dt, tm_);
            float wq0, wq1, wq2;
            {
                float qA = 0.f, qB = 0.f, qC = 0.f;
                if (MODE != TIGRE_ATB_FDK) {
                    const float Eu = fmaf(-cst.z, W0, U0), Ev = fmaf(-cst.w, W0, V0);
                    const float dEu = fmaf(-cst.z, rW.z, rU.z), dEv = fmaf(-cst.w, rW.z, rV.z);
                    const float sW = cst.y * W0, sdW = cst.y * rW.z;
                    qA = fmaf(p.du2 * Eu, Eu, fmaf(p.dv2 * Ev, Ev, sW * W0));
                    qB = 2.f * fmaf(p.du2 * Eu, dEu, fmaf(p.dv2 * Ev, dEv, sW * rW.z));
                    qC = fmaf(p.du2 * dEu, dEu, fmaf(p.dv2 * dEv, dEv, sdW * rW.z));
                }
                float wn[3];
#pragma unroll
                for (int n = 0; n < 3; ++n) {
                    const float kf = H * (float)n;
                    if (MODE == TIGRE_ATB_FDK) {
                        const float ig = rcp_fast(fmaf(kf, rG.z, G0));
                        wn[n] = ig * ig;
                    } else {
                        const float t = rcp_fast(fmaf(kf, rW.z, W0));
                        wn[n] = ((cst.x * t) * (t * t)) * sqrt_fast(fmaf(fmaf(qC, kf, qB), kf, qA));
                    }
                }
                wq0 = wn[0];
                wq2 = ((wn[2] - wn[1]) - (wn[1] - wn[0])) * (0.5f / (H * H));
                wq1 = fmaf(-wq2, H, (wn[1] - wn[0]) * (1.0f / H));
            }
            const float Uh = fmaf(-0.5f, W0, U0), Vh = fmaf(-0.5f, W0, V0);
            const float dUh = fmaf(-0.5f, rW.z, rU.z), dVh = fmaf(-0.5f, rW.z, rV.z);
            const uint32_t col = tiles_s + (uint32_t)(s * stageElems + (p.hu - c0) + (p.hv - c1) * BU) * 4u -
                                 (uint32_t)p.magic * (uint32_t)(BU * 4 + 4);
#pragma unroll
            for (int k = 0; k < ZR; ++k) {
                const float kf = (float)k;
                const float t = fmaf(kf, dt, t0);
                const float Uk = fmaf(kf, dUh, Uh), Vk = fmaf(kf, dVh, Vh);
                const float tmu = fmaf(Uk, t, 12582912.0f), tmv = fmaf(Vk, t, 12582912.0f);
                const float au = fmaf(Uk, t, 0.5f - (tmu - 12582912.0f)), av = fmaf(Vk, t, 0.5f - (tmv - 12582912.0f));
                const uint32_t q = col + __float_as_uint(tmv) * (uint32_t)(BU * 4) + __float_as_uint(tmu) * 4u;
                float p00, p10, p01, p11;
                asm volatile(
                    "ld.shared.f32 %0, [%4];\n\t"
                    "ld.shared.f32 %1, [%4+4];\n\t"
                    "ld.shared.f32 %2, [%4+%5];\n\t"
                    "ld.shared.f32 %3, [%4+%6];"
                    : "=f"(p00), "=f"(p10), "=f"(p01), "=f"(p11)
                    : "r"(q), "n"(BU * 4), "n"(BU * 4 + 4));
                const float r0 = fmaf(au, p10 - p00, p00), r1 = fmaf(au, p11 - p01, p01);
                const float val = fmaf(av, r1 - r0, r0);
                acc[k] = fmaf(fmaf(fmaf(wq2, kf, wq1), kf, wq0), val, acc[k]);
            }
        } else {
            // general view (tilted detector): U, V, W all vary along the z-run, so each voxel has its own reciprocal.
            // (1) the -1/2 of floor_magic is folded into the rows: fu - 1/2 = (U - W/2) t, so round(fu - 1/2) + magic is ONE
            //     FFMA, and au = (U - W/2) t + (1/2 - round) another;
            // (2) both tap indices enter the address as the raw bits of those sums (two integer multiply-adds; the biases
            //     are folded into `col` as in the branch above);
            // (3) matched weight: eu = fu - fus = Eu t with Eu = U - fus W linear in k, so
            //     sx2 + du^2 eu^2 + dv^2 ev^2 = t^2 Q(k), Q = sx2 W^2 + du^2 Eu^2 + dv^2 Ev^2 quadratic in k (Horner), w = km t^3 sqrt(Q).
            const float Uh = fmaf(-0.5f, W0, U0), Vh = fmaf(-0.5f, W0, V0);
            const float dUh = fmaf(-0.5f, rW.z, rU.z), dVh = fmaf(-0.5f, rW.z, rV.z);
            float qA = 0.f, qB = 0.f, qC = 0.f;
            if (MODE != TIGRE_ATB_FDK) {
                const float Eu = fmaf(-cst.z, W0, U0), Ev = fmaf(-cst.w, W0, V0);
                const float dEu = fmaf(-cst.z, rW.z, rU.z), dEv = fmaf(-cst.w, rW.z, rV.z);
                const float sW = cst.y * W0, sdW = cst.y * rW.z;
                qA = fmaf(p.du2 * Eu, Eu, fmaf(p.dv2 * Ev, Ev, sW * W0));
                qB = 2.f * fmaf(p.du2 * Eu, dEu, fmaf(p.dv2 * Ev, dEv, sW * rW.z));
                qC = fmaf(p.du2 * dEu, dEu, fmaf(p.dv2 * dEv, dEv, sdW * rW.z));
            }
            const uint32_t col = tiles_s + (uint32_t)(s * stageElems + (p.hu - c0) + (p.hv - c1) * BU) * 4u -
                                 (uint32_t)p.magic * (uint32_t)(BU * 4 + 4);
#pragma unroll
            for (int k = 0; k < ZR; ++k) {
                const float kf = (float)k;
                const float t = rcp_fast(fmaf(kf, rW.z, W0));
                const float Uk = fmaf(kf, dUh, Uh), Vk = fmaf(kf, dVh, Vh);
                const float tmu = fmaf(Uk, t, 12582912.0f), tmv = fmaf(Vk, t, 12582912.0f);
                const float au = fmaf(Uk, t, 0.5f - (tmu - 12582912.0f)), av = fmaf(Vk, t, 0.5f - (tmv - 12582912.0f));
                const uint32_t q = col + __float_as_uint(tmv) * (uint32_t)(BU * 4) + __float_as_uint(tmu) * 4u;
                float p00, p10, p01, p11;
                asm volatile(
                    "ld.shared.f32 %0, [%4];\n\t"
                    "ld.shared.f32 %1, [%4+4];\n\t"
                    "ld.shared.f32 %2, [%4+%5];\n\t"
                    "ld.shared.f32 %3, [%4+%6];"
                    : "=f"(p00), "=f"(p10), "=f"(p01), "=f"(p11)
                    : "r"(q), "n"(BU * 4), "n"(BU * 4 + 4));
                const float r0 = fmaf(au, p10 - p00, p00), r1 = fmaf(au, p11 - p01, p01);
                const float val = fmaf(av, r1 - r0, r0);
                float w;
                if (MODE == TIGRE_ATB_FDK) {
                    const float ig = rcp_fast(fmaf(kf, rG.z, G0));
                    w = ig * ig;
                } else {
                    w = ((cst.x * t) * (t * t)) * sqrt_fast(fmaf(fmaf(qC, kf, qB), kf, qA));
                }
                acc[k] = fmaf(w, val, acc[k]);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + s);
        if (++s == nStages) s = 0, ph ^= 1;
    }
    if (active) {
        const size_t slice = (size_t)p.nx * p.ny;
#pragma unroll
        for (int k = 0; k < ZR; ++k) {
            if (zb + k < p.nzs) {
                const size_t i = (size_t)(zb + k) * slice + (size_t)iy * p.nx + ix;
                if (FUSE) {   // F2: the same arithmetic as update_t_kernel, on the accumulator instead of a stored gradient
                    float v = fmaf(p.lambda * (p.V ? __ldg(p.V + i) : 1.f), acc[k], vol[i]);
                    if (p.nonneg) v = fmaxf(v, 0.f);
                    vol[i] = v;
                    p.xT[(size_t)(zb + k) * slice + (size_t)ix * p.ny + iy] = v;
                } else {
                    vol[i] = p.accumulate ? vol[i] + acc[k] : acc[k];
                }
            }
        }
    }
}

// ------------------------------------------------------------------------------------------ host side
namespace {

typedef TensorMapEncodeTiledFn EncodeTiledFn;
inline EncodeTiledFn encode_fn() { return tensor_map_encoder(); }

// footprint extent (pixels) of the tile of voxel centres [x0,x0+bx-1] x [y0,..] x [z0,..] in one view
void tile_extent(const VoxView& v, double cx, double cy, double cz, int x0, int y0, int z0, int bx, int by, int bz, double& eu,
                 double& ev) {
    double ulo = 1e300, uhi = -1e300, vlo = 1e300, vhi = -1e300;
    for (int c = 0; c < 8; ++c) {
        const double x = x0 + ((c & 1) ? bx - 1 : 0) - cx, y = y0 + ((c & 2) ? by - 1 : 0) - cy, z = z0 + ((c & 4) ? bz - 1 : 0) - cz;
        const double W = v.rowW[0] * x + v.rowW[1] * y + v.rowW[2] * z + v.rowW[3];
        const double U = v.rowU[0] * x + v.rowU[1] * y + v.rowU[2] * z + v.rowU[3];
        const double V = v.rowV[0] * x + v.rowV[1] * y + v.rowV[2] * z + v.rowV[3];
        if (!(W > 1e-12)) {
            eu = ev = 1e9;
            return;
        }
        ulo = std::fmin(ulo, U / W), uhi = std::fmax(uhi, U / W), vlo = std::fmin(vlo, V / W), vhi = std::fmax(vhi, V / W);
    }
    eu = uhi - ulo, ev = vhi - vlo;
}

struct TmaArgs {
    CUtensorMap map;
    const float* proj;
    const VoxView* d_views;
    int nViews, BV, nStages;
    AtbP p;
    float* vol;
    cudaStream_t st;
};

template <int MODE, int WX, int WY, int ZR, int BU>
int tma_launch(const TmaArgs& A) {
    const size_t stageElems = ((size_t)BU * A.BV + 31) & ~(size_t)31;
    const size_t smem = A.nStages * stageElems * sizeof(float) + 2 * TMA_STAGES_MAX * sizeof(uint64_t) + TMA_STAGES_MAX * sizeof(StageInfo);
    auto kern = A.p.fuse ? atb_tma_kernel<MODE, WX, WY, ZR, BU, true> : atb_tma_kernel<MODE, WX, WY, ZR, BU, false>;
    TG_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 block(32, WX * WY + 1), grid((A.p.nx + 8 * WX - 1) / (8 * WX), (A.p.ny + 4 * WY - 1) / (4 * WY), (A.p.nzs + ZR - 1) / ZR);
    if (grid.y > 65535 || grid.z > 65535) return TIGRE_ERR_ARG;
    int4* boxes = nullptr;
    if (g_atb_box_meta) {   // tigre_Atb_boxes: report the tiling; write the boxes if the caller's buffer is there
        int* m = g_atb_box_meta;
        m[0] = 8 * WX, m[1] = 4 * WY, m[2] = ZR, m[3] = BU, m[4] = A.BV, m[5] = (int)grid.x, m[6] = (int)grid.y, m[7] = (int)grid.z;
        boxes = reinterpret_cast<int4*>(g_atb_boxes);
        if (!boxes) return TIGRE_OK;   // size query only
    }
    kern<<<grid, block, smem, A.st>>>(A.map, A.proj, A.d_views, A.nViews, A.p, A.BV, A.nStages, A.vol, boxes);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}
template <int MODE, int WX, int WY, int ZR>
int tma_launch_bu(int BU, const TmaArgs& A) {
    switch (BU) {
        case 48: return tma_launch<MODE, WX, WY, ZR, 48>(A);
        case 80: return tma_launch<MODE, WX, WY, ZR, 80>(A);
        case 112: return tma_launch<MODE, WX, WY, ZR, 112>(A);
        case 144: return tma_launch<MODE, WX, WY, ZR, 144>(A);
        case 176: return tma_launch<MODE, WX, WY, ZR, 176>(A);
        case 240: return tma_launch<MODE, WX, WY, ZR, 240>(A);
    }
    return 1;
}

// one tile configuration: sizes the staged box from the geometry, encodes the tensor map, launches
template <int WX, int WY, int ZR>
int tma_config(EncodeTiledFn enc, const float* proj, const Grid& g, const VoxView* d_views, const VoxView* h_views, int nViews,
               int mode, const AtbP& p, float* vol, cudaStream_t st) {
    constexpr int BX = 8 * WX, BY = 4 * WY;
    if (g.nx < BX || g.ny < BY || nViews < 2) return 1;   // not worth staging
    // box size: the largest footprint of a tile over a sample of tile positions (corner, edge and centre tiles of
    // the slab) and all views; tiles that still do not fit fall back per view inside the kernel
    const double cx = 0.5 * (g.nx - 1), cy = 0.5 * (g.ny - 1), cz = 0.5 * (g.nz - 1);
    double eu = 0, ev = 0;
    const int xs[3] = {0, std::max(0, (g.nx / 2 / BX) * BX), std::max(0, ((g.nx - 1) / BX) * BX)};
    const int ys[3] = {0, std::max(0, (g.ny / 2 / BY) * BY), std::max(0, ((g.ny - 1) / BY) * BY)};
    const int zs[3] = {p.z0, p.z0 + std::max(0, (p.nzs / 2 / ZR) * ZR), p.z0 + std::max(0, ((p.nzs - 1) / ZR) * ZR)};
    for (int a = 0; a < nViews; ++a)
        for (int i = 0; i < 27; ++i) {
            double e1, e2;
            tile_extent(h_views[a], cx, cy, cz, xs[i % 3], ys[(i / 3) % 3], zs[i / 9], BX, BY, ZR, e1, e2);
            eu = std::fmax(eu, e1), ev = std::fmax(ev, e2);
        }
    if (!(eu < 240.0) || !(ev < 240.0)) return 1;
    if (g_atb_path == 2) eu *= 0.45, ev *= 0.7;   // test hook: most views no longer fit and take the in-kernel fallback
    const int need = (int)std::ceil(eu) + 5 + 3;   // +3: 16-byte aligned origin
    TmaArgs A;
    A.BV = (int)std::ceil(ev) + 5;
    int BU = 0;
    for (int c : {48, 80, 112, 144, 176, 240})
        if (c >= need) {
            BU = c;
            break;
        }
    if (!BU || A.BV > 256) return 1;
    const size_t stageB = (((size_t)BU * A.BV + 31) & ~(size_t)31) * sizeof(float);
    int nStages = TMA_STAGES_MAX;
    while (nStages > 2 && nStages * stageB > 100 * 1024) --nStages;
    if (nStages * stageB > 200 * 1024) return 1;
    A.nStages = std::min(nStages, std::max(2, nViews));
    const cuuint64_t gdim[3] = {(cuuint64_t)g.nu, (cuuint64_t)p.nrows, (cuuint64_t)nViews};
    const cuuint64_t gstr[2] = {(cuuint64_t)g.nu * sizeof(float), (cuuint64_t)g.nu * p.nrows * sizeof(float)};
    const cuuint32_t box[3] = {(cuuint32_t)BU, (cuuint32_t)A.BV, 1};
    const cuuint32_t estr[3] = {1, 1, 1};
    if (enc(&A.map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(proj), gdim, gstr, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) != CUDA_SUCCESS)
        return 1;
    A.proj = proj, A.d_views = d_views, A.nViews = nViews, A.p = p, A.vol = vol, A.st = st;
    if (mode == TIGRE_ATB_FDK) return tma_launch_bu<TIGRE_ATB_FDK, WX, WY, ZR>(BU, A);
    return tma_launch_bu<TIGRE_ATB_MATCHED, WX, WY, ZR>(BU, A);
}

}  // namespace

// Returns TIGRE_OK if the TMA kernel was launched, 1 if this problem does not qualify (caller falls back to the
// gather kernel), a negative status on a CUDA error.
int launch_atb_tma(const float* proj, const Grid& g, const VoxView* d_views, const VoxView* h_views, int nViews, int mode,
                   const AtbP& p, float* vol, cudaStream_t st) {
    EncodeTiledFn enc = encode_fn();
    if (!enc || !h_views || !proj) return 1;
    if ((g.nu & 3) || (reinterpret_cast<uintptr_t>(proj) & 15) || p.nrows < 1) return 1;   // TMA: 16-byte rows and base
    // tile = 4 x 3 consumer warps of 8 x 4 voxel columns, 32 voxels along z per thread (32 x 12 x 32 voxels per CTA, 13 warps,
    // 2 CTAs per SM): the per-view work of a thread (table entry, projective map of its column, weights, barrier round trip) is
    // spread over 32 voxels instead of 16.  Measured on C3 / C2 / C4 (profiles/r1_atb_tma.md): 1160 / 1204 / 861 GUPS against
    // 950 / 918 / 818 for the former 4 x 4 x 16 tile, which stays for thin slabs: there a 32-voxel run would be mostly empty
    // (chosen when the z-extent rounded up to 32 exceeds 1.2 x the z-extent rounded up to 16).
    const int up32 = (p.nzs + 31) / 32 * 32, up16 = (p.nzs + 15) / 16 * 16;
    if (up32 * 10 <= up16 * 12) {
        const int rc = tma_config<4, 3, 32>(enc, proj, g, d_views, h_views, nViews, mode, p, vol, st);
        if (rc != 1) return rc;   // launched, or a CUDA error; 1 = the taller footprint does not fit a stage: try the flatter tile
    }
    return tma_config<4, 4, 16>(enc, proj, g, d_views, h_views, nViews, mode, p, vol, st);
}

}  // namespace tg
