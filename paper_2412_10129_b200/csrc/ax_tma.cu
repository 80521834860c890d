// ax_tma.cu — the interpolated forward projector (reading P9; BASELINE.json north_star "software fp32 trilinear") with the
// volume staged into shared memory by TMA.
//
// Why: the L1 kernel of ax.cu issues eight scalar gathers per sample and sits at 84 % of the L1 data pipe (22 wavefronts per
// 32 samples on C2: every request touches 2-3 lines, and the two x-taps of a row touch the same lines twice).  Shared memory
// serves a 32-lane gather of neighbouring words in ONE wavefront, and the eight taps of a sample become eight LDS with
// immediate offsets off one address.
//
// How: a CTA owns 32 x 4 detector pixels of one view: four consumer warps (one detector row each) and one producer warp.
// All its rays read ONE layout (the volume, or its (x,y)-transposed copy when the beam runs along x), in which Y is the axis
// the beam runs along.  The beam is cut into WINDOWS of R = 8 rows of Y (absolute, aligned to multiples of R).  For each
// window the producer evaluates the four corner rays of the pixel tile at the window's two bounding rows (ray positions at a
// fixed row are projective-linear in the pixel index, so the corners bound all of them), and issues one
// cp.async.bulk.tensor.3d of the BX x (R + 2) x BZ box that holds every tap of every sample of the tile in that window into
// a ring of stages (mbarrier full / empty pairs).  Each consumer lane takes the INTERIOR samples of its own ray whose row
// falls into the window (the same samples, in the same per-ray order, as the L1 kernel: only the order in which the warp
// visits them differs from ray to ray) and reads its taps from the stage without bounds checks.  A window whose taps do not
// fit the box (the producer says so), CTAs whose rays do not all run the same way along Y, and the few bounds-checked samples
// at the two ends of every ray take the L1 path of ax.cu's kernel, restated here.
//
// The samples themselves (positions, count, order of summation per ray) are those of ax_interp_kernel: same interp_setup().
#include "ax_common.cuh"
#include "tma.cuh"

namespace tg {

namespace {

constexpr int AXT_R = 8;               // sample rows per window
constexpr int AXT_BY = AXT_R + 2;      // staged rows: the window's rows, the upper tap row, and one row on the side the
                                       // conservative window test defers samples to
#ifndef AXT_STAGES_N
#define AXT_STAGES_N 1
#endif
constexpr int AXT_STAGES = AXT_STAGES_N;   // ONE stage per CTA: a second one halves the CTAs per SM (shared memory is what limits them: 2 CTAs =
                                           // 15 % of the warps with two 29 KB stages on C2, 242 against 352 G samples/s); the other CTAs of the SM cover a load's latency
constexpr int AXT_NW = AX_TV;          // consumer warps
#ifndef AXTMB
#define AXTMB 6
#endif

struct AxtStage {
    int bx, by, bz;   // centred index of the box origin (voxel index minus n >> 1, per axis of the layout)
    int fits;
};

// position (centred index coordinates of the layout: X fastest, Y rows) of pixel (iu, iv)'s ray on row plane Y = yc
__host__ __device__ inline void ray_xz_at_row(const RayView& rv, double iu, double iv, bool useT, int hx, int hy, int hz, double yc,
                                              double& x, double& z, double& dY) {
    double S[3], d[3];
    for (int k = 0; k < 3; ++k) {
        S[k] = rv.S[k] + iu * rv.dSU[k] + iv * rv.dSV[k];
        d[k] = rv.P0[k] + iu * rv.dU[k] + iv * rv.dV[k] - S[k];
    }
    const double SX = useT ? S[1] : S[0], SY = useT ? S[0] : S[1], dX = useT ? d[1] : d[0];
    dY = useT ? d[0] : d[1];
    const double t = (dY != 0.0) ? ((yc + 0.5 + hy) - SY) / dY : 0.0;
    x = SX + t * dX - 0.5 - hx;
    z = S[2] + t * d[2] - 0.5 - hz;
}

}  // namespace

template <int BX>
__global__ void __launch_bounds__(32 * (AXT_NW + 1), AXTMB)
ax_interp_tma_kernel(const __grid_constant__ CUtensorMap mapV, const __grid_constant__ CUtensorMap mapT, const float* __restrict__ vol,
                     const float* __restrict__ volT, const RayView* __restrict__ views, int nViews, AxP p, int BZ, uint32_t magic,
                     float* __restrict__ proj) {
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int PLANE = BX * AXT_BY;
    const int stageElems = PLANE * BZ;   // BX * 40 bytes * BZ: a multiple of 128 bytes for BX a multiple of 16
    float* tiles = reinterpret_cast<float*>(smem_raw);
    uint64_t* full = reinterpret_cast<uint64_t*>(tiles + (size_t)AXT_STAGES * stageElems);
    uint64_t* empty = full + AXT_STAGES;
    AxtStage* info = reinterpret_cast<AxtStage*>(empty + AXT_STAGES);
    int* range = reinterpret_cast<int*>(info + AXT_STAGES);   // [0] = lowest window, [1] = highest window of the CTA

    const int lane = threadIdx.x, warp = threadIdx.y;
    // tile decode (u-tile fastest, then view, then v-band: ax_decode's order, kept for the L2)
    long long tb = blockIdx.x;
    const int ut = (int)(tb % p.nUt);
    tb /= p.nUt;
    const int view = (int)(tb % nViews), vt = (int)(tb / nViews);
    const int iu0 = ut * AX_TU, iv0 = p.iv0 + vt * AX_TV;
    const RayView& rv = views[view];
    // the tile's central ray picks the layout and the direction of travel for the whole CTA
    const double cu = fmin((double)iu0 + 15.5, (double)(p.nu - 1)), cv = fmin((double)iv0 + 0.5 * (AX_TV - 1), (double)(p.iv1 - 1));
    bool useT;
    {
        const double dx = rv.P0[0] + cu * rv.dU[0] + cv * rv.dV[0] - (rv.S[0] + cu * rv.dSU[0] + cv * rv.dSV[0]);
        const double dy = rv.P0[1] + cu * rv.dU[1] + cv * rv.dV[1] - (rv.S[1] + cu * rv.dSU[1] + cv * rv.dSV[1]);
        useT = fabs(dx) > fabs(dy);
    }
    const int nX = useT ? p.ny : p.nx, nY = useT ? p.nx : p.ny;
    const int hx = nX >> 1, hy = nY >> 1, hz = p.nz >> 1;
    bool wup;
    {
        double x, z, dY;
        ray_xz_at_row(rv, cu, cv, useT, hx, hy, hz, 0.0, x, z, dY);
        wup = dY > 0.0;
    }
    if (lane == 0 && warp == 0) {
        for (int s = 0; s < AXT_STAGES; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, AXT_NW);
        }
        range[0] = 0x7fffffff, range[1] = (int)0x80000000;
        mbar_fence_init();
    }
    __syncthreads();

    // ---------------------------------------------------------------- per-ray set-up (consumers)
    const bool consumer = warp < AXT_NW;
    const int iu = iu0 + lane, iv = iv0 + warp;
    const bool mine = consumer && iu < p.nu && iv < p.iv1;
    InterpRay r;
    r.x0 = r.y0 = r.z0 = r.sx = r.sy = r.sz = 0.f;
    r.k0 = r.kA = r.kB = r.Kuse = 0;
    r.useT = useT;
    uint32_t cnt = 0;
    if (mine) interp_setup<false, false>(rv, p, iu, iv, useT ? 1 : 0, r, cnt);
    const bool live = r.kB > r.kA;
    const bool steep = fabsf(r.sy) > 0.05f * (fabsf(r.sx) + fabsf(r.sz));
    const bool okdir = !live || (steep && ((r.sy >= 0.f) == wup));
    // rows (array index) of the first and last interior sample; the windows they fall into
    int w0 = 0x7fffffff, w1 = (int)0x80000000;
    if (live) {
        const int ja = (int)floorf(fmaf((float)r.kA + 0.5f, r.sy, r.y0)) + hy, jb = (int)floorf(fmaf((float)r.kB - 0.5f, r.sy, r.y0)) + hy;
        const int jl = min(ja, jb) - 1, jh = max(ja, jb) + 1;   // one row of slack for the rounding of these two positions
        w0 = (jl >= 0 ? jl : jl - (AXT_R - 1)) / AXT_R, w1 = (jh >= 0 ? jh : jh - (AXT_R - 1)) / AXT_R;
    }
    w0 = __reduce_min_sync(0xffffffffu, w0), w1 = __reduce_max_sync(0xffffffffu, w1);
    if (lane == 0 && consumer && w0 <= w1) atomicMin(range, w0), atomicMax(range + 1, w1);
    const int lock = __syncthreads_and(okdir ? 1 : 0);   // (also orders the two atomics before the reads below)
    const int wlo = range[0], whi = range[1];
    const int nWin = (lock && wlo <= whi) ? whi - wlo + 1 : 0;

    if (!consumer) {
        // ------------------------------------------------------------ producer warp
        // lanes 0..3 own the corner rays of the pixel tile
        const double pu = (lane & 1) ? fmin((double)(iu0 + AX_TU - 1), (double)(p.nu - 1)) : (double)iu0;
        const double pv = (lane & 2) ? fmin((double)(iv0 + AX_TV - 1), (double)(p.iv1 - 1)) : (double)iv0;
        const CUtensorMap* map = useT ? &mapT : &mapV;
        int s = 0;
        uint32_t ph = 1;
        for (int i = 0; i < nWin; ++i) {
            const int w = wup ? wlo + i : whi - i;
            // box rows (array index): the window's R rows and the upper tap row, plus one row on the side samples are deferred to
            const int byA = wup ? w * AXT_R - 1 : w * AXT_R;
            double xa, za, xb, zb, dY;
            ray_xz_at_row(rv, pu, pv, useT, hx, hy, hz, (double)(byA - hy), xa, za, dY);
            ray_xz_at_row(rv, pu, pv, useT, hx, hy, hz, (double)(byA + AXT_BY - 1 - hy), xb, zb, dY);
            float xlo = (float)fmin(xa, xb), xhi = (float)fmax(xa, xb), zlo = (float)fmin(za, zb), zhi = (float)fmax(za, zb);
#pragma unroll
            for (int o = 2; o > 0; o >>= 1) {
                xlo = fminf(xlo, __shfl_xor_sync(0xffffffffu, xlo, o)), xhi = fmaxf(xhi, __shfl_xor_sync(0xffffffffu, xhi, o));
                zlo = fminf(zlo, __shfl_xor_sync(0xffffffffu, zlo, o)), zhi = fmaxf(zhi, __shfl_xor_sync(0xffffffffu, zhi, o));
            }
            if (lane == 0) {
                int fits = 0, bx = 0, bz = 0;
                if (fabsf(xlo) < 1.0e6f && fabsf(xhi) < 1.0e6f && fabsf(zlo) < 1.0e6f && fabsf(zhi) < 1.0e6f) {
                    // one voxel of slack below the lowest tap; TMA wants the box to start on a 16-byte boundary of the row
                    bx = (((int)floorf(xlo) - 1 + hx) & ~3) - hx, bz = (int)floorf(zlo) - 1;
                    fits = ((int)floorf(xhi) + 3 - bx <= BX) && ((int)floorf(zhi) + 3 - bz <= BZ);
                }
                if (i >= AXT_STAGES) mbar_wait(empty + s, ph);
                info[s].bx = bx, info[s].by = byA - hy, info[s].bz = bz, info[s].fits = fits;
                if (fits) {
                    mbar_arrive_expect_tx(full + s, (uint32_t)(stageElems * sizeof(float)));
                    tma_load_3d(tiles + (size_t)s * stageElems, map, bx + hx, byA, bz + hz - p.zs0, full + s);
                } else {
                    mbar_arrive(full + s);
                }
            }
            __syncwarp();
            if (++s == AXT_STAGES) s = 0, ph ^= 1;
        }
        return;
    }

    // ---------------------------------------------------------------- consumers
    const size_t out = ((size_t)view * p.nv + iv) * p.nu + iu;
    const float* __restrict__ base = useT ? volT : vol;
    const int pitchY = nX;
    const long long pitchZ = (long long)p.nx * p.ny;
    const float* __restrict__ org = base + ((long long)(hz - p.zs0) * pitchZ + (long long)hy * pitchY + hx);
    float acc = 0.f;
    // L1 path, interior sample (ax.cu's, 64-bit offsets): windows that do not fit, CTAs that are not marched in lockstep
    auto interior_l1 = [&](float t) {
        const float x = fmaf(t, r.sx, r.x0), y = fmaf(t, r.sy, r.y0), z = fmaf(t, r.sz, r.z0);
        const float mx = (x - 0.5f) + 12582912.0f, my = (y - 0.5f) + 12582912.0f, mz = (z - 0.5f) + 12582912.0f;
        const float ax = x - (mx - 12582912.0f), ay = y - (my - 12582912.0f), az = z - (mz - 12582912.0f);
        const int ix = __float_as_int(mx) - 0x4B400000, iy = __float_as_int(my) - 0x4B400000, iz = __float_as_int(mz) - 0x4B400000;
        const float* q = org + ((long long)iz * pitchZ + (long long)iy * pitchY + (long long)ix);
        const float v000 = __ldg(q), v100 = __ldg(q + 1), v010 = __ldg(q + pitchY), v110 = __ldg(q + pitchY + 1);
        const float v001 = __ldg(q + pitchZ), v101 = __ldg(q + pitchZ + 1), v011 = __ldg(q + pitchZ + pitchY), v111 = __ldg(q + pitchZ + pitchY + 1);
        const float c00 = fmaf(ax, v100 - v000, v000), c10 = fmaf(ax, v110 - v010, v010);
        const float c01 = fmaf(ax, v101 - v001, v001), c11 = fmaf(ax, v111 - v011, v011);
        const float c0 = fmaf(ay, c10 - c00, c00), c1 = fmaf(ay, c11 - c01, c01);
        acc += fmaf(az, c1 - c0, c0);
    };
    // bounds-checked sample without branches (the two ends of the ray): an outside tap gets weight zero and a clamped address
    auto edge = [&](int k) {
        const float t = (float)k + 0.5f;
        const float x = fmaf(t, r.sx, r.x0), y = fmaf(t, r.sy, r.y0), z = fmaf(t, r.sz, r.z0);
        const float mx = (x - 0.5f) + 12582912.0f, my = (y - 0.5f) + 12582912.0f, mz = (z - 0.5f) + 12582912.0f;
        const float ax = x - (mx - 12582912.0f), ay = y - (my - 12582912.0f), az = z - (mz - 12582912.0f);
        const int jx = __float_as_int(mx) - 0x4B400000 + hx, jy = __float_as_int(my) - 0x4B400000 + hy,
                  jz = __float_as_int(mz) - 0x4B400000 + hz - p.zs0;
        const unsigned ex = (unsigned)(nX - 1), ey = (unsigned)(nY - 1), ez = (unsigned)(p.zs1 - p.zs0 - 1);
        const bool x0 = (unsigned)jx <= ex, x1 = (unsigned)(jx + 1) <= ex;
        const bool y0 = (unsigned)jy <= ey, y1 = (unsigned)(jy + 1) <= ey;
        const bool z0 = (unsigned)jz <= ez, z1 = (unsigned)(jz + 1) <= ez;
        const float wx0 = x0 ? 1.f - ax : 0.f, wx1 = x1 ? ax : 0.f;
        const float wy0 = y0 ? 1.f - ay : 0.f, wy1 = y1 ? ay : 0.f;
        const float wz0 = z0 ? 1.f - az : 0.f, wz1 = z1 ? az : 0.f;
        const int cx0 = x0 ? jx : 0, cx1 = x1 ? jx + 1 : 0;
        const long long oy0 = (long long)(y0 ? jy : 0) * pitchY, oy1 = (long long)(y1 ? jy + 1 : 0) * pitchY;
        const long long oz0 = (long long)(z0 ? jz : 0) * pitchZ, oz1 = (long long)(z1 ? jz + 1 : 0) * pitchZ;
        const float *r00 = base + (oz0 + oy0), *r10 = base + (oz0 + oy1), *r01 = base + (oz1 + oy0), *r11 = base + (oz1 + oy1);
        const float c00 = fmaf(wx1, __ldg(r00 + cx1), wx0 * __ldg(r00 + cx0)), c10 = fmaf(wx1, __ldg(r10 + cx1), wx0 * __ldg(r10 + cx0));
        const float c01 = fmaf(wx1, __ldg(r01 + cx1), wx0 * __ldg(r01 + cx0)), c11 = fmaf(wx1, __ldg(r11 + cx1), wx0 * __ldg(r11 + cx0));
        const float c0 = fmaf(wy1, c10, wy0 * c00), c1 = fmaf(wy1, c11, wy0 * c01);
        acc += fmaf(wz1, c1, wz0 * c0);
    };

    int k = r.kA;
    if (nWin > 0) {
        // samples of window w: those of the ray's interior whose row lies below the window's far boundary (in the direction of
        // travel) and that earlier windows have not taken.  The test is biased by 4e-3 samples towards "later": a sample within
        // rounding of the boundary goes to the next window, whose box holds one more row on that side.
        const float isy = live ? 1.0f / r.sy : 0.f, cc = live ? fmaf(-r.y0, isy, -0.5f) - 4.0e-3f : 0.f;
        const uint32_t tiles_s = smem_u32(tiles);
        int s = 0;
        uint32_t ph = 0;
        for (int i = 0; i < nWin; ++i) {
            const int w = wup ? wlo + i : whi - i;
            const float Yb = (float)((wup ? (w + 1) * AXT_R : w * AXT_R) - hy);   // far boundary, centred coordinates
            const int kend = live ? (int)fminf(fmaxf(ceilf(fmaf(Yb, isy, cc)), (float)k), (float)r.kB) : k;
            mbar_wait(full + s, ph);
            if (info[s].fits) {
                // smem byte address of tap (0,0,0) of a sample = qb + 4 (bits(mz) PLANE + bits(my) BX + bits(mx)), the biases of
                // the three magic numbers and the box origin folded into qb (mod 2^32)
                const uint32_t qb = tiles_s + 4u * (uint32_t)(s * stageElems) -
                                    4u * (magic * (uint32_t)(PLANE + BX + 1) +   // magic = 0x4B400000, passed as data: as a literal ptxas splits the
                                                                                 // constant and re-adds part of it before every one of the 8 loads
                                          (uint32_t)(info[s].bz * PLANE + info[s].by * BX + info[s].bx));
                float t = (float)k + 0.5f;
                for (; k < kend; ++k, t += 1.f) {
                    const float x = fmaf(t, r.sx, r.x0), y = fmaf(t, r.sy, r.y0), z = fmaf(t, r.sz, r.z0);
                    const float mx = (x - 0.5f) + 12582912.0f, my = (y - 0.5f) + 12582912.0f, mz = (z - 0.5f) + 12582912.0f;
                    const float ax = x - (mx - 12582912.0f), ay = y - (my - 12582912.0f), az = z - (mz - 12582912.0f);
                    const uint32_t q = qb + 4u * (__float_as_uint(mz) * (uint32_t)PLANE + __float_as_uint(my) * (uint32_t)BX + __float_as_uint(mx));
#ifdef AXT_CHECK   // debug build (nvcc -DAXT_CHECK): every tap of every staged sample must lie inside the box the producer loaded
                    {
                        const int cx = __float_as_int(mx) - 0x4B400000 - info[s].bx, cy = __float_as_int(my) - 0x4B400000 - info[s].by,
                                  cz = __float_as_int(mz) - 0x4B400000 - info[s].bz;
                        if (cx < 0 || cx + 1 >= BX || cy < 0 || cy + 1 >= AXT_BY || cz < 0 || cz + 1 >= BZ) __trap();
                    }
#endif
                    float v000, v100, v010, v110, v001, v101, v011, v111;
                    asm volatile(
                        "ld.shared.f32 %0, [%8];\n\t"
                        "ld.shared.f32 %1, [%8+4];\n\t"
                        "ld.shared.f32 %2, [%8+%9];\n\t"
                        "ld.shared.f32 %3, [%8+%10];\n\t"
                        "ld.shared.f32 %4, [%8+%11];\n\t"
                        "ld.shared.f32 %5, [%8+%12];\n\t"
                        "ld.shared.f32 %6, [%8+%13];\n\t"
                        "ld.shared.f32 %7, [%8+%14];"
                        : "=f"(v000), "=f"(v100), "=f"(v010), "=f"(v110), "=f"(v001), "=f"(v101), "=f"(v011), "=f"(v111)
                        : "r"(q), "n"(BX * 4), "n"(BX * 4 + 4), "n"(PLANE * 4), "n"(PLANE * 4 + 4), "n"((PLANE + BX) * 4),
                          "n"((PLANE + BX) * 4 + 4));
                    const float c00 = fmaf(ax, v100 - v000, v000), c10 = fmaf(ax, v110 - v010, v010);
                    const float c01 = fmaf(ax, v101 - v001, v001), c11 = fmaf(ax, v111 - v011, v011);
                    const float c0 = fmaf(ay, c10 - c00, c00), c1 = fmaf(ay, c11 - c01, c01);
                    acc += fmaf(az, c1 - c0, c0);
                }
            } else {
                float t = (float)k + 0.5f;
                for (; k < kend; ++k, t += 1.f) interior_l1(t);
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
            if (++s == AXT_STAGES) s = 0, ph ^= 1;
        }
    }
    // interior samples no window took (CTAs that are not marched in lockstep; none otherwise), then the two ends
    {
        float t = (float)k + 0.5f;
        for (; k < r.kB; ++k, t += 1.f) interior_l1(t);
    }
    for (int q = r.k0; q < r.kA; ++q) edge(q);
    for (int q = r.kB; q < r.Kuse; ++q) edge(q);
    if (mine) {
        const float result = acc * (float)p.delta;
        proj[out] = p.accumulate ? proj[out] + result : result;
    }
}

// ------------------------------------------------------------------------------------------ host side
namespace {

struct AxtArgs {
    CUtensorMap mapV, mapT;
    const float *vol, *volT;
    const RayView* d_views;
    int nViews, BZ;
    AxP p;
    float* proj;
    cudaStream_t st;
};

template <int BX>
int axt_launch(const AxtArgs& A) {
    const size_t smem = (size_t)AXT_STAGES * BX * AXT_BY * A.BZ * sizeof(float) + 2 * AXT_STAGES * sizeof(uint64_t) +
                        AXT_STAGES * sizeof(AxtStage) + 2 * sizeof(int);
    auto kern = ax_interp_tma_kernel<BX>;
    TG_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const long long nblk = (long long)A.p.nUt * A.p.nVt * A.nViews;
    dim3 block(32, AXT_NW + 1), grid((unsigned)nblk);
    kern<<<grid, block, smem, A.st>>>(A.mapV, A.mapT, A.vol, A.volT, A.d_views, A.nViews, A.p, A.BZ, 0x4B400000u, A.proj);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace

int g_ax_interp_path = 0;   // 0 = TMA-staged kernel for narrow beams that qualify, 1 = L1 kernel only, 2 = TMA-staged kernel for wide beams too (tigre_set_ax_path)

// Returns TIGRE_OK if the TMA kernel was launched, 1 if this problem does not qualify (the caller runs the L1 kernel),
// a negative status on a CUDA error.  h_views: host copy of the views' table (sizes the staged box).
int launch_ax_interp_tma(const float* vol, const float* volT, const Grid& g, const RayView* d_views, const RayView* h_views,
                         int nViews, const AxP& p, float* proj, cudaStream_t st) {
    if (g_ax_interp_path == 1 || !h_views || !vol || !volT || !tensor_map_encoder()) return 1;
    const int nzs = p.zs1 - p.zs0;
    if ((g.nx & 3) || (g.ny & 3) || g.nx < 16 || g.ny < 16 || nzs < 2 || nViews < 1) return 1;
    if ((reinterpret_cast<uintptr_t>(vol) & 15) || (reinterpret_cast<uintptr_t>(volT) & 15)) return 1;
    // box size: the largest extent, over a sample of views, tiles and windows, of the four corner rays of a pixel tile
    // between the two bounding rows of a window (what the producer evaluates); windows that still do not fit fall back
    // to the L1 path inside the kernel
    double ex = 0.0, ez = 0.0, ex1 = 0.0;   // ex1: extent along ONE row (how far apart the 32 rays of a warp are)
    const int vstep = std::max(1, nViews / 24);
    for (int a = 0; a < nViews; a += vstep) {
        const RayView& rv = h_views[a];
        for (int ti = 0; ti < 9; ++ti) {
            const int iu0 = std::min((g.nu - 1) / AX_TU, (ti % 3) * ((g.nu / AX_TU) / 2)) * AX_TU;
            const int nvt = (p.iv1 - p.iv0 + AX_TV - 1) / AX_TV;
            const int iv0 = p.iv0 + std::min(nvt - 1, (ti / 3) * (nvt / 2)) * AX_TV;
            const double cu = std::min(iu0 + 15.5, (double)(g.nu - 1)), cv = std::min(iv0 + 1.5, (double)(p.iv1 - 1));
            const double dx = rv.P0[0] + cu * rv.dU[0] + cv * rv.dV[0] - (rv.S[0] + cu * rv.dSU[0] + cv * rv.dSV[0]);
            const double dy = rv.P0[1] + cu * rv.dU[1] + cv * rv.dV[1] - (rv.S[1] + cu * rv.dSU[1] + cv * rv.dSV[1]);
            const bool useT = std::fabs(dx) > std::fabs(dy);
            const int nX = useT ? g.ny : g.nx, nY = useT ? g.nx : g.ny;
            const int hx = nX >> 1, hy = nY >> 1, hz = g.nz >> 1;
            for (int wi = 0; wi < 3; ++wi) {
                const int row = std::min(nY - AXT_BY, wi * (nY / 2));
                double xlo = 1e300, xhi = -1e300, zlo = 1e300, zhi = -1e300, x1lo = 1e300, x1hi = -1e300;
                for (int c = 0; c < 4; ++c) {
                    const double pu = (c & 1) ? std::min(iu0 + AX_TU - 1, g.nu - 1) : iu0;
                    const double pv = (c & 2) ? std::min(iv0 + AX_TV - 1, p.iv1 - 1) : iv0;
                    for (int e = 0; e < 2; ++e) {
                        double x, z, dY;
                        ray_xz_at_row(rv, pu, pv, useT, hx, hy, hz, (double)(row + e * (AXT_BY - 1) - hy), x, z, dY);
                        xlo = std::min(xlo, x), xhi = std::max(xhi, x), zlo = std::min(zlo, z), zhi = std::max(zhi, z);
                        if (e == 0) x1lo = std::min(x1lo, x), x1hi = std::max(x1hi, x);
                    }
                }
                if (std::isfinite(xlo) && std::isfinite(xhi)) ex = std::max(ex, xhi - xlo), ez = std::max(ez, zhi - zlo), ex1 = std::max(ex1, x1hi - x1lo);
            }
        }
    }
    const int needX = (int)std::ceil(ex) + 4 + 3, needZ = (int)std::ceil(ez) + 4;   // taps, slack, 16-byte aligned origin
    // Row pitch and shared-memory banks: the lanes of a warp sit on two adjacent rows of the box.  Where neighbouring rays are
    // about one voxel apart (32 lanes = 32 distinct columns) a pitch of 0 mod 32 keeps lanes of different rows on different
    // banks (16 mod 32 made lanes l and l + 16 collide: 46 % more wavefronts on C2); where two lanes share a column (rays half
    // a voxel apart) it is the other way round.
    const bool wide = ex1 > 27.0;   // (C3-like detectors: up to 24 voxels along an oblique row at the far side of the volume; C2, C4: 32-47)
    // Measured (B200, profiles/r2_ax_interp_tma.md): where the 32 rays of a warp are about a voxel apart (C2, C4: 33-47 voxels
    // along an oblique row) a tap request cannot be served in one shared-memory wavefront either (lanes 32 columns apart
    // share a bank: 17.6 wavefronts per warp-sample against the L1 kernel's 22) and the 54 KB stages leave 4 CTAs per SM:
    // 302 / 365 G samples/s against the L1 kernel's 352 / 381.  Narrow beams (rays half a voxel apart, C3's detector) gain:
    // 510 against 459.  Wide beams therefore keep the L1 kernel unless the hook asks for this one (tigre_set_ax_path(2)).
    if (wide && g_ax_interp_path != 2) return 1;
    int BX = 0;
    for (int c : {48, 64, 80, 96, 112, 128})
        if (c >= needX && ((c % 32 == 0) == wide)) {
            BX = c;
            break;
        }
    if (!BX || needZ > 24) return 1;
    AxtArgs A;
    A.BZ = std::max(4, needZ);
    if ((size_t)AXT_STAGES * BX * AXT_BY * A.BZ * sizeof(float) > 96 * 1024) return 1;
    const cuuint32_t box[3] = {(cuuint32_t)BX, (cuuint32_t)AXT_BY, (cuuint32_t)A.BZ};
    const cuuint64_t dimV[3] = {(cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)nzs};
    const cuuint64_t strV[2] = {(cuuint64_t)g.nx * sizeof(float), (cuuint64_t)g.nx * g.ny * sizeof(float)};
    const cuuint64_t dimT[3] = {(cuuint64_t)g.ny, (cuuint64_t)g.nx, (cuuint64_t)nzs};
    const cuuint64_t strT[2] = {(cuuint64_t)g.ny * sizeof(float), (cuuint64_t)g.nx * g.ny * sizeof(float)};
    if (!encode_f32_map(&A.mapV, vol, 3, dimV, strV, box) || !encode_f32_map(&A.mapT, volT, 3, dimT, strT, box)) return 1;
    A.vol = vol, A.volT = volT, A.d_views = d_views, A.nViews = nViews, A.p = p, A.proj = proj, A.st = st;
    switch (BX) {
        case 48: return axt_launch<48>(A);
        case 64: return axt_launch<64>(A);
        case 80: return axt_launch<80>(A);
        case 96: return axt_launch<96>(A);
        case 112: return axt_launch<112>(A);
        case 128: return axt_launch<128>(A);
    }
    return 1;
}

}  // namespace tg

extern "C" int tigre_set_ax_path(int path) {
    if (path < 0 || path > 2) return TIGRE_ERR_ARG;
    tg::g_ax_interp_path = path;
    return TIGRE_OK;
}
