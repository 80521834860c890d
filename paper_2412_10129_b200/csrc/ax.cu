// ax.cu — forward projection b = A x (§2.1 eq. 1), ray-driven, one thread per
// detector pixel.  Two modes (BASELINE.json north_star; DESIGN.md O-A / O-B):
//
//  Siddon (exact intersection lengths).  Instead of the textbook per-ray "next plane" walk, every
//  ray is marched slab by slab along ITS dominant axis D (|d_D| = max): between two consecutive
//  D-planes a ray moves by |m_E|,|m_F| <= 1 voxel along the two other axes, so it crosses at most
//  one E-plane and one F-plane and meets at most three voxels.  The three (length, voxel) pairs
//  of a slab are formed branch-free.  This keeps the 32 lanes of a warp in lock step (same slab
//  index, neighbouring voxels -> few L1 wavefronts per gather) and makes the trip count uniform.
//  The sum of the lengths is exactly the Siddon sum: only the order of summation differs.
//  The lanes of a warp share a detector row, so they cross the z-planes (rarely, and) in nearly the same slabs: the
//  interior runs in warp-uniform groups of AXG slabs, and a group in which no lane crosses a z-plane (one vote) takes
//  a two-voxel slab step with a third fewer instructions and bitwise the same sum.
//  Per-ray set-up (entry/exit, slopes, first slab) is fp64; the march is fp32 with positions
//  recomputed from the integer slab counter (never accumulated) in volume-centred coordinates.
//
//  Interpolated (fixed step, software fp32 trilinear, zero border; reading P9): samples at
//  l_k = l_in + (k+1/2) delta inside the box grown by half a voxel.
#include <cmath>
#include "common.cuh"

#include "ax_siddon.cuh"

namespace tg {


// TRACK (tigre_Ax_index): the march runs as for a gather, without touching the volume, and records per ray the first and
// last voxel it gives a non-zero length to (canonical linear index (iz ny + iy) nx + ix, -1 if none) into track[2 * ray]
// and the number of such voxels into counts[ray]: what reading P19(a) compares with the oracle, from the march itself.
template <typename IdxT, bool UNIT, bool COUNT, bool SCATTER, bool TRACK = false>
__global__ void __launch_bounds__(AX_TU* AX_TV, AXMB)
ax_siddon_kernel(const float* __restrict__ vol, const float* __restrict__ volT, const RayView* __restrict__ views,
                 int nViews, AxP p, float* __restrict__ proj, uint32_t* __restrict__ counts, long long* __restrict__ track = nullptr) {
    int view, iu, iv;
    const bool mine = ax_decode(p, nViews, view, iu, iv);
    // lanes of this warp that own a pixel, taken while all 32 lanes are still here (the mask of every warp vote below)
    const unsigned wmask = __ballot_sync(0xffffffffu, mine);
    if (!mine) return;
    const RayView& rv = views[view];
    const size_t out = ((size_t)view * p.nv + iv) * p.nu + iu;

    // ---- per-ray set-up, fp64: declares the marching state r, base, the slab ranges i0 / nslab / kA / kB, the start cell, ...
#include "ax_siddon_setup.inc"
    if (COUNT) {
        counts[out] = cnt;
        return;
    }
    asm volatile("" : "+l"(base));   // keep the selected pointer in registers (else it is re-selected per slab)
    if (SCATTER) {
        // exact adjoint (vol / volT are the OUTPUTS, proj the input): every length of this ray times its value
        r.ys = proj[out] * scale;
        if (r.ys == 0.f) nslab = 0, kA = 0, kB = 0;
    }
    // ---- the march.  Neighbouring rays enter the volume at different depths; if every lane started its
    // unchecked slabs at its own first one, the warp would be spread over many rows of the volume.  So the head
    // (clipped, bounds-checked slabs) of each lane is stretched to the deepest start in the warp: from there on
    // all lanes are in the SAME absolute slab in every iteration of the interior loop.
    int jmax;
    {
        const bool any = kB > kA;
        jmax = __reduce_max_sync(wmask, any ? i0 + kA : (int)0x80000000);
        if (any) kA = min(max(kA, jmax - i0), kB);
    }
#ifdef AX_PREFETCH
    const IdxT pfo = (IdxT)AXG * r.sD + (IdxT)(int)((float)AXG * 1.5f * fabsf(1.0f / r.imE) + 0.5f) * r.stE;
#endif
    const int last = nslab - 1;
    int k = 0;
    for (; k < kA; ++k)
        siddon_slab_checked<IdxT, UNIT, SCATTER, TRACK>(base, r, ie, jf, diE, diF, nE, nF, k == 0 ? slo0 : 0.f, k == last ? shiN : 1.f);
    const bool ranFast = kB > k;
    {
        // Warp-uniform part of the interior: groups of AXG slabs up to the shallowest end in the warp.  The lanes of a warp share a
        // detector row, so they meet the (rare) z-plane crossings in nearly the same slabs: one vote per group tells whether ANY
        // lane crosses an F-plane in its next AXG slabs (next crossing at hF/mF - k <= AXG slabs ahead; "<=" is conservative under the
        // rounding of that FFMA); if none does, the group runs the two-voxel slab.  All lanes with interior slabs are at absolute
        // slab jmax here.
        const int jendmin = __reduce_min_sync(wmask, ranFast ? i0 + kB : 0x7fffffff);
        const int groups = jendmin == 0x7fffffff ? 0 : (jendmin - jmax) / AXG;
        if (SCATTER) {
            r.fm = __ballot_sync(wmask, ranFast);
            const unsigned tm = __ballot_sync(wmask, base == volT), ln = threadIdx.x & 31u, q = ln ^ 1u;
            r.pok = ((r.fm >> q) & 1u) && ((tm >> q) & 1u) == ((tm >> ln) & 1u);
        }
        for (int g = 0; g < groups; ++g) {
#ifdef AX_PREFETCH
            if (!UNIT && !SCATTER && !TRACK && ranFast) {
                // the rows the next group will read, one L1 prefetch per row (a line holds 32 voxels along E: the drift of the
                // ray over the group is folded into pfo)
                const float* pf = base + (r.off + pfo);
#pragma unroll
                for (int j = 0; j < AXG; ++j) asm volatile("prefetch.global.L1 [%0];" ::"l"(pf + (IdxT)j * r.sD));
            }
#endif
            const bool nearF = ranFast && fmaf(r.hF, r.imF, -r.kf) <= (float)AXG;
            if (__any_sync(wmask, nearF)) {
                if (ranFast) {
#pragma unroll
                    for (int j = 0; j < AXG; ++j) siddon_slab_fast<IdxT, UNIT, SCATTER, TRACK, SCATTER>(base, r);
                }
            } else if (ranFast) {
#pragma unroll
                for (int j = 0; j < AXG; ++j) siddon_slab_e_only<IdxT, UNIT, SCATTER, TRACK, SCATTER>(base, r);
            }
        }
        if (ranFast) k += AXG * groups;
    }
    for (; k < kB; ++k) siddon_slab_fast<IdxT, UNIT, SCATTER, TRACK>(base, r);
    if (k < nslab) {
        // recover the cell indices from the plane state for the checked tail: hE has moved by one per crossing
        if (ranFast) {
            if (r.hE < 1.0e38f) ie = ie0 + (int)rint((double)r.hE - hE0);
            if (r.hF < 1.0e38f) jf = jf0 + (int)rint((double)r.hF - hF0);
        }
        for (; k < nslab; ++k)
            siddon_slab_checked<IdxT, UNIT, SCATTER, TRACK>(base, r, ie, jf, diE, diF, nE, nF, k == 0 ? slo0 : 0.f, k == last ? shiN : 1.f);
    }
    if (TRACK) {
        // offsets are in the layout this ray marched through: bring those of the transposed copy [z][x][y] back to [z][y][x]
        const bool useT = base == volT;
        const long long nxy = (long long)p.nx * p.ny;
        long long fl[2] = {r.first, r.last};
#pragma unroll
        for (int q = 0; q < 2; ++q)
            if (fl[q] >= 0 && useT) {
                const long long z = fl[q] / nxy, rem = fl[q] - z * nxy, x = rem / p.ny, y = rem - x * p.ny;
                fl[q] = z * nxy + y * p.nx + x;
            }
        // the march runs towards increasing D whichever way the ray points: "first" is the voxel nearest the source
        const bool rev = dD < 0.0;
        track[2 * out] = rev ? fl[1] : fl[0], track[2 * out + 1] = rev ? fl[0] : fl[1];
        counts[out] = r.nseg;
        return;
    }
    if (!SCATTER) {
        const float result = r.acc * scale;
        proj[out] = p.accumulate ? proj[out] + result : result;
    }
}

// (x,y) transpose of every z-slice: volT[z][x][y] = vol[z][y][x]
__global__ void __launch_bounds__(256) transpose_xy_kernel(const float* __restrict__ in, float* __restrict__ out, int nx, int ny) {
    __shared__ float tile[32][33];
    const size_t slice = (size_t)nx * ny * blockIdx.z;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int x = x0 + threadIdx.x, y = y0 + j;
        if (x < nx && y < ny) tile[j][threadIdx.x] = in[slice + (size_t)y * nx + x];
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int y = y0 + threadIdx.x, x = x0 + j;
        if (x < nx && y < ny) out[slice + (size_t)x * ny + y] = tile[threadIdx.x][j];
    }
}

template <typename IdxT, bool UNIT, bool COUNT, bool SCATTER>
__global__ void __launch_bounds__(AX_TU* AX_TV, AXIMB)
ax_interp_kernel(const float* __restrict__ vol, const float* __restrict__ volT, const RayView* __restrict__ views, int nViews,
                 AxP p, float* __restrict__ proj, uint32_t* __restrict__ counts) {
    int view, iu, iv;
    const bool mine = ax_decode(p, nViews, view, iu, iv);
    // lanes of this warp that own a pixel, taken while all 32 lanes are still here (the mask of every warp vote below)
    const unsigned wmask = __ballot_sync(0xffffffffu, mine);
    if (!mine) return;
    const RayView& rv = views[view];
    const size_t out = ((size_t)view * p.nv + iv) * p.nu + iu;
    uint32_t cnt = 0;
    InterpRay r;
    interp_setup<UNIT, COUNT>(rv, p, iu, iv, volT != nullptr ? -1 : 0, r, cnt);
    const int nX = r.useT ? p.ny : p.nx, nY = r.useT ? p.nx : p.ny;
    const int hx = nX >> 1, hy = nY >> 1, hz = p.nz >> 1;
    if (COUNT) {
        counts[out] = cnt;
        return;
    }
    const float* __restrict__ base = r.useT ? volT : vol;
    const IdxT pitchY = nX, pitchZ = (IdxT)p.nx * p.ny;
    // address of the voxel with centred index (0,0,0), relative to the first slice present
    const float* __restrict__ org = base + ((IdxT)(hz - p.zs0) * pitchZ + (IdxT)hy * pitchY + hx);
    float acc = 0.f;
    const float ys = SCATTER ? proj[out] * (float)p.delta : 0.f;   // exact adjoint: vol / volT are outputs, proj the input
    if (SCATTER && ys == 0.f) r.k0 = r.kA = r.kB = r.Kuse = 0;
    // bounds-checked sample (entry / exit ends of the ray, and the row-sum variant)
    auto checked = [&](int k) {
        const float t = (float)k + 0.5f;
        const float x = fmaf(t, r.sx, r.x0), y = fmaf(t, r.sy, r.y0), z = fmaf(t, r.sz, r.z0);
        const float fx = floorf(x), fy = floorf(y), fz = floorf(z);
        const float ax = x - fx, ay = y - fy, az = z - fz;
        const int ix = (int)fx + hx, iy = (int)fy + hy, iz = (int)fz + hz;
        float v = 0.f;
        if (UNIT) {
            const float wx = ((unsigned)ix < (unsigned)nX ? 1.f - ax : 0.f) + ((unsigned)(ix + 1) < (unsigned)nX ? ax : 0.f);
            const float wy = ((unsigned)iy < (unsigned)nY ? 1.f - ay : 0.f) + ((unsigned)(iy + 1) < (unsigned)nY ? ay : 0.f);
            const float wz = ((unsigned)(iz - p.zs0) < (unsigned)(p.zs1 - p.zs0) ? 1.f - az : 0.f) +
                             ((unsigned)(iz + 1 - p.zs0) < (unsigned)(p.zs1 - p.zs0) ? az : 0.f);
            v = wx * wy * wz;
        } else {
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                const int jx = ix + (c & 1), jy = iy + ((c >> 1) & 1), jz = iz + (c >> 2);
                if ((unsigned)jx < (unsigned)nX && (unsigned)jy < (unsigned)nY && (unsigned)(jz - p.zs0) < (unsigned)(p.zs1 - p.zs0)) {
                    const float w = ((c & 1) ? ax : 1.f - ax) * ((c & 2) ? ay : 1.f - ay) * ((c & 4) ? az : 1.f - az);
                    const IdxT at = (IdxT)(jz - p.zs0) * pitchZ + (IdxT)jy * pitchY + jx;
                    if (SCATTER) red_add_global(const_cast<float*>(base) + at, w * ys);   // exact adjoint: same weight, added
                    else v = fmaf(w, __ldg(base + at), v);
                }
            }
        }
        acc += v;
    };
    // interior sample: no bounds checks; floor without the conversion pipe (see floor_magic in atb_common.cuh).
    // The element index is formed from the raw bits of (c - 1/2) + 1.5*2^23 (two integer multiply-adds, the
    // bias of the magic number is folded into `bias`), and the four tap rows are four fixed base pointers.
    const float *org0 = org, *orgY = org + pitchY, *orgZ = org + pitchZ, *orgYZ = org + pitchZ + pitchY;
    // keep them four independent 64-bit bases (one IMAD.WIDE per tap row); left to itself the compiler folds
    // them back into one base plus 64-bit index arithmetic with carry chains in the loop
    asm volatile("" : "+l"(org0), "+l"(orgY), "+l"(orgZ), "+l"(orgYZ));
    const uint32_t upY = (uint32_t)pitchY, upZ = (uint32_t)pitchZ, bias = 0x4B400000u * (upZ + upY + 1u);
    auto interior = [&](float t) {
        const float x = fmaf(t, r.sx, r.x0), y = fmaf(t, r.sy, r.y0), z = fmaf(t, r.sz, r.z0);
        const float mx = (x - 0.5f) + 12582912.0f, my = (y - 0.5f) + 12582912.0f, mz = (z - 0.5f) + 12582912.0f;
        const float ax = x - (mx - 12582912.0f), ay = y - (my - 12582912.0f), az = z - (mz - 12582912.0f);
        float v000, v100, v010, v110, v001, v101, v011, v111;
        if (sizeof(IdxT) == 4) {
            const int idx = (int)(__float_as_uint(mz) * upZ + __float_as_uint(my) * upY + __float_as_uint(mx) - bias);
            v000 = __ldg(org0 + idx), v100 = __ldg(org0 + idx + 1);
            v010 = __ldg(orgY + idx), v110 = __ldg(orgY + idx + 1);
            v001 = __ldg(orgZ + idx), v101 = __ldg(orgZ + idx + 1);
            v011 = __ldg(orgYZ + idx), v111 = __ldg(orgYZ + idx + 1);
        } else {
            const int ix = __float_as_int(mx) - 0x4B400000, iy = __float_as_int(my) - 0x4B400000, iz = __float_as_int(mz) - 0x4B400000;
            const float* q = org + ((IdxT)iz * pitchZ + (IdxT)iy * pitchY + (IdxT)ix);
            v000 = __ldg(q), v100 = __ldg(q + 1);
            v010 = __ldg(q + pitchY), v110 = __ldg(q + pitchY + 1);
            v001 = __ldg(q + pitchZ), v101 = __ldg(q + pitchZ + 1);
            v011 = __ldg(q + pitchZ + pitchY), v111 = __ldg(q + pitchZ + pitchY + 1);
        }
        const float c00 = fmaf(ax, v100 - v000, v000), c10 = fmaf(ax, v110 - v010, v010);
        const float c01 = fmaf(ax, v101 - v001, v001), c11 = fmaf(ax, v111 - v011, v011);
        const float c0 = fmaf(ay, c10 - c00, c00), c1 = fmaf(ay, c11 - c01, c01);
        acc += fmaf(az, c1 - c0, c0);
    };
    // the same sample, scattered (exact adjoint): the eight trilinear weights times the ray's value
    auto interior_scatter = [&](float t) {
        const float x = fmaf(t, r.sx, r.x0), y = fmaf(t, r.sy, r.y0), z = fmaf(t, r.sz, r.z0);
        const float mx = (x - 0.5f) + 12582912.0f, my = (y - 0.5f) + 12582912.0f, mz = (z - 0.5f) + 12582912.0f;
        const float ax = x - (mx - 12582912.0f), ay = y - (my - 12582912.0f), az = z - (mz - 12582912.0f);
        const int ix = __float_as_int(mx) - 0x4B400000, iy = __float_as_int(my) - 0x4B400000, iz = __float_as_int(mz) - 0x4B400000;
        float* q = const_cast<float*>(org) + ((IdxT)iz * pitchZ + (IdxT)iy * pitchY + (IdxT)ix);
        const float w0 = (1.f - az) * ys, w1 = az * ys;
        const float w00 = (1.f - ay) * w0, w10 = ay * w0, w01 = (1.f - ay) * w1, w11 = ay * w1;
        red_add_global(q, (1.f - ax) * w00), red_add_global(q + 1, ax * w00);
        red_add_global(q + pitchY, (1.f - ax) * w10), red_add_global(q + pitchY + 1, ax * w10);
        red_add_global(q + pitchZ, (1.f - ax) * w01), red_add_global(q + pitchZ + 1, ax * w01);
        red_add_global(q + pitchZ + pitchY, (1.f - ax) * w11), red_add_global(q + pitchZ + pitchY + 1, ax * w11);
    };
    // bounds-checked sample without branches (gather only): every tap index is tested once per axis; an outside tap gets
    // weight zero and a clamped (valid) address
    auto edge = [&](int k) {
        const float t = (float)k + 0.5f;
        const float x = fmaf(t, r.sx, r.x0), y = fmaf(t, r.sy, r.y0), z = fmaf(t, r.sz, r.z0);
        const float mx = (x - 0.5f) + 12582912.0f, my = (y - 0.5f) + 12582912.0f, mz = (z - 0.5f) + 12582912.0f;
        const float ax = x - (mx - 12582912.0f), ay = y - (my - 12582912.0f), az = z - (mz - 12582912.0f);
        // array indices of the lower taps (relative to the first slice present; may be out of range)
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
        const IdxT oy0 = (IdxT)(y0 ? jy : 0) * pitchY, oy1 = (IdxT)(y1 ? jy + 1 : 0) * pitchY;
        const IdxT oz0 = (IdxT)(z0 ? jz : 0) * pitchZ, oz1 = (IdxT)(z1 ? jz + 1 : 0) * pitchZ;
        const float *r00 = base + (oz0 + oy0), *r10 = base + (oz0 + oy1), *r01 = base + (oz1 + oy0), *r11 = base + (oz1 + oy1);
        const float c00 = fmaf(wx1, __ldg(r00 + cx1), wx0 * __ldg(r00 + cx0)), c10 = fmaf(wx1, __ldg(r10 + cx1), wx0 * __ldg(r10 + cx0));
        const float c01 = fmaf(wx1, __ldg(r01 + cx1), wx0 * __ldg(r01 + cx0)), c11 = fmaf(wx1, __ldg(r11 + cx1), wx0 * __ldg(r11 + cx0));
        const float c0 = fmaf(wy1, c10, wy0 * c00), c1 = fmaf(wy1, c11, wy0 * c01);
        acc += fmaf(wz1, c1, wz0 * c0);
    };
    // unchecked samples [k, kend) of the interior [kA, kB)
    auto inner = [&](int& k, int kend) {
        if (k < kend) {
            float t = (float)k + 0.5f;
            for (; k < kend; ++k, t += 1.f) {
                if (SCATTER) interior_scatter(t);
                else interior(t);
            }
        }
    };

    // The samples of a ray are fixed by the definition (l_in + (k+1/2) delta from ITS entry point), but the
    // order in which a warp visits them is free.  Neighbouring rays enter the volume at different depths, so
    // visiting sample k of every lane together scatters the warp over many rows of the volume.  Instead the
    // warp advances along Y (the in-plane axis the rays run along) AXI_ROWS rows at a time: in each step every
    // lane takes the INTERIOR samples of its own ray that fall into the current rows (16 to 23 of them at a
    // step of half a voxel; the lanes' trip counts differ by at most one), and all lanes stay within AXI_ROWS + 1
    // adjacent rows of the (transposed) volume.  (Two rows per step, the first design, kept the footprint smallest but
    // lost one trip in five to the uneven counts and paid the step's overhead every 4-5 samples.)  The few bounds-checked samples at the two ends of each ray
    // ([k0, kA) and [kB, Kuse)) are left out of the march and taken afterwards by all lanes together: inside the march
    // they ran a lane or three at a time (rays of one warp enter and leave the volume in different rows) and cost a
    // quarter of the kernel's issue slots.
    int k = r.kA;
    const bool live = r.kB > r.kA, up = r.sy >= 0.f;
    const unsigned liveM = __ballot_sync(wmask, live), upM = __ballot_sync(wmask, live && up);
    const bool steep = fabsf(r.sy) > 0.05f * (fabsf(r.sx) + fabsf(r.sz));
    const bool lock = liveM != 0 && (upM == liveM || upM == 0) && __ballot_sync(wmask, live && !steep) == 0;
    if (lock) {
        const bool wup = upM != 0;
        const float isy = live ? 1.0f / r.sy : 0.f, cc = live ? fmaf(-r.y0, isy, -0.5f) : 0.f;
        const int j0 = live ? (int)floorf(fmaf((float)r.kA + 0.5f, r.sy, r.y0)) : (wup ? 0x7fffffff : (int)0x80000000);
        const int jw = wup ? __reduce_min_sync(wmask, j0) : __reduce_max_sync(wmask, j0);
        float Yb = wup ? (float)(jw + AXI_ROWS) : (float)(jw + 1 - AXI_ROWS);   // far side of the current rows in the direction of travel
        const float dY = wup ? (float)AXI_ROWS : -(float)AXI_ROWS;
        for (int it = 0; it < nY / AXI_ROWS + 8; ++it) {
            const float kf = ceilf(fmaf(Yb, isy, cc));
            const int kend = live ? (int)fminf(fmaxf(kf, (float)k), (float)r.kB) : k;
            inner(k, kend);
            Yb += dY;
            if (!__any_sync(wmask, k < r.kB)) break;
        }
    }
    inner(k, r.kB);   // rays not marched in lockstep (mixed directions, rays across Y), leftovers
    for (int q = r.k0; q < r.kA; ++q) {
        if (UNIT || SCATTER) checked(q);
        else edge(q);
    }
    for (int q = r.kB; q < r.Kuse; ++q) {
        if (UNIT || SCATTER) checked(q);
        else edge(q);
    }
    if (!SCATTER) {
        const float result = acc * (float)p.delta;
        proj[out] = p.accumulate ? proj[out] + result : result;
    }
}

// Row sums A 1 of the Siddon projector in closed form: the intersection lengths of a ray with
// the voxels add up to the length of its segment inside the volume box, so a unit volume needs no march: clip the
// segment S -> P (parameter [0,1]) against the box [0,n]^3 in voxel-index coordinates, in fp64.
__global__ void __launch_bounds__(AX_TU* AX_TV)
ax_siddon_unit_kernel(const RayView* __restrict__ views, int nViews, AxP p, float* __restrict__ proj) {
    int view, iu, iv;
    if (!ax_decode(p, nViews, view, iu, iv)) return;
    const RayView& rv = views[view];
    const size_t out = ((size_t)view * p.nv + iv) * p.nu + iu;
    const double n[3] = {(double)p.nx, (double)p.ny, (double)p.nz};
    const double h[3] = {p.hxd, p.hyd, p.hzd};
    double t0 = 0.0, t1 = 1.0, L2 = 0.0;
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        const double S = rv.S[k] + iu * rv.dSU[k] + iv * rv.dSV[k];
        const double d = rv.P0[k] + iu * rv.dU[k] + iv * rv.dV[k] - S;
        L2 += d * h[k] * d * h[k];
        if (d != 0.0) {
            const double a = (0.0 - S) / d, b = (n[k] - S) / d;
            t0 = fmax(t0, fmin(a, b)), t1 = fmin(t1, fmax(a, b));
        } else if (S < 0.0 || S >= n[k]) {
            t1 = -1.0;   // parallel to this pair of faces and outside (a ray IN a face goes to the upper voxel, reading P8)
        }
    }
    const float result = t1 > t0 ? (float)((t1 - t0) * sqrt(L2)) : 0.f;
    proj[out] = p.accumulate ? proj[out] + result : result;
}

// test hook (tigre_set_index_path): 1 = take the 64-bit element-index instantiations (volumes or slabs of >= 2^31 voxels, the
// C5 regime) for every volume, so that they can be compared with the 32-bit ones and with the oracle on small volumes
static int g_index_path = 0;
void set_index_path(int path) { g_index_path = path; }
static bool use_idx64(size_t nvox) { return g_index_path == 1 || nvox >= (1ull << 31); }

template <typename IdxT>
static void ax_dispatch(const float* vol, const float* volT, const RayView* v, int nViews, const AxP& p, int mode, bool unit,
                        float* proj, uint32_t* counts, cudaStream_t st) {
    dim3 block(AX_TU, AX_TV);
    const long long nblk = (long long)p.nUt * p.nVt * nViews;
    dim3 grid((unsigned)nblk);
    if (mode == TIGRE_AX_SIDDON) {
        if (counts) ax_siddon_kernel<IdxT, false, true, false><<<grid, block, 0, st>>>(vol, volT, v, nViews, p, proj, counts);
        else if (unit) ax_siddon_unit_kernel<<<grid, block, 0, st>>>(v, nViews, p, proj);
        else ax_siddon_kernel<IdxT, false, false, false><<<grid, block, 0, st>>>(vol, volT, v, nViews, p, proj, counts);
    } else {
        if (counts) ax_interp_kernel<IdxT, false, true, false><<<grid, block, 0, st>>>(vol, volT, v, nViews, p, proj, counts);
        else if (unit) ax_interp_kernel<IdxT, true, false, false><<<grid, block, 0, st>>>(vol, volT, v, nViews, p, proj, counts);
        else ax_interp_kernel<IdxT, false, false, false><<<grid, block, 0, st>>>(vol, volT, v, nViews, p, proj, counts);
    }
}

int launch_ax_interp_tma(const float* vol, const float* volT, const Grid& g, const RayView* d_views, const RayView* h_views,
                         int nViews, const AxP& p, float* proj, cudaStream_t st);   // ax_tma.cu
int launch_ax_siddon_tma(const float* vol, const float* volT, const Grid& g, const RayView* d_views, const RayView* h_views, int nViews,
                         const AxP& p, float* proj, cudaStream_t st);   // ax_siddon_tma.cu

int launch_ax(const float* vol, const Grid& g, const RayView* d_views, int nViews, int mode, bool unit_vol,
              bool accumulate, float* proj, uint32_t* count_out, cudaStream_t st, const AxSub* sub, const float* volT_in,
              const RayView* h_views) {
    if (mode != TIGRE_AX_SIDDON && mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    if (sub && (sub->row0 < 0 || sub->row0 + sub->nrows > g.nv || sub->zs0 < 0 || sub->zs0 + sub->nzs > g.nz)) return TIGRE_ERR_ARG;
    if (sub && (sub->nrows <= 0 || sub->nzs <= 0)) return TIGRE_OK;   // nothing of this slab reaches the detector
    AxP p;
    p.nx = g.nx, p.ny = g.ny, p.nz = g.nz, p.nu = g.nu, p.nv = g.nv;
    p.hx = (float)g.dx, p.hy = (float)g.dy, p.hz = (float)g.dz;
    p.hxd = g.dx, p.hyd = g.dy, p.hzd = g.dz;
    p.delta = g.accuracy * fmin(g.dx, fmin(g.dy, g.dz));
    p.iv0 = sub ? sub->row0 : 0, p.iv1 = sub ? sub->row0 + sub->nrows : g.nv;
    p.zs0 = sub ? sub->zs0 : 0, p.zs1 = sub ? sub->zs0 + sub->nzs : g.nz;
    if (mode == TIGRE_AX_SIDDON && (p.zs0 != 0 || p.zs1 != g.nz)) return TIGRE_ERR_ARG;   // Siddon slabs are sub-grids
    p.nUt = (g.nu + AX_TU - 1) / AX_TU, p.nVt = (p.iv1 - p.iv0 + AX_TV - 1) / AX_TV;
    p.accumulate = accumulate ? 1 : 0;
    const long long nblk = (long long)p.nUt * p.nVt * nViews;
    if (nblk <= 0 || nblk > 0x7fffffffLL) return TIGRE_ERR_ARG;
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    TempBuf vt;
    const float* volT = nullptr;
    int launches = 1;
    // an (x,y)-transposed copy of the volume (of the slab present, in the chunked path) serves the x-dominant rays
    const int nzT = p.zs1 - p.zs0;
    const bool wantT = !unit_vol && !count_out && vol && g.nx > 1 && g.ny > 1;
    if (wantT && volT_in) volT = volT_in;            // the caller keeps a transposed copy up to date (OS-SART plan)
    else if (wantT && vt.alloc((size_t)g.nx * g.ny * nzT * sizeof(float), st) == TIGRE_OK) volT = vt.as<float>(), launches = 2;
    ProfScope ps(PK_AX, st, launches);
    if (volT && !volT_in) {
        dim3 tb(32, 8), tg_((g.nx + 31) / 32, (g.ny + 31) / 32, nzT);
        if (tg_.y > 65535 || tg_.z > 65535) volT = nullptr;
        else transpose_xy_kernel<<<tg_, tb, 0, st>>>(vol, vt.as<float>(), g.nx, g.ny);
    }
    if (mode == TIGRE_AX_INTERP && !unit_vol && !count_out && volT && h_views && g_index_path == 0) {
        const int rc = launch_ax_interp_tma(vol, volT, g, d_views, h_views, nViews, p, proj, st);
        if (rc <= 0) return rc;   // launched, or a CUDA error; rc > 0: does not qualify
    }
    if (mode == TIGRE_AX_SIDDON && !unit_vol && !count_out && volT && h_views && g_index_path == 0 && !use_idx64(nvox)) {
        const int rc = launch_ax_siddon_tma(vol, volT, g, d_views, h_views, nViews, p, proj, st);
        if (rc <= 0) return rc;
    }
    if (!use_idx64(nvox)) ax_dispatch<int>(vol, volT, d_views, nViews, p, mode, unit_vol, proj, count_out, st);
    else ax_dispatch<long long>(vol, volT, d_views, nViews, p, mode, unit_vol, proj, count_out, st);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

// tigre_Ax_index: the Siddon march without the volume; per ray the first / last voxel with a non-zero length and their number
int launch_ax_track(const Grid& g, const RayView* d_views, int nViews, uint32_t* counts, long long* track, cudaStream_t st) {
    AxP p;
    p.nx = g.nx, p.ny = g.ny, p.nz = g.nz, p.nu = g.nu, p.nv = g.nv;
    p.hx = (float)g.dx, p.hy = (float)g.dy, p.hz = (float)g.dz;
    p.hxd = g.dx, p.hyd = g.dy, p.hzd = g.dz;
    p.delta = g.accuracy * fmin(g.dx, fmin(g.dy, g.dz));
    p.iv0 = 0, p.iv1 = g.nv, p.zs0 = 0, p.zs1 = g.nz;
    p.nUt = (g.nu + AX_TU - 1) / AX_TU, p.nVt = (g.nv + AX_TV - 1) / AX_TV;
    p.accumulate = 0;
    const long long nblk = (long long)p.nUt * p.nVt * nViews;
    if (nblk <= 0 || nblk > 0x7fffffffLL) return TIGRE_ERR_ARG;
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    // the march only forms offsets from these two bases (it never dereferences them); they select the layout each ray walks,
    // exactly as in launch_ax: x-dominant rays take the transposed one whenever launch_ax would make it
    const float* fakeV = reinterpret_cast<const float*>(0x1000);
    const float* fakeT = (g.nx > 1 && g.ny > 1) ? reinterpret_cast<const float*>(0x2000) : nullptr;
    dim3 block(AX_TU, AX_TV), grid((unsigned)nblk);
    ProfScope ps(PK_AX, st);
    if (!use_idx64(nvox)) ax_siddon_kernel<int, true, false, false, true><<<grid, block, 0, st>>>(fakeV, fakeT, d_views, nViews, p, nullptr, counts, track);
    else ax_siddon_kernel<long long, true, false, false, true><<<grid, block, 0, st>>>(fakeV, fakeT, d_views, nViews, p, nullptr, counts, track);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

// the transposed copy alone (for callers that maintain it themselves); returns TIGRE_ERR_ARG if the grid does not fit
int launch_transpose_xy(const float* vol, float* volT, const Grid& g, cudaStream_t st) {
    dim3 tb(32, 8), tg_((g.nx + 31) / 32, (g.ny + 31) / 32, g.nz);
    if (tg_.y > 65535 || tg_.z > 65535) return TIGRE_ERR_ARG;
    ProfScope ps(PK_AX, st);
    transpose_xy_kernel<<<tg_, tb, 0, st>>>(vol, volT, g.nx, g.ny);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

// vol[z][y][x] += volT[z][x][y]
__global__ void __launch_bounds__(256) transpose_add_kernel(const float* __restrict__ inT, float* __restrict__ out, int nx, int ny) {
    __shared__ float tile[32][33];
    const size_t slice = (size_t)nx * ny * blockIdx.z;
    const int x0 = blockIdx.x * 32, y0 = blockIdx.y * 32;
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int y = y0 + threadIdx.x, x = x0 + j;
        if (x < nx && y < ny) tile[j][threadIdx.x] = inT[slice + (size_t)x * ny + y];
    }
    __syncthreads();
    for (int j = threadIdx.y; j < 32; j += 8) {
        const int x = x0 + threadIdx.x, y = y0 + j;
        if (x < nx && y < ny) out[slice + (size_t)y * nx + x] += tile[threadIdx.x][j];
    }
}

// Exact adjoint of launch_ax ("matched" pairs for the Krylov family): the
// same ray march, every (length or trilinear weight) x ray value ADDED to its voxel (red.global.add.f32).
// x-dominant rays scatter into a transposed scratch volume that is added back at the end.
int launch_ax_adjoint(const float* proj, const Grid& g, const RayView* d_views, int nViews, int mode, float* vol,
                      cudaStream_t st) {
    if (mode != TIGRE_AX_SIDDON && mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    AxP p;
    p.nx = g.nx, p.ny = g.ny, p.nz = g.nz, p.nu = g.nu, p.nv = g.nv;
    p.hx = (float)g.dx, p.hy = (float)g.dy, p.hz = (float)g.dz;
    p.hxd = g.dx, p.hyd = g.dy, p.hzd = g.dz;
    p.delta = g.accuracy * fmin(g.dx, fmin(g.dy, g.dz));
    p.iv0 = 0, p.iv1 = g.nv, p.zs0 = 0, p.zs1 = g.nz;
    p.nUt = (g.nu + AX_TU - 1) / AX_TU, p.nVt = (g.nv + AX_TV - 1) / AX_TV;
    p.accumulate = 0;
    const long long nblk = (long long)p.nUt * p.nVt * nViews;
    if (nblk <= 0 || nblk > 0x7fffffffLL) return TIGRE_ERR_ARG;
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    TempBuf vt;
    float* volT = nullptr;
    dim3 tb(32, 8), tgd((g.nx + 31) / 32, (g.ny + 31) / 32, g.nz);
    if (g.nx > 1 && g.ny > 1 && tgd.y <= 65535 && tgd.z <= 65535 && vt.alloc(nvox * sizeof(float), st) == TIGRE_OK) volT = vt.as<float>();
    ProfScope ps(PK_ATB, st, volT ? 2 : 1);
    TG_CUDA(cudaMemsetAsync(vol, 0, nvox * sizeof(float), st));
    if (volT) TG_CUDA(cudaMemsetAsync(volT, 0, nvox * sizeof(float), st));
    dim3 block(AX_TU, AX_TV), grid((unsigned)nblk);
    float* pin = const_cast<float*>(proj);   // read only by the SCATTER instantiations
    if (!use_idx64(nvox)) {
        if (mode == TIGRE_AX_SIDDON) ax_siddon_kernel<int, false, false, true><<<grid, block, 0, st>>>(vol, volT, d_views, nViews, p, pin, nullptr);
        else ax_interp_kernel<int, false, false, true><<<grid, block, 0, st>>>(vol, volT, d_views, nViews, p, pin, nullptr);
    } else {
        if (mode == TIGRE_AX_SIDDON) ax_siddon_kernel<long long, false, false, true><<<grid, block, 0, st>>>(vol, volT, d_views, nViews, p, pin, nullptr);
        else ax_interp_kernel<long long, false, false, true><<<grid, block, 0, st>>>(vol, volT, d_views, nViews, p, pin, nullptr);
    }
    if (volT) transpose_add_kernel<<<tgd, tb, 0, st>>>(volT, vol, g.nx, g.ny);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg
