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
//  Per-ray set-up (entry/exit, slopes, first slab) is fp64; the march is fp32 with positions
//  recomputed from the integer slab counter (never accumulated) in volume-centred coordinates.
//
//  Interpolated (fixed step, software fp32 trilinear, zero border; reading P9): samples at
//  l_k = l_in + (k+1/2) delta inside the box grown by half a voxel.
#include <cmath>
#include "common.cuh"

namespace tg {

struct AxP {
    int nx, ny, nz, nu, nv;
    float hx, hy, hz;     // voxel pitch, mm
    double hxd, hyd, hzd;
    double delta;         // interpolated step, mm
    int nUt, nVt;         // tiles per view
    int accumulate;
};

constexpr int AX_TU = 32, AX_TV = 4;

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
    iv = vt * AX_TV + threadIdx.y;
    return iu < p.nu && iv < p.nv;
}

template <typename IdxT, bool UNIT, bool COUNT>
__global__ void __launch_bounds__(AX_TU* AX_TV)
ax_siddon_kernel(const float* __restrict__ vol, const RayView* __restrict__ views, int nViews, AxP p,
                 float* __restrict__ proj, uint32_t* __restrict__ counts) {
    int view, iu, iv;
    if (!ax_decode(p, nViews, view, iu, iv)) return;
    const RayView& rv = views[view];
    const size_t out = ((size_t)view * p.nv + iv) * p.nu + iu;

    // ---- per-ray set-up, fp64
    double S[3], d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        S[k] = rv.S[k];
        d[k] = rv.P0[k] + iu * rv.dU[k] + iv * rv.dV[k] - S[k];
    }
    const double Lmm = sqrt(d[0] * p.hxd * d[0] * p.hxd + d[1] * p.hyd * d[1] * p.hyd + d[2] * p.hzd * d[2] * p.hzd);
    const double a0 = fabs(d[0]), a1 = fabs(d[1]), a2 = fabs(d[2]);
    const int D = (a0 >= a1 && a0 >= a2) ? 0 : (a1 >= a2 ? 1 : 2);
    const int E = (D + 1) % 3, F = (D + 2) % 3;
    const double dD = sel3(D, d[0], d[1], d[2]), dE = sel3(E, d[0], d[1], d[2]), dF = sel3(F, d[0], d[1], d[2]);
    const double SD = sel3(D, S[0], S[1], S[2]), SE = sel3(E, S[0], S[1], S[2]), SF = sel3(F, S[0], S[1], S[2]);
    const int nD = D == 0 ? p.nx : (D == 1 ? p.ny : p.nz);
    const int nE = E == 0 ? p.nx : (E == 1 ? p.ny : p.nz);
    const int nF = F == 0 ? p.nx : (F == 1 ? p.ny : p.nz);
    float result = 0.f;
    uint32_t cnt = 0;
    if (dD != 0.0) {
        const double mE = dE / dD, mF = dF / dD;
        // range of xi_D covered by the segment S->P, clipped to the volume box on all three axes
        double lo = fmin(SD, SD + dD), hi = fmax(SD, SD + dD);
        lo = fmax(lo, 0.0), hi = fmin(hi, (double)nD);
        bool miss = false;
        if (mE != 0.0) {
            const double t1 = SD + (0.0 - SE) / mE, t2 = SD + ((double)nE - SE) / mE;
            lo = fmax(lo, fmin(t1, t2)), hi = fmin(hi, fmax(t1, t2));
        } else if (SE < 0.0 || SE > (double)nE) miss = true;
        if (mF != 0.0) {
            const double t1 = SD + (0.0 - SF) / mF, t2 = SD + ((double)nF - SF) / mF;
            lo = fmax(lo, fmin(t1, t2)), hi = fmin(hi, fmax(t1, t2));
        } else if (SF < 0.0 || SF > (double)nF) miss = true;
        if (!miss && hi > lo) {
            if (COUNT) {
                // exact number of voxels met = |dix|+|diy|+|diz|+1 between entry and exit voxel
                const double eps = 1e-9 * (hi - lo);
                const double l0 = lo + eps, l1 = hi - eps;
                int c = 1;
                c += abs((int)floor(l1) - (int)floor(l0));
                c += abs((int)floor(SE + (l1 - SD) * mE) - (int)floor(SE + (l0 - SD) * mE));
                c += abs((int)floor(SF + (l1 - SD) * mF) - (int)floor(SF + (l0 - SD) * mF));
                cnt = (uint32_t)c;
            } else {
                int i0 = (int)floor(lo), i1 = (int)ceil(hi);
                i0 = max(i0, 0), i1 = min(i1, nD);
                const int nslab = i1 - i0;
                const int hE = nE >> 1, hF = nF >> 1;   // volume-centred coordinates: |e| <= n/2
                // state at the START of slab i0 (s = 0), fp64: position, cell index, next plane ahead
                const double eS = SE + ((double)i0 - SD) * mE, fS = SF + ((double)i0 - SD) * mF;
                int ie = (int)floor(eS), jf = (int)floor(fS);
                const bool upE = mE > 0.0, upF = mF > 0.0;
                const float eref = (float)(eS - (double)hE), fref = (float)(fS - (double)hF);
                const float mEf = (float)mE, mFf = (float)mF;
                // slab-local parameter of the next E / F plane: s = (next - e0) / m, saturated to [0,1];
                // a ray parallel to the planes (m = 0) never crosses: next = +huge, 1/m := 1
                const float imE = mE != 0.0 ? (float)(1.0 / mE) : 1.f, imF = mF != 0.0 ? (float)(1.0 / mF) : 1.f;
                float nextE = mE != 0.0 ? (float)((upE ? ie + 1 : ie) - hE) : 3.0e38f;
                float nextF = mF != 0.0 ? (float)((upF ? jf + 1 : jf) - hF) : 3.0e38f;
                const float sgE = upE ? 1.f : -1.f, sgF = upF ? 1.f : -1.f;
                const float slo0 = (float)(lo - (double)i0), shiN = (float)(hi - (double)(i1 - 1));
                const IdxT sD = D == 0 ? 1 : (D == 1 ? (IdxT)p.nx : (IdxT)p.nx * p.ny);
                const IdxT sE = E == 0 ? 1 : (E == 1 ? (IdxT)p.nx : (IdxT)p.nx * p.ny);
                const IdxT sF = F == 0 ? 1 : (F == 1 ? (IdxT)p.nx : (IdxT)p.nx * p.ny);
                const IdxT stE = upE ? sE : -sE, stF = upF ? sF : -sF;
                const int diE = upE ? 1 : -1, diF = upF ? 1 : -1;
                IdxT off = (IdxT)i0 * sD + (IdxT)ie * sE + (IdxT)jf * sF;   // may be out of range: guarded below
                float acc = 0.f;
                float kf = 0.f;
                const int last = nslab - 1;
                for (int k = 0; k < nslab; ++k) {
                    const float e0 = fmaf(kf, mEf, eref), f0 = fmaf(kf, mFf, fref);
                    kf += 1.0f;
                    const float se = __saturatef((nextE - e0) * imE);
                    const float sf = __saturatef((nextF - f0) * imF);
                    const bool cE = se < 1.0f, cF = sf < 1.0f;
                    float s1 = fminf(se, sf), s2 = fmaxf(se, sf);
                    float slo = 0.f, shi = 1.f;
                    if (k == 0 || k == last) {   // only the end slabs are clipped to the segment / box
                        slo = (k == 0) ? slo0 : 0.f;
                        shi = (k == last) ? shiN : 1.f;
                        s1 = fminf(fmaxf(s1, slo), shi);
                        s2 = fminf(fmaxf(s2, slo), shi);
                    }
                    const bool vEA = (unsigned)ie < (unsigned)nE, vFA = (unsigned)jf < (unsigned)nF;
                    const int ieC = cE ? ie + diE : ie, jfC = cF ? jf + diF : jf;
                    const IdxT offC = off + (cE ? stE : (IdxT)0) + (cF ? stF : (IdxT)0);
                    const bool vEC = (unsigned)ieC < (unsigned)nE, vFC = (unsigned)jfC < (unsigned)nF;
                    const float lenA = s1 - slo, lenC = shi - s2;
                    if (lenA > 0.f && vEA && vFA) acc = fmaf(lenA, UNIT ? 1.f : __ldg(vol + off), acc);
                    if (__any_sync(__activemask(), cE && cF)) {
                        // some lane crosses both planes inside this slab: a middle voxel between the two crossings
                        // (for a lane with one crossing the middle voxel IS the end voxel and lenC = 0)
                        const float lenB = s2 - s1;
                        const bool eFirst = se < sf;
                        const IdxT offB = eFirst ? off + stE : off + stF;
                        const bool vB = eFirst ? (vEC && vFA) : (vEA && vFC);
                        if (lenB > 0.f && vB) acc = fmaf(lenB, UNIT ? 1.f : __ldg(vol + offB), acc);
                        if (lenC > 0.f && vEC && vFC) acc = fmaf(lenC, UNIT ? 1.f : __ldg(vol + offC), acc);
                    } else {
                        // at most one crossing: [s1, shi] lies in the end voxel (s2 == shi when nothing else crosses)
                        const float lenBC = shi - s1;
                        if (lenBC > 0.f && vEC && vFC) acc = fmaf(lenBC, UNIT ? 1.f : __ldg(vol + offC), acc);
                    }
                    if (cE) nextE += sgE;
                    if (cF) nextF += sgF;
                    ie = ieC, jf = jfC;
                    off = offC + sD;
                }
                result = acc * (float)(Lmm / fabs(dD));
            }
        }
    }
    if (COUNT) {
        counts[out] = cnt;
    } else {
        proj[out] = p.accumulate ? proj[out] + result : result;
    }
}

// ------------------------------------------------------------------------------------------
template <typename IdxT, bool UNIT, bool COUNT>
__global__ void __launch_bounds__(AX_TU* AX_TV)
ax_interp_kernel(const float* __restrict__ vol, const RayView* __restrict__ views, int nViews, AxP p,
                 float* __restrict__ proj, uint32_t* __restrict__ counts) {
    int view, iu, iv;
    if (!ax_decode(p, nViews, view, iu, iv)) return;
    const RayView& rv = views[view];
    const size_t out = ((size_t)view * p.nv + iv) * p.nu + iu;
    // fp64 set-up in voxel-index coordinates (voxel centres at integer + 1/2)
    double S[3], d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        S[k] = rv.S[k];
        d[k] = rv.P0[k] + iu * rv.dU[k] + iv * rv.dV[k] - S[k];
    }
    const double h[3] = {p.hxd, p.hyd, p.hzd};
    const int n[3] = {p.nx, p.ny, p.nz};
    const double Lmm = sqrt(d[0] * h[0] * d[0] * h[0] + d[1] * h[1] * d[1] * h[1] + d[2] * h[2] * d[2] * h[2]);
    float result = 0.f;
    uint32_t cnt = 0;
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
            if (COUNT) {
                cnt = (uint32_t)K;
            } else {
                // centre-index coordinates relative to the volume centre: c = xi - 1/2 - (n-1)/2... kept
                // as (xi - 1/2) - hn with hn = n/2 so floor() stays an exact integer shift
                const int hx = p.nx >> 1, hy = p.ny >> 1, hz = p.nz >> 1;
                const float x0 = (float)(S[0] + lin * d[0] / Lmm - 0.5 - hx);
                const float y0 = (float)(S[1] + lin * d[1] / Lmm - 0.5 - hy);
                const float z0 = (float)(S[2] + lin * d[2] / Lmm - 0.5 - hz);
                const float sx = (float)(p.delta * d[0] / Lmm), sy = (float)(p.delta * d[1] / Lmm),
                            sz = (float)(p.delta * d[2] / Lmm);
                const IdxT pitchY = p.nx, pitchZ = (IdxT)p.nx * p.ny;
                // samples beyond the detector end of the segment are dropped (l_k > |p-S|)
                const long long Kmax = (long long)floor((Lmm - lin) / p.delta - 0.5) + 1;
                const int Kuse = (int)min(K, max(Kmax, 0LL));
                float acc = 0.f;
                for (int k = 0; k < Kuse; ++k) {
                    const float t = (float)k + 0.5f;
                    const float x = fmaf(t, sx, x0), y = fmaf(t, sy, y0), z = fmaf(t, sz, z0);
                    const float fx = floorf(x), fy = floorf(y), fz = floorf(z);
                    const float ax = x - fx, ay = y - fy, az = z - fz;
                    const int ix = (int)fx + hx, iy = (int)fy + hy, iz = (int)fz + hz;
                    float v = 0.f;
                    if (UNIT) {
                        const float wx = ((unsigned)ix < (unsigned)p.nx ? 1.f - ax : 0.f) + ((unsigned)(ix + 1) < (unsigned)p.nx ? ax : 0.f);
                        const float wy = ((unsigned)iy < (unsigned)p.ny ? 1.f - ay : 0.f) + ((unsigned)(iy + 1) < (unsigned)p.ny ? ay : 0.f);
                        const float wz = ((unsigned)iz < (unsigned)p.nz ? 1.f - az : 0.f) + ((unsigned)(iz + 1) < (unsigned)p.nz ? az : 0.f);
                        v = wx * wy * wz;
                    } else if (ix >= 0 && ix + 1 < p.nx && iy >= 0 && iy + 1 < p.ny && iz >= 0 && iz + 1 < p.nz) {
                        const float* q = vol + ((IdxT)iz * pitchZ + (IdxT)iy * pitchY + ix);
                        const float v000 = __ldg(q), v100 = __ldg(q + 1);
                        const float v010 = __ldg(q + pitchY), v110 = __ldg(q + pitchY + 1);
                        const float v001 = __ldg(q + pitchZ), v101 = __ldg(q + pitchZ + 1);
                        const float v011 = __ldg(q + pitchZ + pitchY), v111 = __ldg(q + pitchZ + pitchY + 1);
                        const float c00 = fmaf(ax, v100 - v000, v000), c10 = fmaf(ax, v110 - v010, v010);
                        const float c01 = fmaf(ax, v101 - v001, v001), c11 = fmaf(ax, v111 - v011, v011);
                        const float c0 = fmaf(ay, c10 - c00, c00), c1 = fmaf(ay, c11 - c01, c01);
                        v = fmaf(az, c1 - c0, c0);
                    } else {
#pragma unroll
                        for (int c = 0; c < 8; ++c) {
                            const int jx = ix + (c & 1), jy = iy + ((c >> 1) & 1), jz = iz + (c >> 2);
                            if ((unsigned)jx < (unsigned)p.nx && (unsigned)jy < (unsigned)p.ny && (unsigned)jz < (unsigned)p.nz) {
                                const float w = ((c & 1) ? ax : 1.f - ax) * ((c & 2) ? ay : 1.f - ay) * ((c & 4) ? az : 1.f - az);
                                v = fmaf(w, __ldg(vol + ((IdxT)jz * pitchZ + (IdxT)jy * pitchY + jx)), v);
                            }
                        }
                    }
                    acc += v;
                }
                result = acc * (float)p.delta;
            }
        }
    }
    if (COUNT) {
        counts[out] = cnt;
    } else {
        proj[out] = p.accumulate ? proj[out] + result : result;
    }
}

template <typename IdxT>
static void ax_dispatch(const float* vol, const RayView* v, int nViews, const AxP& p, int mode, bool unit,
                        float* proj, uint32_t* counts, cudaStream_t st) {
    dim3 block(AX_TU, AX_TV);
    const long long nblk = (long long)p.nUt * p.nVt * nViews;
    dim3 grid((unsigned)nblk);
    if (mode == TIGRE_AX_SIDDON) {
        if (counts) ax_siddon_kernel<IdxT, false, true><<<grid, block, 0, st>>>(vol, v, nViews, p, proj, counts);
        else if (unit) ax_siddon_kernel<IdxT, true, false><<<grid, block, 0, st>>>(vol, v, nViews, p, proj, counts);
        else ax_siddon_kernel<IdxT, false, false><<<grid, block, 0, st>>>(vol, v, nViews, p, proj, counts);
    } else {
        if (counts) ax_interp_kernel<IdxT, false, true><<<grid, block, 0, st>>>(vol, v, nViews, p, proj, counts);
        else if (unit) ax_interp_kernel<IdxT, true, false><<<grid, block, 0, st>>>(vol, v, nViews, p, proj, counts);
        else ax_interp_kernel<IdxT, false, false><<<grid, block, 0, st>>>(vol, v, nViews, p, proj, counts);
    }
}

int launch_ax(const float* vol, const Grid& g, const RayView* d_views, int nViews, int mode, bool unit_vol,
              bool accumulate, float* proj, uint32_t* count_out, cudaStream_t st) {
    if (mode != TIGRE_AX_SIDDON && mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    AxP p;
    p.nx = g.nx, p.ny = g.ny, p.nz = g.nz, p.nu = g.nu, p.nv = g.nv;
    p.hx = (float)g.dx, p.hy = (float)g.dy, p.hz = (float)g.dz;
    p.hxd = g.dx, p.hyd = g.dy, p.hzd = g.dz;
    p.delta = g.accuracy * fmin(g.dx, fmin(g.dy, g.dz));
    p.nUt = (g.nu + AX_TU - 1) / AX_TU, p.nVt = (g.nv + AX_TV - 1) / AX_TV;
    p.accumulate = accumulate ? 1 : 0;
    const long long nblk = (long long)p.nUt * p.nVt * nViews;
    if (nblk <= 0 || nblk > 0x7fffffffLL) return TIGRE_ERR_ARG;
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    ProfScope ps(PK_AX, st);
    if (nvox < (1ull << 31)) ax_dispatch<int>(vol, d_views, nViews, p, mode, unit_vol, proj, count_out, st);
    else ax_dispatch<long long>(vol, d_views, nViews, p, mode, unit_vol, proj, count_out, st);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg
