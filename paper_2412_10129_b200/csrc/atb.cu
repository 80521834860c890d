// atb.cu — voxel-driven backprojection x = A^T b (eq. 4, 135 eq. 6; DESIGN.md O-C).
// For each voxel centre and each view: project to the detector with a 3x4 projective map,
// bilinear interpolation with zero border, weight
//   matched  w = (dx dy dz)/(du dv) * R^2/(r^2 cos g) = km * t^2 * R(u,v)     (reading P10)
//   FDK      w = (DSO/(DSO - X'_x))^2 = 1/G^2
// Each thread owns a run of ZR voxels along z at fixed (x,y); accumulators stay in registers
// while the kernel loops over the views.
//
// Two kernels:
//   atb_gather_kernel   any geometry; detector taps gathered through L1/L2 (general fall-back and
//                       the path used when a view's footprint does not fit the staged box)
//   atb_tma_kernel      (atb_tma.cu) footprints staged into shared memory by TMA
#include <cmath>
#include "atb_common.cuh"

namespace tg {

template <int MODE, bool UNIT, bool CLAMP, int ZR>
__global__ void __launch_bounds__(ATB_BX* ATB_BY)
atb_gather_kernel(const float* __restrict__ proj, const VoxView* __restrict__ views, int nViews, AtbP p,
                  float* __restrict__ vol) {
    const int ix = blockIdx.x * ATB_BX + threadIdx.x;
    const int iy = blockIdx.y * ATB_BY + threadIdx.y;
    const int zb = blockIdx.z * ZR;  // relative to z0
    if (ix >= p.nx || iy >= p.ny) return;
    const float cxf = (float)ix - p.cx, cyf = (float)iy - p.cy, czf = (float)(p.z0 + zb) - p.cz;
    float acc[ZR];
#pragma unroll
    for (int k = 0; k < ZR; ++k) acc[k] = 0.f;
    const size_t per = (size_t)p.nu * p.nrows;
    const unsigned nu1 = (unsigned)(p.nu - 1), nr1 = (unsigned)(p.nrows - 1);
    for (int a = 0; a < nViews; ++a) {
        const float4* vp = reinterpret_cast<const float4*>(views + a);
        const float4 rU = __ldg(vp), rV = __ldg(vp + 1), rW = __ldg(vp + 2), rG = __ldg(vp + 3), cst = __ldg(vp + 4);
        const float U0 = fmaf(rU.x, cxf, fmaf(rU.y, cyf, fmaf(rU.z, czf, rU.w)));
        const float V0 = fmaf(rV.x, cxf, fmaf(rV.y, cyf, fmaf(rV.z, czf, rV.w)));
        const float W0 = fmaf(rW.x, cxf, fmaf(rW.y, cyf, fmaf(rW.z, czf, rW.w)));
        const float G0 = fmaf(rG.x, cxf, fmaf(rG.y, cyf, fmaf(rG.z, czf, rG.w)));
        const float* pa = proj + (size_t)a * per;
#pragma unroll
        for (int k = 0; k < ZR; ++k) {
            const float kf = (float)k;
            const TapW tw = voxel_view<MODE, CLAMP>(fmaf(kf, rU.z, U0), fmaf(kf, rV.z, V0), fmaf(kf, rW.z, W0),
                                                    fmaf(kf, rG.z, G0), cst, p);
            const int iu = tw.iu, iv = tw.iv;
            float val;
            if (UNIT) {
                // zero border on the true detector bounds: sum of the in-range tap weights
                const bool u0 = (unsigned)iu < (unsigned)p.nu, u1 = (unsigned)(iu + 1) < (unsigned)p.nu;
                const bool v0 = (unsigned)iv < (unsigned)p.nv, v1 = (unsigned)(iv + 1) < (unsigned)p.nv;
                val = ((u0 ? 1.f - tw.au : 0.f) + (u1 ? tw.au : 0.f)) * ((v0 ? 1.f - tw.av : 0.f) + (v1 ? tw.av : 0.f));
            } else {
                const int lv = iv - p.row0;
                const float* q = pa + (ptrdiff_t)lv * p.nu + iu;
                float p00, p10, p01, p11;
                if ((unsigned)iu < nu1 && (unsigned)lv < nr1) {   // all four taps inside
                    p00 = __ldg(q), p10 = __ldg(q + 1), p01 = __ldg(q + p.nu), p11 = __ldg(q + p.nu + 1);
                } else {
                    const bool u0 = (unsigned)iu < (unsigned)p.nu, u1 = (unsigned)(iu + 1) < (unsigned)p.nu;
                    const bool v0 = (unsigned)lv < (unsigned)p.nrows, v1 = (unsigned)(lv + 1) < (unsigned)p.nrows;
                    p00 = (u0 && v0) ? __ldg(q) : 0.f;
                    p10 = (u1 && v0) ? __ldg(q + 1) : 0.f;
                    p01 = (u0 && v1) ? __ldg(q + p.nu) : 0.f;
                    p11 = (u1 && v1) ? __ldg(q + p.nu + 1) : 0.f;
                }
                const float r0 = fmaf(tw.au, p10 - p00, p00), r1 = fmaf(tw.au, p11 - p01, p01);
                val = fmaf(tw.av, r1 - r0, r0);
            }
            acc[k] = fmaf(tw.w, val, acc[k]);
        }
    }
    const size_t slice = (size_t)p.nx * p.ny;
#pragma unroll
    for (int k = 0; k < ZR; ++k) {
        if (zb + k < p.nzs) {
            float* o = vol + (size_t)(zb + k) * slice + (size_t)iy * p.nx + ix;
            *o = p.accumulate ? *o + acc[k] : acc[k];
        }
    }
}

// largest |fu|, |fv| any voxel of the box can reach (projective map with W > 0: extrema at the corners)
bool vox_needs_clamp(const Grid& g, const VoxView* hv, int n) {
    const double cx = 0.5 * g.nx, cy = 0.5 * g.ny, cz = 0.5 * g.nz;
    for (int a = 0; a < n; ++a) {
        const VoxView& v = hv[a];
        for (int i = 0; i < 8; ++i) {
            const double c[3] = {(i & 1) ? cx : -cx, (i & 2) ? cy : -cy, (i & 4) ? cz : -cz};
            const double W = v.rowW[0] * c[0] + v.rowW[1] * c[1] + v.rowW[2] * c[2] + v.rowW[3];
            const double U = v.rowU[0] * c[0] + v.rowU[1] * c[1] + v.rowU[2] * c[2] + v.rowU[3];
            const double V = v.rowV[0] * c[0] + v.rowV[1] * c[1] + v.rowV[2] * c[2] + v.rowV[3];
            if (!(W > 0.0) || std::fabs(U / W) > 1.0e6 || std::fabs(V / W) > 1.0e6) return true;
        }
    }
    return false;
}

template <int MODE, bool UNIT>
static void atb_gather_launch(dim3 grid, dim3 block, cudaStream_t st, bool clamp, const float* proj, const VoxView* v,
                              int nViews, const AtbP& p, float* vol) {
    constexpr int ZR = 8;
    if (clamp) atb_gather_kernel<MODE, UNIT, true, ZR><<<grid, block, 0, st>>>(proj, v, nViews, p, vol);
    else atb_gather_kernel<MODE, UNIT, false, ZR><<<grid, block, 0, st>>>(proj, v, nViews, p, vol);
}

int launch_atb_tma(const float* proj, const Grid& g, const VoxView* d_views, const VoxView* h_views, int nViews, int mode,
                   const AtbP& p, float* vol, cudaStream_t st);   // atb_tma.cu
int g_atb_path = 0;   // 0 = TMA-staged kernel when the problem qualifies, 1 = gather kernel only, 2 = TMA, box undersized, 3 = TMA without the linearised z-runs

int launch_atb(const float* proj, const Grid& g, const VoxView* d_views, int nViews, int mode, bool unit_proj,
               float* vol, int z0, int nzs, bool accumulate, int row0, int nrows, bool clamp, cudaStream_t st,
               const VoxView* h_views, const AtbFuse* fuse) {
    if (mode != TIGRE_ATB_MATCHED && mode != TIGRE_ATB_FDK) return TIGRE_ERR_ARG;
    AtbP p;
    p.nx = g.nx, p.ny = g.ny, p.nz = g.nz, p.nu = g.nu, p.nv = g.nv;
    p.z0 = z0, p.nzs = nzs, p.row0 = row0, p.nrows = nrows;
    p.cx = 0.5f * (g.nx - 1), p.cy = 0.5f * (g.ny - 1), p.cz = 0.5f * (g.nz - 1);
    p.du2 = (float)(g.du * g.du), p.dv2 = (float)(g.dv * g.dv);
    p.hu = g.nu / 2, p.hv = g.nv / 2;
    p.accumulate = accumulate ? 1 : 0;
    p.magic = 0x4B400000;
    p.lin_ok = g_atb_path != 3;
    p.fuse = fuse ? 1 : 0, p.nonneg = fuse ? fuse->nonneg : 0, p.lambda = fuse ? fuse->lambda : 0.f, p.V = fuse ? fuse->V : nullptr, p.xT = fuse ? fuse->xT : nullptr;
    if (fuse && (unit_proj || accumulate || !h_views || g_atb_path == 1)) return 2;
    constexpr int ZR = 8;
    dim3 block(ATB_BX, ATB_BY);
    dim3 grid((g.nx + ATB_BX - 1) / ATB_BX, (g.ny + ATB_BY - 1) / ATB_BY, (nzs + ZR - 1) / ZR);
    if (grid.y > 65535 || grid.z > 65535) return TIGRE_ERR_ARG;
    ProfScope ps(PK_ATB, st);
    if (!unit_proj && h_views && g_atb_path != 1) {
        const int rc = launch_atb_tma(proj, g, d_views, h_views, nViews, mode, p, vol, st);
        if (rc <= 0) return rc;   // launched, or a CUDA error; rc > 0: does not qualify
    }
    if (fuse) return 2;   // the gather kernel has no fused epilogue
    if (unit_proj) {
        if (mode == TIGRE_ATB_FDK) atb_gather_launch<TIGRE_ATB_FDK, true>(grid, block, st, clamp, proj, d_views, nViews, p, vol);
        else atb_gather_launch<TIGRE_ATB_MATCHED, true>(grid, block, st, clamp, proj, d_views, nViews, p, vol);
    } else {
        if (mode == TIGRE_ATB_FDK) atb_gather_launch<TIGRE_ATB_FDK, false>(grid, block, st, clamp, proj, d_views, nViews, p, vol);
        else atb_gather_launch<TIGRE_ATB_MATCHED, false>(grid, block, st, clamp, proj, d_views, nViews, p, vol);
    }
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg

extern "C" int tigre_set_atb_path(int path) {
    if (path < 0 || path > 3) return TIGRE_ERR_ARG;
    tg::g_atb_path = path;
    return TIGRE_OK;
}
