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
#include "common.cuh"

namespace tg {

struct AtbP {
    int nx, ny, nz;       // full volume size (centred coordinates refer to it)
    int nu, nv;
    int z0, nzs;          // z-slices written: [z0, z0+nzs); vol points at slice z0
    int row0, nrows;      // detector rows present in the projection buffer
    float cx, cy, cz;     // (n-1)/2
    float du2, dv2;       // pixel pitch squared, mm^2
    int hu, hv;           // nu/2, nv/2
    int accumulate;
};

constexpr int ATB_BX = 32, ATB_BY = 8;

template <int MODE, bool UNIT, int ZR>
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
            const float W = fmaf(kf, rW.z, W0);
            const float t = 1.0f / W;
            const float fu = fmaf(kf, rU.z, U0) * t, fv = fmaf(kf, rV.z, V0) * t;   // minus nu/2, nv/2
            float w;
            if (MODE == TIGRE_ATB_FDK) {
                const float G = fmaf(kf, rG.z, G0);
                const float ig = 1.0f / G;
                w = ig * ig;
            } else {
                const float eu = fu - cst.z, ev = fv - cst.w;
                w = cst.x * t * t * sqrtf(fmaf(p.du2 * eu, eu, fmaf(p.dv2 * ev, ev, cst.y)));
            }
            const float flu = floorf(fu), flv = floorf(fv);
            const float au = fu - flu, av = fv - flv;
            const int iu = (int)flu + p.hu, iv = (int)flv + p.hv;
            // zero border on the true detector bounds
            const bool u0 = (unsigned)iu < (unsigned)p.nu, u1 = (unsigned)(iu + 1) < (unsigned)p.nu;
            const bool v0 = (unsigned)iv < (unsigned)p.nv, v1 = (unsigned)(iv + 1) < (unsigned)p.nv;
            float val;
            if (UNIT) {
                val = ((u0 ? 1.f - au : 0.f) + (u1 ? au : 0.f)) * ((v0 ? 1.f - av : 0.f) + (v1 ? av : 0.f));
            } else {
                const float* q = pa + (ptrdiff_t)(iv - p.row0) * p.nu + iu;
                const float p00 = (u0 && v0) ? __ldg(q) : 0.f;
                const float p10 = (u1 && v0) ? __ldg(q + 1) : 0.f;
                const float p01 = (u0 && v1) ? __ldg(q + p.nu) : 0.f;
                const float p11 = (u1 && v1) ? __ldg(q + p.nu + 1) : 0.f;
                const float r0 = fmaf(au, p10 - p00, p00), r1 = fmaf(au, p11 - p01, p01);
                val = fmaf(av, r1 - r0, r0);
            }
            acc[k] = fmaf(w, val, acc[k]);
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

int launch_atb(const float* proj, const Grid& g, const VoxView* d_views, int nViews, int mode, bool unit_proj,
               float* vol, int z0, int nzs, bool accumulate, int row0, int nrows, cudaStream_t st) {
    if (mode != TIGRE_ATB_MATCHED && mode != TIGRE_ATB_FDK) return TIGRE_ERR_ARG;
    AtbP p;
    p.nx = g.nx, p.ny = g.ny, p.nz = g.nz, p.nu = g.nu, p.nv = g.nv;
    p.z0 = z0, p.nzs = nzs, p.row0 = row0, p.nrows = nrows;
    p.cx = 0.5f * (g.nx - 1), p.cy = 0.5f * (g.ny - 1), p.cz = 0.5f * (g.nz - 1);
    p.du2 = (float)(g.du * g.du), p.dv2 = (float)(g.dv * g.dv);
    p.hu = g.nu / 2, p.hv = g.nv / 2;
    p.accumulate = accumulate ? 1 : 0;
    constexpr int ZR = 8;
    dim3 block(ATB_BX, ATB_BY);
    dim3 grid((g.nx + ATB_BX - 1) / ATB_BX, (g.ny + ATB_BY - 1) / ATB_BY, (nzs + ZR - 1) / ZR);
    if (grid.y > 65535 || grid.z > 65535) return TIGRE_ERR_ARG;
    ProfScope ps(PK_ATB, st);
    if (unit_proj) {
        if (mode == TIGRE_ATB_FDK) atb_gather_kernel<TIGRE_ATB_FDK, true, ZR><<<grid, block, 0, st>>>(proj, d_views, nViews, p, vol);
        else atb_gather_kernel<TIGRE_ATB_MATCHED, true, ZR><<<grid, block, 0, st>>>(proj, d_views, nViews, p, vol);
    } else {
        if (mode == TIGRE_ATB_FDK) atb_gather_kernel<TIGRE_ATB_FDK, false, ZR><<<grid, block, 0, st>>>(proj, d_views, nViews, p, vol);
        else atb_gather_kernel<TIGRE_ATB_MATCHED, false, ZR><<<grid, block, 0, st>>>(proj, d_views, nViews, p, vol);
    }
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg
