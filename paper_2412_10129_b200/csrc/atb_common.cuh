// atb_common.cuh — arithmetic shared by the two voxel-driven backprojection kernels (atb.cu: taps
// gathered through L1/L2; atb_tma.cu: detector footprints staged into shared memory by TMA).
// Weights (reading P10 of DESIGN.md; PAPER.md:90, 114 for FDK):
//   matched  w = (dx dy dz)/(du dv) * R^2/(r^2 cos g) = km * t^2 * R(u,v)
//   FDK      w = (DSO/(DSO - X'_x))^2 = 1/G^2
#pragma once
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
    int magic;            // 0x4B400000 = bits of 1.5*2^23 (floor_magic), passed as data (see atb_tma.cu)
    int lin_ok;           // atb_tma.cu: tilted views may take the linearised z-run (0 = always the per-voxel reciprocal: tigre_set_atb_path(3))
    // fusion F2: the kernel's output IS the SART update.  With fuse != 0, `vol` is the iterate x (slab pointer, like
    // the output otherwise): x <- max(0, x + lambda V .* (A^T r)) is formed in the epilogue from the accumulators, and the (x,y)-transposed
    // copy xT gets the new value too; V and xT are slab pointers like vol.  The backprojector is issue-bound and leaves HBM idle, so the
    // update's traffic hides behind the other CTAs' arithmetic, and the gradient volume is neither written nor read.
    int fuse, nonneg;
    float lambda;
    const float* V;
    float* xT;
};

constexpr int ATB_BX = 32, ATB_BY = 8;

// ---- arithmetic shared by the gather and the TMA kernels -------------------------------------
// 1/x and sqrt(x) from the SFU approximations (max rel. error ~1 ulp / ~2 ulp): the IEEE sequences
// cost 8-10 issue slots each and the kernels are issue-bound (profiles/r1_baseline_ncu_full.md).
__device__ __forceinline__ float rcp_fast(float x) {
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_fast(float x) {
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
// floor(x) and its integer value for |x| < 2^21 without the conversion pipe: adding 1.5*2^23 leaves
// round-to-nearest(x - 1/2) in the low mantissa bits.  At exact integers the result may be x-1 with
// fraction 1, which gives the same bilinear value.  Callers clamp x when the geometry allows |x| >= 2^21.
__device__ __forceinline__ float floor_magic(float x, int& i) {
    const float m = 12582912.0f;   // 1.5 * 2^23 = 0x4B400000
    const float t = (x - 0.5f) + m;
    i = __float_as_int(t) - 0x4B400000;
    return t - m;
}

struct TapW {   // per voxel-view: bilinear fractions, integer tap (detector index), weight
    float au, av, w;
    int iu, iv;
};
template <int MODE, bool CLAMP>
__device__ __forceinline__ TapW voxel_view(float U, float V, float W, float G, const float4& cst, const AtbP& p) {
    TapW o;
    const float t = rcp_fast(W);
    float fu = U * t, fv = V * t;   // detector index minus nu/2, nv/2
    if (MODE == TIGRE_ATB_FDK) {
        const float ig = rcp_fast(G);
        o.w = ig * ig;
    } else {
        const float eu = fu - cst.z, ev = fv - cst.w;
        o.w = (cst.x * t) * t * sqrt_fast(fmaf(p.du2 * eu, eu, fmaf(p.dv2 * ev, ev, cst.y)));
    }
    if (CLAMP) {
        fu = fminf(fmaxf(fu, -2.0e6f), 2.0e6f);
        fv = fminf(fmaxf(fv, -2.0e6f), 2.0e6f);
    }
    int iu, iv;
    const float flu = floor_magic(fu, iu), flv = floor_magic(fv, iv);
    o.au = fu - flu, o.av = fv - flv;
    o.iu = iu + p.hu, o.iv = iv + p.hv;
    return o;
}

// bilinear value of one view at tap (iu, iv) (absolute detector indices), zero border, through L1/L2.
// pa points at the view's first present row (row0); nrows rows of nu pixels are present.
__device__ __forceinline__ float bilinear_global(const float* __restrict__ pa, int iu, int iv, float au, float av,
                                                 const AtbP& p) {
    const int lv = iv - p.row0;
    const float* q = pa + (ptrdiff_t)lv * p.nu + iu;
    float p00, p10, p01, p11;
    if ((unsigned)iu < (unsigned)(p.nu - 1) && (unsigned)lv < (unsigned)(p.nrows - 1)) {   // all four taps inside
        p00 = __ldg(q), p10 = __ldg(q + 1), p01 = __ldg(q + p.nu), p11 = __ldg(q + p.nu + 1);
    } else {
        const bool u0 = (unsigned)iu < (unsigned)p.nu, u1 = (unsigned)(iu + 1) < (unsigned)p.nu;
        const bool v0 = (unsigned)lv < (unsigned)p.nrows, v1 = (unsigned)(lv + 1) < (unsigned)p.nrows;
        p00 = (u0 && v0) ? __ldg(q) : 0.f;
        p10 = (u1 && v0) ? __ldg(q + 1) : 0.f;
        p01 = (u0 && v1) ? __ldg(q + p.nu) : 0.f;
        p11 = (u1 && v1) ? __ldg(q + p.nu + 1) : 0.f;
    }
    const float r0 = fmaf(au, p10 - p00, p00), r1 = fmaf(au, p11 - p01, p01);
    return fmaf(av, r1 - r0, r0);
}

}  // namespace tg
