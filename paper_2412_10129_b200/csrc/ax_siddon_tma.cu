// ax_siddon_tma.cu — the Siddon forward projector (ax.cu, reading O-A) with the INTERIOR of the march staged into shared
// memory by TMA ("fetch the beam's box with one cp.async.bulk.tensor.3d per group into a shared-memory
// ring, gather from shared memory, keep the voted two-voxel step").
//
// A CTA owns 32 x 4 detector pixels of one view: four consumer warps (one detector row each) and one producer warp.  When all
// its rays run along the same in-plane axis D (x through the transposed copy, or y), the part of the march that every ray of
// the CTA spends inside the volume away from its faces -- absolute slabs [J0, J1) -- is cut into WINDOWS of AXS_SG slabs.
// For each window the producer evaluates the four corner rays of the pixel tile at the window's two bounding D-planes (ray
// positions at a fixed plane are projective-linear in the pixel index, so the corners bound all of them) and issues ONE
// cp.async.bulk.tensor.3d of the BX x AXS_SG x BZ box (E contiguous, D rows, F planes) that holds every voxel the tile's rays
// meet in those slabs.  The consumers march the window's slabs exactly as ax_siddon_kernel does (same state, same lengths,
// same order of summation per ray), with the element offset replaced by a byte offset into the stage: one LDS per voxel, no
// 64-bit address arithmetic, no L1 miss.  Head and tail of every ray (bounds-checked slabs, slabs before J0 and after the
// last whole window), windows whose box does not fit, and CTAs whose rays do not share D take the L1 path of ax.cu.
//
// MEASURED AND NOT THE DEFAULT (profiles/r2_ax_siddon.md): 1176 G samples/s on C3 against the L1 kernel's 1352, results bitwise
// the same.  (1) The march costs as many instructions from shared memory as through L1 (14 against 14.5 per two-voxel slab:
// the L1 kernel's address is one IMAD.WIDE per voxel already), and the window bookkeeping (wait, cell indices, address, arrive:
// 75 instructions per warp and 12 slabs) comes on top: 13.8e9 warp-instructions per launch against 10.2e9, issue slots 77 %
// busy.  (2) A box is 4-5 times the voxels its rays meet (oblique rays drift a voxel per slab along E; slack; 16-byte origin):
// with the L1 kernel's 32 x 4 tile the boxes move 172 GB per launch from L2 (9.8 bytes per ray-sample, 10.3 TB/s: the bound,
// 1022 G samples/s); 32 x 16 tiles bring that to 79 GB.  tigre_set_siddon_path(1) selects this kernel (tests, bench --siddon-path).
#include "ax_siddon.cuh"
#include "tma.cuh"

namespace tg {

namespace {

#ifndef AXS_SG_N
#define AXS_SG_N 12
#endif
#ifndef AXS_STAGES_N
#define AXS_STAGES_N 2
#endif
#ifndef AXS_TV_N
#define AXS_TV_N 16
#endif
#ifndef AXSMB
#define AXSMB 2
#endif
constexpr int AXS_SG = AXS_SG_N;           // slabs per window: a multiple of AXG
constexpr int AXS_STAGES = AXS_STAGES_N;
constexpr int AXS_TV = AXS_TV_N;           // detector rows per CTA: the box of a window is shared by 32 x AXS_TV rays (a 32 x 4 tile moves
                                           // 9.8 bytes per ray-sample from L2 into its boxes -- 10 TB/s, the kernel's bound; 32 x 16 moves 2.5)
constexpr int AXS_NW = AXS_TV;             // consumer warps
static_assert(AXS_SG % AXG == 0, "a window is a whole number of voted groups");
static_assert(AX_TU == 32, "one warp per detector row of the tile");

struct AxsStage {
    int bx, bz;   // voxel index (along E, F) of the box origin
    int fits, pad;
};

// spin on an mbarrier phase with the address in a register (tma.cuh's mbar_wait re-forms it after every failed try)
__device__ __forceinline__ void mbar_wait_addr(uint32_t bar, uint32_t parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "AXS_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra AXS_DONE;\n"
        "bra AXS_WAIT;\n"
        "AXS_DONE:\n"
        "}\n" ::"r"(bar),
        "r"(parity)
        : "memory");
}

// r.off is an absolute 32-bit shared-memory ADDRESS in the window march (stage base folded in): one LDS, no address arithmetic.
// (Through a pointer plus a byte offset nvcc re-formed stage * stageBytes + base before every load: three instructions per voxel.)
__device__ __forceinline__ float lds_b(int, int addr) {
    float v;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(v) : "r"(addr));
    return v;
}

// The interior slab steps of ax_siddon.cuh with the voxel offset a BYTE offset into the staged box (strides r.stE, r.stF, r.sD
// in bytes too): the same lengths and the same operations on the values.
__device__ __forceinline__ void slab_fast_s(int tb, SidRay<int>& r) {
    const float se = __saturatef(fmaf(r.hE, r.imE, -r.kf)), sf = __saturatef(fmaf(r.hF, r.imF, -r.kf));
    r.kf += 1.0f;
    const bool cE = se < 1.0f, cF = sf < 1.0f;
    const float s1 = fminf(se, sf);
    const int offC = r.off + (cE ? r.stE : 0) + (cF ? r.stF : 0);
    const bool both = cE && cF;
    const float s2 = both ? fmaxf(se, sf) : s1;
    const float vA = lds_b(tb, r.off);
    float vC = vA;
    if (cE || cF) vC = lds_b(tb, offC);
    r.acc = fmaf(s1, vA, r.acc);
    if (both) r.vB = lds_b(tb, r.off + ((se < sf) ? r.stE : r.stF));
    r.acc = fmaf(s2 - s1, r.vB, r.acc);
    r.acc = fmaf(1.0f - s2, vC, r.acc);
    if (cE) r.hE += r.sgE;
    if (cF) r.hF += r.sgF;
    r.off = offC + r.sD;
}
__device__ __forceinline__ void slab_e_only_s(int tb, SidRay<int>& r) {
    const float se = __saturatef(fmaf(r.hE, r.imE, -r.kf));
    r.kf += 1.0f;
    const bool cE = se < 1.0f;
    const int offC = r.off + (cE ? r.stE : 0);
    const float vA = lds_b(tb, r.off);
    float vC = vA;
    if (cE) vC = lds_b(tb, offC);
    r.acc = fmaf(se, vA, r.acc);
    r.acc = fmaf(1.0f - se, vC, r.acc);
    if (cE) r.hE += r.sgE;
    r.off = offC + r.sD;
}

}  // namespace

__global__ void __launch_bounds__(32 * (AXS_NW + 1), AXSMB)
ax_siddon_tma_kernel(const __grid_constant__ CUtensorMap mapV, const __grid_constant__ CUtensorMap mapT, const float* __restrict__ vol,
                     const float* __restrict__ volT, const RayView* __restrict__ views, int nViews, AxP p, int BX, int BZ,
                     float* __restrict__ proj) {   // p.nVt counts THIS kernel's tiles of AXS_TV rows
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int PLANE = BX * AXS_SG;            // elements per F-plane of a stage
    const int stageBytes = PLANE * BZ * 4;    // a multiple of 128 (BX a multiple of 4, AXS_SG a multiple of 6: checked by the launcher)
    unsigned char* tiles = smem_raw;
    uint64_t* full = reinterpret_cast<uint64_t*>(tiles + (size_t)AXS_STAGES * stageBytes);
    uint64_t* empty = full + AXS_STAGES;
    AxsStage* info = reinterpret_cast<AxsStage*>(empty + AXS_STAGES);
    int* range = reinterpret_cast<int*>(info + AXS_STAGES);   // [0] = J0: first slab of the first window, [1] = J1: end of the common interior

    const int lane = threadIdx.x, warp = threadIdx.y;
    long long tb = blockIdx.x;   // ax_decode's tile order
    const int ut = (int)(tb % p.nUt);
    tb /= p.nUt;
    const int view = (int)(tb % nViews), vt = (int)(tb / nViews);
    const int iu0 = ut * AX_TU, iv0 = p.iv0 + vt * AXS_TV;
    const RayView& rv = views[view];
    if (lane == 0 && warp == 0) {
        for (int s = 0; s < AXS_STAGES; ++s) {
            mbar_init(full + s, 1);
            mbar_init(empty + s, AXS_NW);
        }
        range[0] = (int)0x80000000, range[1] = 0x7fffffff;
        mbar_fence_init();
    }
    __syncthreads();

    // ---- per-ray set-up (consumers), fp64: ax_siddon.cuh
    const bool consumer = warp < AXS_NW;
    const int iu = iu0 + lane, iv = iv0 + warp;
    const bool mine = consumer && iu < p.nu && iv < p.iv1;
    SidRay<int> r;
    SidSetup q;
    q.D = 1, q.i0 = 0, q.nslab = 0, q.kA = 0, q.kB = 0, q.ie = q.jf = q.ie0 = q.jf0 = 0, q.diE = q.diF = 1, q.nE = q.nF = 1;
    q.slo0 = 0.f, q.shiN = 1.f, q.scale = 0.f, q.hE0 = q.hF0 = 0.0, q.useT = false;
    r.imE = r.imF = 1.f, r.sgE = r.sgF = 1.f, r.hE = r.hF = 3.0e38f, r.stE = r.stF = r.sD = 0, r.kf = 0.f, r.acc = 0.f, r.vB = 0.f, r.off = 0;
    if (mine) siddon_setup<int, false>(rv, p, iu, iv, true, r, q);
    const int i0 = q.i0, nslab = q.nslab, kB = q.kB;
    int kA = q.kA, ie = q.ie, jf = q.jf;
    const float hEinit = r.hE, hFinit = r.hF;
    // the head (bounds-checked slabs) of every lane is stretched to the deepest start in its warp, as in ax_siddon_kernel
    int jmax;
    {
        const bool any = kB > kA;
        jmax = __reduce_max_sync(0xffffffffu, any ? i0 + kA : (int)0x80000000);
        if (any) kA = min(max(kA, jmax - i0), kB);
    }
    const bool ranFast = kB > kA;
    const int jendmin = __reduce_min_sync(0xffffffffu, ranFast ? i0 + kB : 0x7fffffff);
    if (consumer && lane == 0 && jendmin != 0x7fffffff) atomicMax(range, jmax), atomicMin(range + 1, jendmin);
    // windows need every marching ray of the CTA on the same in-plane dominant axis (hence in the same layout, E contiguous)
    const int allY = __syncthreads_and((!ranFast || q.D == 1) ? 1 : 0);
    const int allX = __syncthreads_and((!ranFast || q.D == 0) ? 1 : 0);   // (also orders the atomics before the reads below)
    const bool useT = allX && !allY;
    const int J0 = range[0], J1 = range[1];
    const int nWin = ((allX || allY) && J1 > J0) ? (J1 - J0) / AXS_SG : 0;

    if (!consumer) {
        // ---------------------------------------------------------------- producer warp: lanes 0..3 own the tile's corner rays
        if (nWin == 0) return;
        const double pu = (lane & 1) ? fmin((double)(iu0 + AX_TU - 1), (double)(p.nu - 1)) : (double)iu0;
        const double pv = (lane & 2) ? fmin((double)(iv0 + AXS_TV - 1), (double)(p.iv1 - 1)) : (double)iv0;
        double S[3], d[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            S[k] = rv.S[k] + pu * rv.dSU[k] + pv * rv.dSV[k];
            d[k] = rv.P0[k] + pu * rv.dU[k] + pv * rv.dV[k] - S[k];
        }
        const double SD = useT ? S[0] : S[1], SE = useT ? S[1] : S[0], dD = useT ? d[0] : d[1], dE = useT ? d[1] : d[0];
        const double mE = dD != 0.0 ? dE / dD : 0.0, mF = dD != 0.0 ? d[2] / dD : 0.0;
        const CUtensorMap* map = useT ? &mapT : &mapV;
        int s = 0;
        uint32_t ph = 1;
        for (int w = 0; w < nWin; ++w) {
            const int yA = J0 + w * AXS_SG;
            const double ea = SE + ((double)yA - SD) * mE, eb = SE + ((double)(yA + AXS_SG) - SD) * mE;
            const double fa = S[2] + ((double)yA - SD) * mF, fb = S[2] + ((double)(yA + AXS_SG) - SD) * mF;
            float elo = (float)fmin(ea, eb), ehi = (float)fmax(ea, eb), flo = (float)fmin(fa, fb), fhi = (float)fmax(fa, fb);
#pragma unroll
            for (int o = 2; o > 0; o >>= 1) {
                elo = fminf(elo, __shfl_xor_sync(0xffffffffu, elo, o)), ehi = fmaxf(ehi, __shfl_xor_sync(0xffffffffu, ehi, o));
                flo = fminf(flo, __shfl_xor_sync(0xffffffffu, flo, o)), fhi = fmaxf(fhi, __shfl_xor_sync(0xffffffffu, fhi, o));
            }
            if (lane == 0) {
                int fits = 0, bx = 0, bz = 0;
                if (fabsf(elo) < 1.0e6f && fabsf(ehi) < 1.0e6f && fabsf(flo) < 1.0e6f && fabsf(fhi) < 1.0e6f) {
                    // one voxel of slack on either side (the march decides its crossings in fp32); origin on a 16-byte boundary
                    bx = ((int)floorf(elo) - 1) & ~3, bz = (int)floorf(flo) - 1;
                    fits = ((int)floorf(ehi) + 2 - bx <= BX) && ((int)floorf(fhi) + 2 - bz <= BZ);
                }
                if (w >= AXS_STAGES) mbar_wait_addr(smem_u32(empty + s), ph);
                info[s].bx = bx, info[s].bz = bz, info[s].fits = fits;
                if (fits) {
                    mbar_arrive_expect_tx(full + s, (uint32_t)stageBytes);
                    tma_load_3d(tiles + (size_t)s * stageBytes, map, bx, yA, bz, full + s);
                } else {
                    mbar_arrive(full + s);
                }
            }
            __syncwarp();
            if (++s == AXS_STAGES) s = 0, ph ^= 1;
        }
        return;
    }

    // ---------------------------------------------------------------- consumers
    const size_t out = ((size_t)view * p.nv + iv) * p.nu + iu;
    const float* base = q.useT ? volT : vol;
    asm volatile("" : "+l"(base));
    const int diE = q.diE, diF = q.diF, nE = q.nE, nF = q.nF;
    const int last = nslab - 1;
    int k = 0;
    for (; k < kA; ++k)
        siddon_slab_checked<int, false, false, false>(base, r, ie, jf, diE, diF, nE, nF, k == 0 ? q.slo0 : 0.f, k == last ? q.shiN : 1.f);
    int jcur = jmax;   // absolute slab the marching lanes of this warp stand at (warp-uniform)
    if (nWin > 0) {   // every consumer warp takes part in the ring, with or without marching lanes
        const unsigned fmask = __ballot_sync(0xffffffffu, ranFast);
        // up to the first window through L1 (at most a few slabs: the warps of a tile start within a voxel or two of each other)
        if (ranFast)
            for (int j = jcur; j < J0; ++j) siddon_slab_fast<int, false, false, false>(base, r);
        if (ranFast) k += J0 - jcur;
        jcur = J0;
        const int gD = r.sD, gE = r.stE, gF = r.stF;   // global element strides, put back after the windows
        const int sE = gE > 0 ? 4 : -4, sF = gF > 0 ? PLANE * 4 : -PLANE * 4, sD = BX * 4;
        const uint32_t full_s = smem_u32(full), tiles_s = smem_u32(tiles);
        int s = 0;
        uint32_t ph = 0;
        for (int w = 0; w < nWin; ++w) {
            mbar_wait_addr(full_s + 8u * (uint32_t)s, ph);
            if (ranFast) {
                // the cell this ray stands in at the start of the window, from the plane state (moves by one per crossing)
                const int ieW = r.hE < 1.0e38f ? q.ie0 + __float2int_rn(r.hE - hEinit) : q.ie0;
                const int jfW = r.hF < 1.0e38f ? q.jf0 + __float2int_rn(r.hF - hFinit) : q.jf0;
                if (info[s].fits) {
                    const int tb = 0;
                    r.stE = sE, r.stF = sF, r.sD = sD;
                    // row 0 of the box = this window's first slab
                    r.off = (int)tiles_s + s * stageBytes + 4 * ((jfW - info[s].bz) * PLANE + (ieW - info[s].bx));
#ifdef AXS_CHECK   // debug build: the ray's cell must lie inside the box with a voxel to spare at the start of every window
                    if (ieW - info[s].bx < 1 || ieW - info[s].bx > BX - 2 || jfW - info[s].bz < 1 || jfW - info[s].bz > BZ - 2) __trap();
#endif
#pragma unroll
                    for (int g = 0; g < AXS_SG / AXG; ++g) {
                        const bool nearF = fmaf(r.hF, r.imF, -r.kf) <= (float)AXG;
                        if (__any_sync(fmask, nearF)) {
#pragma unroll
                            for (int j = 0; j < AXG; ++j) slab_fast_s(tb, r);
                        } else {
#pragma unroll
                            for (int j = 0; j < AXG; ++j) slab_e_only_s(tb, r);
                        }
                    }
                    r.stE = gE, r.stF = gF, r.sD = gD;
                } else {
                    r.off = (jcur + w * AXS_SG) * gD + ieW * (gE > 0 ? gE : -gE) + jfW * (gF > 0 ? gF : -gF);
                    for (int j = 0; j < AXS_SG; ++j) siddon_slab_fast<int, false, false, false>(base, r);
                }
            }
            __syncwarp();
            if (lane == 0) mbar_arrive(empty + s);
            if (++s == AXS_STAGES) s = 0, ph ^= 1;
        }
        if (ranFast) {
            k += nWin * AXS_SG;
            const int ieW = r.hE < 1.0e38f ? q.ie0 + __float2int_rn(r.hE - hEinit) : q.ie0;
            const int jfW = r.hF < 1.0e38f ? q.jf0 + __float2int_rn(r.hF - hFinit) : q.jf0;
            r.off = (i0 + k) * gD + ieW * (gE > 0 ? gE : -gE) + jfW * (gF > 0 ? gF : -gF);
        }
        jcur = J0 + nWin * AXS_SG;
    }
    {
        // the rest of the warp's common interior in voted groups through L1, as in ax_siddon_kernel
        const int groups = jendmin == 0x7fffffff ? 0 : (jendmin - jcur) / AXG;
        for (int g = 0; g < groups; ++g) {
            const bool nearF = ranFast && fmaf(r.hF, r.imF, -r.kf) <= (float)AXG;
            if (__any_sync(0xffffffffu, nearF)) {
                if (ranFast) {
#pragma unroll
                    for (int j = 0; j < AXG; ++j) siddon_slab_fast<int, false, false, false>(base, r);
                }
            } else if (ranFast) {
#pragma unroll
                for (int j = 0; j < AXG; ++j) siddon_slab_e_only<int, false, false, false>(base, r);
            }
        }
        if (ranFast) k += AXG * groups;
    }
    for (; k < kB; ++k) siddon_slab_fast<int, false, false, false>(base, r);
    if (k < nslab) {
        if (ranFast) {
            if (r.hE < 1.0e38f) ie = q.ie0 + (int)rint((double)r.hE - q.hE0);
            if (r.hF < 1.0e38f) jf = q.jf0 + (int)rint((double)r.hF - q.hF0);
        }
        for (; k < nslab; ++k)
            siddon_slab_checked<int, false, false, false>(base, r, ie, jf, diE, diF, nE, nF, k == 0 ? q.slo0 : 0.f, k == last ? q.shiN : 1.f);
    }
    if (mine) {
        const float result = r.acc * q.scale;
        proj[out] = p.accumulate ? proj[out] + result : result;
    }
}

int g_ax_siddon_path = 0;   // 0 = L1 kernel of ax.cu (faster: see the head of this file), 1 = this kernel where the problem qualifies (tigre_set_siddon_path)

// Returns TIGRE_OK if the staged kernel was launched, 1 if this problem does not qualify (the caller runs the L1 kernel), a
// negative status on a CUDA error.  h_views: host copy of the views' table (sizes the staged box).
int launch_ax_siddon_tma(const float* vol, const float* volT, const Grid& g, const RayView* d_views, const RayView* h_views, int nViews,
                         const AxP& p, float* proj, cudaStream_t st) {
    if (g_ax_siddon_path != 1 || !h_views || !vol || !volT || !tensor_map_encoder()) return 1;
    if ((g.nx & 3) || (g.ny & 3) || g.nx < 2 * AXS_SG || g.ny < 2 * AXS_SG || g.nz < 2 || nViews < 1) return 1;
    if ((reinterpret_cast<uintptr_t>(vol) & 15) || (reinterpret_cast<uintptr_t>(volT) & 15)) return 1;
    if (p.iv0 != 0 || p.iv1 != g.nv) return 1;   // (row bands of the chunked path keep the L1 kernel)
    // box size: the largest extent, over a sample of views, tiles and windows, of the four corner rays of a pixel tile between
    // the two bounding planes of a window (what the producer evaluates); windows that still do not fit take the L1 path
    double ex = 0.0, ez = 0.0;
    const int vstep = std::max(1, nViews / 24);
    for (int a = 0; a < nViews; a += vstep) {
        const RayView& rv = h_views[a];
        for (int ti = 0; ti < 9; ++ti) {
            const int iu0 = std::min((g.nu - 1) / AX_TU, (ti % 3) * ((g.nu / AX_TU) / 2)) * AX_TU;
            const int nvt = (g.nv + AXS_TV - 1) / AXS_TV;
            const int iv0 = std::min(nvt - 1, (ti / 3) * (nvt / 2)) * AXS_TV;
            double S[4][3], d[4][3];
            for (int c = 0; c < 4; ++c) {
                const double pu = (c & 1) ? std::min(iu0 + AX_TU - 1, g.nu - 1) : iu0, pv = (c & 2) ? std::min(iv0 + AXS_TV - 1, g.nv - 1) : iv0;
                for (int k = 0; k < 3; ++k) {
                    S[c][k] = rv.S[k] + pu * rv.dSU[k] + pv * rv.dSV[k];
                    d[c][k] = rv.P0[k] + pu * rv.dU[k] + pv * rv.dV[k] - S[c][k];
                }
            }
            const bool useT = std::fabs(d[0][0]) > std::fabs(d[0][1]);
            const int iD = useT ? 0 : 1, iE = useT ? 1 : 0, nD = useT ? g.nx : g.ny;
            for (int wi = 0; wi < 3; ++wi) {
                const double yA = std::min(nD - AXS_SG, wi * (nD / 2));
                double elo = 1e300, ehi = -1e300, flo = 1e300, fhi = -1e300;
                for (int c = 0; c < 4; ++c) {
                    if (d[c][iD] == 0.0) continue;
                    for (int e = 0; e < 2; ++e) {
                        const double t = (yA + e * AXS_SG - S[c][iD]) / d[c][iD];
                        const double pe = S[c][iE] + t * d[c][iE], pf = S[c][2] + t * d[c][2];
                        elo = std::min(elo, pe), ehi = std::max(ehi, pe), flo = std::min(flo, pf), fhi = std::max(fhi, pf);
                    }
                }
                if (std::isfinite(elo) && std::isfinite(ehi) && ehi >= elo) ex = std::max(ex, ehi - elo), ez = std::max(ez, fhi - flo);
            }
        }
    }
    const int needX = (int)std::ceil(ex) + 7, needZ = (int)std::ceil(ez) + 4;   // floor span, a voxel of slack either side, 16-byte aligned origin
    // plane pitch of 16 mod 32 words: the lanes of a warp sit in one row of at most two adjacent F-planes, ~17 columns wide
    int BX = (needX + 3) & ~3;
    for (int c = BX; c < BX + 32; c += 4)
        if ((c * AXS_SG) % 32 == 16) {
            BX = c;
            break;
        }
    const int BZ = (std::max(4, needZ) + 1) & ~1;
    const size_t stage = (size_t)BX * AXS_SG * BZ * sizeof(float);
    if (BX > 256 || BZ > 64 || AXS_STAGES * stage > 100 * 1024) return 1;
    CUtensorMap mapV, mapT;
    const cuuint32_t box[3] = {(cuuint32_t)BX, (cuuint32_t)AXS_SG, (cuuint32_t)BZ};
    const cuuint64_t dimV[3] = {(cuuint64_t)g.nx, (cuuint64_t)g.ny, (cuuint64_t)g.nz};
    const cuuint64_t strV[2] = {(cuuint64_t)g.nx * sizeof(float), (cuuint64_t)g.nx * g.ny * sizeof(float)};
    const cuuint64_t dimT[3] = {(cuuint64_t)g.ny, (cuuint64_t)g.nx, (cuuint64_t)g.nz};
    const cuuint64_t strT[2] = {(cuuint64_t)g.ny * sizeof(float), (cuuint64_t)g.nx * g.ny * sizeof(float)};
    if (!encode_f32_map(&mapV, vol, 3, dimV, strV, box) || !encode_f32_map(&mapT, volT, 3, dimT, strT, box)) return 1;
    const size_t smem = AXS_STAGES * stage + 2 * AXS_STAGES * sizeof(uint64_t) + AXS_STAGES * sizeof(AxsStage) + 2 * sizeof(int);
    TG_CUDA(cudaFuncSetAttribute(ax_siddon_tma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    AxP ps = p;
    ps.nVt = (g.nv + AXS_TV - 1) / AXS_TV;
    const long long nblk = (long long)ps.nUt * ps.nVt * nViews;
    dim3 block(32, AXS_NW + 1), grid((unsigned)nblk);
    ax_siddon_tma_kernel<<<grid, block, smem, st>>>(mapV, mapT, vol, volT, d_views, nViews, ps, BX, BZ, proj);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg

extern "C" TIGRE_API int tigre_set_siddon_path(int path) {
    if (path < 0 || path > 1) return TIGRE_ERR_ARG;
    tg::g_ax_siddon_path = path;
    return TIGRE_OK;
}
