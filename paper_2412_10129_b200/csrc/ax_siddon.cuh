// ax_siddon.cuh — the Siddon march shared by ax.cu (volume gathered through L1) and ax_siddon_tma.cu (interior of the march staged
// into shared memory by TMA): per-ray state, the three slab steps, and the fp64 per-ray set-up as a function.  See the head of
// ax.cu for the method.  (The set-up's text lives in ax_siddon_setup.inc and is included by ax_siddon_kernel directly and by siddon_setup() here.)
#pragma once
#include <cmath>
#include "ax_common.cuh"

namespace tg {

// Per-ray marching state shared by the checked (end slabs) and unchecked (interior) slab steps.
template <typename IdxT>
struct SidRay {
    float imE, imF, sgE, sgF;                       // 1/mE, 1/mF (1 if the ray never crosses), plane step +-1
    IdxT stE, stF, sD;                              // signed element strides of one step along E, F, D
    // distance (in voxels along E / F) from the ray's position at the start of slab 0 to the next E / F plane
    // ahead of it.  Grows by exactly +-1 per crossing (magnitudes <= n: the adds are exact up to one ulp of the
    // largest value, they do not accumulate); the crossing's position inside slab k is hE/mE - k, one FFMA.
    float hE, hF;
    float kf, acc, vB;
    float ys;                                       // scatter (exact adjoint): ray value times the length scale
    IdxT off;                                       // element offset of the current voxel
    // TRACK instantiation only (tigre_Ax_index, reading P19(a)): element offsets of the first / last voxel met with a
    // non-zero length, and the number of such voxels
    long long first, last;
    uint32_t nseg;
    bool pok;      // SCATTER only: lane ^ 1 is in fm and scatters into the same array
    unsigned fm;   // SCATTER only: the lanes of the warp that run the warp-uniform groups of the interior together
    __device__ __forceinline__ void note(IdxT o, float len) {
        if (len > 0.f) {
            if (nseg == 0) first = (long long)o;
            last = (long long)o;
            ++nseg;
        }
    }
};

// Exact-adjoint scatter inside the warp-uniform groups: the lanes named in fm execute this together and are in the same slab.
// Neighbouring rays are less than a voxel apart on most geometries, so lanes 2j and 2j + 1 often add to the SAME voxel; then the
// even lane adds both values in one REDG (the L1 -> L2 reduction path, not the issue slots, is what binds the scatter kernels:
// profiles/r2_scatter.md).  Any pairing is correct; runs that straddle a pair boundary just stay two operations.  pok: the
// partner lane runs the groups too AND adds into the same array (vol or its transposed copy) -- equal offsets then mean one voxel.
// (Merging runs of up to three lanes at any alignment -- 3 shuffles, a vote and a CLZ per REDG -- was measured slower than no
// merging at all: 582 against 700 G samples/s on C3; this two-shuffle pairing gives 785.)
#ifndef AX_NO_PAIR
template <typename IdxT>
__device__ __forceinline__ void red_pair(float* out, IdxT off, float v, unsigned fm, bool pok) {
    const IdxT o2 = __shfl_xor_sync(fm, off, 1);
    const float v2 = __shfl_xor_sync(fm, v, 1);
    const bool same = pok && o2 == off;
    if (same && (threadIdx.x & 1u)) return;   // blockDim.x is a multiple of 32: the parity of threadIdx.x is the lane's
    red_add_global(out + off, same ? v + v2 : v);
}
#else
template <typename IdxT>
__device__ __forceinline__ void red_pair(float* out, IdxT off, float v, unsigned, bool) { red_add_global(out + off, v); }
#endif

// One D-slab, interior of the volume: the whole slab [0,1] lies inside the ray's clipped range and at
// least 1e-3 voxel away from the lateral faces, so no clipping and no bounds checks are needed.
template <typename IdxT, bool UNIT, bool SCATTER, bool TRACK = false, bool PAIR = false>
__device__ __forceinline__ void siddon_slab_fast(const float* __restrict__ base, SidRay<IdxT>& r) {
    // slab-local parameter of the next E / F plane crossing, saturated to [0,1] (1 = not in this slab)
    const float se = __saturatef(fmaf(r.hE, r.imE, -r.kf)), sf = __saturatef(fmaf(r.hF, r.imF, -r.kf));
    r.kf += 1.0f;
    const bool cE = se < 1.0f, cF = sf < 1.0f;
    const float s1 = fminf(se, sf);
    const IdxT offC = r.off + (cE ? r.stE : (IdxT)0) + (cF ? r.stF : (IdxT)0);
    // a lane that crosses both planes inside this slab meets a middle voxel between the two crossings; for
    // the other lanes the middle piece has zero length
    const bool both = cE && cF;
    const float s2 = both ? fmaxf(se, sf) : s1;
    if (TRACK) {
        r.note(r.off, s1);
        if (both) r.note(r.off + ((se < sf) ? r.stE : r.stF), s2 - s1);
        r.note(offC, 1.0f - s2);
    } else if (SCATTER) {
        // exact adjoint: the same three lengths, added to the voxels instead of gathered from them
        float* out = const_cast<float*>(base);
        if (PAIR) red_pair(out, r.off, s1 * r.ys, r.fm, r.pok);
        else red_add_global(out + r.off, s1 * r.ys);
        if (both) red_add_global(out + (r.off + ((se < sf) ? r.stE : r.stF)), (s2 - s1) * r.ys);
        if (PAIR) red_pair(out, offC, (1.0f - s2) * r.ys, r.fm, r.pok);
        else red_add_global(out + offC, (1.0f - s2) * r.ys);
    } else {
        const float vA = UNIT ? 1.f : __ldg(base + r.off);
        float vC = vA;   // a lane that stays in its voxel does not load it twice
        if (!UNIT && (cE || cF)) vC = __ldg(base + offC);
        r.acc = fmaf(s1, vA, r.acc);
        // (the middle weight multiplies the last value loaded when this lane has no middle voxel: times zero)
        if (both && !UNIT) r.vB = __ldg(base + (r.off + ((se < sf) ? r.stE : r.stF)));
        r.acc = fmaf(s2 - s1, UNIT ? 1.f : r.vB, r.acc);
        r.acc = fmaf(1.0f - s2, vC, r.acc);
    }
    if (cE) r.hE += r.sgE;
    if (cF) r.hF += r.sgF;
    r.off = offC + r.sD;
}

// One interior D-slab of a ray that is known not to cross an F-plane in it (sf = 1 in siddon_slab_fast): the same two
// lengths and the same operations on them as there, without the middle voxel and the F bookkeeping (bitwise the same sum).
template <typename IdxT, bool UNIT, bool SCATTER, bool TRACK = false, bool PAIR = false>
__device__ __forceinline__ void siddon_slab_e_only(const float* __restrict__ base, SidRay<IdxT>& r) {
    const float se = __saturatef(fmaf(r.hE, r.imE, -r.kf));
    r.kf += 1.0f;
    const bool cE = se < 1.0f;
    const IdxT offC = r.off + (cE ? r.stE : (IdxT)0);
    if (TRACK) {
        r.note(r.off, se);
        r.note(offC, 1.0f - se);
    } else if (SCATTER) {
        float* out = const_cast<float*>(base);
        if (PAIR) red_pair(out, r.off, se * r.ys, r.fm, r.pok), red_pair(out, offC, (1.0f - se) * r.ys, r.fm, r.pok);
        else red_add_global(out + r.off, se * r.ys), red_add_global(out + offC, (1.0f - se) * r.ys);
    } else {
        const float vA = UNIT ? 1.f : __ldg(base + r.off);
        float vC = vA;   // a lane that stays in its voxel does not load it twice (the L1 data pipe is co-critical)
        if (!UNIT && cE) vC = __ldg(base + offC);
        r.acc = fmaf(se, vA, r.acc);
        r.acc = fmaf(1.0f - se, vC, r.acc);
    }
    if (cE) r.hE += r.sgE;
    r.off = offC + r.sD;
}

// One D-slab with clipping to [slo, shi] and per-voxel bounds checks (first / last slabs of a ray and
// slabs that run within 1e-3 voxel of a lateral face).
template <typename IdxT, bool UNIT, bool SCATTER, bool TRACK = false>
__device__ __forceinline__ void siddon_slab_checked(const float* __restrict__ base, SidRay<IdxT>& r, int& ie, int& jf,
                                                    int diE, int diF, int nE, int nF, float slo, float shi) {
    const float se = __saturatef(fmaf(r.hE, r.imE, -r.kf)), sf = __saturatef(fmaf(r.hF, r.imF, -r.kf));
    r.kf += 1.0f;
    const bool cE = se < 1.0f, cF = sf < 1.0f;
    const float s1 = fminf(fmaxf(fminf(se, sf), slo), shi);
    const float s2 = fminf(fmaxf(fmaxf(se, sf), slo), shi);
    const bool vEA = (unsigned)ie < (unsigned)nE, vFA = (unsigned)jf < (unsigned)nF;
    const int ieC = cE ? ie + diE : ie, jfC = cF ? jf + diF : jf;
    const IdxT offC = r.off + (cE ? r.stE : (IdxT)0) + (cF ? r.stF : (IdxT)0);
    const bool vEC = (unsigned)ieC < (unsigned)nE, vFC = (unsigned)jfC < (unsigned)nF;
    const bool eFirst = se < sf;
    const IdxT offB = eFirst ? r.off + r.stE : r.off + r.stF;
    const bool vB = eFirst ? (vEC && vFA) : (vEA && vFC);
    const float lenA = s1 - slo, lenB = s2 - s1, lenC = shi - s2;
    // with a single crossing [s1, shi] lies in the end voxel: lenB + lenC = shi - s1
    const float lenE = (cE && cF) ? lenC : lenB + lenC;
    if (TRACK) {
        if (vEA && vFA) r.note(r.off, lenA);
        if (cE && cF && vB) r.note(offB, lenB);
        if (vEC && vFC) r.note(offC, lenE);
    } else if (SCATTER) {
        float* out = const_cast<float*>(base);
        if (lenA > 0.f && vEA && vFA) red_add_global(out + r.off, lenA * r.ys);
        if (cE && cF && lenB > 0.f && vB) red_add_global(out + offB, lenB * r.ys);
        if (lenE > 0.f && vEC && vFC) red_add_global(out + offC, lenE * r.ys);
    } else {
        if (lenA > 0.f && vEA && vFA) r.acc = fmaf(lenA, UNIT ? 1.f : __ldg(base + r.off), r.acc);
        if (cE && cF && lenB > 0.f && vB) r.acc = fmaf(lenB, UNIT ? 1.f : __ldg(base + offB), r.acc);
        if (lenE > 0.f && vEC && vFC) r.acc = fmaf(lenE, UNIT ? 1.f : __ldg(base + offC), r.acc);
    }
    if (cE) r.hE += r.sgE;
    if (cF) r.hF += r.sgF;
    ie = ieC, jf = jfC;
    r.off = offC + r.sD;
}

// What the fp64 set-up of one ray leaves besides the marching state: the slab ranges and the cell the march starts in.
struct SidSetup {
    int D;                         // dominant axis of this ray
    int i0, nslab, kA, kB;         // first slab (absolute), number of slabs, unchecked slabs k in [kA, kB)
    int ie, jf, ie0, jf0, diE, diF, nE, nF;
    float slo0, shiN, scale;
    double hE0, hF0;
    double SD, SE, SF, mE, mF;     // start of the ray and its slopes in (D, E, F) index coordinates
    bool useT;                     // the ray reads the (x,y)-transposed copy
    bool rev;                      // the ray points towards decreasing D (the march always runs towards increasing D)
    uint32_t cnt;                  // COUNT: exact number of voxels met
};

template <typename IdxT, bool COUNT>
__device__ __forceinline__ void siddon_setup(const RayView& rv, const AxP& p, int iu, int iv, bool haveT, SidRay<IdxT>& rout, SidSetup& q) {
    // stand-ins for the two volume pointers the text selects `base` from (never dereferenced here)
    const float* const vol = nullptr;
    const float* const volT = haveT ? reinterpret_cast<const float*>(sizeof(float)) : nullptr;
#include "ax_siddon_setup.inc"
    rout = r;
    q.D = D, q.i0 = i0, q.nslab = nslab, q.kA = kA, q.kB = kB, q.ie = ie, q.jf = jf, q.ie0 = ie0, q.jf0 = jf0, q.diE = diE, q.diF = diF;
    q.nE = nE, q.nF = nF, q.slo0 = slo0, q.shiN = shiN, q.scale = scale, q.hE0 = hE0, q.hF0 = hF0;
    q.SD = SD, q.SE = SE, q.SF = SF, q.mE = dD != 0.0 ? dE / dD : 0.0, q.mF = dD != 0.0 ? dF / dD : 0.0;
    q.useT = haveT && base == volT, q.rev = dD < 0.0, q.cnt = cnt;
    (void)Lmm, (void)nD;
}

}  // namespace tg
