// ax_siddon.cuh — the Siddon march shared by ax.cu (volume gathered through L1) and ax_siddon_tma.cu (interior of the march staged
// into shared memory by TMA): per-ray state, the three slab steps, and the fp64 per-ray set-up as a function.  See the head of
// ax.cu for the method.  (ax_siddon_kernel of ax.cu keeps its own inline copy of the set-up below: handing the twenty values
// through a struct costs that kernel 1-2 % in spills at its 56-register budget; the two texts must stay the same.)
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
__device__ __forceinline__ void siddon_setup(const RayView& rv, const AxP& p, int iu, int iv, bool haveT, SidRay<IdxT>& r, SidSetup& q) {
    q.useT = false;
    // ---- per-ray set-up, fp64
    double S[3], d[3];
#pragma unroll
    for (int k = 0; k < 3; ++k) {
        S[k] = rv.S[k] + iu * rv.dSU[k] + iv * rv.dSV[k];   // parallel beam: every ray has its own start (P29)
        d[k] = rv.P0[k] + iu * rv.dU[k] + iv * rv.dV[k] - S[k];
    }
    const double Lmm = sqrt(d[0] * p.hxd * d[0] * p.hxd + d[1] * p.hyd * d[1] * p.hyd + d[2] * p.hzd * d[2] * p.hzd);
    const double a0 = fabs(d[0]), a1 = fabs(d[1]), a2 = fabs(d[2]);
    const int D = (a0 >= a1 && a0 >= a2) ? 0 : (a1 >= a2 ? 1 : 2);
    q.D = D;
    // F is the z axis unless the ray itself runs along z: along a detector row (= a warp) the rays cross the z-planes in nearly
    // the same slabs, which the march below uses
    const int E = D == 0 ? 1 : 0, F = D == 2 ? 1 : 2;
    const double dD = sel3(D, d[0], d[1], d[2]), dE = sel3(E, d[0], d[1], d[2]), dF = sel3(F, d[0], d[1], d[2]);
    q.rev = dD < 0.0;
    const double SD = sel3(D, S[0], S[1], S[2]), SE = sel3(E, S[0], S[1], S[2]), SF = sel3(F, S[0], S[1], S[2]);
    q.SD = SD, q.SE = SE, q.SF = SF, q.mE = dD != 0.0 ? dE / dD : 0.0, q.mF = dD != 0.0 ? dF / dD : 0.0;
    const int nD = D == 0 ? p.nx : (D == 1 ? p.ny : p.nz);
    const int nE = q.nE = E == 0 ? p.nx : (E == 1 ? p.ny : p.nz);
    const int nF = q.nF = F == 0 ? p.nx : (F == 1 ? p.ny : p.nz);
    uint32_t& cnt = q.cnt;
    cnt = 0;
    // marching state, filled by the set-up below; a ray that misses the volume keeps nslab = 0
    r.imE = r.imF = 1.f, r.sgE = r.sgF = 1.f, r.hE = r.hF = 3.0e38f, r.stE = r.stF = r.sD = 0;
    r.kf = 0.f, r.acc = 0.f, r.vB = 0.f, r.ys = 0.f, r.off = 0;
    r.first = r.last = -1, r.nseg = 0, r.fm = 0, r.pok = false;
    int &i0 = q.i0, &nslab = q.nslab, &kA = q.kA, &kB = q.kB, &ie = q.ie, &jf = q.jf, &ie0 = q.ie0, &jf0 = q.jf0, &diE = q.diE, &diF = q.diF;
    i0 = 0, nslab = 0, kA = 0, kB = 0, ie = 0, jf = 0, ie0 = 0, jf0 = 0, diE = 1, diF = 1;
    float &slo0 = q.slo0, &shiN = q.shiN, &scale = q.scale;
    slo0 = 0.f, shiN = 1.f, scale = 0.f;
    double &hE0 = q.hE0, &hF0 = q.hF0;   // fp64 values r.hE / r.hF start from (0 for a ray that never crosses)
    hE0 = 0.0, hF0 = 0.0;
    if (dD != 0.0) {
        const double mE = dE / dD, mF = dF / dD;
        // range of xi_D covered by the segment S->P, clipped to the volume box on all three axes;
        // [sa, sb]: sub-range that also stays >= margin away from the lateral faces (unchecked slabs)
        const double margin = 1e-3;
        double lo = fmin(SD, SD + dD), hi = fmax(SD, SD + dD);
        lo = fmax(lo, 0.0), hi = fmin(hi, (double)nD);
        double sa = lo, sb = hi;
        bool miss = false;
        if (mE != 0.0) {
            const double t1 = SD + (0.0 - SE) / mE, t2 = SD + ((double)nE - SE) / mE;
            lo = fmax(lo, fmin(t1, t2)), hi = fmin(hi, fmax(t1, t2));
            const double u1 = SD + (margin - SE) / mE, u2 = SD + ((double)nE - margin - SE) / mE;
            sa = fmax(sa, fmin(u1, u2)), sb = fmin(sb, fmax(u1, u2));
        } else {
            if (SE < 0.0 || SE > (double)nE) miss = true;
            if (SE < margin || SE > (double)nE - margin) sb = sa - 1.0;
        }
        if (mF != 0.0) {
            const double t1 = SD + (0.0 - SF) / mF, t2 = SD + ((double)nF - SF) / mF;
            lo = fmax(lo, fmin(t1, t2)), hi = fmin(hi, fmax(t1, t2));
            const double u1 = SD + (margin - SF) / mF, u2 = SD + ((double)nF - margin - SF) / mF;
            sa = fmax(sa, fmin(u1, u2)), sb = fmin(sb, fmax(u1, u2));
        } else {
            if (SF < 0.0 || SF > (double)nF) miss = true;
            if (SF < margin || SF > (double)nF - margin) sb = sa - 1.0;
        }
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
                int i1 = (int)ceil(hi);
                i0 = max((int)floor(lo), 0), i1 = min(i1, nD);
                nslab = i1 - i0;
                // unchecked slabs: k in [kA, kB), each fully inside [max(lo,sa), min(hi,sb)]
                kA = (int)ceil(fmax(lo, sa)) - i0, kB = (int)floor(fmin(hi, sb)) - i0;
                kA = min(max(kA, 0), nslab), kB = min(max(kB, kA), nslab);
                // state at the START of slab i0 (s = 0), fp64: position, cell index, next plane ahead
                const double eS = SE + ((double)i0 - SD) * mE, fS = SF + ((double)i0 - SD) * mF;
                ie0 = (int)floor(eS), jf0 = (int)floor(fS);
                ie = ie0, jf = jf0;
                const bool upE = mE > 0.0, upF = mF > 0.0;
                // x-dominant rays read the (x,y)-transposed copy so that neighbouring lanes (which differ
                // mostly in y) touch neighbouring addresses
                const bool useT = (D == 0) && haveT;
                q.useT = useT;
                const IdxT pX = useT ? (IdxT)p.ny : (IdxT)1, pY = useT ? (IdxT)1 : (IdxT)p.nx, pZ = (IdxT)p.nx * p.ny;
                const IdxT sD = D == 0 ? pX : (D == 1 ? pY : pZ);
                const IdxT sE = E == 0 ? pX : (E == 1 ? pY : pZ);
                const IdxT sF = F == 0 ? pX : (F == 1 ? pY : pZ);
                // a ray parallel to the planes (m = 0) never crosses: next plane at +huge, 1/m := 1
                r.imE = mE != 0.0 ? (float)(1.0 / mE) : 1.f, r.imF = mF != 0.0 ? (float)(1.0 / mF) : 1.f;
                hE0 = mE != 0.0 ? (double)(upE ? ie0 + 1 : ie0) - eS : 0.0;
                hF0 = mF != 0.0 ? (double)(upF ? jf0 + 1 : jf0) - fS : 0.0;
                r.hE = mE != 0.0 ? (float)hE0 : 3.0e38f, r.hF = mF != 0.0 ? (float)hF0 : 3.0e38f;
                r.sgE = upE ? 1.f : -1.f, r.sgF = upF ? 1.f : -1.f;
                r.stE = upE ? sE : -sE, r.stF = upF ? sF : -sF, r.sD = sD;
                r.off = (IdxT)i0 * sD + (IdxT)ie * sE + (IdxT)jf * sF;   // may be out of range in checked slabs
                diE = upE ? 1 : -1, diF = upF ? 1 : -1;
                slo0 = (float)(lo - (double)i0), shiN = (float)(hi - (double)(i1 - 1));
                scale = (float)(Lmm / fabs(dD));
            }
        }
    }
}

}  // namespace tg
