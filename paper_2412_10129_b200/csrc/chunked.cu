// chunked.cu — single-GPU host-chunking path (§2.5 "split the problem
// into pieces that fit" is prior art for other GPUs: here the split is sized for one B200's HBM).
//
// Volume and projections live in PINNED host memory and are larger than the device budget.
//   Ax   outer loop: batches of views whose projections stay resident on the device;
//        inner loop: z-slabs of the volume streamed H2D (double buffered) on a copy stream while the
//        previous slab is projected; every slab ADDS its partial line integrals, and only to the band of
//        detector rows it can reach (Siddon: the slab is projected as its own sub-grid — intersection
//        lengths are additive over voxels; interpolated: the sample positions are those of the full
//        volume and taps outside the slab count as zero, so the sum over slabs is the same set of terms).
//        Finished batches go back D2H on a second copy stream.
//   A^T b outer loop: z-slabs of the output volume resident on the device;
//        inner loop: view batches, of which only the slab's detector-row band is copied in
//        (one strided 2-D copy per batch, double buffered); slabs go back D2H on the second copy stream.
// Same kernels as the in-HBM path (launch_ax / launch_atb): results agree up to summation order.
#include <algorithm>
#include <cmath>
#include <cstring>
#include "common.cuh"

namespace tg {

static size_t g_budget = 0;
size_t chunk_budget() { return g_budget; }
// bytes copied and chunk counts of the most recent chunked call (tigre_chunk_stats)
static unsigned long long g_h2d = 0, g_d2h = 0;
static int g_nslabs = 0, g_nbatches = 0;

namespace {

struct Side {   // side streams and the events that order them against the caller's stream
    cudaStream_t h2d = nullptr, d2h = nullptr;
    cudaEvent_t ready[2] = {nullptr, nullptr}, freed[2] = {nullptr, nullptr}, done = nullptr, out[2] = {nullptr, nullptr},
                start = nullptr;
    int init() {
        TG_CUDA(cudaStreamCreateWithFlags(&h2d, cudaStreamNonBlocking));
        TG_CUDA(cudaStreamCreateWithFlags(&d2h, cudaStreamNonBlocking));
        cudaEvent_t* all[] = {&ready[0], &ready[1], &freed[0], &freed[1], &done, &out[0], &out[1], &start};
        for (cudaEvent_t* e : all) TG_CUDA(cudaEventCreateWithFlags(e, cudaEventDisableTiming));
        return TIGRE_OK;
    }
    ~Side() {
        cudaEvent_t all[] = {ready[0], ready[1], freed[0], freed[1], done, out[0], out[1], start};
        for (cudaEvent_t e : all)
            if (e) cudaEventDestroy(e);
        if (h2d) cudaStreamDestroy(h2d);
        if (d2h) cudaStreamDestroy(d2h);
    }
};

// Declared AFTER the device buffers of a chunked call, so that it is destroyed FIRST: on an early error return the side
// streams may still be copying into / out of those buffers, and they must be idle before the buffers go back to the pool.
struct DrainSide {
    Side& s;
    ~DrainSide() {
        if (s.h2d) cudaStreamSynchronize(s.h2d);
        if (s.d2h) cudaStreamSynchronize(s.d2h);
        (void)cudaGetLastError();
    }
};

size_t device_budget() {
    if (g_budget) return g_budget;
    // a caller-owned workspace IS the budget (its largest free block, less room for the view tables and alignment)
    if (workspace_active()) {
        const size_t f = workspace_free_bytes();
        return f > ((size_t)64 << 20) ? f - ((size_t)32 << 20) : f / 2;
    }
    size_t fr = 0, tot = 0;
    if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) {
        (void)cudaGetLastError();
        return (size_t)8 << 30;
    }
    return fr / 4 * 3;
}

// union over views [a0, a0+na) of the detector-row bands of the z-slices [z0, z0+nzs)
void band_union(const Grid& g, const std::vector<ViewH>& views, int a0, int na, int z0, int nzs, int& row0, int& nrows) {
    int lo = g.nv, hi = 0;
    for (int a = a0; a < a0 + na; ++a) {
        int r0, nr;
        row_band(g, views[a], z0, nzs, r0, nr);
        if (nr > 0) lo = std::min(lo, r0), hi = std::max(hi, r0 + nr);
    }
    row0 = hi > lo ? lo : 0, nrows = hi > lo ? hi - lo : 0;
}

}  // namespace

// What the chunked SIRT driver (tigre_sirt_chunked) adds to the two passes.
//   pass 1 (chunked_ax_impl): once a view batch holds A x, it becomes r = W .* (b - A x) before it goes home (to r_host):
//     W = 1/(A 1) for the batch (closed form for Siddon), b uploaded on the copy stream, ||b - A x||^2 accumulated in *d_nrm2.
//   pass 2 (chunked_atb_impl): per z-slab G = A^T r (streamed bands, as chunked_atb), U = A^T 1 from a device buffer of ones
//     through the same TMA kernel, x slab uploaded, x <- max(0, x + lambda G / U) where U > thr, x slab sent home.
//     vmax_only: only max(A^T 1) over the volume is formed (the threshold of reading P13 needs it before any update).
struct SirtCtx {
    const float* h_b = nullptr;     // pass 1: measured projections (pinned)
    double* d_nrm2 = nullptr;       // pass 1: device accumulator of ||b - A x||^2
    float lambda = 1.f;             // pass 2
    int nonneg = 1;
    float thr = 0.f;                // pass 2: U <= thr -> V = 0
    bool vmax_only = false;         // pass 2 variant: *d_vmax = max over the volume of A^T 1, nothing written home
    float* d_vmax = nullptr;
};

static int chunked_ax_impl(const float* h_vol, const tigre_geo* geo, const double* angles, int nA, int mode, float* h_proj,
                           cudaStream_t st, const SirtCtx* sirt) {
    Grid g;
    std::vector<ViewH> views;
    TG_TRY(tables_prep(geo, angles, nA, g, views));
    const size_t per = (size_t)g.nu * g.nv, slice = (size_t)g.nx * g.ny;
    const size_t perB = per * sizeof(float), sliceB = slice * sizeof(float);
    const size_t budget = device_budget();
    // launch_ax keeps an (x,y)-transposed copy of the slab it projects: one more slab of room
    const size_t nbufV = 3;
    // Even when everything would fit, large problems are cut into a few pieces so that the pipeline has
    // something to overlap: >= 2 view batches (the D2H of one hides behind the kernels of the next; the price is
    // one more H2D pass over the volume, itself hidden) and >= 4 z-slabs (the first upload is the only exposed one).
    const size_t big = (size_t)256 << 20;
    const int nExtra = sirt ? 2 : 0;   // SIRT: one batch-sized buffer for W and one for b
    int nAb, nPb;
    if (perB * nA * (1 + nExtra) + nbufV * sliceB * std::min(g.nz, 8) <= budget && perB * nA <= big) nAb = nA, nPb = 1;
    else {
        nAb = (int)std::min<size_t>((size_t)nA, std::max<size_t>(1, budget / 2 / ((2 + nExtra) * perB))), nPb = 2;
        nAb = std::min(nAb, std::max(1, (nA + 1) / 2));
    }
    const size_t projB = (size_t)(nPb + nExtra) * nAb * perB;
    if (projB + nbufV * sliceB > budget) return TIGRE_ERR_WORKSPACE;
    int nzs = (int)std::min<size_t>((size_t)g.nz, (budget - projB) / (nbufV * sliceB));
    if ((size_t)g.nz * sliceB > big) nzs = std::min(nzs, std::max(1, (g.nz + 3) / 4));
    // slabs stay below 2^31 voxels, so the ray-driven kernels keep 32-bit element offsets (their 64-bit instantiations
    // run 20 % slower: 1086 against 1353 G samples/s on C3); a ray only meets the one or two slabs its detector row can reach
    nzs = std::min<long long>(nzs, std::max<long long>(1, ((1ll << 31) - 1) / (long long)slice));
    const int nSlabs = (g.nz + nzs - 1) / nzs;
    nzs = (g.nz + nSlabs - 1) / nSlabs;   // even slabs
    const int nBatches = (nA + nAb - 1) / nAb;
    const int nVb = nSlabs > 1 ? 2 : 1;

    g_h2d = g_d2h = 0, g_nslabs = nSlabs, g_nbatches = nBatches;
    Side sd;
    TG_TRY(sd.init());
    TempBuf vb[2], pb[2], wb, bb;
    cudaEvent_t evB = nullptr, evBfree = nullptr;   // SIRT: b batch has arrived / its buffer is free again
    struct EvGuard {
        cudaEvent_t &a, &b;
        ~EvGuard() {
            if (a) cudaEventDestroy(a);
            if (b) cudaEventDestroy(b);
        }
    } evg{evB, evBfree};
    DrainSide drain{sd};
    for (int i = 0; i < nVb; ++i) TG_TRY(vb[i].alloc((size_t)nzs * sliceB, st));
    for (int i = 0; i < nPb; ++i) TG_TRY(pb[i].alloc((size_t)nAb * perB, st));
    if (sirt) {
        TG_TRY(wb.alloc((size_t)nAb * perB, st));
        TG_TRY(bb.alloc((size_t)nAb * perB, st));
        TG_CUDA(cudaEventCreateWithFlags(&evB, cudaEventDisableTiming));
        TG_CUDA(cudaEventCreateWithFlags(&evBfree, cudaEventDisableTiming));
    }
    const double epsW = 1e-2 * std::min(g.dx, std::min(g.dy, g.dz));   // reading P13
    TG_CUDA(cudaEventRecord(sd.start, st));          // buffers exist from here on in stream order
    TG_CUDA(cudaStreamWaitEvent(sd.h2d, sd.start, 0));
    TG_CUDA(cudaStreamWaitEvent(sd.d2h, sd.start, 0));

    long long islab = 0;   // running slab-upload counter (selects the volume buffer)
    for (int b = 0; b < nBatches; ++b) {
        const int a0 = b * nAb, na = std::min(nAb, nA - a0);
        float* P = pb[b % nPb].as<float>();
        if (b >= nPb) TG_CUDA(cudaStreamWaitEvent(st, sd.out[b % nPb], 0));   // its previous contents are home
        TG_CUDA(cudaMemsetAsync(P, 0, (size_t)na * perB, st));
        std::vector<RayView> hr(na);
        for (int i = 0; i < na; ++i) build_ray_view(g, views[a0 + i], hr[i]);
        TempBuf tab;
        if (mode == TIGRE_AX_INTERP || sirt) TG_TRY(upload(tab, hr.data(), sizeof(RayView) * na, st));
        if (sirt) {   // this batch's measured projections come up on the copy stream, ahead of the slabs
            if (b > 0) TG_CUDA(cudaStreamWaitEvent(sd.h2d, evBfree, 0));
            TG_CUDA(cudaMemcpyAsync(bb.p, sirt->h_b + (size_t)a0 * per, (size_t)na * perB, cudaMemcpyHostToDevice, sd.h2d));
            g_h2d += (unsigned long long)na * perB;
            TG_CUDA(cudaEventRecord(evB, sd.h2d));
        }
        for (int s = 0; s < nSlabs; ++s) {
            const int z0 = s * nzs, nz_s = std::min(nzs, g.nz - z0);
            float* V = vb[islab % nVb].as<float>();
            if (nSlabs > 1 || b == 0) {   // a volume that fits in one slab is uploaded once
                if (islab >= nVb) TG_CUDA(cudaStreamWaitEvent(sd.h2d, sd.freed[islab % nVb], 0));
                TG_CUDA(cudaMemcpyAsync(V, h_vol + (size_t)z0 * slice, (size_t)nz_s * sliceB, cudaMemcpyHostToDevice, sd.h2d));
                g_h2d += (unsigned long long)nz_s * sliceB;
                TG_CUDA(cudaEventRecord(sd.ready[islab % nVb], sd.h2d));
                TG_CUDA(cudaStreamWaitEvent(st, sd.ready[islab % nVb], 0));
            }
            AxSub sub;
            band_union(g, views, a0, na, z0, nz_s, sub.row0, sub.nrows);
            if (mode == TIGRE_AX_SIDDON) {
                // the slab as its own grid: same voxels, z origin moved to its first slice
                Grid gs = g;
                gs.nz = nz_s;
                std::vector<RayView> hs(hr);
                for (RayView& r : hs) r.S[2] -= (double)z0, r.P0[2] -= (double)z0;
                TempBuf tabs;
                TG_TRY(upload(tabs, hs.data(), sizeof(RayView) * na, st));
                sub.zs0 = 0, sub.nzs = nz_s;
                TG_TRY(launch_ax(V, gs, tabs.as<RayView>(), na, mode, false, true, P, nullptr, st, &sub));
            } else {
                sub.zs0 = z0, sub.nzs = nz_s;
                TG_TRY(launch_ax(V, g, tab.as<RayView>(), na, mode, false, true, P, nullptr, st, &sub, nullptr, hr.data()));
            }
            if (nSlabs > 1) {
                TG_CUDA(cudaEventRecord(sd.freed[islab % nVb], st));
                ++islab;
            }
        }
        if (sirt) {
            // r = W .* (b - A x) in place over the batch; W = 1/(A 1) of the FULL volume for these views
            float* Wd = wb.as<float>();
            TG_TRY(launch_ax(nullptr, g, tab.as<RayView>(), na, mode, true, false, Wd, nullptr, st));
            TG_TRY(launch_invert_rows(Wd, (size_t)na * per, (float)epsW, st));
            TG_CUDA(cudaStreamWaitEvent(st, evB, 0));
            TG_TRY(launch_residual(bb.as<float>(), nullptr, P, Wd, P, per, na, sirt->d_nrm2, st));
            TG_CUDA(cudaEventRecord(evBfree, st));
        }
        TG_CUDA(cudaEventRecord(sd.done, st));
        TG_CUDA(cudaStreamWaitEvent(sd.d2h, sd.done, 0));
        TG_CUDA(cudaMemcpyAsync(h_proj + (size_t)a0 * per, P, (size_t)na * perB, cudaMemcpyDeviceToHost, sd.d2h));
        g_d2h += (unsigned long long)na * perB;
        TG_CUDA(cudaEventRecord(sd.out[b % nPb], sd.d2h));
    }
    for (int i = 0; i < std::min(nPb, nBatches); ++i) TG_CUDA(cudaStreamWaitEvent(st, sd.out[i], 0));
    TG_CUDA(cudaEventRecord(sd.done, sd.h2d));
    TG_CUDA(cudaStreamWaitEvent(st, sd.done, 0));
    for (int i = 0; i < 2; ++i) vb[i].release(), pb[i].release();
    wb.release(), bb.release();
    TG_CUDA(cudaStreamSynchronize(st));
    return TIGRE_OK;
}

int chunked_ax(const float* h_vol, const tigre_geo* geo, const double* angles, int nA, int mode, float* h_proj, cudaStream_t st) {
    return chunked_ax_impl(h_vol, geo, angles, nA, mode, h_proj, st, nullptr);
}

// h_proj: the projections backprojected (SIRT: the weighted residual r); h_vol: the result (SIRT: the iterate, read AND written)
static int chunked_atb_impl(const float* h_proj, const tigre_geo* geo, const double* angles, int nA, int mode, float* h_vol,
                            cudaStream_t st, const SirtCtx* sirt) {
    Grid g;
    std::vector<ViewH> views;
    TG_TRY(tables_prep(geo, angles, nA, g, views));
    const size_t per = (size_t)g.nu * g.nv, slice = (size_t)g.nx * g.ny;
    const size_t sliceB = slice * sizeof(float);
    const size_t budget = device_budget();
    // the per-view voxel -> detector tables of all views, once
    std::vector<VoxView> hv(nA);
    for (int a = 0; a < nA; ++a) TG_TRY(build_vox_view(g, views[a], hv[a]));
    const bool clamp = vox_needs_clamp(g, hv.data(), nA);
    TempBuf tab;
    TG_TRY(upload(tab, hv.data(), sizeof(VoxView) * nA, st));

    // volume slabs: the whole volume if it fits in half of the budget, else two buffers in that half
    // (large volumes are cut into >= 2 slabs even if they fit, so that the D2H of one hides behind the next)
    const size_t big = (size_t)256 << 20;
    // slab-sized buffers: two output slabs (plain A^T b); SIRT: G, U and two slabs of the iterate
    const int nSlabBufs = sirt ? (sirt->vmax_only ? 1 : 4) : 2;
    int nzs;
    if ((size_t)g.nz * sliceB * (sirt ? nSlabBufs : 1) <= budget / 2 && (size_t)g.nz * sliceB <= big) nzs = g.nz;
    else nzs = (int)std::min<size_t>(budget / 2 / (nSlabBufs * sliceB), (size_t)std::max(1, (g.nz + 1) / 2));
    if (nzs < 1) return TIGRE_ERR_WORKSPACE;
    const int nSlabs = (g.nz + nzs - 1) / nzs;
    nzs = (g.nz + nSlabs - 1) / nSlabs;
    const int nVb = nSlabs > 1 ? 2 : 1;
    const size_t volB = (size_t)(sirt ? nSlabBufs : nVb) * nzs * sliceB;
    // view batches: two buffers of nAb row bands; size them for the widest band of any slab
    std::vector<int> r0s(nSlabs), nrs(nSlabs);
    int nrMax = 1;
    for (int s = 0; s < nSlabs; ++s) {
        const int z0 = s * nzs, nz_s = std::min(nzs, g.nz - z0);
        band_union(g, views, 0, nA, z0, nz_s, r0s[s], nrs[s]);
        nrMax = std::max(nrMax, nrs[s]);
    }
    const size_t bandB = (size_t)nrMax * g.nu * sizeof(float);
    const int nBandBufs = sirt ? 3 : 2;   // SIRT: a third band buffer full of ones (A^T 1 through the same kernel)
    if (volB + nBandBufs * bandB > budget) return TIGRE_ERR_WORKSPACE;
    int nAb = (int)std::min<size_t>((size_t)nA, (budget - volB) / (nBandBufs * bandB));
    if (bandB * nA > ((size_t)64 << 20)) nAb = std::min(nAb, std::max(1, (nA + 3) / 4));   // >= 4 batches to overlap
    const int nBatches = (nA + nAb - 1) / nAb;
    const int nPb = nBatches * nSlabs > 1 ? 2 : 1;

    g_h2d = g_d2h = 0, g_nslabs = nSlabs, g_nbatches = nBatches;
    Side sd;
    TG_TRY(sd.init());
    TempBuf vb[2], pb[2], gb, ub, ones;
    DrainSide drain{sd};
    if (!sirt) {
        for (int i = 0; i < nVb; ++i) TG_TRY(vb[i].alloc((size_t)nzs * sliceB, st));
    } else {
        TG_TRY(ub.alloc((size_t)nzs * sliceB, st));
        if (!sirt->vmax_only) {
            TG_TRY(gb.alloc((size_t)nzs * sliceB, st));
            for (int i = 0; i < nVb; ++i) TG_TRY(vb[i].alloc((size_t)nzs * sliceB, st));   // slabs of the iterate
        }
        TG_TRY(ones.alloc((size_t)nAb * bandB, st));
        TG_TRY(launch_fill(ones.as<float>(), 1.0f, (size_t)nAb * bandB / sizeof(float), st));
    }
    if (!sirt || !sirt->vmax_only)
        for (int i = 0; i < nPb; ++i) TG_TRY(pb[i].alloc((size_t)nAb * bandB, st));
    TG_CUDA(cudaEventRecord(sd.start, st));
    TG_CUDA(cudaStreamWaitEvent(sd.h2d, sd.start, 0));
    TG_CUDA(cudaStreamWaitEvent(sd.d2h, sd.start, 0));

    long long ib = 0;   // running batch-upload counter (selects the projection buffer)
    for (int s = 0; s < nSlabs; ++s) {
        const int z0 = s * nzs, nz_s = std::min(nzs, g.nz - z0);
        // V: where A^T (h_proj) of this slab is formed: an output slab, or (SIRT) the gradient buffer G
        float* V = sirt ? gb.as<float>() : vb[s % nVb].as<float>();
        float* X = sirt ? vb[s % nVb].as<float>() : nullptr;   // SIRT: the slab of the iterate
        if (s >= nVb) TG_CUDA(cudaStreamWaitEvent(st, sd.out[s % nVb], 0));
        const int row0 = r0s[s], nrows = nrs[s];
        if (sirt && sirt->vmax_only) {
            // max over this slab of A^T 1
            if (nrows > 0) {
                for (int b = 0; b < nBatches; ++b) {
                    const int a0 = b * nAb, na = std::min(nAb, nA - a0);
                    TG_TRY(launch_atb(ones.as<float>(), g, tab.as<VoxView>() + a0, na, mode, false, ub.as<float>(), z0, nz_s, b > 0, row0,
                                      nrows, clamp, st, hv.data() + a0));
                }
                TG_TRY(launch_max(ub.as<float>(), (size_t)nz_s * slice, sirt->d_vmax, st));
            }
            continue;
        }
        if (nrows <= 0) {
            TG_CUDA(cudaMemsetAsync(V, 0, (size_t)nz_s * sliceB, st));   // this slab sees no detector row
            if (sirt) TG_CUDA(cudaMemsetAsync(ub.p, 0, (size_t)nz_s * sliceB, st));
        } else {
            for (int b = 0; b < nBatches; ++b, ++ib) {
                const int a0 = b * nAb, na = std::min(nAb, nA - a0);
                float* P = pb[ib % nPb].as<float>();
                if (ib >= nPb) TG_CUDA(cudaStreamWaitEvent(sd.h2d, sd.freed[ib % nPb], 0));
                const size_t rowBytes = (size_t)nrows * g.nu * sizeof(float);
                TG_CUDA(cudaMemcpy2DAsync(P, rowBytes, h_proj + ((size_t)a0 * g.nv + row0) * g.nu, per * sizeof(float), rowBytes,
                                          (size_t)na, cudaMemcpyHostToDevice, sd.h2d));
                g_h2d += (unsigned long long)rowBytes * na;
                TG_CUDA(cudaEventRecord(sd.ready[ib % nPb], sd.h2d));
                TG_CUDA(cudaStreamWaitEvent(st, sd.ready[ib % nPb], 0));
                TG_TRY(launch_atb(P, g, tab.as<VoxView>() + a0, na, mode, false, V, z0, nz_s, b > 0, row0, nrows, clamp, st, hv.data() + a0));
                TG_CUDA(cudaEventRecord(sd.freed[ib % nPb], st));
                if (sirt)   // U += A^T 1 of the same views, through the same kernel, from the buffer of ones
                    TG_TRY(launch_atb(ones.as<float>(), g, tab.as<VoxView>() + a0, na, mode, false, ub.as<float>(), z0, nz_s, b > 0, row0,
                                      nrows, clamp, st, hv.data() + a0));
            }
        }
        if (sirt) {
            // x_slab <- max(0, x_slab + lambda G / U) where U > thr (readings P13, P14); the slab of the iterate comes up on the
            // caller's stream (a small share of the slab's time) and goes home from its own buffer
            TG_CUDA(cudaMemcpyAsync(X, h_vol + (size_t)z0 * slice, (size_t)nz_s * sliceB, cudaMemcpyHostToDevice, st));
            g_h2d += (unsigned long long)nz_s * sliceB;
            TG_TRY(launch_invert_rows(ub.as<float>(), (size_t)nz_s * slice, sirt->thr, st));
            TG_TRY(launch_update(X, V, ub.as<float>(), sirt->lambda, sirt->nonneg, (size_t)nz_s * slice, st));
            V = X;
        }
        TG_CUDA(cudaEventRecord(sd.done, st));
        TG_CUDA(cudaStreamWaitEvent(sd.d2h, sd.done, 0));
        TG_CUDA(cudaMemcpyAsync(h_vol + (size_t)z0 * slice, V, (size_t)nz_s * sliceB, cudaMemcpyDeviceToHost, sd.d2h));
        g_d2h += (unsigned long long)nz_s * sliceB;
        TG_CUDA(cudaEventRecord(sd.out[s % nVb], sd.d2h));
    }
    if (!(sirt && sirt->vmax_only))
        for (int i = 0; i < std::min(nVb, nSlabs); ++i) TG_CUDA(cudaStreamWaitEvent(st, sd.out[i], 0));
    TG_CUDA(cudaEventRecord(sd.done, sd.h2d));
    TG_CUDA(cudaStreamWaitEvent(st, sd.done, 0));
    for (int i = 0; i < 2; ++i) vb[i].release(), pb[i].release();
    gb.release(), ub.release(), ones.release();
    TG_CUDA(cudaStreamSynchronize(st));
    return TIGRE_OK;
}

int chunked_atb(const float* h_proj, const tigre_geo* geo, const double* angles, int nA, int mode, float* h_vol, cudaStream_t st) {
    return chunked_atb_impl(h_proj, geo, angles, nA, mode, h_vol, st, nullptr);
}

// One or more SIRT iterations on pinned host arrays larger than the device budget (BASELINE.json configs[4]; PAPER.md:115,
// 135 eq. 6 with one subset, 203): x <- max(0, x + lambda V .* A^T(W .* (b - A x))), W = 1/(A 1), V = 1/(A^T 1) thresholded as in
// reading P13 (the threshold of V needs max(A^T 1) over the whole volume: one extra pass of A^T 1, once per call).
int chunked_sirt(const float* h_b, const tigre_geo* geo, const double* angles, int nA, int n_iter, float lambda, int nonneg,
                 int ax_mode, int atb_mode, float* h_x, float* h_r, double* resid_hist, cudaStream_t st) {
    TempBuf sc;
    TG_TRY(sc.alloc(sizeof(double) * (size_t)(std::max(n_iter, 1) + 1), st));
    TG_CUDA(cudaMemsetAsync(sc.p, 0, sizeof(double) * (size_t)(std::max(n_iter, 1) + 1), st));
    double* d_nrm = sc.as<double>();
    float* d_vmax = reinterpret_cast<float*>(d_nrm + std::max(n_iter, 1));
    unsigned long long h2d = 0, d2h = 0;
    SirtCtx c;
    c.lambda = lambda, c.nonneg = nonneg;
    if (n_iter > 0) {
        c.vmax_only = true, c.d_vmax = d_vmax;
        TG_TRY(chunked_atb_impl(h_r, geo, angles, nA, atb_mode, h_x, st, &c));
        float vmax = 0.f;
        TG_CUDA(cudaMemcpyAsync(&vmax, d_vmax, sizeof(float), cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        c.thr = 1e-6f * vmax;
        c.vmax_only = false;
    }
    for (int it = 0; it < n_iter; ++it) {
        c.h_b = h_b, c.d_nrm2 = d_nrm + it;
        TG_TRY(chunked_ax_impl(h_x, geo, angles, nA, ax_mode, h_r, st, &c));
        h2d += g_h2d, d2h += g_d2h;
        TG_TRY(chunked_atb_impl(h_r, geo, angles, nA, atb_mode, h_x, st, &c));
        h2d += g_h2d, d2h += g_d2h;
    }
    g_h2d = h2d, g_d2h = d2h;
    if (resid_hist && n_iter > 0) {
        std::vector<double> h(n_iter);
        TG_CUDA(cudaMemcpyAsync(h.data(), d_nrm, sizeof(double) * n_iter, cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        for (int it = 0; it < n_iter; ++it) resid_hist[it] = std::sqrt(h[it]);
    }
    return TIGRE_OK;
}

}  // namespace tg

extern "C" int tigre_chunk_stats(uint64_t* h2d_bytes, uint64_t* d2h_bytes, int* n_slabs, int* n_batches) {
    if (h2d_bytes) *h2d_bytes = tg::g_h2d;
    if (d2h_bytes) *d2h_bytes = tg::g_d2h;
    if (n_slabs) *n_slabs = tg::g_nslabs;
    if (n_batches) *n_batches = tg::g_nbatches;
    return TIGRE_OK;
}

extern "C" int tigre_set_chunk_budget(size_t bytes) {
    tg::g_budget = bytes;
    return TIGRE_OK;
}
