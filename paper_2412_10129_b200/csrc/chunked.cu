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

size_t device_budget() {
    if (g_budget) return g_budget;
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

int chunked_ax(const float* h_vol, const tigre_geo* geo, const double* angles, int nA, int mode, float* h_proj,
               cudaStream_t st) {
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
    int nAb, nPb;
    if (perB * nA + nbufV * sliceB * std::min(g.nz, 8) <= budget && perB * nA <= big) nAb = nA, nPb = 1;
    else {
        nAb = (int)std::min<size_t>((size_t)nA, std::max<size_t>(1, budget / 2 / (2 * perB))), nPb = 2;
        nAb = std::min(nAb, std::max(1, (nA + 1) / 2));
    }
    const size_t projB = (size_t)nPb * nAb * perB;
    if (projB + nbufV * sliceB > budget) return TIGRE_ERR_WORKSPACE;
    int nzs = (int)std::min<size_t>((size_t)g.nz, (budget - projB) / (nbufV * sliceB));
    if ((size_t)g.nz * sliceB > big) nzs = std::min(nzs, std::max(1, (g.nz + 3) / 4));
    const int nSlabs = (g.nz + nzs - 1) / nzs;
    nzs = (g.nz + nSlabs - 1) / nSlabs;   // even slabs
    const int nBatches = (nA + nAb - 1) / nAb;
    const int nVb = nSlabs > 1 ? 2 : 1;

    g_h2d = g_d2h = 0, g_nslabs = nSlabs, g_nbatches = nBatches;
    Side sd;
    TG_TRY(sd.init());
    TempBuf vb[2], pb[2];
    for (int i = 0; i < nVb; ++i) TG_TRY(vb[i].alloc((size_t)nzs * sliceB, st));
    for (int i = 0; i < nPb; ++i) TG_TRY(pb[i].alloc((size_t)nAb * perB, st));
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
        if (mode == TIGRE_AX_INTERP) TG_TRY(upload(tab, hr.data(), sizeof(RayView) * na, st));
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
                TG_TRY(launch_ax(V, g, tab.as<RayView>(), na, mode, false, true, P, nullptr, st, &sub));
            }
            if (nSlabs > 1) {
                TG_CUDA(cudaEventRecord(sd.freed[islab % nVb], st));
                ++islab;
            }
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
    TG_CUDA(cudaStreamSynchronize(st));
    return TIGRE_OK;
}

int chunked_atb(const float* h_proj, const tigre_geo* geo, const double* angles, int nA, int mode, float* h_vol,
                cudaStream_t st) {
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
    int nzs;
    if ((size_t)g.nz * sliceB <= budget / 2 && (size_t)g.nz * sliceB <= big) nzs = g.nz;
    else nzs = (int)std::min<size_t>(budget / 2 / (2 * sliceB), (size_t)std::max(1, (g.nz + 1) / 2));
    if (nzs < 1) return TIGRE_ERR_WORKSPACE;
    const int nSlabs = (g.nz + nzs - 1) / nzs;
    nzs = (g.nz + nSlabs - 1) / nSlabs;
    const int nVb = nSlabs > 1 ? 2 : 1;
    const size_t volB = (size_t)nVb * nzs * sliceB;
    // view batches: two buffers of nAb row bands; size them for the widest band of any slab
    std::vector<int> r0s(nSlabs), nrs(nSlabs);
    int nrMax = 1;
    for (int s = 0; s < nSlabs; ++s) {
        const int z0 = s * nzs, nz_s = std::min(nzs, g.nz - z0);
        band_union(g, views, 0, nA, z0, nz_s, r0s[s], nrs[s]);
        nrMax = std::max(nrMax, nrs[s]);
    }
    const size_t bandB = (size_t)nrMax * g.nu * sizeof(float);
    if (volB + 2 * bandB > budget) return TIGRE_ERR_WORKSPACE;
    int nAb = (int)std::min<size_t>((size_t)nA, (budget - volB) / (2 * bandB));
    if (bandB * nA > ((size_t)64 << 20)) nAb = std::min(nAb, std::max(1, (nA + 3) / 4));   // >= 4 batches to overlap
    const int nBatches = (nA + nAb - 1) / nAb;
    const int nPb = nBatches * nSlabs > 1 ? 2 : 1;

    g_h2d = g_d2h = 0, g_nslabs = nSlabs, g_nbatches = nBatches;
    Side sd;
    TG_TRY(sd.init());
    TempBuf vb[2], pb[2];
    for (int i = 0; i < nVb; ++i) TG_TRY(vb[i].alloc((size_t)nzs * sliceB, st));
    for (int i = 0; i < nPb; ++i) TG_TRY(pb[i].alloc((size_t)nAb * bandB, st));
    TG_CUDA(cudaEventRecord(sd.start, st));
    TG_CUDA(cudaStreamWaitEvent(sd.h2d, sd.start, 0));
    TG_CUDA(cudaStreamWaitEvent(sd.d2h, sd.start, 0));

    long long ib = 0;   // running batch-upload counter (selects the projection buffer)
    for (int s = 0; s < nSlabs; ++s) {
        const int z0 = s * nzs, nz_s = std::min(nzs, g.nz - z0);
        float* V = vb[s % nVb].as<float>();
        if (s >= nVb) TG_CUDA(cudaStreamWaitEvent(st, sd.out[s % nVb], 0));
        const int row0 = r0s[s], nrows = nrs[s];
        if (nrows <= 0) {
            TG_CUDA(cudaMemsetAsync(V, 0, (size_t)nz_s * sliceB, st));   // this slab sees no detector row
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
            }
        }
        TG_CUDA(cudaEventRecord(sd.done, st));
        TG_CUDA(cudaStreamWaitEvent(sd.d2h, sd.done, 0));
        TG_CUDA(cudaMemcpyAsync(h_vol + (size_t)z0 * slice, V, (size_t)nz_s * sliceB, cudaMemcpyDeviceToHost, sd.d2h));
        g_d2h += (unsigned long long)nz_s * sliceB;
        TG_CUDA(cudaEventRecord(sd.out[s % nVb], sd.d2h));
    }
    for (int i = 0; i < std::min(nVb, nSlabs); ++i) TG_CUDA(cudaStreamWaitEvent(st, sd.out[i], 0));
    TG_CUDA(cudaEventRecord(sd.done, sd.h2d));
    TG_CUDA(cudaStreamWaitEvent(st, sd.done, 0));
    for (int i = 0; i < 2; ++i) vb[i].release(), pb[i].release();
    TG_CUDA(cudaStreamSynchronize(st));
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
