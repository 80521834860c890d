// api.cu — the C ABI of libtigre_b200 (include/tigre_b200.h): argument checks, per-view table
// upload, kernel launches and the SIRT/OS-SART, CGLS and FDK drivers (DESIGN.md O-D..O-F).
// No CPU fallback anywhere: without a device every compute call returns TIGRE_ERR_NO_DEVICE.
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstring>
#include <map>
#include <memory>
#include <mutex>
#include <string>
#include <array>
#include <vector>
#include "common.cuh"

namespace tg {

static thread_local std::string g_last_cuda_error;
void set_cuda_error(cudaError_t e, const char* file, int line) {
    char buf[512];
    snprintf(buf, sizeof buf, "%s (%s) at %s:%d", cudaGetErrorName(e), cudaGetErrorString(e), file, line);
    g_last_cuda_error = buf;
    (void)cudaGetLastError();  // clear the non-sticky error state
}

// ---------------------------------------------------------------- profiling hook
struct ProfRec {
    cudaEvent_t a, b;
    int kind;
};
static std::mutex g_prof_mu;
static bool g_prof_on = false;
static std::vector<ProfRec*> g_prof_recs;
static unsigned long long g_prof_launches[PK_N] = {0, 0, 0};

ProfScope::ProfScope(int k, cudaStream_t s, int launches) : kind(k), st(s), rec(nullptr) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_prof_launches[k] += launches;
    if (!g_prof_on) return;
    ProfRec* r = new ProfRec;
    r->kind = k;
    if (cudaEventCreate(&r->a) != cudaSuccess || cudaEventCreate(&r->b) != cudaSuccess) {
        (void)cudaGetLastError();
        delete r;
        return;
    }
    cudaEventRecord(r->a, s);
    rec = r;
}
ProfScope::~ProfScope() {
    if (!rec) return;
    ProfRec* r = (ProfRec*)rec;
    cudaEventRecord(r->b, st);
    std::lock_guard<std::mutex> lk(g_prof_mu);
    g_prof_recs.push_back(r);
}

// ---------------------------------------------------------------- caller-owned workspace (tigre_set_workspace)
// "the library allocates nothing persistent; volume / projection / workspace memory is the caller's".
// When a workspace is set every temporary and every plan buffer is carved from it by this first-fit free list (host-side
// bookkeeping only, 256-byte granules, neighbours coalesced on release) and the library makes no cudaMallocAsync call.
// Re-use of a released block is ordered by the stream the calls are enqueued on, as with the stream-ordered pool.
struct Workspace {
    std::mutex mu;
    char* base = nullptr;
    size_t size = 0, in_use = 0, high = 0;
    std::map<size_t, size_t> free_;     // offset -> length of every free block
    std::map<size_t, size_t> used;      // offset -> length of every live block
    unsigned long long pool_allocs = 0; // cudaMallocAsync calls made since the last tigre_set_workspace
    void* take(size_t bytes) {
        bytes = (bytes + 255) & ~(size_t)255;
        for (auto it = free_.begin(); it != free_.end(); ++it) {
            if (it->second < bytes) continue;
            const size_t off = it->first, len = it->second;
            free_.erase(it);
            if (len > bytes) free_[off + bytes] = len - bytes;
            used[off] = bytes;
            in_use += bytes, high = std::max(high, in_use);
            return base + off;
        }
        return nullptr;
    }
    void give(void* p) {
        const size_t off = (size_t)((char*)p - base);
        auto u = used.find(off);
        if (u == used.end()) return;
        size_t o = off, len = u->second;
        in_use -= len;
        used.erase(u);
        auto nx = free_.lower_bound(o);
        if (nx != free_.end() && o + len == nx->first) len += nx->second, nx = free_.erase(nx);
        if (nx != free_.begin()) {
            auto pv = std::prev(nx);
            if (pv->first + pv->second == o) o = pv->first, len += pv->second, free_.erase(pv);
        }
        free_[o] = len;
    }
};
static Workspace g_ws;
size_t workspace_free_bytes() {   // largest free block of the workspace (0: none set)
    std::lock_guard<std::mutex> lk(g_ws.mu);
    size_t m = 0;
    for (auto& f : g_ws.free_) m = std::max(m, f.second);
    return g_ws.base ? m : 0;
}
bool workspace_active() { return g_ws.base != nullptr; }

int TempBuf::alloc(size_t bytes, cudaStream_t st) {
    release();
    s = st;
    if (bytes == 0) bytes = 16;
    {
        std::lock_guard<std::mutex> lk(g_ws.mu);
        if (g_ws.base) {
            p = g_ws.take(bytes);
            ws = true;
            if (!p) {
                ws = false;
                g_last_cuda_error = "caller-owned workspace too small (tigre_set_workspace)";
                return TIGRE_ERR_WORKSPACE;
            }
            return TIGRE_OK;
        }
        ++g_ws.pool_allocs;
    }
    ws = false;
    cudaError_t e = cudaMallocAsync(&p, bytes, st);
    if (e != cudaSuccess) {
        p = nullptr;
        set_cuda_error(e, __FILE__, __LINE__);
        return TIGRE_ERR_WORKSPACE;
    }
    return TIGRE_OK;
}
void TempBuf::release() {
    if (p) {
        if (ws) {
            std::lock_guard<std::mutex> lk(g_ws.mu);
            g_ws.give(p);
        } else {
            cudaFreeAsync(p, s);
        }
    }
    p = nullptr, ws = false;
}
int upload(TempBuf& buf, const void* host, size_t bytes, cudaStream_t st) {
    TG_TRY(buf.alloc(bytes, st));
    // pageable source: the runtime stages the bytes before returning, so `host` may die afterwards
    TG_CUDA(cudaMemcpyAsync(buf.p, host, bytes, cudaMemcpyHostToDevice, st));
    return TIGRE_OK;
}

static int ensure_device() {
    static std::once_flag once;
    static int status = TIGRE_OK;
    std::call_once(once, [] {
        int n = 0;
        if (cudaGetDeviceCount(&n) != cudaSuccess || n <= 0) {
            (void)cudaGetLastError();
            status = TIGRE_ERR_NO_DEVICE;
            return;
        }
        // keep freed temporaries in the pool instead of returning them to the OS at every sync
        int dev = 0;
        cudaGetDevice(&dev);
        cudaMemPool_t pool;
        if (cudaDeviceGetDefaultMemPool(&pool, dev) == cudaSuccess) {
            unsigned long long thr = ~0ull;
            cudaMemPoolSetAttribute(pool, cudaMemPoolAttrReleaseThreshold, &thr);
        }
        (void)cudaGetLastError();
    });
    return status;
}

enum MemKind { MEM_DEVICE, MEM_PINNED, MEM_PAGEABLE };
static MemKind mem_kind(const void* p) {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        (void)cudaGetLastError();
        return MEM_PAGEABLE;
    }
    if (at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged) return MEM_DEVICE;
    if (at.type == cudaMemoryTypeHost) return MEM_PINNED;
    return MEM_PAGEABLE;
}

// ---------------------------------------------------------------- per-view tables on the device
struct Tables {
    std::vector<ViewH> views;
    Grid g;
    TempBuf ray, vox;
    std::vector<VoxView> hvox;   // host copy of the table in `vox` (sizes the TMA boxes)
    std::vector<RayView> hray;   // host copy of the table in `ray` (sizes the boxes of the interpolated projector)
    bool clamp = false;
    int build_ray(const int32_t* idx, int n, cudaStream_t st) {
        std::vector<RayView>& h = hray;
        h.resize(n);
        for (int i = 0; i < n; ++i) build_ray_view(g, views[idx ? idx[i] : i], h[i]);
        return upload(ray, h.data(), sizeof(RayView) * n, st);
    }
    int build_vox(const int32_t* idx, int n, cudaStream_t st) {
        std::vector<VoxView>& h = hvox;
        h.resize(n);
        for (int i = 0; i < n; ++i) TG_TRY(build_vox_view(g, views[idx ? idx[i] : i], h[i]));
        clamp = vox_needs_clamp(g, h.data(), n);
        return upload(vox, h.data(), sizeof(VoxView) * n, st);
    }
};

int tables_prep(const tigre_geo* geo, const double* angles, int nA, Grid& g, std::vector<ViewH>& views) {
    TG_TRY(validate_geo(geo, angles, nA));
    TG_TRY(ensure_device());
    g = make_grid(geo);
    resolve_views(geo, angles, nA, views);
    return TIGRE_OK;
}
static int prep(const tigre_geo* geo, const double* angles, int nA, Tables& t) {
    return tables_prep(geo, angles, nA, t.g, t.views);
}

static int device_ax(const float* vol, Tables& t, const int32_t* idx, int n, int mode, bool unit, float* proj,
                     cudaStream_t st) {
    TG_TRY(t.build_ray(idx, n, st));
    return launch_ax(vol, t.g, t.ray.as<RayView>(), n, mode, unit, false, proj, nullptr, st, nullptr, nullptr, t.hray.data());
}
static int device_atb(const float* proj, Tables& t, const int32_t* idx, int n, int mode, bool unit, float* vol,
                      cudaStream_t st) {
    TG_TRY(t.build_vox(idx, n, st));
    return launch_atb(proj, t.g, t.vox.as<VoxView>(), n, mode, unit, vol, 0, t.g.nz, false, 0, t.g.nv, t.clamp, st,
                      t.hvox.data());
}

}  // namespace tg

using namespace tg;

extern "C" {

int tigre_version(void) { return 100; }

int tigre_profile(int enable) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    for (ProfRec* r : g_prof_recs) {
        cudaEventDestroy(r->a);
        cudaEventDestroy(r->b);
        delete r;
    }
    g_prof_recs.clear();
    for (int k = 0; k < PK_N; ++k) g_prof_launches[k] = 0;
    g_prof_on = enable != 0;
    return TIGRE_OK;
}
int tigre_profile_read(double* ms, uint64_t* launches) {
    std::lock_guard<std::mutex> lk(g_prof_mu);
    double acc[PK_N] = {0, 0, 0};
    for (ProfRec* r : g_prof_recs) {
        TG_CUDA(cudaEventSynchronize(r->b));
        float t = 0.f;
        TG_CUDA(cudaEventElapsedTime(&t, r->a, r->b));
        acc[r->kind] += t;
    }
    for (int k = 0; k < PK_N; ++k) {
        if (ms) ms[k] = acc[k];
        if (launches) launches[k] = g_prof_launches[k];
    }
    return TIGRE_OK;
}

const char* tigre_strerror(int code) {
    switch (code) {
        case TIGRE_OK: return "ok";
        case TIGRE_ERR_ARG: return "invalid argument";
        case TIGRE_ERR_GEOMETRY: return "invalid geometry (non-positive size/distance, or volume at/behind the source)";
        case TIGRE_ERR_MEMSPACE: return "data pointer in the wrong memory space (need device, or pinned host for the chunked path)";
        case TIGRE_ERR_WORKSPACE: return "temporary device allocation failed";
        case TIGRE_ERR_CUDA: return "CUDA error (see tigre_last_cuda_error)";
        case TIGRE_ERR_NO_DEVICE: return "no CUDA device (libtigre_b200 has no CPU fallback)";
        case TIGRE_ERR_TOO_LARGE: return "size exceeds the fixed scratch array of a no-allocation entry point (tigre_residual_noalloc: n > TIGRE_RESIDUAL_NOALLOC_MAX_N = 2^28 elements); nothing was launched";
    }
    return "unknown error";
}
const char* tigre_last_cuda_error(void) { return g_last_cuda_error.c_str(); }

int tigre_Ax(const float* vol, const tigre_geo* geo, const double* angles, int nA, int mode, float* proj,
             void* cuda_stream) {
    if (!vol || !proj) return TIGRE_ERR_ARG;
    if (mode != TIGRE_AX_SIDDON && mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const MemKind kv = mem_kind(vol), kp = mem_kind(proj);
    if (kv == MEM_PINNED && kp == MEM_PINNED) return chunked_ax(vol, geo, angles, nA, mode, proj, st);
    if (kv != MEM_DEVICE || kp != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    return device_ax(vol, t, nullptr, nA, mode, false, proj, st);
}

int tigre_Atb(const float* proj, const tigre_geo* geo, const double* angles, int nA, int mode, float* vol,
              void* cuda_stream) {
    if (!vol || !proj) return TIGRE_ERR_ARG;
    if (mode < TIGRE_ATB_MATCHED || mode > TIGRE_ATB_EXACT_INTERP) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const MemKind kv = mem_kind(vol), kp = mem_kind(proj);
    if (mode >= TIGRE_ATB_EXACT_SIDDON) {   // ray-driven exact transpose: device arrays only
        if (kv != MEM_DEVICE || kp != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
        TG_TRY(t.build_ray(nullptr, nA, st));
        return launch_ax_adjoint(proj, t.g, t.ray.as<RayView>(), nA, mode - TIGRE_ATB_EXACT_SIDDON, vol, st);
    }
    if (kv == MEM_PINNED && kp == MEM_PINNED) return chunked_atb(proj, geo, angles, nA, mode, vol, st);
    if (kv != MEM_DEVICE || kp != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    return device_atb(proj, t, nullptr, nA, mode, false, vol, st);
}

// ---------------------------------------------------------------- z-slab entry points (multi-GPU sharding)
int tigre_slab_row_band(const tigre_geo* geo, const double* angles, int nA, int z0, int nzs, int* row0, int* nrows) {
    if (!row0 || !nrows) return TIGRE_ERR_ARG;
    TG_TRY(validate_geo(geo, angles, nA));      // host arithmetic only: no device needed
    const Grid g = make_grid(geo);
    if (z0 < 0 || nzs <= 0 || z0 + nzs > g.nz) return TIGRE_ERR_ARG;
    std::vector<ViewH> views;
    resolve_views(geo, angles, nA, views);
    int lo = g.nv, hi = 0;
    for (int a = 0; a < nA; ++a) {
        int r0, nr;
        row_band(g, views[a], z0, nzs, r0, nr);
        if (nr > 0) lo = std::min(lo, r0), hi = std::max(hi, r0 + nr);
    }
    *row0 = hi > lo ? lo : 0, *nrows = hi > lo ? hi - lo : 0;
    return TIGRE_OK;
}

int tigre_Ax_slab(const float* vol_slab, const tigre_geo* geo, const double* angles, int nA, int mode, int z0, int nzs,
                  float* proj, void* cuda_stream) {
    if (!vol_slab || !proj) return TIGRE_ERR_ARG;
    if (mode != TIGRE_AX_SIDDON && mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    const Grid& g = t.g;
    if (z0 < 0 || nzs <= 0 || z0 + nzs > g.nz) return TIGRE_ERR_ARG;
    if (mem_kind(vol_slab) != MEM_DEVICE || mem_kind(proj) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    TG_CUDA(cudaMemsetAsync(proj, 0, sizeof(float) * (size_t)nA * g.nu * g.nv, st));
    AxSub sub;
    {
        int lo = g.nv, hi = 0;
        for (int a = 0; a < nA; ++a) {
            int r0, nr;
            row_band(g, t.views[a], z0, nzs, r0, nr);
            if (nr > 0) lo = std::min(lo, r0), hi = std::max(hi, r0 + nr);
        }
        sub.row0 = hi > lo ? lo : 0, sub.nrows = hi > lo ? hi - lo : 0;
    }
    if (sub.nrows == 0) return TIGRE_OK;
    std::vector<RayView> hr(nA);
    for (int i = 0; i < nA; ++i) build_ray_view(g, t.views[i], hr[i]);
    if (mode == TIGRE_AX_SIDDON) {
        // the slab as its own grid: same voxels, z origin moved to its first slice (intersection lengths are additive)
        Grid gs = g;
        gs.nz = nzs;
        for (RayView& r : hr) r.S[2] -= (double)z0, r.P0[2] -= (double)z0;
        TG_TRY(upload(t.ray, hr.data(), sizeof(RayView) * nA, st));
        sub.zs0 = 0, sub.nzs = nzs;
        return launch_ax(vol_slab, gs, t.ray.as<RayView>(), nA, mode, false, true, proj, nullptr, st, &sub);
    }
    // interpolated: the sample positions are those of the full volume; taps outside the slab count as zero
    TG_TRY(upload(t.ray, hr.data(), sizeof(RayView) * nA, st));
    sub.zs0 = z0, sub.nzs = nzs;
    return launch_ax(vol_slab, g, t.ray.as<RayView>(), nA, mode, false, true, proj, nullptr, st, &sub, nullptr, hr.data());
}

int tigre_Atb_slab(const float* proj, const tigre_geo* geo, const double* angles, int nA, int mode, int z0, int nzs,
                   float* vol_slab, void* cuda_stream) {
    if (!vol_slab || !proj) return TIGRE_ERR_ARG;
    if (mode != TIGRE_ATB_MATCHED && mode != TIGRE_ATB_FDK) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    const Grid& g = t.g;
    if (z0 < 0 || nzs <= 0 || z0 + nzs > g.nz) return TIGRE_ERR_ARG;
    if (mem_kind(vol_slab) != MEM_DEVICE || mem_kind(proj) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    TG_TRY(t.build_vox(nullptr, nA, st));
    return launch_atb(proj, g, t.vox.as<VoxView>(), nA, mode, false, vol_slab, z0, nzs, false, 0, g.nv, t.clamp, st,
                      t.hvox.data());
}

int tigre_row_weights(const tigre_geo* geo, const double* angles, int nA, int ax_mode, float* W, void* cuda_stream) {
    if (!W) return TIGRE_ERR_ARG;
    if (ax_mode != TIGRE_AX_SIDDON && ax_mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(W) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    TG_TRY(device_ax(nullptr, t, nullptr, nA, ax_mode, true, W, st));
    const double eps = 1e-2 * std::min(t.g.dx, std::min(t.g.dy, t.g.dz));
    return launch_invert_rows(W, (size_t)nA * t.g.nu * t.g.nv, (float)eps, st);
}

int tigre_col_weights(const tigre_geo* geo, const double* angles, int nA, int atb_mode, float* V, void* cuda_stream) {
    if (!V) return TIGRE_ERR_ARG;
    if (atb_mode != TIGRE_ATB_MATCHED && atb_mode != TIGRE_ATB_FDK) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(V) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    TG_TRY(device_atb(nullptr, t, nullptr, nA, atb_mode, true, V, st));
    return launch_invert_cols(V, (size_t)t.g.nx * t.g.ny * t.g.nz, 1e-6f, st);
}

int tigre_residual(const float* b, const float* Ax, const float* W, float* r, size_t n, double* nrm2, void* cuda_stream) {
    if (n == 0) {
        if (nrm2) *nrm2 = 0.0;
        return TIGRE_OK;
    }
    if (!b || !Ax || !r) return TIGRE_ERR_ARG;
    TG_TRY(ensure_device());
    cudaStream_t st = (cudaStream_t)cuda_stream;
    TempBuf acc;
    if (nrm2) {
        TG_TRY(acc.alloc(sizeof(double), st));
        TG_CUDA(cudaMemsetAsync(acc.p, 0, sizeof(double), st));
    }
    TG_TRY(launch_residual(b, nullptr, Ax, W, r, n, 1, nrm2 ? acc.as<double>() : nullptr, st));
    if (nrm2) {
        TG_CUDA(cudaMemcpyAsync(nrm2, acc.p, sizeof(double), cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
    }
    return TIGRE_OK;
}

int tigre_update(float* x, const float* g, const float* V, float lambda, int nonneg, size_t n, void* cuda_stream) {
    if (n == 0) return TIGRE_OK;
    if (!x || !g) return TIGRE_ERR_ARG;
    TG_TRY(ensure_device());
    return launch_update(x, g, V, lambda, nonneg, n, (cudaStream_t)cuda_stream);
}

int tigre_Ax_count(const tigre_geo* geo, const double* angles, int nA, int mode, uint32_t* counts, uint64_t* total,
                   void* cuda_stream) {
    if (mode != TIGRE_AX_SIDDON && mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)nA * t.g.nu * t.g.nv;
    TempBuf own, tot;
    uint32_t* c = counts;
    if (!c) {
        TG_TRY(own.alloc(n * sizeof(uint32_t), st));
        c = own.as<uint32_t>();
    } else if (mem_kind(counts) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    TG_TRY(t.build_ray(nullptr, nA, st));
    TG_TRY(launch_ax(nullptr, t.g, t.ray.as<RayView>(), nA, mode, false, false, nullptr, c, st));
    if (total) {
        TG_TRY(tot.alloc(sizeof(unsigned long long), st));
        TG_TRY(launch_count_reduce(c, n, tot.as<unsigned long long>(), st));
        unsigned long long h = 0;
        TG_CUDA(cudaMemcpyAsync(&h, tot.p, sizeof h, cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        *total = h;
    }
    return TIGRE_OK;
}

int tigre_Ax_index(const tigre_geo* geo, const double* angles, int nA, int64_t* first_last, uint32_t* nseg, void* cuda_stream) {
    if (!first_last || !nseg) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(first_last) != MEM_DEVICE || mem_kind(nseg) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    TG_TRY(t.build_ray(nullptr, nA, st));
    static_assert(sizeof(long long) == sizeof(int64_t), "int64_t is long long here");
    return launch_ax_track(t.g, t.ray.as<RayView>(), nA, nseg, reinterpret_cast<long long*>(first_last), st);
}

int tigre_set_workspace(void* dev_ptr, size_t bytes) {
    std::lock_guard<std::mutex> lk(g_ws.mu);
    if (!g_ws.used.empty()) return TIGRE_ERR_ARG;   // a plan or a call in flight still holds blocks of the current workspace
    if (dev_ptr && bytes < 4096) return TIGRE_ERR_ARG;
    if (dev_ptr && mem_kind(dev_ptr) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    g_ws.free_.clear();
    g_ws.in_use = g_ws.high = 0, g_ws.pool_allocs = 0;
    if (!dev_ptr) {
        g_ws.base = nullptr, g_ws.size = 0;
        return TIGRE_OK;
    }
    // carve from the first 256-byte boundary inside the block
    const size_t mis = (size_t)((uintptr_t)dev_ptr & 255), skip = mis ? 256 - mis : 0;
    g_ws.base = (char*)dev_ptr + skip, g_ws.size = (bytes - skip) & ~(size_t)255;
    g_ws.free_[0] = g_ws.size;
    return TIGRE_OK;
}

int tigre_workspace_stats(size_t* in_use, size_t* high_water, uint64_t* pool_allocs) {
    std::lock_guard<std::mutex> lk(g_ws.mu);
    if (in_use) *in_use = g_ws.in_use;
    if (high_water) *high_water = g_ws.high;
    if (pool_allocs) *pool_allocs = g_ws.pool_allocs;
    return TIGRE_OK;
}

int tigre_microbench(int kind, double* value, void* cuda_stream) {
    if (!value) return TIGRE_ERR_ARG;
    TG_TRY(ensure_device());
    return microbench(kind, value, (cudaStream_t)cuda_stream);
}

// test hook (tigre_set_plan_v_path): 0 = store V_s per subset when they fit (default), 1 = always store, 2 = always recompute
static int g_plan_v_path = 0;
static int g_plan_fuse = 1;   // 1 = the OS-SART update runs in the backprojector's epilogue where it can (fusion F2), 0 = always as its own kernel (tigre_set_plan_fuse)
}  // extern "C"
namespace tg {
extern int* g_atb_box_meta;
extern int32_t* g_atb_boxes;
}
extern "C" {
int tigre_Atb_boxes(const float* proj, const tigre_geo* geo, const double* angles, int nA, int mode, float* vol, int32_t* meta,
                    int32_t* boxes, void* cuda_stream) {
    if (!proj || !vol || !meta) return TIGRE_ERR_ARG;
    if (mode != TIGRE_ATB_MATCHED && mode != TIGRE_ATB_FDK) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(proj) != MEM_DEVICE || mem_kind(vol) != MEM_DEVICE || (boxes && mem_kind(boxes) != MEM_DEVICE)) return TIGRE_ERR_MEMSPACE;
    for (int i = 0; i < 8; ++i) meta[i] = 0;
    g_atb_box_meta = meta, g_atb_boxes = boxes;
    const int rc = device_atb(proj, t, nullptr, nA, mode, false, vol, (cudaStream_t)cuda_stream);
    g_atb_box_meta = nullptr, g_atb_boxes = nullptr;
    return rc;
}

int tigre_set_plan_v_path(int path) {
    if (path < 0 || path > 2) return TIGRE_ERR_ARG;
    g_plan_v_path = path;
    return TIGRE_OK;
}

int tigre_set_plan_fuse(int on) {
    if (on != 0 && on != 1) return TIGRE_ERR_ARG;
    g_plan_fuse = on;
    return TIGRE_OK;
}

int tigre_set_index_path(int path) {
    if (path != 0 && path != 1) return TIGRE_ERR_ARG;
    set_index_path(path);
    return TIGRE_OK;
}

// ---------------------------------------------------------------- OS-SART / SIRT
// A plan holds what does not change between iterations: the per-subset view tables, the row weights
// W_s = 1/(A_s 1) and column weights V_s = 1/(A_s^T 1) (P13, P16) and the scratch buffers.
struct tigre_plan {
    Tables t;
    int nA = 0, nSubsets = 0, maxs = 0, ax_mode = 0, atb_mode = 0;
    std::vector<int32_t> idx, off;
    std::vector<TempBuf> ray, vox;
    std::vector<std::vector<VoxView>> hvox;
    std::vector<std::vector<RayView>> hray;
    TempBuf W, V, Axb, grad, d_idx, d_acc;
    size_t bytes = 0;
    bool clamp = false;
    // Column weights: one volume per subset while nSubsets volumes fit the plan's share of the device (C3: 20 x 537 MB), else
    // ONE volume that every subset step refills (A_s^T 1 through the same TMA kernel, from a buffer of ones: one more
    // backprojection per subset).  Single-view subsets (SART, ASD-POCS, SART-TV) of a 512^3 problem would need 386 GB stored.
    bool v_stored = true;
    // V_s of subset s, ready to use on the stream (stored: a pointer; otherwise computed now into the one volume)
    int col_weights(int s, float** out, cudaStream_t st) {
        const Grid& g = t.g;
        const size_t nvox = (size_t)g.nx * g.ny * g.nz, per = (size_t)g.nu * g.nv;
        if (v_stored) {
            *out = V.as<float>() + nvox * s;
            return TIGRE_OK;
        }
        const int n = off[s + 1] - off[s];
        float* ones = Axb.as<float>();   // free between two subset steps
        TG_TRY(launch_fill(ones, 1.0f, per * n, st));
        TG_TRY(launch_atb(ones, g, vox[s].as<VoxView>(), n, atb_mode, false, V.as<float>(), 0, g.nz, false, 0, g.nv, clamp, st, hvox[s].data()));
        TG_TRY(launch_invert_cols(V.as<float>(), nvox, 1e-6f, st));
        *out = V.as<float>();
        return TIGRE_OK;
    }
};

int tigre_plan_create(const tigre_geo* geo, const double* angles, int nA, const int32_t* subset_idx,
                      const int32_t* subset_off, int nSubsets, int ax_mode, int atb_mode, void* cuda_stream,
                      tigre_plan** out) {
    return tigre_plan_create_ex(geo, angles, nA, subset_idx, subset_off, nSubsets, ax_mode, atb_mode, 0, cuda_stream, out);
}

int tigre_plan_create_ex(const tigre_geo* geo, const double* angles, int nA, const int32_t* subset_idx,
                         const int32_t* subset_off, int nSubsets, int ax_mode, int atb_mode, int redundancy,
                         void* cuda_stream, tigre_plan** out) {
    if (!out || !subset_idx || !subset_off || nSubsets <= 0) return TIGRE_ERR_ARG;
    *out = nullptr;
    if (ax_mode != TIGRE_AX_SIDDON && ax_mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    if (atb_mode != TIGRE_ATB_MATCHED && atb_mode != TIGRE_ATB_FDK) return TIGRE_ERR_ARG;
    std::unique_ptr<tigre_plan> P(new tigre_plan);
    TG_TRY(prep(geo, angles, nA, P->t));
    cudaStream_t st = (cudaStream_t)cuda_stream;
    P->nA = nA, P->nSubsets = nSubsets, P->ax_mode = ax_mode, P->atb_mode = atb_mode;
    for (int s = 0; s < nSubsets; ++s) {
        const int n = subset_off[s + 1] - subset_off[s];
        if (n <= 0) return TIGRE_ERR_ARG;
        P->maxs = std::max(P->maxs, n);
        for (int k = subset_off[s]; k < subset_off[s + 1]; ++k)
            if (subset_idx[k] < 0 || subset_idx[k] >= nA) return TIGRE_ERR_ARG;
    }
    const int nIdx = subset_off[nSubsets];
    P->idx.assign(subset_idx, subset_idx + nIdx);
    P->off.assign(subset_off, subset_off + nSubsets + 1);
    const Grid& g = P->t.g;
    const size_t per = (size_t)g.nu * g.nv, nvox = (size_t)g.nx * g.ny * g.nz;
    TG_TRY(P->W.alloc(sizeof(float) * per * nIdx, st));
    {
        // store V_s per subset if that takes at most half of what is free now (or of the caller's workspace)
        size_t fr = 0, tot = 0;
        if (workspace_active()) fr = workspace_free_bytes();
        else if (cudaMemGetInfo(&fr, &tot) != cudaSuccess) fr = 0, (void)cudaGetLastError();
        P->v_stored = nSubsets == 1 || sizeof(float) * nvox * (size_t)nSubsets <= fr / 2;
        if (g_plan_v_path == 1) P->v_stored = true;
        if (g_plan_v_path == 2) P->v_stored = false;
    }
    TG_TRY(P->V.alloc(sizeof(float) * nvox * (P->v_stored ? nSubsets : 1), st));
    TG_TRY(P->Axb.alloc(sizeof(float) * per * P->maxs, st));
    TG_TRY(P->grad.alloc(sizeof(float) * nvox, st));
    TG_TRY(upload(P->d_idx, subset_idx, sizeof(int32_t) * nIdx, st));
    P->bytes = sizeof(float) * (per * nIdx + nvox * (P->v_stored ? nSubsets : 1) + per * P->maxs + nvox);
    P->ray = std::vector<TempBuf>(nSubsets);
    P->vox = std::vector<TempBuf>(nSubsets);
    P->hvox.resize(nSubsets);
    P->hray.resize(nSubsets);
    const double epsW = 1e-2 * std::min(g.dx, std::min(g.dy, g.dz));
    std::vector<double> red;
    if (redundancy) TG_TRY(fdk_weights(g, P->t.views, TIGRE_FDK_WANG, red));   // [nA][nu], reading P17 / P28
    for (int s = 0; s < nSubsets; ++s) {
        const int32_t* idx = subset_idx + subset_off[s];
        const int n = subset_off[s + 1] - subset_off[s];
        std::vector<RayView>& hr = P->hray[s];
        hr.resize(n);
        std::vector<VoxView>& hv = P->hvox[s];
        hv.resize(n);
        for (int i = 0; i < n; ++i) {
            build_ray_view(g, P->t.views[idx[i]], hr[i]);
            TG_TRY(build_vox_view(g, P->t.views[idx[i]], hv[i]));
        }
        TG_TRY(upload(P->ray[s], hr.data(), sizeof(RayView) * n, st));
        P->clamp = P->clamp || vox_needs_clamp(g, hv.data(), n);
        TG_TRY(upload(P->vox[s], hv.data(), sizeof(VoxView) * n, st));
        float* Ws = P->W.as<float>() + per * subset_off[s];
        TG_TRY(launch_ax(nullptr, g, P->ray[s].as<RayView>(), n, ax_mode, true, false, Ws, nullptr, st));
        TG_TRY(launch_invert_rows(Ws, per * n, (float)epsW, st));
        if (redundancy) {
            std::vector<float> cw((size_t)n * g.nu);
            for (int i = 0; i < n; ++i)
                for (int iu = 0; iu < g.nu; ++iu) cw[(size_t)i * g.nu + iu] = (float)red[(size_t)idx[i] * g.nu + iu];
            TempBuf tc;
            TG_TRY(upload(tc, cw.data(), sizeof(float) * cw.size(), st));
            TG_TRY(launch_scale_columns(Ws, tc.as<float>(), n, g.nv, g.nu, st));
        }
        if (P->v_stored) {
            // A_s^T 1 as the backprojection of a buffer of ones through the TMA kernel (4 ms per C3 subset; the gather kernel's
            // unit-projection variant, which it replaces here, took 6)
            float* Vs = P->V.as<float>() + nvox * s;
            TG_TRY(launch_fill(P->Axb.as<float>(), 1.0f, per * n, st));
            TG_TRY(launch_atb(P->Axb.as<float>(), g, P->vox[s].as<VoxView>(), n, atb_mode, false, Vs, 0, g.nz, false, 0, g.nv, P->clamp, st,
                              hv.data()));
            TG_TRY(launch_invert_cols(Vs, nvox, 1e-6f, st));
        }
    }
    *out = P.release();
    return TIGRE_OK;
}

int tigre_plan_destroy(tigre_plan* plan) {
    delete plan;   // TempBuf destructors return the buffers to the stream-ordered pool
    return TIGRE_OK;
}

size_t tigre_plan_bytes(const tigre_plan* plan) { return plan ? plan->bytes : 0; }

static int plan_ossart_impl(tigre_plan* P, const float* b, float* x, int n_iter, float lambda, int nonneg, double* resid_hist,
                            void* cuda_stream, int s_begin, int s_end);

int tigre_plan_ossart(tigre_plan* P, const float* b, float* x, int n_iter, float lambda, int nonneg,
                      double* resid_hist, void* cuda_stream) {
    if (!P) return TIGRE_ERR_ARG;
    return plan_ossart_impl(P, b, x, n_iter, lambda, nonneg, resid_hist, cuda_stream, 0, P->nSubsets);
}

int tigre_plan_ossart_subsets(tigre_plan* P, const float* b, float* x, int s_begin, int s_end, float lambda, int nonneg,
                              void* cuda_stream) {
    if (!P || s_begin < 0 || s_end > P->nSubsets || s_begin > s_end) return TIGRE_ERR_ARG;
    if (s_begin == s_end) return TIGRE_OK;
    return plan_ossart_impl(P, b, x, 1, lambda, nonneg, nullptr, cuda_stream, s_begin, s_end);
}

// z-slices [zlo, zhi] of the volume that rays of detector rows [r0, r1) of these cone-beam views can meet (zlo > zhi: none), or
// false if no bound is formed (parallel beam, source or detector over the volume's (x,y) footprint).  The points such rays reach
// inside the footprint are (pyramid over the band from the source) n (footprint x all z), a convex polytope: its z-extremes are at
// corner rays clipped to the footprint, or where a vertical edge of the footprint meets one of the pyramid's four side planes
// (all eight taken, whether or not inside the face: a superset).  RayView is in voxel-index coordinates.  Three slices of margin.
static bool band_z_range(const RayView* hv, int nViews, const Grid& g, int r0, int r1, int& zlo, int& zhi) {
    double lo = 1e300, hi = -1e300;
    const double bx[2] = {0.0, (double)g.nx}, by[2] = {0.0, (double)g.ny};
    for (int a = 0; a < nViews; ++a) {
        const RayView& rv = hv[a];
        for (int k = 0; k < 3; ++k)
            if (rv.dSU[k] != 0.0 || rv.dSV[k] != 0.0) return false;
        const double* S = rv.S;
        if (S[0] >= bx[0] && S[0] <= bx[1] && S[1] >= by[0] && S[1] <= by[1]) return false;
        double d[4][3];
        for (int c = 0; c < 4; ++c) {
            const double iu = (c & 1) ? g.nu - 1 : 0, iv = (c & 2) ? r1 - 1 : r0;
            for (int k = 0; k < 3; ++k) d[c][k] = rv.P0[k] + iu * rv.dU[k] + iv * rv.dV[k] - S[k];
            double t0 = 0.0, t1 = 1.0;
            for (int k = 0; k < 2; ++k) {
                const double n = k == 0 ? bx[1] : by[1];
                if (d[c][k] != 0.0) {
                    const double ta = (0.0 - S[k]) / d[c][k], tb = (n - S[k]) / d[c][k];
                    t0 = std::max(t0, std::min(ta, tb)), t1 = std::min(t1, std::max(ta, tb));
                } else if (S[k] < 0.0 || S[k] > n) {
                    t1 = -1.0;
                }
            }
            if (t1 >= t0) {
                if (t1 >= 1.0) return false;   // the detector pixel itself lies over the footprint
                const double za = S[2] + t0 * d[c][2], zb = S[2] + t1 * d[c][2];
                lo = std::min(lo, std::min(za, zb)), hi = std::max(hi, std::max(za, zb));
            }
        }
        const int face[4][2] = {{0, 1}, {2, 3}, {0, 2}, {1, 3}};   // bottom row, top row, first column, last column
        for (int f = 0; f < 4; ++f) {
            const double* p = d[face[f][0]];
            const double* q = d[face[f][1]];
            const double n[3] = {p[1] * q[2] - p[2] * q[1], p[2] * q[0] - p[0] * q[2], p[0] * q[1] - p[1] * q[0]};
            const double nn = std::sqrt(n[0] * n[0] + n[1] * n[1] + n[2] * n[2]);
            if (!(std::fabs(n[2]) > 1e-9 * nn)) continue;   // a vertical face holds no isolated point of a vertical edge
            for (int e = 0; e < 4; ++e) {
                const double z = S[2] - (n[0] * (bx[e & 1] - S[0]) + n[1] * (by[e >> 1] - S[1])) / n[2];
                lo = std::min(lo, z), hi = std::max(hi, z);
            }
        }
    }
    if (hi < lo) {
        zlo = 0, zhi = -1;
        return true;
    }
    zlo = (int)std::max(0.0, std::floor(std::max(lo, -1e8)) - 3.0), zhi = (int)std::min((double)g.nz - 1.0, std::floor(std::min(hi, 1e8)) + 3.0);
    return true;
}

int tigre_band_z_range(const tigre_geo* geo, const double* angles, int nA, int row0, int row1, int32_t* zlo, int32_t* zhi) {
    if (!zlo || !zhi) return TIGRE_ERR_ARG;
    TG_TRY(validate_geo(geo, angles, nA));
    const Grid g = make_grid(geo);
    if (row0 < 0 || row1 > g.nv || row0 >= row1) return TIGRE_ERR_ARG;
    std::vector<ViewH> views;
    resolve_views(geo, angles, nA, views);
    std::vector<RayView> h(nA);
    for (int i = 0; i < nA; ++i) build_ray_view(g, views[i], h[i]);
    int lo = 0, hi = -1;
    if (!band_z_range(h.data(), nA, g, row0, row1, lo, hi)) return 1;
    *zlo = lo, *zhi = hi;
    return TIGRE_OK;
}

static int plan_ossart_impl(tigre_plan* P, const float* b, float* x, int n_iter, float lambda, int nonneg, double* resid_hist,
                            void* cuda_stream, int s_begin, int s_end) {
    if (!P || !b || !x || n_iter < 0) return TIGRE_ERR_ARG;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = P->t.g;
    const size_t per = (size_t)g.nu * g.nv, nvox = (size_t)g.nx * g.ny * g.nz;
    // b and x may live in device memory, or both in pinned host memory (end-to-end path: the
    // projections and the iterate are copied in, the iterate is copied back, all on `st`)
    const MemKind kb = mem_kind(b), kx = mem_kind(x);
    TempBuf db, dx, xT;
    const float* bd = b;
    float* xd = x;
    constexpr int X_BANDS = 8, AX_ROW_ALIGN = 4;   // bands of detector rows of the first projection (multiples of the Ax kernels' 4-row tiles; 4 bands: +1.1 ms on C3)
    constexpr int X_DOWN = 4;                      // z-ranges of the last update, downloaded one behind the other
    bool banded = false, downloaded = false;
    std::vector<std::vector<std::array<size_t, 2>>> bandRuns;   // per band (and one more for the rest): runs {first slice, count} of the iterate
    std::vector<int> bandRow0, bandRows;
    int sbase = 1;
    // end-to-end path: the projections go up on a side stream in the order the subsets need them (one event per subset:
    // the first sweep's residual of subset s waits for its views only), so all but the first subset's upload hides
    // behind the kernels; the iterate goes up first on the caller's stream
    cudaStream_t up = nullptr;
    std::vector<cudaEvent_t> ev;
    struct Cleanup {
        cudaStream_t& s;
        std::vector<cudaEvent_t>& e;
        ~Cleanup() {   // destroyed before db / dx (declared after them): the upload stream is idle before they are released
            if (s) cudaStreamSynchronize(s);
            for (cudaEvent_t x : e) cudaEventDestroy(x);
            if (s) cudaStreamDestroy(s);
            (void)cudaGetLastError();
        }
    } cleanup{up, ev};
    if (kb == MEM_PINNED && kx == MEM_PINNED) {
        TG_TRY(db.alloc(sizeof(float) * per * P->nA, st));
        TG_TRY(dx.alloc(sizeof(float) * nvox, st));
        bd = db.as<float>(), xd = dx.as<float>();
        // The iterate: the first subset's projection is cut into bands of detector rows, each of which meets only a range of z-slices
        // (band_z_range); the slices go up on the side stream in the order the bands need them, one event per band, so the first
        // band's rays start when a quarter of the volume has arrived instead of all of it.  Without a bound (or without the
        // transposed copy, which the bands fill slice range by slice range) the iterate goes up whole on the caller's stream.
        const size_t slice = (size_t)g.nx * g.ny;
        if (n_iter > 0 && g.nz >= 4 * X_BANDS && g.nx > 1 && g.ny > 1 && xT.alloc(sizeof(float) * nvox, st) == TIGRE_OK) {
            const int rows = ((g.nv + X_BANDS - 1) / X_BANDS + AX_ROW_ALIGN - 1) / AX_ROW_ALIGN * AX_ROW_ALIGN;
            std::vector<char> sent(g.nz, 0);
            banded = true;
            for (int bnd = 0; bnd < X_BANDS && banded; ++bnd) {
                const int r0 = std::min(bnd * rows, g.nv), r1 = std::min(r0 + rows, g.nv);
                int zlo = 0, zhi = -1;
                if (r1 > r0 && !band_z_range(P->hray[s_begin].data(), P->off[s_begin + 1] - P->off[s_begin], g, r0, r1, zlo, zhi)) banded = false;
                bandRow0.push_back(r0), bandRows.push_back(r1 - r0);
                bandRuns.emplace_back();
                for (int z = zlo; z <= zhi; ++z) {
                    if (sent[z]) continue;
                    int z1 = z;
                    while (z1 <= zhi && !sent[z1]) sent[z1++] = 1;
                    bandRuns.back().push_back(std::array<size_t, 2>{(size_t)z, (size_t)(z1 - z)});
                    z = z1 - 1;
                }
            }
            if (banded) {
                bandRuns.emplace_back();   // the slices no band asked for
                for (int z = 0; z < g.nz; ++z) {
                    if (sent[z]) continue;
                    int z1 = z;
                    while (z1 < g.nz && !sent[z1]) sent[z1++] = 1;
                    bandRuns.back().push_back(std::array<size_t, 2>{(size_t)z, (size_t)(z1 - z)});
                    z = z1 - 1;
                }
            } else {
                bandRuns.clear(), bandRow0.clear(), bandRows.clear();
            }
        }
        if (!banded) TG_CUDA(cudaMemcpyAsync(dx.p, x, sizeof(float) * nvox, cudaMemcpyHostToDevice, st));
        if (n_iter > 0) {
            TG_CUDA(cudaStreamCreateWithFlags(&up, cudaStreamNonBlocking));
            cudaEvent_t start;
            TG_CUDA(cudaEventCreateWithFlags(&start, cudaEventDisableTiming));
            ev.push_back(start);
            TG_CUDA(cudaEventRecord(start, st));               // the buffer exists from here on in stream order
            TG_CUDA(cudaStreamWaitEvent(up, start, 0));
            for (size_t bnd = 0; bnd < bandRuns.size(); ++bnd) {
                for (const auto& run : bandRuns[bnd])
                    TG_CUDA(cudaMemcpyAsync(dx.as<float>() + run[0] * slice, x + run[0] * slice, sizeof(float) * slice * run[1], cudaMemcpyHostToDevice, up));
                cudaEvent_t e;
                TG_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
                ev.push_back(e);
                TG_CUDA(cudaEventRecord(e, up));
            }
            sbase = (int)ev.size();   // ev[sbase + s - s_begin]: subset s's projections have arrived
            for (int s = s_begin; s < s_end; ++s) {
                for (int k = P->off[s]; k < P->off[s + 1]; ++k) {
                    const size_t o = per * (size_t)P->idx[k];
                    TG_CUDA(cudaMemcpyAsync(db.as<float>() + o, b + o, sizeof(float) * per, cudaMemcpyHostToDevice, up));
                }
                cudaEvent_t e;
                TG_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
                ev.push_back(e);
                TG_CUDA(cudaEventRecord(e, up));
            }
        }
    } else if (kb != MEM_DEVICE || kx != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    TG_TRY(P->d_acc.alloc(sizeof(double) * std::max(n_iter, 1), st));
    TG_CUDA(cudaMemsetAsync(P->d_acc.p, 0, sizeof(double) * std::max(n_iter, 1), st));
    // the (x,y)-transposed copy of the iterate that the Ax kernels read for x-dominant rays is kept up to date by the
    // update kernel (one pass over the volume per subset instead of two)
    float* xTd = nullptr;
    if (banded) xTd = xT.as<float>();   // filled band by band below
    else if (n_iter > 0 && g.nx > 1 && g.ny > 1 && (xT.p || xT.alloc(sizeof(float) * nvox, st) == TIGRE_OK) &&
             launch_transpose_xy(xd, xT.as<float>(), g, st) == TIGRE_OK)
        xTd = xT.as<float>();
    for (int it = 0; it < n_iter; ++it) {
        for (int s = s_begin; s < s_end; ++s) {
            const int n = P->off[s + 1] - P->off[s];
            float* Ws = P->W.as<float>() + per * P->off[s];
            float* Vs = nullptr;
            float* A = P->Axb.as<float>();
            TG_TRY(P->col_weights(s, &Vs, st));   // (when V_s is not stored this uses A as scratch: before this subset's projection)
            if (banded && it == 0 && s == s_begin) {
                const size_t slice = (size_t)g.nx * g.ny;
                for (size_t bnd = 0; bnd < bandRuns.size(); ++bnd) {
                    TG_CUDA(cudaStreamWaitEvent(st, ev[1 + bnd], 0));   // this band's slices of the iterate have arrived
                    for (const auto& run : bandRuns[bnd]) {
                        Grid gs = g;
                        gs.nz = (int)run[1];
                        TG_TRY(launch_transpose_xy(xd + run[0] * slice, xTd + run[0] * slice, gs, st));
                    }
                    if (bnd < bandRows.size() && bandRows[bnd] > 0) {
                        const AxSub sub{bandRow0[bnd], bandRows[bnd], 0, g.nz};
                        TG_TRY(launch_ax(xd, g, P->ray[s].as<RayView>(), n, P->ax_mode, false, false, A, nullptr, st, &sub, xTd, P->hray[s].data()));
                    }
                }
            } else {
                TG_TRY(launch_ax(xd, g, P->ray[s].as<RayView>(), n, P->ax_mode, false, false, A, nullptr, st, nullptr, xTd, P->hray[s].data()));
            }
            if (up && it == 0) TG_CUDA(cudaStreamWaitEvent(st, ev[sbase + s - s_begin], 0));   // this subset's projections have arrived
            // r = W_s .* (b_s - A_s x) in place over A; b is gathered through the subset's view list
            TG_TRY(launch_residual(bd, P->d_idx.as<int32_t>() + P->off[s], A, Ws, A, per, n, P->d_acc.as<double>() + it, st));
            if (up && xTd && it == n_iter - 1 && s == s_end - 1 && g.nz >= 32 * X_DOWN) {
                // last update of an end-to-end call: backprojection and update go range by range of z-slices (whole 32-slice blocks of
                // the backprojector), and each range of the new iterate starts for the host on the side stream as soon as it is final,
                // behind the ranges still being computed (the same kernels on the same data: the same bits)
                const size_t slice = (size_t)g.nx * g.ny;
                const int step = (g.nz / X_DOWN + 31) / 32 * 32;
                for (int z0 = 0; z0 < g.nz; z0 += step) {
                    const int nzs = std::min(step, g.nz - z0);
                    const size_t o = (size_t)z0 * slice;
                    const AtbFuse fz{xTd + o, Vs ? Vs + o : nullptr, lambda, nonneg};
                    const int frc = g_plan_fuse ? launch_atb(A, g, P->vox[s].as<VoxView>(), n, P->atb_mode, false, xd + o, z0, nzs, false, 0, g.nv, P->clamp, st,
                                                             P->hvox[s].data(), &fz) : 2;
                    if (frc < 0) return frc;
                    if (frc == 2) {
                        TG_TRY(launch_atb(A, g, P->vox[s].as<VoxView>(), n, P->atb_mode, false, P->grad.as<float>() + o, z0, nzs, false, 0, g.nv, P->clamp, st,
                                          P->hvox[s].data()));
                        TG_TRY(launch_update_t(xd + o, xTd + o, P->grad.as<float>() + o, Vs ? Vs + o : nullptr, lambda, nonneg, g.nx, g.ny, nzs, st));
                    }
                    cudaEvent_t e;
                    TG_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
                    ev.push_back(e);
                    TG_CUDA(cudaEventRecord(e, st));
                    TG_CUDA(cudaStreamWaitEvent(up, e, 0));
                    TG_CUDA(cudaMemcpyAsync(x + o, xd + o, sizeof(float) * slice * nzs, cudaMemcpyDeviceToHost, up));
                }
                cudaEvent_t e;
                TG_CUDA(cudaEventCreateWithFlags(&e, cudaEventDisableTiming));
                ev.push_back(e);
                TG_CUDA(cudaEventRecord(e, up));
                TG_CUDA(cudaStreamWaitEvent(st, e, 0));   // the caller's stream is done when the iterate is on the host
                downloaded = true;
                continue;
            }
            if (xTd && g_plan_fuse) {   // F2: the update in the backprojector's epilogue (where the TMA kernel takes the problem)
                const AtbFuse fz{xTd, Vs, lambda, nonneg};
                const int frc = launch_atb(A, g, P->vox[s].as<VoxView>(), n, P->atb_mode, false, xd, 0, g.nz, false, 0, g.nv, P->clamp, st, P->hvox[s].data(), &fz);
                if (frc < 0) return frc;
                if (frc == TIGRE_OK) continue;
            }
            TG_TRY(launch_atb(A, g, P->vox[s].as<VoxView>(), n, P->atb_mode, false, P->grad.as<float>(), 0, g.nz, false, 0, g.nv, P->clamp, st,
                              P->hvox[s].data()));
            if (xTd) TG_TRY(launch_update_t(xd, xTd, P->grad.as<float>(), Vs, lambda, nonneg, g.nx, g.ny, g.nz, st));
            else TG_TRY(launch_update(xd, P->grad.as<float>(), Vs, lambda, nonneg, nvox, st));
        }
    }
    if (xd != x && !downloaded) TG_CUDA(cudaMemcpyAsync(x, xd, sizeof(float) * nvox, cudaMemcpyDeviceToHost, st));
    if (resid_hist && n_iter > 0) {
        std::vector<double> h(n_iter);
        TG_CUDA(cudaMemcpyAsync(h.data(), P->d_acc.p, sizeof(double) * n_iter, cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        for (int it = 0; it < n_iter; ++it) resid_hist[it] = std::sqrt(h[it]);
    } else if (xd != x) {
        TG_CUDA(cudaStreamSynchronize(st));
    }
    return TIGRE_OK;
}

int tigre_ossart(const float* b, const tigre_geo* geo, const double* angles, int nA, const int32_t* subset_idx,
                 const int32_t* subset_off, int nSubsets, int n_iter, float lambda, int nonneg, int ax_mode,
                 int atb_mode, float* x, double* resid_hist, void* cuda_stream) {
    if (!b || !x) return TIGRE_ERR_ARG;
    tigre_plan* P = nullptr;
    TG_TRY(tigre_plan_create(geo, angles, nA, subset_idx, subset_off, nSubsets, ax_mode, atb_mode, cuda_stream, &P));
    const int rc = tigre_plan_ossart(P, b, x, n_iter, lambda, nonneg, resid_hist, cuda_stream);
    tigre_plan_destroy(P);
    return rc;
}

int tigre_sirt_chunked(const float* b, const tigre_geo* geo, const double* angles, int nA, int n_iter, float lambda, int nonneg,
                       int ax_mode, int atb_mode, float* x_inout, float* r_scratch, double* resid_hist, void* cuda_stream) {
    if (!b || !x_inout || !r_scratch || n_iter < 0) return TIGRE_ERR_ARG;
    if (ax_mode != TIGRE_AX_SIDDON && ax_mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    if (atb_mode != TIGRE_ATB_MATCHED && atb_mode != TIGRE_ATB_FDK) return TIGRE_ERR_ARG;
    if (r_scratch == b && n_iter > 1) return TIGRE_ERR_ARG;   // the residual would overwrite data a later iteration needs
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(b) != MEM_PINNED || mem_kind(x_inout) != MEM_PINNED || mem_kind(r_scratch) != MEM_PINNED) return TIGRE_ERR_MEMSPACE;
    return chunked_sirt(b, geo, angles, nA, n_iter, lambda, nonneg, ax_mode, atb_mode, x_inout, r_scratch, resid_hist,
                        (cudaStream_t)cuda_stream);
}

// ---------------------------------------------------------------- MLEM / OSEM (eq. 5; reading P33)
int tigre_plan_osem(tigre_plan* P, const float* b, float* x, int n_iter, void* cuda_stream) {
    if (!P || !b || !x || n_iter < 0) return TIGRE_ERR_ARG;
    if (mem_kind(b) != MEM_DEVICE || mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = P->t.g;
    const size_t per = (size_t)g.nu * g.nv, nvox = (size_t)g.nx * g.ny * g.nz;
    for (int it = 0; it < n_iter; ++it) {
        for (int s = 0; s < P->nSubsets; ++s) {
            const int n = P->off[s + 1] - P->off[s];
            float* A = P->Axb.as<float>();
            float* Vs = nullptr;
            TG_TRY(P->col_weights(s, &Vs, st));
            TG_TRY(launch_ax(x, g, P->ray[s].as<RayView>(), n, P->ax_mode, false, false, A, nullptr, st, nullptr, nullptr, P->hray[s].data()));
            TG_TRY(launch_ratio(b, P->d_idx.as<int32_t>() + P->off[s], A, A, per, n, st));
            TG_TRY(launch_atb(A, g, P->vox[s].as<VoxView>(), n, P->atb_mode, false, P->grad.as<float>(), 0, g.nz, false, 0, g.nv, P->clamp,
                              st, P->hvox[s].data()));
            TG_TRY(launch_mul_update(x, P->grad.as<float>(), Vs, nvox, st));
        }
    }
    return TIGRE_OK;
}

// ---------------------------------------------------------------- ASD-POCS family (reading P23; oracle/pocs.py)
// Data step = one OS-SART sweep of the plan with relaxation beta; regulariser step = ng normalised steepest-descent
// steps on (Aw)TV.  The control scalars (dd, dp, dg) decide the next step length on the host: two stream
// synchronisations per iteration, against hundreds of kernel launches.
int tigre_plan_asd_pocs(tigre_plan* P, const float* b, float* x, int n_iter, float beta, float beta_red, int ng, float alpha,
                        float alpha_red, float r_max, float epsilon, float delta, float tv_eps, double* hist, int* n_done,
                        void* cuda_stream) {
    if (n_done) *n_done = 0;
    if (!P || !b || !x || n_iter < 0 || ng < 0 || !(tv_eps >= 0.f)) return TIGRE_ERR_ARG;
    if (mem_kind(b) != MEM_DEVICE || mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = P->t.g;
    const size_t per = (size_t)g.nu * g.nv, nvox = (size_t)g.nx * g.ny * g.nz;
    TempBuf x0, xp, acc, tvacc;
    TG_TRY(x0.alloc(sizeof(float) * nvox, st));
    TG_TRY(xp.alloc(sizeof(float) * nvox, st));
    TG_TRY(acc.alloc(sizeof(double) * 4, st));
    TG_TRY(tvacc.alloc(sizeof(double) * std::max(ng, 1), st));
    double* d = acc.as<double>();
    float* G = P->grad.as<float>();
    double dtvg = 0.0;
    for (int it = 0; it < n_iter; ++it) {
        TG_CUDA(cudaMemcpyAsync(x0.p, x, sizeof(float) * nvox, cudaMemcpyDeviceToDevice, st));
        // ---- data step
        for (int s = 0; s < P->nSubsets; ++s) {
            const int n = P->off[s + 1] - P->off[s];
            float* A = P->Axb.as<float>();
            float* Vs = nullptr;
            TG_TRY(P->col_weights(s, &Vs, st));
            TG_TRY(launch_ax(x, g, P->ray[s].as<RayView>(), n, P->ax_mode, false, false, A, nullptr, st, nullptr, nullptr, P->hray[s].data()));
            TG_TRY(launch_residual(b, P->d_idx.as<int32_t>() + P->off[s], A, P->W.as<float>() + per * P->off[s], A, per, n, nullptr, st));
            TG_TRY(launch_atb(A, g, P->vox[s].as<VoxView>(), n, P->atb_mode, false, G, 0, g.nz, false, 0, g.nv, P->clamp, st,
                              P->hvox[s].data()));
            TG_TRY(launch_update(x, G, Vs, beta, 1, nvox, st));
        }
        beta *= beta_red;
        // ---- dd = ||A x - b||, dp = ||x - x0||
        TG_CUDA(cudaMemsetAsync(d + 3, 0, sizeof(double), st));
        for (int s = 0; s < P->nSubsets; ++s) {
            const int n = P->off[s + 1] - P->off[s];
            float* A = P->Axb.as<float>();
            TG_TRY(launch_ax(x, g, P->ray[s].as<RayView>(), n, P->ax_mode, false, false, A, nullptr, st, nullptr, nullptr, P->hray[s].data()));
            TG_TRY(launch_residual(b, P->d_idx.as<int32_t>() + P->off[s], A, nullptr, A, per, n, d + 3, st));
        }
        TG_TRY(launch_diff_stats(x, x0.as<float>(), x0.as<float>(), nvox, d, st));
        double h[4];
        TG_CUDA(cudaMemcpyAsync(h, d, sizeof h, cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        const double dd = std::sqrt(h[3]), dp = std::sqrt(h[0]);
        if (it == 0) dtvg = (double)alpha * dp;
        TG_CUDA(cudaMemcpyAsync(xp.p, x, sizeof(float) * nvox, cudaMemcpyDeviceToDevice, st));
        // ---- regulariser step
        const double used = dtvg;
        if (ng > 0) TG_CUDA(cudaMemsetAsync(tvacc.p, 0, sizeof(double) * ng, st));
        for (int k = 0; k < ng; ++k) {
            TG_TRY(launch_tv_gradient(x, g.nx, g.ny, g.nz, delta, tv_eps, G, nullptr, tvacc.as<double>() + k, st));
            TG_TRY(launch_tv_step(x, G, (float)dtvg, tvacc.as<double>() + k, nvox, st));
        }
        TG_TRY(launch_diff_stats(x, xp.as<float>(), x0.as<float>(), nvox, d, st));
        TG_CUDA(cudaMemcpyAsync(h, d, 3 * sizeof(double), cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        const double dg = std::sqrt(h[0]);
        if (dg > (double)r_max * dp && dd > (double)epsilon) dtvg *= (double)alpha_red;
        const double c = (dg > 0.0 && dp > 0.0) ? h[1] / (dg * dp) : 0.0;
        if (hist) hist[5 * it] = dd, hist[5 * it + 1] = dp, hist[5 * it + 2] = dg, hist[5 * it + 3] = used, hist[5 * it + 4] = c;
        if (n_done) *n_done = it + 1;
        if ((c < -0.99 && dd <= (double)epsilon) || beta < 0.005f) break;
    }
    return TIGRE_OK;
}

// ---------------------------------------------------------------- CGLS (textbook recurrences, O-F)
int tigre_cgls(const float* b, const tigre_geo* geo, const double* angles, int nA, int n_iter, int ax_mode,
               int atb_mode, float* x, double* resid_hist, void* cuda_stream) {
    if (!b || !x || n_iter < 0) return TIGRE_ERR_ARG;
    if (ax_mode != TIGRE_AX_SIDDON && ax_mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    if (atb_mode < TIGRE_ATB_MATCHED || atb_mode > TIGRE_ATB_EXACT_INTERP) return TIGRE_ERR_ARG;
    const bool exact = atb_mode >= TIGRE_ATB_EXACT_SIDDON;
    if (exact && atb_mode - TIGRE_ATB_EXACT_SIDDON != ax_mode) return TIGRE_ERR_ARG;   // the transpose of THIS Ax
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(b) != MEM_DEVICE || mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = t.g;
    const size_t np = (size_t)nA * g.nu * g.nv, nvox = (size_t)g.nx * g.ny * g.nz;
    TempBuf r, q, s, p, sc;
    TG_TRY(r.alloc(sizeof(float) * np, st));
    TG_TRY(q.alloc(sizeof(float) * np, st));
    TG_TRY(s.alloc(sizeof(float) * nvox, st));
    TG_TRY(p.alloc(sizeof(float) * nvox, st));
    // device scalars: [0]=gamma [1]=gamma_new [2]=||q||^2 [3+it]=||r||^2 history
    TG_TRY(sc.alloc(sizeof(double) * (3 + std::max(n_iter, 1)), st));
    double* d = sc.as<double>();
    TG_TRY(t.build_ray(nullptr, nA, st));
    if (!exact) TG_TRY(t.build_vox(nullptr, nA, st));
    const RayView* rv = t.ray.as<RayView>();
    const VoxView* vv = t.vox.as<VoxView>();
    auto AT = [&](const float* y, float* out) -> int {
        if (exact) return launch_ax_adjoint(y, g, rv, nA, ax_mode, out, st);
        return launch_atb(y, g, vv, nA, atb_mode, false, out, 0, g.nz, false, 0, g.nv, t.clamp, st, t.hvox.data());
    };
    TG_CUDA(cudaMemsetAsync(x, 0, sizeof(float) * nvox, st));
    TG_CUDA(cudaMemcpyAsync(r.p, b, sizeof(float) * np, cudaMemcpyDeviceToDevice, st));              // r = b - A 0
    TG_TRY(AT(r.as<float>(), s.as<float>()));
    TG_CUDA(cudaMemcpyAsync(p.p, s.p, sizeof(float) * nvox, cudaMemcpyDeviceToDevice, st));          // p = s
    TG_TRY(launch_dot(s.as<float>(), s.as<float>(), nvox, d + 0, st));                               // gamma
    for (int it = 0; it < n_iter; ++it) {
        TG_TRY(launch_ax(p.as<float>(), g, rv, nA, ax_mode, false, false, q.as<float>(), nullptr, st, nullptr, nullptr, t.hray.data()));   // q = A p
        TG_TRY(launch_dot(q.as<float>(), q.as<float>(), np, d + 2, st));
        TG_TRY(launch_axpy(x, p.as<float>(), d + 0, d + 2, 1.f, nvox, st));                          // x += alpha p
        TG_TRY(launch_axpy(r.as<float>(), q.as<float>(), d + 0, d + 2, -1.f, np, st));               // r -= alpha q
        TG_TRY(AT(r.as<float>(), s.as<float>()));
        TG_TRY(launch_dot(s.as<float>(), s.as<float>(), nvox, d + 1, st));                           // gamma'
        TG_TRY(launch_xpby(p.as<float>(), s.as<float>(), d + 1, d + 0, nvox, st));                   // p = s + beta p
        TG_CUDA(cudaMemcpyAsync(d + 0, d + 1, sizeof(double), cudaMemcpyDeviceToDevice, st));        // gamma = gamma'
        TG_TRY(launch_dot(r.as<float>(), r.as<float>(), np, d + 3 + it, st));
    }
    if (resid_hist && n_iter > 0) {
        std::vector<double> h(n_iter);
        TG_CUDA(cudaMemcpyAsync(h.data(), d + 3, sizeof(double) * n_iter, cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        for (int it = 0; it < n_iter; ++it) resid_hist[it] = std::sqrt(h[it]);
    }
    return TIGRE_OK;
}

// ---------------------------------------------------------------- gradient descent, eq. (4) (reading P32)
int tigre_gradient_descent(const float* b, const tigre_geo* geo, const double* angles, int nA, int n_iter, float lambda, int ax_mode,
                           int atb_mode, float* x, double* resid_hist, void* cuda_stream) {
    if (!b || !x || n_iter < 0) return TIGRE_ERR_ARG;
    if (ax_mode != TIGRE_AX_SIDDON && ax_mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    if (atb_mode < TIGRE_ATB_MATCHED || atb_mode > TIGRE_ATB_EXACT_INTERP) return TIGRE_ERR_ARG;
    const bool exact = atb_mode >= TIGRE_ATB_EXACT_SIDDON;
    if (exact && atb_mode - TIGRE_ATB_EXACT_SIDDON != ax_mode) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(b) != MEM_DEVICE || mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = t.g;
    const size_t np = (size_t)nA * g.nu * g.nv, nvox = (size_t)g.nx * g.ny * g.nz;
    TempBuf r, grad, sc;
    TG_TRY(r.alloc(sizeof(float) * np, st));
    TG_TRY(grad.alloc(sizeof(float) * nvox, st));
    TG_TRY(sc.alloc(sizeof(double) * std::max(n_iter, 1), st));
    TG_CUDA(cudaMemsetAsync(sc.p, 0, sizeof(double) * std::max(n_iter, 1), st));
    TG_TRY(t.build_ray(nullptr, nA, st));
    if (!exact) TG_TRY(t.build_vox(nullptr, nA, st));
    for (int it = 0; it < n_iter; ++it) {
        TG_TRY(launch_ax(x, g, t.ray.as<RayView>(), nA, ax_mode, false, false, r.as<float>(), nullptr, st, nullptr, nullptr, t.hray.data()));
        TG_TRY(launch_residual(b, nullptr, r.as<float>(), nullptr, r.as<float>(), (size_t)g.nu * g.nv, nA, sc.as<double>() + it, st));
        if (exact) TG_TRY(launch_ax_adjoint(r.as<float>(), g, t.ray.as<RayView>(), nA, ax_mode, grad.as<float>(), st));
        else TG_TRY(launch_atb(r.as<float>(), g, t.vox.as<VoxView>(), nA, atb_mode, false, grad.as<float>(), 0, g.nz, false, 0, g.nv, t.clamp, st,
                               t.hvox.data()));
        TG_TRY(launch_update(x, grad.as<float>(), nullptr, lambda, 0, nvox, st));
    }
    if (resid_hist && n_iter > 0) {
        std::vector<double> h(n_iter);
        TG_CUDA(cudaMemcpyAsync(h.data(), sc.p, sizeof(double) * n_iter, cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        for (int it = 0; it < n_iter; ++it) resid_hist[it] = std::sqrt(h[it]);
    }
    return TIGRE_OK;
}

// ---------------------------------------------------------------- FDK (O-D)
static int fdk_filter_impl(const float* b, Tables& t, int nA, float* q, cudaStream_t st) {
    std::vector<double> dd(4 * (size_t)nA);   // DSD, DSO, offDetector (u, v) per view
    for (int a = 0; a < nA; ++a)
        dd[a] = t.views[a].DSD, dd[nA + a] = t.views[a].DSO, dd[2 * nA + 2 * a] = t.views[a].offD[0], dd[2 * nA + 2 * a + 1] = t.views[a].offD[1];
    // parallel beam (P29): no magnification (tau = du) and no cosine weight: the kernels' DSO/DSD = 1, DSD/sqrt(DSD^2 + u^2 + v^2) = 1
    if (t.views[0].parallel) std::fill(dd.begin(), dd.begin() + 2 * nA, 1e15);
    {
        // tensor-core filter (fdk_tc.cu) where the problem qualifies
        std::vector<double> taps;
        fdk_filter_taps(t.g.nu, TIGRE_FILTER_RAM_LAK, taps);
        const std::vector<float> ft(taps.begin(), taps.end());
        const std::vector<double> dsd(dd.begin(), dd.begin() + nA), dso(dd.begin() + nA, dd.begin() + 2 * nA), offd(dd.begin() + 2 * nA, dd.end());
        const int rc = launch_fdk_filter_tc(b, t.g, dsd, dso, offd, nA, ft, nullptr, q, st);
        if (rc <= 0) return rc;
    }
    TempBuf tb;
    TG_TRY(upload(tb, dd.data(), sizeof(double) * dd.size(), st));
    // Ram-Lak, no weights: taps formed in the kernel, odd taps only (fdk.cu)
    return launch_fdk_filter_taps(b, t.g, tb.as<double>(), tb.as<double>() + nA, tb.as<double>() + 2 * nA, nA, nullptr, nullptr, q, st, true);
}
int tigre_fdk_filter(const float* b, const tigre_geo* geo, const double* angles, int nA, float* q, void* cuda_stream) {
    if (!b || !q) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(b) != MEM_DEVICE || mem_kind(q) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    return fdk_filter_impl(b, t, nA, q, (cudaStream_t)cuda_stream);
}
int tigre_fdk(const float* b, const tigre_geo* geo, const double* angles, int nA, float* x, void* cuda_stream) {
    if (!b || !x) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(b) != MEM_DEVICE || mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = t.g;
    TempBuf q;
    TG_TRY(q.alloc(sizeof(float) * (size_t)nA * g.nu * g.nv, st));
    TG_TRY(fdk_filter_impl(b, t, nA, q.as<float>(), st));
    TG_TRY(device_atb(q.as<float>(), t, nullptr, nA, TIGRE_ATB_FDK, false, x, st));
    return launch_scale(x, (float)(M_PI / (double)nA), (size_t)g.nx * g.ny * g.nz, st);
}

// ---------------------------------------------------------------- FDK variants (fdk.cu; P26-P28)
static int fdk_filter_ex_impl(const float* b, Tables& t, int nA, int filter, int weighting, float* q, cudaStream_t st) {
    if (filter < TIGRE_FILTER_RAM_LAK || filter > TIGRE_FILTER_HANN) return TIGRE_ERR_ARG;
    if (weighting < TIGRE_FDK_FULL || weighting > TIGRE_FDK_WANG) return TIGRE_ERR_ARG;
    if (weighting != TIGRE_FDK_FULL && t.views[0].parallel) return TIGRE_ERR_ARG;   // cone-beam redundancy weights
    if (filter == TIGRE_FILTER_RAM_LAK && weighting == TIGRE_FDK_FULL) return fdk_filter_impl(b, t, nA, q, st);
    const int nu = t.g.nu;
    std::vector<double> dd(4 * (size_t)nA), taps, w;   // DSD, DSO, offDetector (u, v) per view
    for (int a = 0; a < nA; ++a)
        dd[a] = t.views[a].DSD, dd[nA + a] = t.views[a].DSO, dd[2 * nA + 2 * a] = t.views[a].offD[0], dd[2 * nA + 2 * a + 1] = t.views[a].offD[1];
    // parallel beam (P29): no magnification (tau = du) and no cosine weight: the kernels' DSO/DSD = 1, DSD/sqrt(DSD^2 + u^2 + v^2) = 1
    if (t.views[0].parallel) std::fill(dd.begin(), dd.begin() + 2 * nA, 1e15);
    fdk_filter_taps(nu, filter, taps);
    std::vector<float> ft(taps.begin(), taps.end()), fw;
    TempBuf tb, tt, tw;
    TG_TRY(upload(tb, dd.data(), sizeof(double) * dd.size(), st));
    TG_TRY(upload(tt, ft.data(), sizeof(float) * ft.size(), st));
    if (weighting != TIGRE_FDK_FULL) {
        TG_TRY(fdk_weights(t.g, t.views, weighting, w));
        fw.resize(w.size());
        const double k = weighting == TIGRE_FDK_WANG ? 2.0 : 1.0;
        for (size_t i = 0; i < w.size(); ++i) fw[i] = (float)(k * w[i]);
        TG_TRY(upload(tw, fw.data(), sizeof(float) * fw.size(), st));
    }
    {
        const std::vector<double> dsd(dd.begin(), dd.begin() + nA), dso(dd.begin() + nA, dd.begin() + 2 * nA), offd(dd.begin() + 2 * nA, dd.end());
        const int rc = launch_fdk_filter_tc(b, t.g, dsd, dso, offd, nA, ft, weighting != TIGRE_FDK_FULL ? tw.as<float>() : nullptr, q, st);
        if (rc <= 0) return rc;
    }
    return launch_fdk_filter_taps(b, t.g, tb.as<double>(), tb.as<double>() + nA, tb.as<double>() + 2 * nA, nA, tt.as<float>(),
                                  weighting != TIGRE_FDK_FULL ? tw.as<float>() : nullptr, q, st, filter == TIGRE_FILTER_RAM_LAK);
}
int tigre_fdk_filter_ex(const float* b, const tigre_geo* geo, const double* angles, int nA, int filter, int weighting, float* q,
                        void* cuda_stream) {
    if (!b || !q) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(b) != MEM_DEVICE || mem_kind(q) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    return fdk_filter_ex_impl(b, t, nA, filter, weighting, q, (cudaStream_t)cuda_stream);
}
int tigre_fdk_ex(const float* b, const tigre_geo* geo, const double* angles, int nA, int filter, int weighting, float* x,
                 void* cuda_stream) {
    if (!b || !x) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(b) != MEM_DEVICE || mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = t.g;
    TempBuf q;
    TG_TRY(q.alloc(sizeof(float) * (size_t)nA * g.nu * g.nv, st));
    TG_TRY(fdk_filter_ex_impl(b, t, nA, filter, weighting, q.as<float>(), st));
    TG_TRY(device_atb(q.as<float>(), t, nullptr, nA, TIGRE_ATB_FDK, false, x, st));
    double scale = M_PI / (double)nA;
    if (weighting == TIGRE_FDK_PARKER) scale = std::fabs(t.views[nA - 1].ang[0] - t.views[0].ang[0]) / (double)(nA - 1);
    return launch_scale(x, (float)scale, (size_t)g.nx * g.ny * g.nz, st);
}
int tigre_flatten_detector(const float* curved, const tigre_geo* geo, const double* angles, int nA, float* flat, void* cuda_stream) {
    if (!curved || !flat || curved == flat) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(curved) != MEM_DEVICE || mem_kind(flat) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    std::vector<double> dd(nA);
    for (int a = 0; a < nA; ++a) dd[a] = t.views[a].DSD;
    TempBuf tb;
    TG_TRY(upload(tb, dd.data(), sizeof(double) * dd.size(), st));
    return launch_flatten(curved, t.g, tb.as<double>(), nA, flat, st);
}
int tigre_fdk_weights(const tigre_geo* geo, const double* angles, int nA, int weighting, double* w) {
    if (!w) return TIGRE_ERR_ARG;
    TG_TRY(validate_geo(geo, angles, nA));      // host arithmetic only: no device needed
    Grid g = make_grid(geo);
    std::vector<ViewH> views;
    resolve_views(geo, angles, nA, views);
    std::vector<double> v;
    TG_TRY(fdk_weights(g, views, weighting, v));
    std::copy(v.begin(), v.end(), w);
    return TIGRE_OK;
}

// ---------------------------------------------------------------- TV / AwTV (tv.cu)
int tigre_awtv_gradient(const float* x, int nx, int ny, int nz, float delta, float eps, float* g, double* value,
                        double* grad_norm2, void* cuda_stream) {
    if (!x || nx <= 0 || ny <= 0 || nz <= 0 || !(eps >= 0.f)) return TIGRE_ERR_ARG;
    TG_TRY(ensure_device());
    if (mem_kind(x) != MEM_DEVICE || (g && mem_kind(g) != MEM_DEVICE)) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    TempBuf acc;
    const bool scal = value || grad_norm2;
    if (scal) {
        TG_TRY(acc.alloc(2 * sizeof(double), st));
        TG_CUDA(cudaMemsetAsync(acc.p, 0, 2 * sizeof(double), st));
    }
    double* d = acc.as<double>();
    TG_TRY(launch_tv_gradient(x, nx, ny, nz, delta, eps, g, value ? d : nullptr, (grad_norm2 && g) ? d + 1 : nullptr, st));
    if (scal) {
        double h[2] = {0, 0};
        TG_CUDA(cudaMemcpyAsync(h, d, sizeof h, cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        if (value) *value = h[0];
        if (grad_norm2) *grad_norm2 = h[1];
    }
    return TIGRE_OK;
}

int tigre_awtv(const float* x, int nx, int ny, int nz, float delta, float eps, double* value, void* cuda_stream) {
    if (!value) return TIGRE_ERR_ARG;
    return tigre_awtv_gradient(x, nx, ny, nz, delta, eps, nullptr, value, nullptr, cuda_stream);
}

int tigre_minimize_awtv(float* x, int nx, int ny, int nz, float delta, float eps, float alpha, int n_steps, void* cuda_stream) {
    if (!x || nx <= 0 || ny <= 0 || nz <= 0 || n_steps < 0 || !(eps >= 0.f)) return TIGRE_ERR_ARG;
    TG_TRY(ensure_device());
    if (mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)nx * ny * nz;
    TempBuf g, acc;
    TG_TRY(g.alloc(n * sizeof(float), st));
    TG_TRY(acc.alloc(sizeof(double) * std::max(n_steps, 1), st));
    TG_CUDA(cudaMemsetAsync(acc.p, 0, sizeof(double) * std::max(n_steps, 1), st));
    for (int it = 0; it < n_steps; ++it) {
        TG_TRY(launch_tv_gradient(x, nx, ny, nz, delta, eps, g.as<float>(), nullptr, acc.as<double>() + it, st));
        TG_TRY(launch_tv_step(x, g.as<float>(), alpha, acc.as<double>() + it, n, st));
    }
    return TIGRE_OK;
}

// ---------------------------------------------------------------- TV proximal operator and FISTA (prox.cu; P24, P25)
static int tv_prox_impl(const float* f, int nx, int ny, int nz, float lam, int n_iter, float tau, float* u, float* p3, float* d,
                        cudaStream_t st) {
    const size_t n = (size_t)nx * ny * nz;
    if (!(lam > 0.f)) {
        if (u != f) TG_CUDA(cudaMemcpyAsync(u, f, sizeof(float) * n, cudaMemcpyDeviceToDevice, st));
        return TIGRE_OK;
    }
    float *px = p3, *py = p3 + n, *pz = p3 + 2 * n;
    TG_CUDA(cudaMemsetAsync(p3, 0, sizeof(float) * 3 * n, st));
    for (int it = 0; it < n_iter; ++it) {
        TG_TRY(launch_prox_div(px, py, pz, f, lam, false, d, nx, ny, nz, st));
        TG_TRY(launch_prox_update(px, py, pz, d, tau, nx, ny, nz, st));
    }
    return launch_prox_div(px, py, pz, f, lam, true, u, nx, ny, nz, st);
}

// SART-TV (reading P31; oracle/pocs.py sart_tv): per iteration the plan's OS-SART sweep with relaxation lambda, then the TV prox
int tigre_plan_sart_tv(tigre_plan* P, const float* b, float* x, int n_iter, float lambda, float lambda_red, float tv_lambda,
                       int tv_iter, float tau, double* resid_hist, void* cuda_stream) {
    if (!P || !b || !x || n_iter < 0 || tv_iter < 0 || !(tv_lambda >= 0.f) || !(tau > 0.f)) return TIGRE_ERR_ARG;
    if (mem_kind(b) != MEM_DEVICE || mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = P->t.g;
    const size_t nvox = (size_t)g.nx * g.ny * g.nz;
    TempBuf p3, dd;
    TG_TRY(p3.alloc(sizeof(float) * 3 * nvox, st));
    TG_TRY(dd.alloc(sizeof(float) * nvox, st));
    for (int it = 0; it < n_iter; ++it) {
        TG_TRY(tigre_plan_ossart(P, b, x, 1, lambda, 1, resid_hist ? resid_hist + it : nullptr, cuda_stream));
        TG_TRY(tv_prox_impl(x, g.nx, g.ny, g.nz, tv_lambda, tv_iter, tau, x, p3.as<float>(), dd.as<float>(), st));
        lambda *= lambda_red;
    }
    return TIGRE_OK;
}

int tigre_tv_prox(const float* f, int nx, int ny, int nz, float lambda, int n_iter, float tau, float* u, void* cuda_stream) {
    if (!f || !u || nx <= 0 || ny <= 0 || nz <= 0 || n_iter < 0 || !(lambda >= 0.f) || !(tau > 0.f)) return TIGRE_ERR_ARG;
    TG_TRY(ensure_device());
    if (mem_kind(f) != MEM_DEVICE || mem_kind(u) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const size_t n = (size_t)nx * ny * nz;
    TempBuf p3, d;
    // 16-byte aligned component arrays need n % 4 == 0; otherwise the launchers take the scalar kernels
    TG_TRY(p3.alloc(sizeof(float) * 3 * n, st));
    TG_TRY(d.alloc(sizeof(float) * n, st));
    return tv_prox_impl(f, nx, ny, nz, lambda, n_iter, tau, u, p3.as<float>(), d.as<float>(), st);
}

int tigre_fista(const float* b, const tigre_geo* geo, const double* angles, int nA, int n_iter, float L, float tv_lambda,
                int tv_iter, float tau, int ax_mode, int atb_mode, float* x, double* resid_hist, void* cuda_stream) {
    if (!b || !x || n_iter < 0 || tv_iter < 0 || !(L > 0.f) || !(tv_lambda >= 0.f) || !(tau > 0.f)) return TIGRE_ERR_ARG;
    if (ax_mode != TIGRE_AX_SIDDON && ax_mode != TIGRE_AX_INTERP) return TIGRE_ERR_ARG;
    if (atb_mode < TIGRE_ATB_MATCHED || atb_mode > TIGRE_ATB_EXACT_INTERP) return TIGRE_ERR_ARG;
    const bool exact = atb_mode >= TIGRE_ATB_EXACT_SIDDON;
    if (exact && atb_mode - TIGRE_ATB_EXACT_SIDDON != ax_mode) return TIGRE_ERR_ARG;
    Tables t;
    TG_TRY(prep(geo, angles, nA, t));
    if (mem_kind(b) != MEM_DEVICE || mem_kind(x) != MEM_DEVICE) return TIGRE_ERR_MEMSPACE;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const Grid& g = t.g;
    const size_t np = (size_t)nA * g.nu * g.nv, nvox = (size_t)g.nx * g.ny * g.nz;
    TempBuf r, y, grad, xn, p3, dd, sc;
    TG_TRY(r.alloc(sizeof(float) * np, st));
    TG_TRY(y.alloc(sizeof(float) * nvox, st));
    TG_TRY(grad.alloc(sizeof(float) * nvox, st));
    TG_TRY(xn.alloc(sizeof(float) * nvox, st));
    TG_TRY(p3.alloc(sizeof(float) * 3 * nvox, st));
    TG_TRY(dd.alloc(sizeof(float) * nvox, st));
    TG_TRY(sc.alloc(sizeof(double) * std::max(n_iter, 1), st));
    TG_CUDA(cudaMemsetAsync(sc.p, 0, sizeof(double) * std::max(n_iter, 1), st));
    TG_TRY(t.build_ray(nullptr, nA, st));
    if (!exact) TG_TRY(t.build_vox(nullptr, nA, st));
    const RayView* rv = t.ray.as<RayView>();
    const VoxView* vv = t.vox.as<VoxView>();
    TG_CUDA(cudaMemcpyAsync(y.p, x, sizeof(float) * nvox, cudaMemcpyDeviceToDevice, st));            // y_0 = x_0
    double tk = 1.0;
    for (int it = 0; it < n_iter; ++it) {
        TG_TRY(launch_ax(y.as<float>(), g, rv, nA, ax_mode, false, false, r.as<float>(), nullptr, st, nullptr, nullptr, t.hray.data()));
        TG_TRY(launch_residual(b, nullptr, r.as<float>(), nullptr, r.as<float>(), (size_t)g.nu * g.nv, nA, sc.as<double>() + it, st));
        if (exact) TG_TRY(launch_ax_adjoint(r.as<float>(), g, rv, nA, ax_mode, grad.as<float>(), st));
        else TG_TRY(launch_atb(r.as<float>(), g, vv, nA, atb_mode, false, grad.as<float>(), 0, g.nz, false, 0, g.nv, t.clamp, st, t.hvox.data()));
        TG_TRY(launch_update(y.as<float>(), grad.as<float>(), nullptr, 2.0f / L, 0, nvox, st));      // y + (2/L) A^T (b - A y)
        TG_TRY(tv_prox_impl(y.as<float>(), g.nx, g.ny, g.nz, tv_lambda, tv_iter, tau, xn.as<float>(), p3.as<float>(), dd.as<float>(), st));
        const double tn = 0.5 * (1.0 + std::sqrt(1.0 + 4.0 * tk * tk));
        TG_TRY(launch_momentum(y.as<float>(), x, xn.as<float>(), (float)((tk - 1.0) / tn), nvox, st));
        tk = tn;
    }
    if (resid_hist && n_iter > 0) {
        std::vector<double> h(n_iter);
        TG_CUDA(cudaMemcpyAsync(h.data(), sc.p, sizeof(double) * n_iter, cudaMemcpyDeviceToHost, st));
        TG_CUDA(cudaStreamSynchronize(st));
        for (int it = 0; it < n_iter; ++it) resid_hist[it] = std::sqrt(h[it]);
    }
    return TIGRE_OK;
}

// Upper bounds (256-byte granules and a megabyte of small tables / scalars included) on the temporaries of one call on
// device-resident data.  OSSART = tigre_ossart / tigre_plan_* with ONE subset (SIRT): tigre_plan_workspace_bytes is the general form.
size_t tigre_workspace_bytes(const tigre_geo* geo, int nA, int op) {
    if (!geo || nA <= 0) return 0;
    const size_t per = (size_t)geo->nDetector[0] * geo->nDetector[1] * sizeof(float);
    const size_t vol = (size_t)geo->nVoxel[0] * geo->nVoxel[1] * geo->nVoxel[2] * sizeof(float);
    const size_t tab = (size_t)nA * (sizeof(RayView) + sizeof(VoxView) + 4 * sizeof(double)) + ((size_t)1 << 20);
    switch (op) {
        case TIGRE_OP_AX: return tab + vol;                       // the (x,y)-transposed copy of the volume
        case TIGRE_OP_ATB: return tab + vol;                      // exact modes: the transposed scratch volume
        case TIGRE_OP_OSSART: return tigre_plan_workspace_bytes(geo, nA, 1, nA, 0);
        case TIGRE_OP_CGLS: return tab + per * nA * 2 + vol * 3;  // r, q; s, p; transposed copy / scratch
        case TIGRE_OP_FDK: return tab + per * nA + (size_t)geo->nDetector[0] * (nA + 1) * sizeof(float);
    }
    return 0;
}

size_t tigre_plan_workspace_bytes(const tigre_geo* geo, int nA, int nSubsets, int max_subset_views, int host_data) {
    if (!geo || nA <= 0 || nSubsets <= 0 || max_subset_views <= 0) return 0;
    const size_t per = (size_t)geo->nDetector[0] * geo->nDetector[1] * sizeof(float);
    const size_t vol = (size_t)geo->nVoxel[0] * geo->nVoxel[1] * geo->nVoxel[2] * sizeof(float);
    const size_t tab = (size_t)nA * (sizeof(RayView) + sizeof(VoxView) + sizeof(int32_t) + sizeof(float) * geo->nDetector[0]) +
                       (size_t)nSubsets * 1024 + ((size_t)1 << 20);
    // plan: W (all views), V (one volume per subset), one subset's Ax / residual, A^T r; iteration: transposed iterate;
    // pinned-host data (end-to-end path): device copies of b and x
    size_t n = tab + per * nA + vol * nSubsets + per * max_subset_views + vol + vol;
    if (host_data) n += per * nA + vol;
    return n;
}

}  // extern "C"
