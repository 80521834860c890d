// common.cuh — shared declarations of libtigre_b200 (CUDA path only; nothing here is used by,
// or taken from, oracle/).  Geometry follows PAPER.md:543-566 (App. B Table B1) and §2.4
// (lines 179-197) under the readings P1-P6 listed in DESIGN.md.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include <stddef.h>
#include <vector>
#include "../../include/tigre_b200.h"

namespace tg {

// ---------------------------------------------------------------- errors
void set_cuda_error(cudaError_t e, const char* file, int line);
#define TG_CUDA(expr)                                                     \
    do {                                                                  \
        cudaError_t _e = (expr);                                          \
        if (_e != cudaSuccess) {                                          \
            tg::set_cuda_error(_e, __FILE__, __LINE__);                   \
            return (_e == cudaErrorMemoryAllocation) ? TIGRE_ERR_WORKSPACE : TIGRE_ERR_CUDA; \
        }                                                                 \
    } while (0)
#define TG_TRY(expr)                 \
    do {                             \
        int _s = (expr);             \
        if (_s != TIGRE_OK) return _s; \
    } while (0)

// ---------------------------------------------------------------- host geometry (fp64)
struct ViewH {  // one projection's resolved parameters (everything but sizes per view)
    double DSD, DSO, COR;
    double offO[3], offD[2], rotD[3], ang[3];
    int parallel;   // tigre_geo.mode == TIGRE_GEO_PARALLEL (reading P29)
};

// Ray-driven per-view table, in VOXEL-INDEX coordinates xi = (X - volume_min)/dVoxel, so voxel
// (ix,iy,iz) is the cube [ix,ix+1) x [iy,iy+1) x [iz,iz+1).  fp64: per-ray set-up is done in
// double on the device (about 1/600 of the work of a ray).
struct RayView {
    double S[3];    // source
    double P0[3];   // centre of pixel (0,0)
    double dU[3];   // step per pixel along u
    double dV[3];   // step per pixel along v
    double dSU[3];  // step of the ray's START per pixel along u / v: zero for cone beam (all rays start at S),
    double dSV[3];  // = dU / dV for parallel beam (S is then the start of pixel (0,0)'s ray)
};

// Voxel-driven per-view table (fp32, built in fp64).  With c = centred voxel index
// (ix-(nx-1)/2, iy-(ny-1)/2, iz-(nz-1)/2):
//   W  = rowW.c + rowW[3]   (normalised detector-normal depth, t = 1/W is the magnification)
//   fu - nu/2 = (rowU.c + rowU[3]) / W ,  fv - nv/2 likewise   (integer shifts: floor() commutes)
//   G  = rowG.c + rowG[3]   = (DSO - X'_x)/DSO   (FDK distance weight = 1/G^2)
//   matched weight = km * t^2 * sqrt(sx2 + du^2*(fuh-fus)^2 + dv^2*(fvh-fvs)^2), fuh = fu - nu/2
struct alignas(16) VoxView {
    float rowU[4], rowV[4], rowW[4], rowG[4];
    float km, sx2, fus, fvs;
};

struct Grid {
    int nx, ny, nz, nu, nv;
    double dx, dy, dz, du, dv, accuracy;
};

int validate_geo(const tigre_geo* geo, const double* angles, int nA);
Grid make_grid(const tigre_geo* geo);
void resolve_views(const tigre_geo* geo, const double* angles, int nA, std::vector<ViewH>& out);
void build_ray_view(const Grid& g, const ViewH& v, RayView& r);
// returns TIGRE_ERR_GEOMETRY if a corner of the (z-restricted) volume is at/behind the source
int build_vox_view(const Grid& g, const ViewH& v, VoxView& o);
// detector rows the z-slices [z0,z0+nzs) can reach in view v (with the interpolation support and slack)
void row_band(const Grid& g, const ViewH& v, int z0, int nzs, int& row0, int& nrows);

// ---------------------------------------------------------------- stream-ordered temporaries
struct TempBuf {  // RAII: a block of the caller's workspace (tigre_set_workspace) if one is set, else cudaMallocAsync / cudaFreeAsync on one stream
    void* p = nullptr;
    cudaStream_t s = nullptr;
    bool ws = false;
    TempBuf() {}
    TempBuf(const TempBuf&) = delete;
    TempBuf& operator=(const TempBuf&) = delete;
    ~TempBuf() { release(); }
    int alloc(size_t bytes, cudaStream_t st);
    void release();
    template <class T> T* as() { return reinterpret_cast<T*>(p); }
};
// copy a small host table to a fresh device buffer on the stream (host data is staged before return)
int upload(TempBuf& buf, const void* host, size_t bytes, cudaStream_t st);

// ---------------------------------------------------------------- in-library timing (bench.py's roofline leg)
// When enabled with tigre_profile(1) every launcher brackets its kernels with CUDA events on the
// launching stream; tigre_profile_read() sums the elapsed times per kind.  Launch counts are kept always.
enum ProfKind { PK_AX = 0, PK_ATB = 1, PK_EW = 2, PK_N = 3 };
struct ProfScope {
    int kind;
    cudaStream_t st;
    void* rec;
    ProfScope(int kind, cudaStream_t st, int launches = 1);
    ~ProfScope();
};

// ---------------------------------------------------------------- kernel launchers (device pointers)
// forward projection of nViews views given their RayView table (device), out contiguous [nViews][nv][nu]
//   unit_vol: treat the volume as all ones (row sums A 1), vol may be NULL
//   count_out: if non-NULL, write per-ray sample counts instead of projecting (measurement helper)
//   accumulate: proj += instead of proj = (partial projections of a z-slab, chunked path)
//   sub (chunked path): compute detector rows [row0,row0+nrows) only; interpolated mode: `vol` holds the
//   z-slices [zs0,zs0+nzs) of a volume of height g.nz and points at slice zs0 (other slices count as 0)
struct AxSub {
    int row0, nrows, zs0, nzs;
};
//   h_views: host copy of the same table; when given (and the problem qualifies) the interpolated mode runs the kernel of
//   ax_tma.cu (boxes of the volume staged into shared memory by TMA), otherwise the L1 gather kernel of ax.cu
int launch_ax(const float* vol, const Grid& g, const RayView* d_views, int nViews, int mode, bool unit_vol,
              bool accumulate, float* proj, uint32_t* count_out, cudaStream_t st, const AxSub* sub = nullptr,
              const float* volT_in = nullptr,    // volT_in: an up-to-date (x,y)-transposed copy of vol, if the caller has one
              const RayView* h_views = nullptr);
int launch_transpose_xy(const float* vol, float* volT, const Grid& g, cudaStream_t st);
// Siddon march without the volume: counts[ray] = voxels met with a non-zero length, track[2 ray], [2 ray + 1] = first / last of them
int launch_ax_track(const Grid& g, const RayView* d_views, int nViews, uint32_t* counts, long long* track, cudaStream_t st);
void set_index_path(int path);
// exact adjoint of launch_ax (ray-driven scatter of the same weights); vol [nz][ny][nx] is overwritten
int launch_ax_adjoint(const float* proj, const Grid& g, const RayView* d_views, int nViews, int mode, float* vol,
                      cudaStream_t st);
// backprojection of nViews views given their VoxView table (device) into z-slices [z0, z0+nzs) of a
// volume whose full height is g.nz; vol points at slice z0.  accumulate: vol += instead of vol =.
//   unit_proj: treat projections as all ones (column sums A^T 1), proj may be NULL
//   row0/nrows: the projection buffer holds detector rows [row0,row0+nrows) only (chunked path)
//   h_views: host copy of the same table; when given (and the problem qualifies) the TMA-staged kernel of
//   atb_tma.cu runs, otherwise the L1/L2 gather kernel of atb.cu
struct AtbFuse {   // launch_atb with the SART update in the backprojector's epilogue (atb_common.cuh, AtbP::fuse): vol = the iterate's slab
    float* xT;     // slab of the (x,y)-transposed copy of the iterate, updated too
    const float* V;   // slab of the column weights (may be null = ones)
    float lambda;
    int nonneg;
};
// Returns 2 (nothing launched) when `fuse` is given and the TMA kernel does not take the problem: the caller then runs the two steps.
int launch_atb(const float* proj, const Grid& g, const VoxView* d_views, int nViews, int mode, bool unit_proj,
               float* vol, int z0, int nzs, bool accumulate, int row0, int nrows, bool clamp, cudaStream_t st,
               const VoxView* h_views = nullptr, const AtbFuse* fuse = nullptr);
// true if some voxel of the box can project beyond |index| 1e6 in some view (then the kernels clamp)
bool vox_needs_clamp(const Grid& g, const VoxView* host_views, int n);

// elementwise
int launch_residual(const float* b, const int32_t* view_idx, const float* Ax, const float* W, float* r,
                    size_t per_view, int nViews, double* d_nrm2_accum, cudaStream_t st);
int launch_update(float* x, const float* g, const float* V, float lambda, int nonneg, size_t n, cudaStream_t st);
// the same update, which also writes the (x,y)-transposed copy xT[z][x][y] of the new iterate (tiles through shared memory)
int launch_update_t(float* x, float* xT, const float* g, const float* V, float lambda, int nonneg, int nx, int ny, int nz,
                    cudaStream_t st);
int launch_invert_rows(float* w, size_t n, float eps, cudaStream_t st);                 // w = w>eps ? 1/w : 0
int launch_invert_cols(float* v, size_t n, float rel_eps, cudaStream_t st);             // eps = rel_eps*max(v)
int launch_dot(const float* a, const float* b, size_t n, double* d_out, cudaStream_t st);   // *d_out = sum a*b
int launch_axpy(float* y, const float* x, const double* d_num, const double* d_den, float sign, size_t n,
                cudaStream_t st);                                                       // y += sign*(num/den)*x
int launch_xpby(float* p, const float* s, const double* d_num, const double* d_den, size_t n,
                cudaStream_t st);                                                       // p = s + (num/den)*p
int launch_scale(float* x, float a, size_t n, cudaStream_t st);
int launch_fill(float* x, float a, size_t n, cudaStream_t st);                          // x = a
int launch_max(const float* v, size_t n, float* d_max, cudaStream_t st);                // *d_max = max(*d_max, max v), v >= 0
int launch_scale_columns(float* W, const float* colw, int nViews, int nv, int nu, cudaStream_t st);
int launch_ratio(const float* b, const int32_t* view_idx, const float* Ax, float* q, size_t per_view, int nViews, cudaStream_t st);
int launch_mul_update(float* x, const float* g, const float* V, size_t n, cudaStream_t st);
int launch_diff_stats(const float* a, const float* b, const float* c, size_t n, double* d_out3, cudaStream_t st);
void fdk_filter_taps(int nu, int filter, std::vector<double>& g);
int fdk_weights(const Grid& g, const std::vector<ViewH>& views, int weighting, std::vector<double>& w);
int launch_fdk_filter_taps(const float* b, const Grid& g, const double* d_dsd, const double* d_dso, const double* d_offd, int nViews,
                           const float* d_taps, const float* d_colw, float* q, cudaStream_t st, bool odd_only = false);
// the same filter on the tensor cores (fdk_tc.cu); returns 1 if the problem does not qualify (then the kernel above runs)
int launch_fdk_filter_tc(const float* b, const Grid& g, const std::vector<double>& dsd, const std::vector<double>& dso,
                         const std::vector<double>& offd, int nViews, const std::vector<float>& h_taps, const float* d_colw, float* q,
                         cudaStream_t st);
int launch_flatten(const float* curved, const Grid& g, const double* d_dsd, int nViews, float* flat, cudaStream_t st);
int launch_count_reduce(const uint32_t* c, size_t n, unsigned long long* d_total, cudaStream_t st);

// TV / AwTV (tv.cu): value and/or gradient in one pass (g, d_val, d_gg may be NULL; accumulators pre-zeroed);
// normalised descent step x -= alpha g / sqrt(*d_gg)
int launch_tv_gradient(const float* x, int nx, int ny, int nz, float delta, float eps, float* g, double* d_val, double* d_gg,
                       cudaStream_t st);
int launch_prox_div(const float* px, const float* py, const float* pz, const float* f, float lam, bool final, float* out, int nx,
                    int ny, int nz, cudaStream_t st);
int launch_prox_update(float* px, float* py, float* pz, const float* d, float tau, int nx, int ny, int nz, cudaStream_t st);
int launch_momentum(float* y, float* x, const float* xn, float c, size_t n, cudaStream_t st);
int launch_tv_step(float* x, const float* g, float alpha, const double* d_gg, size_t n, cudaStream_t st);

int microbench(int kind, double* value, cudaStream_t st);   // peaks.cu

// chunked (pinned host) path
int chunked_ax(const float* h_vol, const tigre_geo* geo, const double* angles, int nA, int mode, float* h_proj,
               cudaStream_t st);
int chunked_atb(const float* h_proj, const tigre_geo* geo, const double* angles, int nA, int mode, float* h_vol,
                cudaStream_t st);
int chunked_sirt(const float* h_b, const tigre_geo* geo, const double* angles, int nA, int n_iter, float lambda, int nonneg,
                 int ax_mode, int atb_mode, float* h_x, float* h_r, double* resid_hist, cudaStream_t st);
size_t chunk_budget();
size_t workspace_free_bytes();   // largest free block of the caller's workspace (0: none set)
bool workspace_active();
int tables_prep(const tigre_geo* geo, const double* angles, int nA, Grid& g, std::vector<ViewH>& views);

}  // namespace tg
