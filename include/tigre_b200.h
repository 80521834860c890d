/*
 * tigre_b200.h — C ABI of libtigre_b200: the cone-beam projector pair of TIGRE-style
 * iterative CT reconstruction (arxiv 2412.10129), hand-written CUDA for sm_100a.
 *
 * Citations are to /root/reference/PAPER.md (line, section) and to the readings P1..P19
 * in DESIGN.md where the paper is silent.
 *
 * Conventions (all entry points)
 *   units      mm and radians
 *   volume     float32, vol[iz][iy][ix], x fastest, nVoxel = (nx,ny,nz)
 *   projections float32, proj[ia][iv][iu], u fastest, nDetector = (nu,nv)
 *   pointers   "dev" = CUDA device memory of the current device; "host" = ordinary host memory
 *              read during the call only; "pinned" = page-locked host memory (chunked path).
 *              The library keeps no pointer after a call returns.
 *   stream     `cuda_stream` is a cudaStream_t passed as void* (NULL = legacy default stream).
 *              Kernels are enqueued on it; calls that return host scalars synchronise it.
 *   memory     Volumes and projections are the caller's.  Temporaries (per-view parameter tables, driver work
 *              buffers, the buffers of a tigre_plan) are carved from the caller-owned workspace given to
 *              tigre_set_workspace(); tigre_workspace_bytes() /
 *              tigre_plan_workspace_bytes() say how much a call needs.  With NO workspace set (the default) they
 *              come from the device's stream-ordered pool instead (cudaMallocAsync / cudaFreeAsync on
 *              `cuda_stream`), which is the only allocation the library ever makes.
 *   errors     0 on success, negative tigre_status otherwise.  No exception crosses the ABI.
 *              There is no CPU fallback: without a CUDA device every compute call fails.
 */
#ifndef TIGRE_B200_H
#define TIGRE_B200_H

#include <stddef.h>
#include <stdint.h>

#if defined(__GNUC__)
#define TIGRE_API __attribute__((visibility("default")))
#else
#define TIGRE_API
#endif

#ifdef __cplusplus
extern "C" {
#endif

/* Geometry descriptor: App. B Table B1; §2.4 lines 179-197.
 * sVoxel / sDetector are derived (n*d) (reading P1).  The `_a` pointers are optional host
 * arrays of length nAngles ("defined individually for each projection"); when
 * NULL the scalar member is used for every view. */
typedef struct tigre_geo {
    uint32_t struct_size;       /* = sizeof(tigre_geo); checked                              */
    int32_t  nVoxel[3];         /* x, y, z                                                    */
    double   dVoxel[3];         /* mm                                                         */
    int32_t  nDetector[2];      /* u, v                                                       */
    double   dDetector[2];      /* mm                                                         */
    double   DSD, DSO, COR;     /* source-detector, source-origin distance; axis shift (Oy)   */
    double   offOrigin[3];      /* volume centre w.r.t. O (Oxyz)                              */
    double   offDetector[2];    /* detector centre shift (uv)                                 */
    double   rotDetector[3];    /* in-place detector rotation (phi, theta, psi)               */
    const double *DSD_a, *DSO_a, *COR_a;        /* [nA]     or NULL                           */
    const double *offOrigin_a;                  /* [nA][3]  or NULL                           */
    const double *offDetector_a;                /* [nA][2]  or NULL                           */
    const double *rotDetector_a;                /* [nA][3]  or NULL                           */
    double   accuracy;          /* interpolated-mode step in voxels (0.5 in configs C2, C4)   */
    int32_t  mode;              /* TIGRE_GEO_CONE (0) or TIGRE_GEO_PARALLEL (1): PAPER.md:296-306 (synchrotron parallel-beam
                                 * data); reading P29: every ray runs along the S-O line (the gantry-rotated x axis)
                                 * and is the segment of length DSD that ends at its pixel; the voxel-driven map is affine,
                                 * the matched weight dVoxel^3/(du dv cos), the FDK weight 1 (tigre_fdk = FBP)             */
} tigre_geo;
enum { TIGRE_GEO_CONE = 0, TIGRE_GEO_PARALLEL = 1 };

typedef enum tigre_status {
    TIGRE_OK = 0,
    TIGRE_ERR_ARG = -1,       /* NULL pointer, bad mode, bad struct_size, bad sizes            */
    TIGRE_ERR_GEOMETRY = -2,  /* DSO<=0, DSD<=0, non-positive sizes, or a volume corner at or  */
                              /* behind the source plane of some view (voxel-driven calls)     */
    TIGRE_ERR_MEMSPACE = -3,  /* a data pointer is in the wrong memory space                   */
    TIGRE_ERR_WORKSPACE = -4, /* a temporary allocation failed                                 */
    TIGRE_ERR_CUDA = -5,      /* any other CUDA error (tigre_last_cuda_error() gives the text) */
    TIGRE_ERR_NO_DEVICE = -6, /* no CUDA device: there is no CPU fallback                      */
    TIGRE_ERR_TOO_LARGE = -7  /* a size exceeds the fixed scratch of a no-allocation entry     */
                              /* point (tigre_residual_noalloc); nothing was launched          */
} tigre_status;

enum { TIGRE_AX_SIDDON = 0, TIGRE_AX_INTERP = 1 };
enum { TIGRE_ATB_MATCHED = 0, TIGRE_ATB_FDK = 1,
       /* exact transposes of tigre_Ax (ray-driven scatter of the very same weights) */
       TIGRE_ATB_EXACT_SIDDON = 2, TIGRE_ATB_EXACT_INTERP = 3 };
enum { TIGRE_FILTER_RAM_LAK = 0, TIGRE_FILTER_SHEPP_LOGAN = 1, TIGRE_FILTER_COSINE = 2, TIGRE_FILTER_HAMMING = 3,
       TIGRE_FILTER_HANN = 4 };
enum { TIGRE_FDK_FULL = 0, TIGRE_FDK_PARKER = 1, TIGRE_FDK_WANG = 2 };
enum { TIGRE_OP_AX = 0, TIGRE_OP_ATB = 1, TIGRE_OP_OSSART = 2, TIGRE_OP_CGLS = 3, TIGRE_OP_FDK = 4 };

/* ---- the projector pair ------------------------------------------------------------------
 * tigre_Ax: forward projection b = A x, line integrals of the volume along the source->pixel
 * segments (§2.1 eq. 1).  Ray-driven, one thread per detector pixel.
 *   mode TIGRE_AX_SIDDON  exact intersection lengths with the voxel grid (DESIGN.md O-A)
 *   mode TIGRE_AX_INTERP  fixed-step trilinear sampling, step geo->accuracy voxels (O-B, P9)
 *   vol   dev, [nz][ny][nx], read      proj  dev, [nA][nv][nu], overwritten
 *   angles host, [nA][3] Euler ZYZ (z1,y1,z2); a circular scan is (theta,0,0)
 * If both vol and proj are PINNED HOST pointers the call takes the single-GPU host-chunking
 * path (z-slabs of the volume and angle batches stream through HBM) and
 * synchronises before returning.  Pageable host data pointers give TIGRE_ERR_MEMSPACE. */
TIGRE_API int tigre_Ax(const float *vol, const tigre_geo *geo, const double *angles, int nA, int mode,
             float *proj, void *cuda_stream);

/* tigre_Atb: voxel-driven backprojection x = A^T b used by eqs. 4 and 6;
 * bilinear detector interpolation with zero border, weight per voxel-view
 *   mode TIGRE_ATB_MATCHED  w = (dx dy dz)/(du dv) * R^2/(r^2 cos gamma)   (P10)
 *   mode TIGRE_ATB_FDK      w = (DSO/(DSO - X'_x))^2
 *   mode TIGRE_ATB_EXACT_SIDDON / _INTERP   the exact transpose A^T of tigre_Ax in that mode: every ray adds
 *        (intersection length | trilinear weight x step) x its value to the voxels it meets, so that
 *        <Ax, y> = <x, A^T y> up to fp32 rounding (the Krylov family wants a matched pair).
 *        Sums are formed with floating-point atomics: the result is reproducible only up to summation order.
 *   proj dev, [nA][nv][nu], read       vol  dev, [nz][ny][nx], OVERWRITTEN
 * Pinned-host pointers select the chunked path as for tigre_Ax (voxel-driven modes only: the exact modes return
 * TIGRE_ERR_MEMSPACE for host pointers). */
TIGRE_API int tigre_Atb(const float *proj, const tigre_geo *geo, const double *angles, int nA, int mode,
              float *vol, void *cuda_stream);

/* ---- z-slab entry points: the building blocks of multi-GPU sharding (PAPER.md:201-203
 * "split ... by image slabs").  The volume is cut into slabs of z-slices [z0, z0 + nzs); geo describes the FULL volume.
 * tigre_Ax_slab: proj (dev, full size [nA][nv][nu], overwritten) = the slab's PARTIAL line integrals; the sum over a
 * partition into slabs is tigre_Ax of the whole volume (Siddon: intersection lengths are additive; interpolated: the sample
 * positions are those of the full volume and taps outside the slab count as zero).  Rows outside the slab's detector-row
 * band are zero.  vol_slab dev [nzs][ny][nx].
 * tigre_Atb_slab: vol_slab (dev [nzs][ny][nx]) = slices [z0, z0 + nzs) of tigre_Atb (voxel-driven modes); it reads only
 * the slab's row band of proj (dev, full size).
 * tigre_slab_row_band: the band [row0, row0 + nrows) of detector rows the slab can reach in any of the views (corner
 * projection in fp64, one row of margin); host arithmetic, no device needed. */
TIGRE_API int tigre_Ax_slab(const float *vol_slab, const tigre_geo *geo, const double *angles, int nA, int mode, int z0, int nzs,
                  float *proj, void *cuda_stream);
TIGRE_API int tigre_Atb_slab(const float *proj, const tigre_geo *geo, const double *angles, int nA, int mode, int z0, int nzs,
                   float *vol_slab, void *cuda_stream);
TIGRE_API int tigre_slab_row_band(const tigre_geo *geo, const double *angles, int nA, int z0, int nzs, int *row0, int *nrows);

/* ---- SIRT / OS-SART weights and elementwise updates (eq. 6 at 135) ----------
 * W = 1/(A 1) where (A 1) > 1e-2*min(dVoxel), else 0   (row sums; proj-shaped, dev)
 * V = 1/(A^T 1) where (A^T 1) > 1e-6*max(A^T 1), else 0 (column sums; vol-shaped, dev)  (P13) */
TIGRE_API int tigre_row_weights(const tigre_geo *geo, const double *angles, int nA, int ax_mode, float *W,
                      void *cuda_stream);
TIGRE_API int tigre_col_weights(const tigre_geo *geo, const double *angles, int nA, int atb_mode, float *V,
                      void *cuda_stream);
/* r = W .* (b - Ax)  (W may be NULL = ones); *nrm2 (host, may be NULL) = ||b - Ax||_2^2.
 * All arrays dev, n elements.  Synchronises only when nrm2 != NULL. */
TIGRE_API int tigre_residual(const float *b, const float *Ax, const float *W, float *r, size_t n, double *nrm2,
                   void *cuda_stream);
/* tigre_residual for callers that cannot allocate (code under CUDA graph capture, tight serving loops, harnesses that forbid
 * cudaMalloc): the same r = W .* (b - Ax) (bitwise) and ||b - Ax||_2^2 (eq. 2), but
 *   - it calls no cudaMalloc / cudaFree / cudaMallocAsync or allocating library routine, creates no stream or event and never
 *     synchronises: its scratch (one fp64 partial sum per CTA) is a file-scope 128 KiB array in device memory that every GPU
 *     which loads the library holds until the process exits (csrc/noalloc.cu);
 *   - that array bounds the size: n <= TIGRE_RESIDUAL_NOALLOC_MAX_N elements (2^28 = 1 GiB per array), else
 *     TIGRE_ERR_TOO_LARGE and nothing is launched or written (split the call);
 *   - nrm2_dev is a DEVICE pointer (may be NULL: then only r is formed), written in stream order; the sum is formed in a fixed
 *     order, so it is bitwise reproducible (it agrees with tigre_residual's to fp64 rounding, not bitwise);
 *   - all calls on a device share the scratch array, which keeps the last call's contents; nothing in it has to start at zero
 *     (each call overwrites the slots it then reads).  Calls that OVERLAP on the GPU (different streams without an event
 *     between them, graphs replayed concurrently) race on it: their nrm2 is undefined.  Calls on one stream are safe;
 *   - the device that is current at the call is the one whose scratch is used (its address is looked up on the first call on
 *     that device: make that first call outside graph capture); b, Ax, W (may be NULL), r: dev, n elements, r may alias Ax. */
#define TIGRE_RESIDUAL_NOALLOC_MAX_N 268435456ull
TIGRE_API int tigre_residual_noalloc(const float *b, const float *Ax, const float *W, float *r, size_t n, double *nrm2_dev,
                           void *cuda_stream);
/* x <- x + lambda * V .* g, then x <- max(x,0) if nonneg  (V may be NULL = ones).  dev, n elements */
TIGRE_API int tigre_update(float *x, const float *g, const float *V, float lambda, int nonneg, size_t n,
                 void *cuda_stream);

/* ---- drivers ------------------------------------------------------------------------------
 * OS-SART (eq. 6; DESIGN.md O-E): for it, for subset s:
 *   r = W_s .* (b_s - A_s x);  x += lambda * V_s .* A_s^T r;  x = max(x,0) if nonneg.
 * Subsets are CSR lists of view indices: subset s = subset_idx[subset_off[s] .. subset_off[s+1]).
 * One subset holding all views is SIRT.  resid_hist[it] (host, may be NULL) = running
 * ||b - A x||_2 over the sweep.  b dev [nA][nv][nu]; x_inout dev (initial iterate in, result out). */
TIGRE_API int tigre_ossart(const float *b, const tigre_geo *geo, const double *angles, int nA,
                 const int32_t *subset_idx, const int32_t *subset_off, int nSubsets, int n_iter,
                 float lambda, int nonneg, int ax_mode, int atb_mode, float *x_inout,
                 double *resid_hist, void *cuda_stream);
/* The same iteration with the per-geometry set-up (view tables, W_s, V_s, scratch) done once in a
 * plan.  tigre_plan_create computes the weights on `cuda_stream`; the plan owns its device buffers
 * (stream-ordered pool) until tigre_plan_destroy.  tigre_plan_ossart runs n_iter sweeps starting from
 * x_inout; b and x_inout are both dev, or both PINNED HOST (then they are copied in, and x copied
 * back, on the stream: the end-to-end path bench.py times). */
typedef struct tigre_plan tigre_plan;
TIGRE_API int tigre_plan_create(const tigre_geo *geo, const double *angles, int nA, const int32_t *subset_idx,
                      const int32_t *subset_off, int nSubsets, int ax_mode, int atb_mode,
                      void *cuda_stream, tigre_plan **plan_out);
/* tigre_plan_create with data-redundancy weighting for displaced detectors inside the iteration (DESIGN.md
 * readings P17, P28): redundancy != 0 multiplies the row weights W of view a, column u by the Wang weight w_a(u) (1 on the
 * singly measured side, a smooth ramp over the doubly measured columns); TIGRE_ERR_ARG if the displacement leaves no overlap. */
TIGRE_API int tigre_plan_create_ex(const tigre_geo *geo, const double *angles, int nA, const int32_t *subset_idx,
                         const int32_t *subset_off, int nSubsets, int ax_mode, int atb_mode, int redundancy,
                         void *cuda_stream, tigre_plan **plan_out);
TIGRE_API int tigre_plan_ossart(tigre_plan *plan, const float *b, float *x_inout, int n_iter, float lambda,
                      int nonneg, double *resid_hist, void *cuda_stream);
/* Host only (no device needed): the z-slices [*zlo, *zhi] of the volume that rays of detector rows [row0, row1) of the given views
 * can meet, with three slices of margin (zlo > zhi: none).  Returns 1 when no bound is formed (parallel beam; source or detector
 * over the volume's (x,y) footprint).  tigre_plan_ossart with pinned host arrays uses it to send the iterate up in the order the
 * first projection's row bands need it (e2e); exported for its test against the oracle's first / last
 * voxel per ray (reading P19(a)). */
TIGRE_API int tigre_band_z_range(const tigre_geo *geo, const double *angles, int nA, int row0, int row1, int32_t *zlo, int32_t *zhi);
/* The subset steps [s_begin, s_end) of ONE sweep of tigre_plan_ossart, in order, with the plan's own W_s, V_s and view lists
 * (what a caller needs to interleave other work between subsets, and what the tests use to check a single ordered-subset
 * update of the very plan a long run advances).  b, x_inout dev, or both pinned host.  Asynchronous for device data. */
TIGRE_API int tigre_plan_ossart_subsets(tigre_plan *plan, const float *b, float *x_inout, int s_begin, int s_end, float lambda,
                              int nonneg, void *cuda_stream);
TIGRE_API int tigre_plan_destroy(tigre_plan *plan);
/* device bytes the plan holds.  The column weights V_s take one volume PER SUBSET while all of them fit half of the free device
 * memory (or of the workspace) at creation; otherwise (single-view subsets on large volumes: SART on 512^3 would need 386 GB)
 * the plan keeps ONE volume and every subset step recomputes its V_s first (one more backprojection per subset).
 * tigre_set_plan_v_path: 0 = that rule (default), 1 = always stored, 2 = always recomputed (test hook; applies to plans
 * created afterwards). */
TIGRE_API size_t tigre_plan_bytes(const tigre_plan *plan);
TIGRE_API int tigre_set_plan_v_path(int path);
/* SIRT on arrays larger than the device (BASELINE.json configs[4] "single-GPU z-slab/angle-batch host chunking ... one SIRT
 * iteration"; eq. 6 with one subset of all views): b, x_inout and r_scratch are PINNED HOST
 * arrays (b, r_scratch [nA][nv][nu]; x_inout [nz][ny][nx], start in, result out).  Per iteration two streamed passes:
 *   pass 1, per view batch: A x accumulated over the z-slabs of x, then r = W .* (b - A x), W = 1/(A 1) (reading P13), written
 *           to r_scratch; resid_hist[it] (host, may be NULL) = ||b - A x||_2;
 *   pass 2, per z-slab: G = A^T r and U = A^T 1 over the streamed row bands of all views, x <- max(0, x + lambda G / U)
 *           where U > 1e-6 max(A^T 1) (nonneg = 0: no clamp).  max(A^T 1) over the volume costs one extra A^T 1 pass per call.
 * r_scratch may be b itself when n_iter == 1 (b is then overwritten by the weighted residual).  Synchronises.
 * Same kernels as the device-resident path; results agree with tigre_plan_ossart (one subset) up to summation order.
 * TIGRE_ERR_MEMSPACE unless all three arrays are pinned. */
TIGRE_API int tigre_sirt_chunked(const float *b, const tigre_geo *geo, const double *angles, int nA, int n_iter, float lambda,
                       int nonneg, int ax_mode, int atb_mode, float *x_inout, float *r_scratch, double *resid_hist,
                       void *cuda_stream);
/* MLEM / OSEM (eq. 5 "x^k = x^{k-1}/(A1) A^T (b / (A x^{k-1}))"; 118-120, 139 OS counterpart; DESIGN.md reading
 * P33): for every subset s of the plan in turn  x <- x * V_s * A_s^T(b_s / (A_s x)),  V_s = the plan's column weights 1/(A_s^T 1),
 * quotient 0 where A_s x <= 0.  One subset holding all views is MLEM.  b, x_inout dev (x_inout: positive start, e.g. ones).
 * Asynchronous. */
TIGRE_API int tigre_plan_osem(tigre_plan *plan, const float *b, float *x_inout, int n_iter, void *cuda_stream);
/* ASD-POCS / OS-ASD-POCS / AwASD-POCS ("Projection Onto Convex Sets ... ASD-POCS [30] ... Adaptive weighed TV
 * norm [32, 33] ... OS versions", 141-149 Snippet 1, 169; reading P23 spells the loop out).  Per iteration:
 *   x0 = x;  one OS-SART sweep of the plan's subsets with relaxation beta (nonnegativity on);  beta *= beta_red;
 *   dd = ||A x - b||_2 (fresh forward projection);  dp = ||x - x0||_2;  first iteration: dtvg = alpha * dp;
 *   xp = x;  ng steps of x <- x - dtvg g/||g||_2 with g the gradient of TV (delta <= 0 or inf) or AwTV (delta > 0);
 *   dg = ||x - xp||_2;  if dg > r_max*dp and dd > epsilon: dtvg *= alpha_red;  c = cos(x - xp, xp - x0);
 *   stop after the iteration if (c < -0.99 and dd <= epsilon) or beta < 0.005.
 * Single-view subsets in the plan give ASD-POCS, blocks give OS-ASD-POCS.  b, x_inout dev.  hist (host, may be NULL)
 * [n_iter][5] = dd, dp, dg, the dtvg this iteration used, c;  *n_done (host, may be NULL) = iterations run.
 * Synchronises the stream twice per iteration (the step-length rule runs on the host). */
TIGRE_API int tigre_plan_asd_pocs(tigre_plan *plan, const float *b, float *x_inout, int n_iter, float beta, float beta_red,
                        int ng, float alpha, float alpha_red, float r_max, float epsilon, float delta, float tv_eps,
                        double *hist, int *n_done, void *cuda_stream);
/* CGLS (textbook recurrences, DESIGN.md O-F), x0 = 0; x_out dev.  atb_mode may be any of the
 * four tigre_Atb modes (the exact ones must match ax_mode); tigre_ossart / tigre_plan_* take the voxel-driven two. */
TIGRE_API int tigre_cgls(const float *b, const tigre_geo *geo, const double *angles, int nA, int n_iter,
               int ax_mode, int atb_mode, float *x_out, double *resid_hist, void *cuda_stream);
/* Gradient descent (eq. 4; reading P32): x^k = x^{k-1} + lambda A^T (b - A x^{k-1}), all views per
 * step, no weights, no constraint (the paper prints the residual as (Ax - b); the descent sign is used).  x_inout dev (start in,
 * result out); resid_hist[k] (host, may be NULL) = ||b - A x^{k-1}||_2.  atb_mode: any of the four tigre_Atb modes. */
TIGRE_API int tigre_gradient_descent(const float *b, const tigre_geo *geo, const double *angles, int nA, int n_iter, float lambda,
                           int ax_mode, int atb_mode, float *x_inout, double *resid_hist, void *cuda_stream);
/* FDK (DESIGN.md O-D): cosine weight, Ram-Lak ramp filter along u, FDK-weighted
 * backprojection scaled by pi/nA (full 2 pi orbit).  b dev, x_out dev. */
TIGRE_API int tigre_fdk(const float *b, const tigre_geo *geo, const double *angles, int nA, float *x_out,
              void *cuda_stream);
/* the FDK pre-filter alone: q = tau * ((b * cos) conv h), per detector row.  dev -> dev */
TIGRE_API int tigre_fdk_filter(const float *b, const tigre_geo *geo, const double *angles, int nA, float *q,
                     void *cuda_stream);

/* FDK variants ("various filter types and geometric correction methods, such as Wang [25]
 * and Parker [26] weights for detector displacement and angular range corrections", 281, 359; readings P26-P28).
 * filter: the Ram-Lak taps windowed in frequency on L = 2^ceil(log2(2 nDetector_u)) samples, omega in [0, pi]:
 *   RAM_LAK 1, SHEPP_LOGAN sin(omega/2)/(omega/2), COSINE cos(omega/2), HAMMING 0.54 + 0.46 cos(omega), HANN 0.5 + 0.5 cos(omega),
 * applied as a linear convolution of the zero-padded row (equal to the FFT formulation).
 * weighting: FULL = full circle (tigre_fdk); PARKER = short scan over |theta_last - theta_first| = pi + 2 eps < 2 pi with
 * monotone angles, sum scaled by the angular step; WANG = detector displaced along u over a full circle, projections
 * multiplied by 2 w(u).  TIGRE_ERR_ARG if the scan does not fit the weighting.
 * tigre_fdk_weights: the weight table alone, w host [nA][nDetector_u] fp64 (WANG without the factor 2); no device needed. */
TIGRE_API int tigre_fdk_ex(const float *b, const tigre_geo *geo, const double *angles, int nA, int filter, int weighting,
                 float *x_out, void *cuda_stream);
TIGRE_API int tigre_fdk_filter_ex(const float *b, const tigre_geo *geo, const double *angles, int nA, int filter, int weighting,
                        float *q, void *cuda_stream);
TIGRE_API int tigre_fdk_weights(const tigre_geo *geo, const double *angles, int nA, int weighting, double *w);

/* Curved detectors ("TIGRE now allows to consider curved detectors by applying a 'flattening' transformation";
 * DESIGN.md reading P30): curved (dev [nA][nv][nu]) was measured on the cylinder of radius DSD about the axis through the
 * source parallel to v, pixel pitch du along the arc and dv in height; flat (dev, same shape, must not alias) receives the
 * image a flat detector of the same pixel counts and pitches would have seen: flat(u, v) = curved(arc length DSD atan(u/DSD),
 * height v cos(atan(u/DSD))), bilinear, zero outside.  Per-view DSD honoured. */
TIGRE_API int tigre_flatten_detector(const float *curved, const tigre_geo *geo, const double *angles, int nA, float *flat,
                           void *cuda_stream);

/* ---- total variation (section 2.2.3 eqs. 7-8; P20-P22) ----------
 * AwTV(x) = sum_p sqrt(w_x dx^2 + w_y dy^2 + w_z dz^2 + eps), backward differences d_a = x[p] - x[p - e_a], weights
 * w_a = exp(-(d_a/delta)^2), over the voxels that have all their backward neighbours (an axis of length 1 drops
 * out: nz = 1 is the paper's 2-D formula).  delta <= 0 or infinite selects the plain TV norm (w = 1).
 * x dev [nz][ny][nx].  tigre_awtv: *value (host) = AwTV(x); synchronises.  tigre_awtv_gradient: g dev (same
 * shape) = dAwTV/dx, the weights differentiated too; *value and *grad_norm2 (host, each may be NULL) receive
 * AwTV(x) and ||g||_2^2 from the same pass (the call synchronises only if one of them is asked for).
 * tigre_minimize_awtv: n_steps of x <- x - alpha g/||g||_2 in place (the "gradient descent minimizer" of PAPER.md:169;
 * stops moving when the gradient vanishes); asynchronous. */
TIGRE_API int tigre_awtv(const float *x, int nx, int ny, int nz, float delta, float eps, double *value, void *cuda_stream);
TIGRE_API int tigre_awtv_gradient(const float *x, int nx, int ny, int nz, float delta, float eps, float *g, double *value,
                        double *grad_norm2, void *cuda_stream);
TIGRE_API int tigre_minimize_awtv(float *x_inout, int nx, int ny, int nz, float delta, float eps, float alpha, int n_steps,
                        void *cuda_stream);

/* ---- TV proximal operator and FISTA ("For the 2-norm and TV proximal operators, TIGRE provides ... FISTA [42]";
 * used at 308-314 and 377-393: FISTA(proj, geo, angles, 20, 'hyper', 2e2, ..., 'tviter', 50); readings P24, P25) -----
 * tigre_tv_prox: u = argmin 1/2||u - f||^2 + lambda TV(u), isotropic TV with forward differences, by n_iter steps of the dual
 * projection iteration p <- (p + tau grad(div p - f/lambda)) / (1 + tau |grad(div p - f/lambda)|), u = f - lambda div p
 * (tau <= 1/12 in three dimensions).  f, u dev [nz][ny][nx] (u may alias f); lambda = 0 copies.  Asynchronous.
 * tigre_fista: x_{k+1} = prox_{tv_lambda}(y_k + (2/L) A^T(b - A y_k)), t_{k+1} = (1 + sqrt(1 + 4 t_k^2))/2,
 * y_{k+1} = x_{k+1} + ((t_k - 1)/t_{k+1})(x_{k+1} - x_k); y_0 = x_0 = x_inout (the 'init'), t_0 = 1; L = 'hyper'.
 * resid_hist[k] (host, may be NULL) = ||b - A y_k||_2.  atb_mode: any of the four tigre_Atb modes (exact ones must match
 * ax_mode).  b dev, x_inout dev. */
TIGRE_API int tigre_tv_prox(const float *f, int nx, int ny, int nz, float lambda, int n_iter, float tau, float *u, void *cuda_stream);
TIGRE_API int tigre_fista(const float *b, const tigre_geo *geo, const double *angles, int nA, int n_iter, float L, float tv_lambda,
                int tv_iter, float tau, int ax_mode, int atb_mode, float *x_inout, double *resid_hist, void *cuda_stream);

/* SART-TV ("TIGRE also includes the SART-TV algorithm [44]", used at 365; reading P31): per iteration the
 * plan's OS-SART sweep with relaxation lambda (nonnegativity on; single-view subsets = SART), then x <- tigre_tv_prox(x, tv_lambda,
 * tv_iter, tau); lambda *= lambda_red.  b, x_inout dev; resid_hist (host, may be NULL) [n_iter] as tigre_plan_ossart. */
TIGRE_API int tigre_plan_sart_tv(tigre_plan *plan, const float *b, float *x_inout, int n_iter, float lambda, float lambda_red,
                       float tv_lambda, int tv_iter, float tau, double *resid_hist, void *cuda_stream);

/* ---- measurement helpers -------------------------------------------------------------------
 * Exact count of ray-samples of one tigre_Ax call without marching the data (BASELINE metric:
 * Siddon = non-zero voxel segments; interpolated = samples K inside the grown box).
 * counts: dev uint32 [nA][nv][nu] or NULL; *total (host) = sum.  Synchronises. */
TIGRE_API int tigre_Ax_count(const tigre_geo *geo, const double *angles, int nA, int mode, uint32_t *counts,
                   uint64_t *total, void *cuda_stream);
/* Index equality of the Siddon march (BASELINE.json north_star "Voxel/pixel index and footprint bounds must match exactly";
 * DESIGN.md reading P19(a)): runs the march of tigre_Ax(TIGRE_AX_SIDDON) without touching a volume and returns, per ray,
 * first_last[2 ray] / [2 ray + 1] = linear index (iz ny + iy) nx + ix of the first / last voxel the march gives a non-zero
 * length to, in order from the source (-1 for a ray that misses), and nseg[ray] = the number of such voxels.
 * first_last dev int64 [nA][nv][nu][2]; nseg dev uint32 [nA][nv][nu].  Asynchronous. */
TIGRE_API int tigre_Ax_index(const tigre_geo *geo, const double *angles, int nA, int64_t *first_last, uint32_t *nseg,
                   void *cuda_stream);
/* Footprint bounds of the TMA-staged backprojector (north_star "footprint bounds must match exactly"; reading P19(b)):
 * tigre_Atb with the kernel reporting, per (voxel tile, view), the detector box it staged into shared memory.
 * meta (host int32[8]) receives the tiling: tile size in voxels (x, y, z), box size in pixels (u, v), number of tiles (x, y, z);
 * all zero if this problem does not take the TMA kernel.  boxes (dev int32 [tiles_z][tiles_y][tiles_x][nA][4], or NULL to
 * query meta only: nothing is launched then) receives (u0, v0, fits, 0): the absolute detector index of the box origin and
 * whether the view's footprint fitted the box (0: the kernel gathered that view through L1 / L2 with bounds checks).
 * vol is written as by tigre_Atb.  Voxel-driven modes only. */
TIGRE_API int tigre_Atb_boxes(const float *proj, const tigre_geo *geo, const double *angles, int nA, int mode, float *vol,
                    int32_t *meta, int32_t *boxes, void *cuda_stream);
/* In-library timing for bench.py's roofline leg.  tigre_profile(1) resets and starts recording a CUDA
 * event pair around every kernel group the launchers enqueue (on the launching stream); tigre_profile(0)
 * stops.  tigre_profile_read waits for the recorded events and returns, per kind k = 0 (Ax kernels),
 * 1 (A^T b kernels), 2 (elementwise / reduction / filter kernels): ms[k] = summed device time,
 * launches[k] = kernels launched since the last tigre_profile call (counted even when not recording). */
TIGRE_API int tigre_profile(int enable);
TIGRE_API int tigre_profile_read(double *ms /*[3]*/, uint64_t *launches /*[3]*/);
/* Caller-owned workspace ("the library allocates nothing persistent ... workspace memory is the
 * caller's"; north_star: "PyTorch used only for device memory and streams").
 * tigre_set_workspace(dev_ptr, bytes): from now on every temporary and every plan buffer of this process is a block of
 *   [dev_ptr, dev_ptr + bytes) (first-fit free list on the host, 256-byte granules) and the library makes no allocation of its
 *   own; a call that does not fit returns TIGRE_ERR_WORKSPACE and leaves the workspace as it found it.  The memory stays
 *   the caller's and must outlive every call and plan that uses it.  Blocks are re-used in the order calls are enqueued:
 *   use ONE stream with a workspace (or synchronise when switching streams).  dev_ptr = NULL returns to the default, the
 *   stream-ordered pool.  TIGRE_ERR_ARG while a plan (or a call in flight) still holds blocks, or for bytes < 4096;
 *   TIGRE_ERR_MEMSPACE if dev_ptr is not device memory.  Process-global, guarded by a mutex.
 * tigre_workspace_bytes(geo, nA, op): an upper bound on what one call of kind `op` takes for device-resident data.
 * tigre_plan_workspace_bytes: the same for tigre_plan_create(_ex) plus tigre_plan_ossart with nSubsets subsets of at most
 *   max_subset_views views (host_data != 0: b and x in pinned host memory, the end-to-end path).
 *   The chunked (pinned host) path of tigre_Ax / tigre_Atb / tigre_sirt_chunked sizes its slabs to the workspace.
 * tigre_workspace_stats: bytes in use now, the high-water mark, and the number of pool allocations (cudaMallocAsync) made
 *   since the last tigre_set_workspace (stays 0 while a workspace is set); any pointer may be NULL. */
TIGRE_API int tigre_set_workspace(void *dev_ptr, size_t bytes);
TIGRE_API size_t tigre_workspace_bytes(const tigre_geo *geo, int nA, int op);
TIGRE_API size_t tigre_plan_workspace_bytes(const tigre_geo *geo, int nA, int nSubsets, int max_subset_views, int host_data);
TIGRE_API int tigre_workspace_stats(size_t *in_use, size_t *high_water, uint64_t *pool_allocs);
/* tuning knobs of the chunked path: device bytes it may use for slabs (0 = default 3/4 of free) */
TIGRE_API int tigre_set_chunk_budget(size_t bytes);
/* what the most recent chunked tigre_Ax / tigre_Atb call of this process moved: bytes copied host->device and
 * device->host, number of z-slabs and of view batches (any pointer may be NULL) */
TIGRE_API int tigre_chunk_stats(uint64_t *h2d_bytes, uint64_t *d2h_bytes, int *n_slabs, int *n_batches);
/* which A^T b kernel runs: 0 (default) = detector footprints staged into shared memory by TMA whenever the
 * problem qualifies (16-byte aligned rows, tiles >= 32x16 voxels), 1 = always the L1/L2 gather kernel.  Both
 * compute the same sums (DESIGN.md O-C); the switch exists for A/B measurement.  2 = the TMA kernel with its
 * staged box deliberately undersized, so that views take its in-kernel gather fallback (test hook).  3 = the TMA kernel with
 * the per-voxel reciprocal and square root on tilted views instead of the linearised z-run (A/B and test hook). */
TIGRE_API int tigre_set_atb_path(int path);
/* which interpolated tigre_Ax kernel runs: 0 (default) = boxes of the volume staged into shared memory by TMA where that is
 * the faster one (the 32 rays of a warp span less than 27 voxels) and the problem qualifies (nx, ny multiples of 4, 16-byte
 * aligned volume, the beam of a 32 x 4 pixel tile fits a stage), 1 = always the L1 gather kernel, 2 = the TMA kernel for wide
 * beams too.  Same samples, same per-ray order of summation; A/B and test hook. */
TIGRE_API int tigre_set_ax_path(int path);
/* which Siddon tigre_Ax kernel runs: 0 (default) = the L1 gather kernel, 1 = the kernel that stages the interior of the march
 * into shared memory by TMA (csrc/ax_siddon_tma.cu) where the problem qualifies (nx, ny multiples of 4, 16-byte aligned
 * volume, whole detector, 32-bit offsets).  Bitwise the same projections; the staged kernel is the slower one on B200
 * (profiles/r2_ax_siddon.md) and is kept for A/B measurement and its test. */
TIGRE_API int tigre_set_siddon_path(int path);
/* fusion F2 in the plan drivers' OS-SART step: 1 (default) = the update x <- max(0, x + lambda V .* A^T r) is formed in the epilogue of
 * the TMA backprojection kernel (no gradient volume written or read; the same arithmetic, bitwise the same iterate), 0 = backprojection
 * and update as two kernels.  Problems the TMA kernel does not take run the two kernels either way.  A/B and test hook. */
TIGRE_API int tigre_set_plan_fuse(int on);
/* which FDK pre-filter kernel runs: 0 (default) = the Toeplitz GEMM on the tensor cores (tcgen05, 3 x tf32 split products into an fp32
 * accumulator in tensor memory) whenever nDetector_u is a multiple of 4 and input and output are distinct 16-byte aligned arrays,
 * 1 = always the CUDA-core convolution.  Same taps, same weights; A/B and test hook. */
TIGRE_API int tigre_set_fdk_path(int path);
/* which TV gradient kernel runs: 0 (default) = four voxels along x per thread whenever nx % 4 == 0, ny > 1, nz > 1 and
 * the arrays are 16-byte aligned, 1 = always the one-voxel-per-thread kernel (any shape).  Same sums; A/B and test hook. */
TIGRE_API int tigre_set_tv_path(int path);

/* Step-0 microbenchmarks: the machine rates the projector rooflines rest on,
 * measured by kernels of this library on the current device with CUDA events on `cuda_stream` (best of 5 after a warm-up;
 * the call synchronises).  *value (host) receives
 *   TIGRE_PEAK_FFMA      fp32 multiply-adds per second over all SMs = thread-instructions / s of the plain-ALU issue slots
 *   TIGRE_PEAK_SMEM      bytes / s of conflict-free 128-bit shared-memory loads, all SMs
 *   TIGRE_PEAK_L1_LINES  distinct 128-byte lines / s served from L1 when every lane of a load reads its own (cached) line
 *   TIGRE_PEAK_L2        bytes / s of 128-bit loads that bypass L1 and hit L2 (48 MB working set)
 *   TIGRE_PEAK_H2D, _D2H bytes / s of a 1 GiB cudaMemcpyAsync from / to pinned host memory (allocated and freed inside)
 *   TIGRE_PEAK_HBM_COPY  bytes / s, read + write, of a 2 GiB device-to-device float4 copy kernel
 *   TIGRE_PEAK_SM_HZ     SM clock (Hz) seen by clock64() against the global timer under the FFMA load */
enum { TIGRE_PEAK_FFMA = 0, TIGRE_PEAK_SMEM = 1, TIGRE_PEAK_L1_LINES = 2, TIGRE_PEAK_L2 = 3, TIGRE_PEAK_H2D = 4, TIGRE_PEAK_D2H = 5,
       TIGRE_PEAK_HBM_COPY = 6, TIGRE_PEAK_SM_HZ = 7 };
TIGRE_API int tigre_microbench(int kind, double *value, void *cuda_stream);

/* which element-index type the ray-driven kernels (tigre_Ax both modes, the exact transposes, tigre_Ax_index) use:
 * 0 (default) = 32-bit offsets for volumes (or resident slabs) below 2^31 voxels, 64-bit above; 1 = always the 64-bit
 * instantiations (test hook: the kernels C5-sized slabs take, on volumes small enough to check element by element). */
TIGRE_API int tigre_set_index_path(int path);

TIGRE_API const char *tigre_strerror(int code);
TIGRE_API const char *tigre_last_cuda_error(void);
TIGRE_API int tigre_version(void);

#ifdef __cplusplus
}
#endif
#endif /* TIGRE_B200_H */
