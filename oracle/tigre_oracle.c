/*
 * oracle/tigre_oracle.c — TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of what the cone-beam projector pair computes
 * (arxiv 2412.10129, "TIGRE v3"; /root/reference/PAPER.md).  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * build, load or call this file.  It shares no code, header, table or helper with
 * paper_2412_10129_b200/ (the CUDA path) and neither includes the other.
 *
 * What the paper fixes: b = A x with A the discretised line-integral (Radon) operator
 * (§2.1 eq. 1); the geometry parameters (§2.4,
 * 543-566 App. B Table B1).  The paper never describes the inside of the projectors;
 * every convention below that it leaves open is a reading listed as P1..P19 in
 * DESIGN.md ("Readings of the paper"), taken from SURVEY.md §8(c).
 *
 * Pin status (tests/test_oracle_*.py, `-m "not gpu"`):
 *   ax_siddon      pinned: brute-force per-voxel box intersection, unit-volume box chord,
 *                          single voxel, closed-form ellipsoid chords (loose), parallel limit.
 *   ax_interp      pinned on: linear-ramp closed form, single-voxel central ray, convergence
 *                          to Siddon, parallel limit.  The sampling rule itself (step, midpoint
 *                          offset, half-voxel border) is a reading (P9): beyond those pins,
 *                          "parity unpinned".
 *   atb (fdk / matched)  pinned: proj==1 closed form of the weights, linear projections,
 *                          delta-pixel brute force, normalisation against the exact transpose.
 *   atb_exact_*    pinned: <Ax,y> = <x,A^T y> to 1e-12.
 *   fdk_filter     pinned: reconstruction of an analytic ball returns rho; impulse response = tau * cos * Ram-Lak taps with
 *                          the cosine from independent geometry (also with a displaced detector); wide-fan ball needs it.
 *
 * Layout: vol[iz][iy][ix] (x fastest), proj[ia][iv][iu] (u fastest).  Inputs may be
 * float32 or float64 (flag); all arithmetic and all outputs are float64.
 * Build: gcc -O2 -fopenmp -shared -fPIC (see oracle/build.py).  No -ffast-math.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int32_t nx, ny, nz;
    int32_t nu, nv;
    int32_t parallel; /* 0 = cone beam; 1 = parallel beam (reading P29): rays along the S-O line */
    double dx, dy, dz;
    double du, dv;
    double accuracy;
} orc_grid;

/* one projection's geometry: every non-size parameter may differ per view */
typedef struct {
    double DSD, DSO, COR;
    double offO[3];
    double offD[2];
    double rotD[3]; /* phi, theta, psi */
    double ang[3];  /* Euler ZYZ z1, y1, z2 */
} orc_view;

typedef struct {
    const void *p;
    int f32;
} arr_t;
static inline double LD(arr_t a, size_t i) {
    return a.f32 ? (double)((const float *)a.p)[i] : ((const double *)a.p)[i];
}

/* ---------------------------------------------------------------- small linear algebra */
static void rotx(double a, double R[9]) {
    double c = cos(a), s = sin(a);
    double M[9] = {1, 0, 0, 0, c, -s, 0, s, c};
    memcpy(R, M, sizeof M);
}
static void roty(double a, double R[9]) {
    double c = cos(a), s = sin(a);
    double M[9] = {c, 0, s, 0, 1, 0, -s, 0, c};
    memcpy(R, M, sizeof M);
}
static void rotz(double a, double R[9]) {
    double c = cos(a), s = sin(a);
    double M[9] = {c, -s, 0, s, c, 0, 0, 0, 1};
    memcpy(R, M, sizeof M);
}
static void mm(const double A[9], const double B[9], double C[9]) {
    double T[9];
    for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
            double s = 0;
            for (int k = 0; k < 3; k++) s += A[3 * i + k] * B[3 * k + j];
            T[3 * i + j] = s;
        }
    memcpy(C, T, sizeof T);
}
static void mv(const double A[9], const double x[3], double y[3]) {
    double t[3];
    for (int i = 0; i < 3; i++) t[i] = A[3 * i] * x[0] + A[3 * i + 1] * x[1] + A[3 * i + 2] * x[2];
    memcpy(y, t, sizeof t);
}
static void mtv(const double A[9], const double x[3], double y[3]) { /* y = A^T x */
    double t[3];
    for (int i = 0; i < 3; i++) t[i] = A[i] * x[0] + A[3 + i] * x[1] + A[6 + i] * x[2];
    memcpy(y, t, sizeof t);
}

/* ---------------------------------------------------------------- geometry */
/* P6: gantry R_g = Rz(z1) Ry(y1) Rz(z2).  P3: detector R_det = Rz(psi) Ry(theta) Rx(phi). */
static void frames(const orc_view *w, double Rg[9], double Rd[9]) {
    double A[9], B[9], C[9];
    rotz(w->ang[0], A);
    roty(w->ang[1], B);
    rotz(w->ang[2], C);
    mm(A, B, Rg);
    mm(Rg, C, Rg);
    rotz(w->rotD[2], A);
    roty(w->rotD[1], B);
    rotx(w->rotD[0], C);
    mm(A, B, Rd);
    mm(Rd, C, Rd);
}
/* P2 default pose: S0 = (DSO,0,0).  P5: COR translates source and detector by (0,-COR,0). */
static void source_pos(const orc_view *w, const double Rg[9], double S[3]) {
    double S1[3] = {w->DSO, -w->COR, 0.0};
    mv(Rg, S1, S);
}
/* pixel centre (iu,iv) may be fractional.  P4: offDetector in the unrotated uv frame. */
static void pixel_pos(const orc_grid *g, const orc_view *w, const double Rg[9], const double Rd[9],
                      double iu, double iv, double P[3]) {
    double u = (iu + 0.5) * g->du - 0.5 * g->nu * g->du;
    double v = (iv + 0.5) * g->dv - 0.5 * g->nv * g->dv;
    double loc[3] = {0.0, u, v}, r[3];
    mv(Rd, loc, r);
    double p1[3] = {w->DSO - w->DSD + r[0], w->offD[0] + r[1] - w->COR, w->offD[1] + r[2]};
    mv(Rg, p1, P);
}
/* P29 parallel beam: every ray runs along the gantry-rotated x axis (the S-O line); its segment starts DSD in front of
 * its pixel.  Cone beam: all rays start at the source. */
static void ray_start(const orc_grid *g, const orc_view *w, const double Rg[9], const double P[3], double S[3]) {
    if (g->parallel) {
        double e[3] = {w->DSD, 0.0, 0.0}, r[3];
        mv(Rg, e, r);
        for (int k = 0; k < 3; k++) S[k] = P[k] + r[k];
    } else {
        source_pos(w, Rg, S);
    }
}
/* voxel centre X (world) -> continuous detector index (fu,fv) and the weight terms */
typedef struct {
    double fu, fv;
    double depth; /* DSO - X'_x  (scanner frame)            */
    double R, r;  /* |hit - S|, |X - S|                     */
    double cosg;  /* |n.(hit - S)| / R                      */
    int ok;       /* 0 if the voxel is at/behind the source */
} vox_map;
static vox_map voxel_to_det(const orc_grid *g, const orc_view *w, const double Rg[9],
                            const double Rd[9], const double X[3]) {
    vox_map m;
    double Xp[3];
    mtv(Rg, X, Xp);
    Xp[1] += w->COR;
    double Dc[3] = {w->DSO - w->DSD, w->offD[0], w->offD[1]};
    double a[3] = {Xp[0] - Dc[0], Xp[1] - Dc[1], Xp[2] - Dc[2]};
    double b[3] = {w->DSO - Dc[0], 0.0 - Dc[1], 0.0 - Dc[2]};
    double q[3], s[3];
    mtv(Rd, a, q);
    mtv(Rd, b, s);
    if (g->parallel) {
        /* slide the voxel along the ray direction e = R_det^T e_x onto the detector plane q_x = 0 */
        double ex[3] = {1.0, 0.0, 0.0}, e[3];
        mtv(Rd, ex, e);
        double t = q[0] / e[0];
        double u = q[1] - t * e[1], v = q[2] - t * e[2];
        m.fu = (u + 0.5 * g->nu * g->du) / g->du - 0.5;
        m.fv = (v + 0.5 * g->nv * g->dv) / g->dv - 0.5;
        m.depth = w->DSO; /* FDK distance weight (DSO/depth)^2 = 1 */
        m.R = m.r = 1.0;  /* no magnification */
        m.cosg = fabs(e[0]);
        m.ok = 1;
        return m;
    }
    m.depth = w->DSO - Xp[0];
    double den = s[0] - q[0];
    m.ok = (den > 0.0) && (m.depth > 0.0);
    double t = s[0] / den;
    double u = s[1] + t * (q[1] - s[1]);
    double v = s[2] + t * (q[2] - s[2]);
    m.fu = (u + 0.5 * g->nu * g->du) / g->du - 0.5;
    m.fv = (v + 0.5 * g->nv * g->dv) / g->dv - 0.5;
    m.R = sqrt(s[0] * s[0] + (u - s[1]) * (u - s[1]) + (v - s[2]) * (v - s[2]));
    m.r = sqrt((q[0] - s[0]) * (q[0] - s[0]) + (q[1] - s[1]) * (q[1] - s[1]) +
               (q[2] - s[2]) * (q[2] - s[2]));
    m.cosg = fabs(s[0]) / m.R;
    return m;
}
static void voxel_centre(const orc_grid *g, const orc_view *w, int ix, int iy, int iz, double X[3]) {
    X[0] = w->offO[0] + (ix + 0.5) * g->dx - 0.5 * g->nx * g->dx;
    X[1] = w->offO[1] + (iy + 0.5) * g->dy - 0.5 * g->ny * g->dy;
    X[2] = w->offO[2] + (iz + 0.5) * g->dz - 0.5 * g->nz * g->dz;
}

/* ---------------------------------------------------------------- O-A  Siddon, one ray */
static int cmp_d(const void *a, const void *b) {
    double x = *(const double *)a, y = *(const double *)b;
    return (x > y) - (x < y);
}
/* slab method on an axis-aligned box; returns 0 on miss */
static int box_clip(const double S[3], const double d[3], const double b0[3], const double b1[3],
                    double *tin, double *tout) {
    double lo = -INFINITY, hi = INFINITY;
    for (int k = 0; k < 3; k++) {
        if (d[k] == 0.0) {
            if (S[k] < b0[k] || S[k] > b1[k]) return 0;
        } else {
            double t1 = (b0[k] - S[k]) / d[k], t2 = (b1[k] - S[k]) / d[k];
            if (t1 > t2) {
                double t = t1;
                t1 = t2;
                t2 = t;
            }
            if (t1 > lo) lo = t1;
            if (t2 < hi) hi = t2;
        }
    }
    *tin = lo;
    *tout = hi;
    return hi > lo;
}
/* Fills idx[]/len[] (capacity nx+ny+nz+4) with the voxel segments of ray S->P clipped to
 * t in [0,1] (P7).  All plane crossings are collected, sorted, and each consecutive pair is
 * attributed to the voxel containing its midpoint (P8).  Returns the number of segments
 * of non-zero length. */
static int siddon_ray_m(const orc_grid *g, const orc_view *w, const double S[3], const double P[3],
                        double *ts, int64_t *idx, double *len, int *m_out) {
    double d[3] = {P[0] - S[0], P[1] - S[1], P[2] - S[2]};
    double L = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    int n[3] = {g->nx, g->ny, g->nz};
    double h[3] = {g->dx, g->dy, g->dz};
    double b0[3], b1[3];
    for (int k = 0; k < 3; k++) {
        b0[k] = w->offO[k] - 0.5 * n[k] * h[k];
        b1[k] = b0[k] + n[k] * h[k];
    }
    double tin, tout;
    if (!box_clip(S, d, b0, b1, &tin, &tout)) return 0;
    double lo = tin > 0.0 ? tin : 0.0, hi = tout < 1.0 ? tout : 1.0;
    if (!(hi > lo)) return 0;
    int m = 0;
    ts[m++] = lo;
    ts[m++] = hi;
    for (int k = 0; k < 3; k++) {
        if (d[k] == 0.0) continue;
        for (int i = 0; i <= n[k]; i++) {
            double t = (b0[k] + i * h[k] - S[k]) / d[k];
            if (t > lo && t < hi) ts[m++] = t;
        }
    }
    qsort(ts, m, sizeof(double), cmp_d);
    if (m_out) *m_out = m; /* number of sorted crossing parameters left in ts[] (for the knife-edge flags) */
    int ns = 0;
    for (int j = 0; j + 1 < m; j++) {
        double ta = ts[j], tb = ts[j + 1];
        if (!(tb > ta)) continue;
        double tm = 0.5 * (ta + tb);
        int c[3];
        for (int k = 0; k < 3; k++) {
            c[k] = (int)floor((S[k] + tm * d[k] - b0[k]) / h[k]);
            if (c[k] < 0) c[k] = 0;
            if (c[k] > n[k] - 1) c[k] = n[k] - 1;
        }
        idx[ns] = ((int64_t)c[2] * n[1] + c[1]) * n[0] + c[0];
        len[ns] = (tb - ta) * L;
        ns++;
    }
    return ns;
}

static int siddon_ray(const orc_grid *g, const orc_view *w, const double S[3], const double P[3],
                      double *ts, int64_t *idx, double *len) {
    return siddon_ray_m(g, w, S, P, ts, idx, len, NULL);
}

/* ---------------------------------------------------------------- O-B  interpolated, one ray */
/* trilinear interpolant with zero border, xi in index coordinates (voxel centres at integers) */
static double trilinear(const orc_grid *g, arr_t vol, const double xi[3]) {
    int n[3] = {g->nx, g->ny, g->nz};
    int i0[3];
    double f[3];
    for (int k = 0; k < 3; k++) {
        double fl = floor(xi[k]);
        i0[k] = (int)fl;
        f[k] = xi[k] - fl;
    }
    double s = 0.0;
    for (int cz = 0; cz < 2; cz++)
        for (int cy = 0; cy < 2; cy++)
            for (int cx = 0; cx < 2; cx++) {
                int ix = i0[0] + cx, iy = i0[1] + cy, iz = i0[2] + cz;
                if (ix < 0 || ix >= n[0] || iy < 0 || iy >= n[1] || iz < 0 || iz >= n[2]) continue;
                double wgt = (cx ? f[0] : 1.0 - f[0]) * (cy ? f[1] : 1.0 - f[1]) * (cz ? f[2] : 1.0 - f[2]);
                s += wgt * LD(vol, ((size_t)iz * n[1] + iy) * n[0] + ix);
            }
    return s;
}
/* steps 1-5 of SURVEY §8(c) O-B (reading P9).  If scat != NULL the transpose of the same
 * weights is scattered into scat (exact adjoint) with ray value yv. Returns K via *Kout. */
static double interp_ray(const orc_grid *g, const orc_view *w, arr_t vol, const double S[3],
                         const double P[3], double *scat, double yv, int64_t *Kout) {
    double d[3] = {P[0] - S[0], P[1] - S[1], P[2] - S[2]};
    double L = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
    double wd[3] = {d[0] / L, d[1] / L, d[2] / L};
    int n[3] = {g->nx, g->ny, g->nz};
    double h[3] = {g->dx, g->dy, g->dz};
    double c0[3], b0[3], b1[3]; /* c0 = centre of voxel 0; B+ = box grown by half a voxel */
    for (int k = 0; k < 3; k++) {
        double vmin = w->offO[k] - 0.5 * n[k] * h[k];
        c0[k] = vmin + 0.5 * h[k];
        b0[k] = vmin - 0.5 * h[k];
        b1[k] = vmin + n[k] * h[k] + 0.5 * h[k];
    }
    if (Kout) *Kout = 0;
    double lin, lout;
    if (!box_clip(S, wd, b0, b1, &lin, &lout)) return 0.0;
    if (lin < 0.0) lin = 0.0;
    if (lout > L) lout = L;
    if (!(lout > lin)) return 0.0;
    double hmin = h[0] < h[1] ? h[0] : h[1];
    if (h[2] < hmin) hmin = h[2];
    double delta = g->accuracy * hmin;
    int64_t K = (int64_t)ceil((lout - lin) / delta);
    if (Kout) *Kout = K;
    double sum = 0.0;
    for (int64_t k = 0; k < K; k++) {
        double l = lin + (k + 0.5) * delta;
        if (l > L) continue;
        double xi[3];
        for (int a = 0; a < 3; a++) xi[a] = (S[a] + l * wd[a] - c0[a]) / h[a];
        if (!scat) {
            sum += trilinear(g, vol, xi);
        } else {
            int i0[3];
            double f[3];
            for (int a = 0; a < 3; a++) {
                double fl = floor(xi[a]);
                i0[a] = (int)fl;
                f[a] = xi[a] - fl;
            }
            for (int cz = 0; cz < 2; cz++)
                for (int cy = 0; cy < 2; cy++)
                    for (int cx = 0; cx < 2; cx++) {
                        int ix = i0[0] + cx, iy = i0[1] + cy, iz = i0[2] + cz;
                        if (ix < 0 || ix >= n[0] || iy < 0 || iy >= n[1] || iz < 0 || iz >= n[2]) continue;
                        double wgt = (cx ? f[0] : 1.0 - f[0]) * (cy ? f[1] : 1.0 - f[1]) *
                                     (cz ? f[2] : 1.0 - f[2]);
                        scat[((size_t)iz * n[1] + iy) * n[0] + ix] += delta * wgt * yv;
                    }
        }
    }
    return delta * sum;
}

/* ---------------------------------------------------------------- exported: forward projection */
/* mode 0 = Siddon, 1 = interpolated.  ray_ids == NULL: all rays of all views, out[nA*nv*nu];
 * otherwise out[n_rays] for linear ids (ia*nv + iv)*nu + iu.
 * Optional per-ray outputs (may be NULL): nseg (Siddon: non-zero segments; interp: K),
 * first_vox / last_vox (Siddon: linear voxel index of the first/last segment in order of
 * increasing t, -1 if none). */
int orc_ax(const void *vol, int vol_f32, const orc_grid *g, const orc_view *views, int nA, int mode,
           const int64_t *ray_ids, int64_t n_rays, double *out, int64_t *nseg, int64_t *first_vox,
           int64_t *last_vox) {
    arr_t V = {vol, vol_f32};
    int64_t per = (int64_t)g->nu * g->nv;
    int64_t N = ray_ids ? n_rays : per * nA;
    int cap = g->nx + g->ny + g->nz + 8;
#pragma omp parallel
    {
        double *ts = (double *)malloc(sizeof(double) * cap);
        double *len = (double *)malloc(sizeof(double) * cap);
        int64_t *idx = (int64_t *)malloc(sizeof(int64_t) * cap);
#pragma omp for schedule(dynamic, 256)
        for (int64_t r = 0; r < N; r++) {
            int64_t id = ray_ids ? ray_ids[r] : r;
            int ia = (int)(id / per);
            int iv = (int)((id % per) / g->nu), iu = (int)(id % g->nu);
            const orc_view *w = &views[ia];
            double Rg[9], Rd[9], S[3], P[3];
            frames(w, Rg, Rd);
            pixel_pos(g, w, Rg, Rd, iu, iv, P);
            ray_start(g, w, Rg, P, S);
            if (mode == 0) {
                int ns = siddon_ray(g, w, S, P, ts, idx, len);
                double s = 0.0;
                for (int j = 0; j < ns; j++) s += len[j] * LD(V, (size_t)idx[j]);
                out[r] = s;
                if (nseg) nseg[r] = ns;
                if (first_vox) first_vox[r] = ns ? idx[0] : -1;
                if (last_vox) last_vox[r] = ns ? idx[ns - 1] : -1;
            } else {
                int64_t K;
                out[r] = interp_ray(g, w, V, S, P, NULL, 0.0, &K);
                if (nseg) nseg[r] = K;
            }
        }
        free(ts);
        free(len);
        free(idx);
    }
    return 0;
}

/* Index / footprint equality (reading P19(a)): per ray (linear ids as in orc_ax) the number of non-zero segments, the
 * linear voxel index of the first, second, second-to-last and last segment in order of increasing t (-1 if absent), and
 * what a reader needs to call a ray knife-edge: the parameter lengths (t in [0,1] along source -> pixel) of the first and
 * the last segment, and the smallest gap between two consecutive sorted crossing parameters (0 when two planes are
 * crossed at the same point: the ray runs through a voxel edge).  All outputs [n_rays]. */
int orc_siddon_index(const orc_grid *g, const orc_view *views, int nA, const int64_t *ray_ids, int64_t n_rays,
                     int64_t *nseg, int64_t *vox4, double *first_t, double *last_t, double *min_gap) {
    int64_t per = (int64_t)g->nu * g->nv;
    int cap = g->nx + g->ny + g->nz + 8;
    (void)nA;
#pragma omp parallel
    {
        double *ts = (double *)malloc(sizeof(double) * cap);
        double *len = (double *)malloc(sizeof(double) * cap);
        int64_t *idx = (int64_t *)malloc(sizeof(int64_t) * cap);
#pragma omp for schedule(dynamic, 256)
        for (int64_t r = 0; r < n_rays; r++) {
            int64_t id = ray_ids[r];
            int ia = (int)(id / per);
            int iv = (int)((id % per) / g->nu), iu = (int)(id % g->nu);
            const orc_view *w = &views[ia];
            double Rg[9], Rd[9], S[3], P[3];
            frames(w, Rg, Rd);
            pixel_pos(g, w, Rg, Rd, iu, iv, P);
            ray_start(g, w, Rg, P, S);
            int m = 0;
            int ns = siddon_ray_m(g, w, S, P, ts, idx, len, &m);
            double L = sqrt((P[0] - S[0]) * (P[0] - S[0]) + (P[1] - S[1]) * (P[1] - S[1]) + (P[2] - S[2]) * (P[2] - S[2]));
            nseg[r] = ns;
            vox4[4 * r + 0] = ns > 0 ? idx[0] : -1;
            vox4[4 * r + 1] = ns > 1 ? idx[1] : -1;
            vox4[4 * r + 2] = ns > 1 ? idx[ns - 2] : -1;
            vox4[4 * r + 3] = ns > 0 ? idx[ns - 1] : -1;
            first_t[r] = ns > 0 ? len[0] / L : 0.0;
            last_t[r] = ns > 0 ? len[ns - 1] / L : 0.0;
            double mg = INFINITY;
            if (ns > 0)
                for (int j = 0; j + 1 < m; j++)
                    if (ts[j + 1] - ts[j] < mg) mg = ts[j + 1] - ts[j];
            min_gap[r] = mg;
        }
        free(ts);
        free(len);
        free(idx);
    }
    return 0;
}

/* Siddon segments of one ray, for brute-force pins: returns count, fills idx/len (capacity cap) */
int orc_siddon_segments(const orc_grid *g, const orc_view *views, int ia, int iu, int iv,
                        int64_t *idx, double *len, int cap) {
    int need = g->nx + g->ny + g->nz + 8;
    if (cap < need) return -1;
    double *ts = (double *)malloc(sizeof(double) * need);
    const orc_view *w = &views[ia];
    double Rg[9], Rd[9], S[3], P[3];
    frames(w, Rg, Rd);
    pixel_pos(g, w, Rg, Rd, iu, iv, P);
    ray_start(g, w, Rg, P, S);
    int ns = siddon_ray(g, w, S, P, ts, idx, len);
    free(ts);
    return ns;
}

/* exact transposes: ray-driven scatter of the very same weights (P11).  Serial on purpose. */
int orc_atb_exact(const void *proj, int proj_f32, const orc_grid *g, const orc_view *views, int nA,
                  int mode, double *vol_out) {
    arr_t Y = {proj, proj_f32};
    size_t nvox = (size_t)g->nx * g->ny * g->nz;
    memset(vol_out, 0, nvox * sizeof(double));
    int cap = g->nx + g->ny + g->nz + 8;
    double *ts = (double *)malloc(sizeof(double) * cap);
    double *len = (double *)malloc(sizeof(double) * cap);
    int64_t *idx = (int64_t *)malloc(sizeof(int64_t) * cap);
    arr_t none = {NULL, 0};
    for (int ia = 0; ia < nA; ia++) {
        const orc_view *w = &views[ia];
        double Rg[9], Rd[9], S[3], P[3];
        frames(w, Rg, Rd);
        for (int iv = 0; iv < g->nv; iv++)
            for (int iu = 0; iu < g->nu; iu++) {
                double yv = LD(Y, ((size_t)ia * g->nv + iv) * g->nu + iu);
                pixel_pos(g, w, Rg, Rd, iu, iv, P);
                ray_start(g, w, Rg, P, S);
                if (mode == 0) {
                    int ns = siddon_ray(g, w, S, P, ts, idx, len);
                    for (int j = 0; j < ns; j++) vol_out[idx[j]] += len[j] * yv;
                } else {
                    interp_ray(g, w, none, S, P, vol_out, yv, NULL);
                }
            }
    }
    free(ts);
    free(len);
    free(idx);
    return 0;
}

/* ---------------------------------------------------------------- O-C  voxel-driven backprojection */
/* bilinear with taps floor, floor+1 and out-of-range taps = 0 */
static double bilinear(const orc_grid *g, arr_t proj, size_t base, double fu, double fv) {
    double flu = floor(fu), flv = floor(fv);
    int iu = (int)flu, iv = (int)flv;
    double au = fu - flu, av = fv - flv;
    double s = 0.0;
    for (int cv = 0; cv < 2; cv++)
        for (int cu = 0; cu < 2; cu++) {
            int ju = iu + cu, jv = iv + cv;
            if (ju < 0 || ju >= g->nu || jv < 0 || jv >= g->nv) continue;
            s += (cu ? au : 1.0 - au) * (cv ? av : 1.0 - av) * LD(proj, base + (size_t)jv * g->nu + ju);
        }
    return s;
}
/* mode 0 = matched ("pixel-weighted", reading P10):  w = (dx dy dz)/(du dv) * R^2/(r^2 cos g)
 * mode 1 = FDK distance weight:                      w = (DSO/(DSO - X'_x))^2
 * vox_ids == NULL: all voxels, out[nz*ny*nx]; else out[n_vox] for linear ids (iz*ny+iy)*nx+ix.
 * unit_proj != 0: proj is taken as all ones (weights A^T 1) and `proj` is ignored.
 * fuv (may be NULL): [n][nA][2] continuous detector indices, for the footprint checks (P19).
 * Returns -1 if some voxel is at or behind the source plane (geometry error, §8(b)). */
int orc_atb(const void *proj, int proj_f32, int unit_proj, const orc_grid *g, const orc_view *views,
            int nA, int mode, const int64_t *vox_ids, int64_t n_vox, double *out, double *fuv) {
    arr_t Y = {proj, proj_f32};
    int64_t N = vox_ids ? n_vox : (int64_t)g->nx * g->ny * g->nz;
    size_t per = (size_t)g->nu * g->nv;
    int bad = 0;
    double *Rgs = (double *)malloc(sizeof(double) * 18 * (size_t)nA);
    for (int ia = 0; ia < nA; ia++) frames(&views[ia], Rgs + 18 * ia, Rgs + 18 * ia + 9);
    double cvol = (g->dx * g->dy * g->dz) / (g->du * g->dv);
#pragma omp parallel for schedule(dynamic, 1024) reduction(| : bad)
    for (int64_t j = 0; j < N; j++) {
        int64_t id = vox_ids ? vox_ids[j] : j;
        int ix = (int)(id % g->nx), iy = (int)((id / g->nx) % g->ny), iz = (int)(id / ((int64_t)g->nx * g->ny));
        double acc = 0.0;
        for (int ia = 0; ia < nA; ia++) {
            const orc_view *w = &views[ia];
            double X[3];
            voxel_centre(g, w, ix, iy, iz, X);
            vox_map m = voxel_to_det(g, w, Rgs + 18 * ia, Rgs + 18 * ia + 9, X);
            if (!m.ok) {
                bad |= 1;
                continue;
            }
            double wgt = (mode == 1) ? (w->DSO / m.depth) * (w->DSO / m.depth)
                                     : cvol * (m.R * m.R) / (m.r * m.r * m.cosg);
            double val;
            if (unit_proj) {
                /* bilinear of an all-ones image with zero border = sum of in-range tap weights */
                double flu = floor(m.fu), flv = floor(m.fv);
                int iu = (int)flu, iv = (int)flv;
                double au = m.fu - flu, av = m.fv - flv;
                val = 0.0;
                for (int cv = 0; cv < 2; cv++)
                    for (int cu = 0; cu < 2; cu++) {
                        int ju = iu + cu, jv = iv + cv;
                        if (ju < 0 || ju >= g->nu || jv < 0 || jv >= g->nv) continue;
                        val += (cu ? au : 1.0 - au) * (cv ? av : 1.0 - av);
                    }
            } else {
                val = bilinear(g, Y, (size_t)ia * per, m.fu, m.fv);
            }
            acc += wgt * val;
            if (fuv) {
                fuv[((size_t)j * nA + ia) * 2 + 0] = m.fu;
                fuv[((size_t)j * nA + ia) * 2 + 1] = m.fv;
            }
        }
        out[j] = acc;
    }
    free(Rgs);
    return bad ? -1 : 0;
}

/* ---------------------------------------------------------------- O-D  FDK pre-filter (P12) */
/* per projection: p1 = p * DSD/sqrt(DSD^2+u^2+v^2); q = tau * (p1 * h) along u, direct linear
 * convolution with zero padding, tau = du*DSO/DSD, h[0]=1/(4 tau^2), h[odd n] = -1/(pi n tau)^2.
 * (u,v) are measured from the foot of the source's perpendicular on the detector plane (the principal ray of the
 * textbook derivation [24]): detector-local pixel-centre coordinates PLUS offDetector (reading P34; the weight is the
 * cosine between the ray and the detector normal; rotDetector is not taken into it). */
int orc_fdk_filter(const void *proj, int proj_f32, const orc_grid *g, const orc_view *views, int nA,
                   double *out) {
    arr_t Y = {proj, proj_f32};
    int nu = g->nu, nv = g->nv;
#pragma omp parallel
    {
        double *row = (double *)malloc(sizeof(double) * nu);
#pragma omp for collapse(2) schedule(dynamic, 8)
        for (int ia = 0; ia < nA; ia++)
            for (int iv = 0; iv < nv; iv++) {
                const orc_view *w = &views[ia];
                double tau = g->parallel ? g->du : g->du * w->DSO / w->DSD; /* P29: no magnification */
                double v = (iv + 0.5) * g->dv - 0.5 * nv * g->dv + w->offD[1];
                size_t base = ((size_t)ia * nv + iv) * nu;
                for (int iu = 0; iu < nu; iu++) {
                    double u = (iu + 0.5) * g->du - 0.5 * nu * g->du + w->offD[0];
                    row[iu] = LD(Y, base + iu) * (g->parallel ? 1.0 : w->DSD / sqrt(w->DSD * w->DSD + u * u + v * v));
                }
                for (int iu = 0; iu < nu; iu++) {
                    double s = row[iu] / (4.0 * tau * tau);
                    for (int ju = 0; ju < nu; ju++) {
                        int n = iu - ju;
                        if (n & 1) s -= row[ju] / (M_PI * M_PI * (double)n * (double)n * tau * tau);
                    }
                    out[base + iu] = tau * s;
                }
            }
        free(row);
    }
    return 0;
}

/* geometry probes for the pins: world positions of the source and of a pixel centre, and the
 * voxel -> detector map of one voxel centre */
void orc_source_pixel(const orc_grid *g, const orc_view *views, int ia, double iu, double iv,
                      double S[3], double P[3]) {
    double Rg[9], Rd[9];
    frames(&views[ia], Rg, Rd);
    pixel_pos(g, &views[ia], Rg, Rd, iu, iv, P);
    ray_start(g, &views[ia], Rg, P, S);
}
void orc_voxel_map(const orc_grid *g, const orc_view *views, int ia, int ix, int iy, int iz,
                   double X[3], double fuv[2]) {
    double Rg[9], Rd[9];
    frames(&views[ia], Rg, Rd);
    voxel_centre(g, &views[ia], ix, iy, iz, X);
    vox_map m = voxel_to_det(g, &views[ia], Rg, Rd, X);
    fuv[0] = m.fu;
    fuv[1] = m.fv;
}
/* measurement plumbing for bench.py's cpu_baseline (all hardware threads and single thread): no arithmetic */
void orc_set_num_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int orc_num_threads(void) {
    int n = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        n = omp_get_num_threads();
    }
#endif
    return n;
}
