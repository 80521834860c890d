// geometry.cu — host-side fp64 geometry precompute.
// PAPER.md:543-566 Table B1; §2.4; readings P1-P6 of DESIGN.md:
//   default pose  S0 = (DSO,0,0), detector centre D0 = (DSO-DSD,0,0), e_u = +y, e_v = +z   (P2)
//   R_det = Rz(psi) Ry(theta) Rx(phi) about the shifted detector centre                      (P3)
//   offDetector is applied in the unrotated uv frame                                         (P4)
//   COR moves source and detector by (0,-COR,0) in the scanner frame                         (P5)
//   gantry R_g = Rz(z1) Ry(y1) Rz(z2), applied to scanner-frame points                       (P6)
#include <cmath>
#include <cstring>
#include "common.cuh"

namespace tg {

namespace {
struct M3 {
    double m[3][3];
};
M3 mul(const M3& a, const M3& b) {
    M3 c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c.m[i][j] = a.m[i][0] * b.m[0][j] + a.m[i][1] * b.m[1][j] + a.m[i][2] * b.m[2][j];
    return c;
}
M3 transpose(const M3& a) {
    M3 c;
    for (int i = 0; i < 3; ++i)
        for (int j = 0; j < 3; ++j) c.m[i][j] = a.m[j][i];
    return c;
}
void apply(const M3& a, const double x[3], double y[3]) {
    double t[3];
    for (int i = 0; i < 3; ++i) t[i] = a.m[i][0] * x[0] + a.m[i][1] * x[1] + a.m[i][2] * x[2];
    y[0] = t[0], y[1] = t[1], y[2] = t[2];
}
M3 Rx(double a) { return M3{{{1, 0, 0}, {0, std::cos(a), -std::sin(a)}, {0, std::sin(a), std::cos(a)}}}; }
M3 Ry(double a) { return M3{{{std::cos(a), 0, std::sin(a)}, {0, 1, 0}, {-std::sin(a), 0, std::cos(a)}}}; }
M3 Rz(double a) { return M3{{{std::cos(a), -std::sin(a), 0}, {std::sin(a), std::cos(a), 0}, {0, 0, 1}}}; }
M3 gantry(const ViewH& v) { return mul(mul(Rz(v.ang[0]), Ry(v.ang[1])), Rz(v.ang[2])); }
M3 detrot(const ViewH& v) { return mul(mul(Rz(v.rotD[2]), Ry(v.rotD[1])), Rx(v.rotD[0])); }
}  // namespace

Grid make_grid(const tigre_geo* geo) {
    Grid g;
    g.nx = geo->nVoxel[0], g.ny = geo->nVoxel[1], g.nz = geo->nVoxel[2];
    g.nu = geo->nDetector[0], g.nv = geo->nDetector[1];
    g.dx = geo->dVoxel[0], g.dy = geo->dVoxel[1], g.dz = geo->dVoxel[2];
    g.du = geo->dDetector[0], g.dv = geo->dDetector[1];
    g.accuracy = geo->accuracy;
    return g;
}

void resolve_views(const tigre_geo* geo, const double* angles, int nA, std::vector<ViewH>& out) {
    out.resize(nA);
    for (int a = 0; a < nA; ++a) {
        ViewH& v = out[a];
        v.DSD = geo->DSD_a ? geo->DSD_a[a] : geo->DSD;
        v.DSO = geo->DSO_a ? geo->DSO_a[a] : geo->DSO;
        v.COR = geo->COR_a ? geo->COR_a[a] : geo->COR;
        for (int k = 0; k < 3; ++k) v.offO[k] = geo->offOrigin_a ? geo->offOrigin_a[3 * a + k] : geo->offOrigin[k];
        for (int k = 0; k < 2; ++k) v.offD[k] = geo->offDetector_a ? geo->offDetector_a[2 * a + k] : geo->offDetector[k];
        for (int k = 0; k < 3; ++k) v.rotD[k] = geo->rotDetector_a ? geo->rotDetector_a[3 * a + k] : geo->rotDetector[k];
        for (int k = 0; k < 3; ++k) v.ang[k] = angles[3 * a + k];
        v.parallel = geo->mode == TIGRE_GEO_PARALLEL;
    }
}

int validate_geo(const tigre_geo* geo, const double* angles, int nA) {
    if (!geo || !angles || nA <= 0) return TIGRE_ERR_ARG;
    if (geo->struct_size != sizeof(tigre_geo)) return TIGRE_ERR_ARG;
    for (int k = 0; k < 3; ++k)
        if (geo->nVoxel[k] <= 0 || !(geo->dVoxel[k] > 0.0)) return TIGRE_ERR_GEOMETRY;
    for (int k = 0; k < 2; ++k)
        if (geo->nDetector[k] <= 0 || !(geo->dDetector[k] > 0.0)) return TIGRE_ERR_GEOMETRY;
    if (!(geo->accuracy > 0.0)) return TIGRE_ERR_GEOMETRY;
    if (geo->mode != TIGRE_GEO_CONE && geo->mode != TIGRE_GEO_PARALLEL) return TIGRE_ERR_GEOMETRY;
    for (int a = 0; a < nA; ++a) {
        double dsd = geo->DSD_a ? geo->DSD_a[a] : geo->DSD;
        double dso = geo->DSO_a ? geo->DSO_a[a] : geo->DSO;
        if (!(dsd > 0.0) || !(dso > 0.0)) return TIGRE_ERR_GEOMETRY;
    }
    return TIGRE_OK;
}

void build_ray_view(const Grid& g, const ViewH& v, RayView& r) {
    const M3 Rg = gantry(v), Rd = detrot(v);
    const double h[3] = {g.dx, g.dy, g.dz};
    const int n[3] = {g.nx, g.ny, g.nz};
    double vmin[3];
    for (int k = 0; k < 3; ++k) vmin[k] = v.offO[k] - 0.5 * n[k] * h[k];
    // scanner-frame source / pixel (0,0) centre / pixel steps
    const double S1[3] = {v.DSO, -v.COR, 0.0};
    const double u0 = 0.5 * g.du - 0.5 * g.nu * g.du, v0 = 0.5 * g.dv - 0.5 * g.nv * g.dv;
    double loc0[3] = {0.0, u0, v0}, eu[3] = {0.0, g.du, 0.0}, ev[3] = {0.0, 0.0, g.dv};
    double r0[3], ru[3], rv[3];
    apply(Rd, loc0, r0);
    apply(Rd, eu, ru);
    apply(Rd, ev, rv);
    const double p1[3] = {v.DSO - v.DSD + r0[0], v.offD[0] + r0[1] - v.COR, v.offD[1] + r0[2]};
    double S[3], P[3], dU[3], dV[3];
    apply(Rg, S1, S);
    apply(Rg, p1, P);
    apply(Rg, ru, dU);
    apply(Rg, rv, dV);
    if (v.parallel) {   // P29: the ray of a pixel starts DSD in front of it along the gantry-rotated x axis
        const double e1[3] = {v.DSD, 0.0, 0.0};
        double e[3];
        apply(Rg, e1, e);
        for (int k = 0; k < 3; ++k) S[k] = P[k] + e[k];
    }
    for (int k = 0; k < 3; ++k) {
        r.S[k] = (S[k] - vmin[k]) / h[k];
        r.P0[k] = (P[k] - vmin[k]) / h[k];
        r.dU[k] = dU[k] / h[k];
        r.dV[k] = dV[k] / h[k];
        r.dSU[k] = v.parallel ? r.dU[k] : 0.0;
        r.dSV[k] = v.parallel ? r.dV[k] : 0.0;
    }
}

// fp64 rows of the voxel -> detector map of one view (see VoxView in common.cuh); also the detector-frame
// source s (s[0] = distance source -> detector plane) and the scanner-frame x of the volume centre.
struct VoxRows {
    double rowU[4], rowV[4], rowW[4], rowG[4], s[3];
};
static int build_vox_rows(const Grid& g, const ViewH& v, VoxRows& R) {
    const M3 RgT = transpose(gantry(v)), RdT = transpose(detrot(v));
    const double h[3] = {g.dx, g.dy, g.dz};
    // q(c) = M c + q0 : detector-frame position of the voxel with centred index c
    M3 D = {{{h[0], 0, 0}, {0, h[1], 0}, {0, 0, h[2]}}};
    const M3 A = mul(RgT, D);        // scanner-frame X' = A c + RgT offO + (0,COR,0)
    const M3 M = mul(RdT, A);
    double xo[3];
    apply(RgT, v.offO, xo);
    xo[1] += v.COR;
    const double Dc[3] = {v.DSO - v.DSD, v.offD[0], v.offD[1]};
    double a0[3] = {xo[0] - Dc[0], xo[1] - Dc[1], xo[2] - Dc[2]}, q0[3];
    apply(RdT, a0, q0);
    double b0[3] = {v.DSO - Dc[0], -Dc[1], -Dc[2]};
    double* s = R.s;
    apply(RdT, b0, s);
    double *rowW = R.rowW, *rowU = R.rowU, *rowV = R.rowV, *rowG = R.rowG;
    if (v.parallel) {
        // P29: slide the voxel along the ray direction e = R_det^T e_x onto the detector plane q_x = 0: an affine map (W = 1)
        const double ex[3] = {1.0, 0.0, 0.0};
        double e[3];
        apply(RdT, ex, e);
        if (!(std::fabs(e[0]) > 1e-9)) return TIGRE_ERR_GEOMETRY;
        const double oU = 0.5 * (g.nu - 1) - (double)(g.nu / 2), oV = 0.5 * (g.nv - 1) - (double)(g.nv / 2);
        for (int k = 0; k < 3; ++k) {
            rowW[k] = 0.0, rowG[k] = 0.0;
            rowU[k] = (M.m[1][k] - e[1] / e[0] * M.m[0][k]) / g.du;
            rowV[k] = (M.m[2][k] - e[2] / e[0] * M.m[0][k]) / g.dv;
        }
        rowW[3] = 1.0, rowG[3] = 1.0;
        rowU[3] = (q0[1] - e[1] / e[0] * q0[0]) / g.du + oU;
        rowV[3] = (q0[2] - e[2] / e[0] * q0[0]) / g.dv + oV;
        s[0] = std::fabs(e[0]), s[1] = 0.0, s[2] = 0.0;   // s[0] carries the cosine between ray and detector normal
        return TIGRE_OK;
    }
    if (!(s[0] > 0.0)) return TIGRE_ERR_GEOMETRY;
    for (int k = 0; k < 3; ++k) rowW[k] = -M.m[0][k] / s[0];
    rowW[3] = 1.0 - q0[0] / s[0];
    // u*W = s_y*W + (q_y - s_y);  fu = u/du + (nu-1)/2;  fuh = fu - nu/2 = u/du + offU
    const double offU = 0.5 * (g.nu - 1) - (double)(g.nu / 2), offV = 0.5 * (g.nv - 1) - (double)(g.nv / 2);
    for (int k = 0; k < 3; ++k) rowU[k] = (s[1] * rowW[k] + M.m[1][k]) / g.du + offU * rowW[k];
    rowU[3] = (s[1] * rowW[3] + q0[1] - s[1]) / g.du + offU * rowW[3];
    for (int k = 0; k < 3; ++k) rowV[k] = (s[2] * rowW[k] + M.m[2][k]) / g.dv + offV * rowW[k];
    rowV[3] = (s[2] * rowW[3] + q0[2] - s[2]) / g.dv + offV * rowW[3];
    for (int k = 0; k < 3; ++k) rowG[k] = -A.m[0][k] / v.DSO;
    rowG[3] = (v.DSO - xo[0]) / v.DSO;
    return TIGRE_OK;
}

// Detector rows [row0, row0+nrows) that the z-slices [z0, z0+nzs) of the volume can reach in view v:
// the projective map is quasi-linear where W > 0, so the extrema of fv over the slab box (grown by one
// voxel: trilinear support, bilinear taps) are at its corners.  Any corner at W <= 0: all rows.
void row_band(const Grid& g, const ViewH& v, int z0, int nzs, int& row0, int& nrows) {
    row0 = 0, nrows = g.nv;
    VoxRows R;
    if (build_vox_rows(g, v, R) != TIGRE_OK) return;
    const double cx = 0.5 * g.nx + 1.0, cy = 0.5 * g.ny + 1.0;
    const double za = (double)z0 - 0.5 * g.nz - 1.0, zb = (double)(z0 + nzs) - 0.5 * g.nz + 1.0;
    double lo = 1e300, hi = -1e300;
    for (int i = 0; i < 8; ++i) {
        const double c[3] = {(i & 1) ? cx : -cx, (i & 2) ? cy : -cy, (i & 4) ? zb : za};
        const double W = R.rowW[0] * c[0] + R.rowW[1] * c[1] + R.rowW[2] * c[2] + R.rowW[3];
        const double V = R.rowV[0] * c[0] + R.rowV[1] * c[1] + R.rowV[2] * c[2] + R.rowV[3];
        if (!(W > 1e-9)) return;
        lo = std::fmin(lo, V / W), hi = std::fmax(hi, V / W);
    }
    // fv = (V/W) + nv/2 is the continuous row index; taps floor(fv), floor(fv)+1; one row of slack
    const double a = std::floor(lo + (double)(g.nv / 2)) - 1.0, b = std::ceil(hi + (double)(g.nv / 2)) + 2.0;
    const int r0 = (int)std::fmax(0.0, std::fmin(a, (double)g.nv)), r1 = (int)std::fmax(0.0, std::fmin(b, (double)g.nv));
    row0 = r0, nrows = r1 > r0 ? r1 - r0 : 0;
}

int build_vox_view(const Grid& g, const ViewH& v, VoxView& o) {
    VoxRows R;
    TG_TRY(build_vox_rows(g, v, R));
    const double *rowW = R.rowW, *rowU = R.rowU, *rowV = R.rowV, *rowG = R.rowG, *s = R.s;
    const double offU = 0.5 * (g.nu - 1) - (double)(g.nu / 2), offV = 0.5 * (g.nv - 1) - (double)(g.nv / 2);
    // every corner of the volume box must be in front of the source (W>0, G>0)
    const double cx = 0.5 * g.nx, cy = 0.5 * g.ny, cz = 0.5 * g.nz;
    for (int i = 0; i < 8; ++i) {
        const double c[3] = {(i & 1) ? cx : -cx, (i & 2) ? cy : -cy, (i & 4) ? cz : -cz};
        const double W = rowW[0] * c[0] + rowW[1] * c[1] + rowW[2] * c[2] + rowW[3];
        const double G = rowG[0] * c[0] + rowG[1] * c[1] + rowG[2] * c[2] + rowG[3];
        if (!(W > 0.0) || !(G > 0.0)) return TIGRE_ERR_GEOMETRY;
    }
    for (int k = 0; k < 4; ++k) {
        o.rowU[k] = (float)rowU[k];
        o.rowV[k] = (float)rowV[k];
        o.rowW[k] = (float)rowW[k];
        o.rowG[k] = (float)rowG[k];
    }
    if (v.parallel) {
        // constant matched weight dVoxel^3 / (du dv cos) through the SAME kernel arithmetic  km t^2 sqrt(sx2 + du^2 eu^2 +
        // dv^2 ev^2)  (t = 1): sx2 = 2^100 absorbs the other terms exactly in fp32, sqrt(2^100) = 2^50
        o.km = (float)((g.dx * g.dy * g.dz) / (g.du * g.dv) / s[0] / 1125899906842624.0);
        o.sx2 = 1.2676506002282294e30f;
        o.fus = 0.f, o.fvs = 0.f;
        return TIGRE_OK;
    }
    o.km = (float)((g.dx * g.dy * g.dz) / (g.du * g.dv) / s[0]);
    o.sx2 = (float)(s[0] * s[0]);
    o.fus = (float)(s[1] / g.du + offU);
    o.fvs = (float)(s[2] / g.dv + offV);
    return TIGRE_OK;
}

}  // namespace tg
