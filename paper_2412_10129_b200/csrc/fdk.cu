// fdk.cu — the FDK pre-filter (reading P12) and the FDK variants (section 8(f).4; "various filter types and geometric correction methods,
// such as Wang [25] and Parker [26] weights", 281, 359; readings P26-P28).
//
// Filters: the Ram-Lak taps (P12) windowed in frequency on L = 2^ceil(log2(2 nu)) samples.  The product of the taps'
// spectrum with the window is transformed back ON THE HOST (fp64, direct cosine sums: the spectrum is real and even) into
// nu spatial taps for tau = 1; the device then applies them as a direct linear convolution of the zero-padded row, which
// equals the FFT formulation exactly (L >= 2 nu: no wrap) and keeps the kernel free of an FFT dependency.
// Weights: Parker (short scan) and Wang (displaced detector) are per-view, per-column factors built on the host in
// fp64 and multiplied into the cosine-weighted row before the convolution.
#include <algorithm>
#include <cmath>
#include <mutex>
#include <vector>
#include "common.cuh"

namespace tg {

namespace {

// q[iu] = (1/tau) * sum_m row[m] * taps[|iu - m|],  row = b * cosine weight * colw: one CTA per detector row and view.
// The convolution is a dense contraction of nu^2 multiply-adds per row (C3: 2.9e11 per FDK), so it is laid out for the FMA
// pipe: a thread owns FR = 8 consecutive outputs and slides a register window of 8 row values past them, one new value per
// tap index n on each side, so a tap costs ONE broadcast shared-memory load (two LDS.128 per 8 taps) plus one row load per
// side for 16 FMAs.  The row sits in shared memory split into FR planes by (index mod FR), zero-padded on both sides: the
// threads of a warp (consecutive groups of outputs) then read consecutive words of one plane (no bank conflicts) and the
// row's ends need no tests.  ODD = true: Ram-Lak without a window (taps vanish at even n != 0): even n only shift the window.
// taps == NULL: the Ram-Lak taps of reading P12 are formed in the kernel.
constexpr int FR = 8;

__host__ __device__ constexpr int mod8(int x) { return ((x % FR) + FR) % FR; }
__host__ __device__ constexpr int fdiv8(int x) { return (x - mod8(x)) / FR; }

// acc[j] += sum_{d >= 0} T[d] * (src[i0 + A + j - d] + src[i0 + AR + j + d]),  j = 0..7, for an 8-aligned i0: the left window
// runs over taps d <= 8 mL + 7, the right one over d <= 8 mR + 7 (negative: side absent).  src is stored in FR planes by
// (index mod FR), element e at plane e mod FR, offset (e + PAD) / FR; ob = (i0 + PAD) / FR.  A, AR are compile-time so that every
// plane index is: each tap costs one row load per side (consecutive words across the threads of a warp: no bank
// conflict), one broadcast tap (two LDS.128 per 8 taps) and 16 FMAs.
template <int A, int AR>
__device__ __forceinline__ void conv8(const float* __restrict__ src, int PL, int ob, const float* __restrict__ T, int mL, int mR,
                                      float (&acc)[FR]) {
    float L[FR], R[FR];
#pragma unroll
    for (int j = 0; j < FR; ++j) {
        L[j] = src[mod8(A + j) * PL + ob + fdiv8(A + j)];
        R[j] = src[mod8(AR + j) * PL + ob + fdiv8(AR + j)];
    }
    for (int m = 0; m <= mL; ++m) {
        const float4 ta = *reinterpret_cast<const float4*>(T + FR * m), tb = *reinterpret_cast<const float4*>(T + FR * m + 4);
        const float t[FR] = {ta.x, ta.y, ta.z, ta.w, tb.x, tb.y, tb.z, tb.w};
#pragma unroll
        for (int k = 0; k < FR; ++k) {   // tap d = FR * m + k
#pragma unroll
            for (int j = 0; j < FR; ++j) acc[j] = fmaf(t[k], L[j], acc[j]);
#pragma unroll
            for (int j = FR - 1; j > 0; --j) L[j] = L[j - 1];
            L[0] = src[mod8(A - k - 1) * PL + ob - m + fdiv8(A - k - 1)];          // src[i0 + A - (d + 1)]
        }
    }
    for (int m = 0; m <= mR; ++m) {
        const float4 ta = *reinterpret_cast<const float4*>(T + FR * m), tb = *reinterpret_cast<const float4*>(T + FR * m + 4);
        const float t[FR] = {ta.x, ta.y, ta.z, ta.w, tb.x, tb.y, tb.z, tb.w};
#pragma unroll
        for (int k = 0; k < FR; ++k) {
#pragma unroll
            for (int j = 0; j < FR; ++j) acc[j] = fmaf(t[k], R[j], acc[j]);
#pragma unroll
            for (int j = 0; j < FR - 1; ++j) R[j] = R[j + 1];
            R[FR - 1] = src[mod8(AR + k) * PL + ob + m + 1 + fdiv8(AR + k)];       // src[i0 + AR + FR - 1 + (d + 1)]
        }
    }
}

// ODD = false: every tap (windowed filters).  The centre tap is applied separately and T[0] = 0, so both windows start at the
//              output's own position (A = AR = 0).
// ODD = true:  Ram-Lak without a window: the taps vanish at even n != 0, so an output of one parity reads only row elements of
//              the other parity.  The row is stored as two half-rows X0[m] = row[2m], X1[m] = row[2m + 1] and the taps as
//              T[d] = tap[2d + 1]: output 2j reads X1[j - 1 - d] and X1[j + d], output 2j + 1 reads X0[j - d] and X0[j + 1 + d]:
//              two dense half-length convolutions (no skipped taps).
template <bool ODD>
__global__ void __launch_bounds__(128)
fdk_conv_kernel(const float* __restrict__ b, int nu, int nv, float du, float dv, const double* __restrict__ dsd_a,
                const double* __restrict__ dso_a, const double* __restrict__ offd_a, const float* __restrict__ taps,
                const float* __restrict__ colw, float* __restrict__ q, int PAD, int PL, int NT) {
    extern __shared__ __align__(16) float sm[];
    float* tp = sm;              // [NT]  taps (ODD: T[d] = tap[2d + 1]; else tap[n] with tp[0] = 0), zero beyond the row
    float* rw = sm + NT;         // [FR][PL] planes of the row (ODD: [2][FR][PL], the two half-rows)
    const int iv = blockIdx.x, ia = blockIdx.y;
    const float DSD = (float)dsd_a[ia], DSO = (float)dso_a[ia];
    const float itau = DSD / (du * DSO);
    // reading P34: the cosine weight is centred on the principal ray: local pixel coordinates plus offDetector
    const float offu = offd_a ? (float)offd_a[2 * ia] : 0.f, offv = offd_a ? (float)offd_a[2 * ia + 1] : 0.f;
    const float v = ((float)iv + 0.5f) * dv - 0.5f * (float)nv * dv + offv;
    const size_t base = ((size_t)ia * nv + iv) * nu;
    const int nplanes = (ODD ? 2 : 1) * FR * PL;
    for (int i = threadIdx.x; i < nplanes; i += blockDim.x) rw[i] = 0.f;
    for (int n = threadIdx.x; n < NT; n += blockDim.x) {
        const int src = ODD ? 2 * n + 1 : n;
        float t = 0.f;
        if (src >= 1 && src < nu) t = taps ? __ldg(taps + src) : ((src & 1) ? -1.0f / (9.8696044010893586f * (float)src * (float)src) : 0.f);
        tp[n] = t;
    }
    const float tap0 = taps ? __ldg(taps) : 0.25f;
    __syncthreads();
    for (int iu = threadIdx.x; iu < nu; iu += blockDim.x) {
        const float u = ((float)iu + 0.5f) * du - 0.5f * (float)nu * du + offu;
        float r = __ldg(b + base + iu) * DSD * rsqrtf(DSD * DSD + u * u + v * v);
        if (colw) r *= __ldg(colw + (size_t)ia * nu + iu);
        if (ODD) {
            const int m = iu >> 1;
            rw[(iu & 1) * FR * PL + (m % FR) * PL + (m + PAD) / FR] = r;
        } else {
            rw[(iu % FR) * PL + (iu + PAD) / FR] = r;
        }
    }
    __syncthreads();
    if (!ODD) {
        for (int c = threadIdx.x; c * FR < nu; c += blockDim.x) {
            const int i0 = c * FR, ob = (i0 + PAD) / FR;
            float acc[FR];
#pragma unroll
            for (int j = 0; j < FR; ++j) acc[j] = tap0 * rw[j * PL + ob];
            conv8<0, 0>(rw, PL, ob, tp, (i0 + FR - 1) / FR, (nu - 1 - i0) / FR, acc);
#pragma unroll
            for (int j = 0; j < FR; ++j)
                if (i0 + j < nu) q[base + i0 + j] = acc[j] * itau;
        }
    } else {
        const int n0 = (nu + 1) >> 1, n1 = nu >> 1;          // lengths of X0 (even elements) and X1 (odd elements)
        const int C0 = (n0 + FR - 1) / FR, C1 = (n1 + FR - 1) / FR;
        const float* X0 = rw;
        const float* X1 = rw + FR * PL;
        for (int id = threadIdx.x; id < C0 + C1; id += blockDim.x) {
            const int par = id >= C0, j0 = (par ? id - C0 : id) * FR, ob = (j0 + PAD) / FR;
            float acc[FR];
            if (!par) {   // outputs 2j: own half-row X0, neighbours in X1 at j - 1 - d and j + d
#pragma unroll
                for (int j = 0; j < FR; ++j) acc[j] = tap0 * X0[j * PL + ob];
                const int last = n1 - 1 - j0;
                conv8<-1, 0>(X1, PL, ob, tp, (j0 + FR - 2) / FR, last >= 0 ? last / FR : -1, acc);
            } else {      // outputs 2j + 1: own half-row X1, neighbours in X0 at j - d and j + 1 + d
#pragma unroll
                for (int j = 0; j < FR; ++j) acc[j] = tap0 * X1[j * PL + ob];
                const int last = n0 - 2 - j0;
                conv8<0, 1>(X0, PL, ob, tp, (j0 + FR - 1) / FR, last >= 0 ? last / FR : -1, acc);
            }
#pragma unroll
            for (int j = 0; j < FR; ++j) {
                const int i = 2 * (j0 + j) + par;
                if (i < nu) q[base + i] = acc[j] * itau;
            }
        }
    }
}

// curved -> flat detector (reading P30): flat pixel (u, v) reads the curved image at arc length DSD atan(u/DSD) and height
// v cos(atan(u/DSD)), bilinear, zero outside.  One thread per flat pixel; per-column quantities are recomputed (cheap).
__global__ void __launch_bounds__(256)
flatten_kernel(const float* __restrict__ curved, int nu, int nv, float du, float dv, const double* __restrict__ dsd_a,
               float* __restrict__ flat, size_t total) {
    const size_t per = (size_t)nu * nv;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < total; i += (size_t)gridDim.x * blockDim.x) {
        const size_t ia = i / per;
        const int r = (int)(i - ia * per), iv = r / nu, iu = r - iv * nu;
        const float DSD = (float)dsd_a[ia];
        const float u = ((float)iu + 0.5f) * du - 0.5f * (float)nu * du;
        const float v = ((float)iv + 0.5f) * dv - 0.5f * (float)nv * dv;
        const float gamma = atanf(u / DSD);
        const float fi = (DSD * gamma + 0.5f * (float)nu * du) / du - 0.5f;
        const float fj = (v * cosf(gamma) + 0.5f * (float)nv * dv) / dv - 0.5f;
        const float fli = floorf(fi), flj = floorf(fj);
        const int i0 = (int)fli, j0 = (int)flj;
        const float ai = fi - fli, aj = fj - flj;
        const float* src = curved + ia * per;
        float acc = 0.f;
#pragma unroll
        for (int cj = 0; cj < 2; ++cj)
#pragma unroll
            for (int ci = 0; ci < 2; ++ci) {
                const int ii = i0 + ci, jj = j0 + cj;
                if ((unsigned)ii < (unsigned)nu && (unsigned)jj < (unsigned)nv)
                    acc = fmaf((ci ? ai : 1.f - ai) * (cj ? aj : 1.f - aj), __ldg(src + (size_t)jj * nu + ii), acc);
            }
        flat[i] = acc;
    }
}

double window_at(int filter, double om) {
    switch (filter) {
        case TIGRE_FILTER_SHEPP_LOGAN: return om > 0.0 ? std::sin(0.5 * om) / (0.5 * om) : 1.0;
        case TIGRE_FILTER_COSINE: return std::cos(0.5 * om);
        case TIGRE_FILTER_HAMMING: return 0.54 + 0.46 * std::cos(om);
        case TIGRE_FILTER_HANN: return 0.5 + 0.5 * std::cos(om);
        default: return 1.0;
    }
}

}  // namespace

// taps for tau = 1 (the kernel scales by 1/tau: h ~ 1/tau^2, times the tau of the quadrature).  The windowed taps cost two
// O(nu L) cosine sums on the host (4 ms for nu = 1024, while the tensor-core filter of a whole C3 scan takes 7): the last
// (nu, filter) pair is kept.
static void fdk_filter_taps_compute(int nu, int filter, std::vector<double>& g);
void fdk_filter_taps(int nu, int filter, std::vector<double>& g) {
    static std::mutex mu;
    static int c_nu = -1, c_filter = -1;
    static std::vector<double> cache;
    std::lock_guard<std::mutex> lk(mu);
    if (nu != c_nu || filter != c_filter) {
        fdk_filter_taps_compute(nu, filter, cache);
        c_nu = nu, c_filter = filter;
    }
    g = cache;
}
static void fdk_filter_taps_compute(int nu, int filter, std::vector<double>& g) {
    g.assign(nu, 0.0);
    if (filter == TIGRE_FILTER_RAM_LAK) {
        g[0] = 0.25;
        for (int n = 1; n < nu; n += 2) g[n] = -1.0 / (M_PI * M_PI * (double)n * (double)n);
        return;
    }
    int L = 1;
    while (L < 2 * nu) L <<= 1;
    const int half = L / 2;
    std::vector<double> ct(L);
    for (int j = 0; j < L; ++j) ct[j] = std::cos(2.0 * M_PI * (double)j / (double)L);
    std::vector<double> HW(half + 1);
    for (int k = 0; k <= half; ++k) {
        double s = 0.0;
        for (int n = 1; n < half; n += 2) s += -1.0 / (M_PI * M_PI * (double)n * (double)n) * ct[(size_t)((long long)k * n % L)];
        HW[k] = (0.25 + 2.0 * s) * window_at(filter, 2.0 * M_PI * (double)k / (double)L);
    }
    for (int m = 0; m < nu; ++m) {
        double s = 0.0;
        for (int k = 1; k < half; ++k) s += HW[k] * ct[(size_t)((long long)k * m % L)];
        g[m] = (HW[0] + 2.0 * s + HW[half] * ((m & 1) ? -1.0 : 1.0)) / (double)L;
    }
}

// Parker (P27) / Wang (P28, without the factor 2) weights, [nA][nu]; returns TIGRE_ERR_ARG for a scan they do not apply to
int fdk_weights(const Grid& g, const std::vector<ViewH>& views, int weighting, std::vector<double>& w) {
    const int nA = (int)views.size(), nu = g.nu;
    w.assign((size_t)nA * nu, 1.0);
    if (weighting == TIGRE_FDK_FULL) return TIGRE_OK;
    if (weighting == TIGRE_FDK_PARKER) {
        if (nA < 2) return TIGRE_ERR_ARG;
        const double t0 = views[0].ang[0], t1 = views[nA - 1].ang[0];
        const double dir = t1 > t0 ? 1.0 : -1.0;
        for (int a = 1; a < nA; ++a)
            if (!((views[a].ang[0] - views[a - 1].ang[0]) * dir > 0.0)) return TIGRE_ERR_ARG;   // monotone angles only
        const double Theta = std::fabs(t1 - t0), eps = 0.5 * (Theta - M_PI);
        if (!(Theta < 2.0 * M_PI)) return TIGRE_ERR_ARG;
        for (int a = 0; a < nA; ++a) {
            const double beta = std::fabs(views[a].ang[0] - t0);
            for (int iu = 0; iu < nu; ++iu) {
                const double u = (iu + 0.5) * g.du - 0.5 * nu * g.du + views[a].offD[0];
                const double gamma = -dir * std::atan(u / views[a].DSD);
                double v = 1.0;
                if (beta < 2.0 * eps - 2.0 * gamma) {
                    const double s = std::sin(0.25 * M_PI * beta / (eps - gamma));
                    v = s * s;
                } else if (beta > M_PI - 2.0 * gamma) {
                    const double s = std::sin(0.25 * M_PI * (M_PI + 2.0 * eps - beta) / (eps + gamma));
                    v = s * s;
                }
                w[(size_t)a * nu + iu] = v;
            }
        }
        return TIGRE_OK;
    }
    if (weighting == TIGRE_FDK_WANG) {
        for (int a = 0; a < nA; ++a) {
            const double off = views[a].offD[0], s = off >= 0.0 ? 1.0 : -1.0;
            const double u_ov = 0.5 * nu * g.du - std::fabs(off);
            if (!(u_ov > 0.0)) return TIGRE_ERR_ARG;
            const double den = std::atan(u_ov / views[a].DSD);
            for (int iu = 0; iu < nu; ++iu) {
                const double t = ((iu + 0.5) * g.du - 0.5 * nu * g.du + off) * s;
                double v = 0.5 * (std::sin(0.5 * M_PI * std::atan(t / views[a].DSD) / den) + 1.0);
                if (t > u_ov) v = 1.0;
                if (t < -u_ov) v = 0.0;
                w[(size_t)a * nu + iu] = v;
            }
        }
        return TIGRE_OK;
    }
    return TIGRE_ERR_ARG;
}

int launch_flatten(const float* curved, const Grid& g, const double* d_dsd, int nViews, float* flat, cudaStream_t st) {
    ProfScope ps(PK_EW, st);
    const size_t total = (size_t)g.nu * g.nv * nViews;
    if (total == 0) return TIGRE_OK;
    const int blocks = (int)std::min<size_t>((total + 255) / 256, (size_t)148 * 16);
    flatten_kernel<<<blocks, 256, 0, st>>>(curved, g.nu, g.nv, (float)g.du, (float)g.dv, d_dsd, flat, total);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

// d_taps: nu taps for tau = 1 (device) or NULL for the Ram-Lak taps of P12; odd_only: the taps vanish at even n != 0
// d_offd: [nViews][2] offDetector per view (device) or NULL (no displacement)
int launch_fdk_filter_taps(const float* b, const Grid& g, const double* d_dsd, const double* d_dso, const double* d_offd, int nViews,
                           const float* d_taps, const float* d_colw, float* q, cudaStream_t st, bool odd_only) {
    ProfScope ps(PK_EW, st);
    // odd_only: two half-rows of ceil(nu / 2) elements; otherwise one row of nu
    const int len = odd_only ? (g.nu + 1) / 2 : g.nu;
    const int nuC = (len + FR - 1) / FR * FR;
    const int PAD = nuC + 3 * FR;                   // zero padding on each side (multiple of FR)
    int PL = (nuC + 2 * PAD) / FR;                  // words per plane
    PL += (PL % 32 == 1) ? 0 : ((33 - PL % 32) % 32);   // = 1 mod 32: the fill of the planes is then conflict-free as well
    const int NT = nuC + 2 * FR;                    // taps incl. the overshoot of the last block, multiple of 4
    const size_t smem = ((size_t)NT + (size_t)(odd_only ? 2 : 1) * FR * PL) * sizeof(float);
    if (smem > 200 * 1024) return TIGRE_ERR_ARG;
    auto kern = odd_only ? fdk_conv_kernel<true> : fdk_conv_kernel<false>;
    if (smem > 48 * 1024) TG_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid(g.nv, nViews);
    kern<<<grid, 128, smem, st>>>(b, g.nu, g.nv, (float)g.du, (float)g.dv, d_dsd, d_dso, d_offd, d_taps, d_colw, q, PAD, PL, NT);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg
