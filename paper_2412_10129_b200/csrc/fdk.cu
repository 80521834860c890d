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

template <bool ODD>
__global__ void __launch_bounds__(128)
fdk_conv_kernel(const float* __restrict__ b, int nu, int nv, float du, float dv, const double* __restrict__ dsd_a,
                const double* __restrict__ dso_a, const float* __restrict__ taps, const float* __restrict__ colw,
                float* __restrict__ q, int PAD, int PL, int NT) {
    extern __shared__ __align__(16) float sm[];
    float* tp = sm;              // [NT]  taps, tp[0] = 0 (the centre tap is applied separately), zero beyond nu
    float* rw = sm + NT;         // [FR][PL]  row value i at plane (i mod FR), offset (i + PAD) / FR
    const int iv = blockIdx.x, ia = blockIdx.y;
    const float DSD = (float)dsd_a[ia], DSO = (float)dso_a[ia];
    const float itau = DSD / (du * DSO);
    const float v = ((float)iv + 0.5f) * dv - 0.5f * (float)nv * dv;
    const size_t base = ((size_t)ia * nv + iv) * nu;
    for (int i = threadIdx.x; i < FR * PL; i += blockDim.x) rw[i] = 0.f;
    for (int n = threadIdx.x; n < NT; n += blockDim.x) {
        float t = 0.f;
        if (n >= 1 && n < nu) t = taps ? __ldg(taps + n) : ((n & 1) ? -1.0f / (9.8696044010893586f * (float)n * (float)n) : 0.f);
        tp[n] = t;
    }
    const float tap0 = taps ? __ldg(taps) : 0.25f;
    __syncthreads();
    for (int iu = threadIdx.x; iu < nu; iu += blockDim.x) {
        const float u = ((float)iu + 0.5f) * du - 0.5f * (float)nu * du;
        float r = __ldg(b + base + iu) * DSD * rsqrtf(DSD * DSD + u * u + v * v);
        if (colw) r *= __ldg(colw + (size_t)ia * nu + iu);
        rw[(iu % FR) * PL + (iu + PAD) / FR] = r;
    }
    __syncthreads();
    for (int c = threadIdx.x; c * FR < nu; c += blockDim.x) {
        const int i0 = c * FR, ob = (i0 + PAD) / FR;
        float acc[FR], L[FR], R[FR];
#pragma unroll
        for (int j = 0; j < FR; ++j) {
            L[j] = rw[j * PL + ob];          // window at n = 0: row[i0 + j]
            R[j] = L[j];
            acc[j] = tap0 * L[j];
        }
        // left side: row[i0 + j - n]; taps with n > i0 + FR - 1 meet only the zero padding
        const int mL = (i0 + FR - 1) / FR, mR = (nu - 1 - i0) / FR;
        for (int m = 0; m <= mL; ++m) {
            const float4 ta = *reinterpret_cast<const float4*>(tp + FR * m), tb = *reinterpret_cast<const float4*>(tp + FR * m + 4);
            const float t[FR] = {ta.x, ta.y, ta.z, ta.w, tb.x, tb.y, tb.z, tb.w};
#pragma unroll
            for (int k = 0; k < FR; ++k) {   // n = FR * m + k
                if (!ODD || (k & 1)) {
#pragma unroll
                    for (int j = 0; j < FR; ++j) acc[j] = fmaf(t[k], L[j], acc[j]);
                }
#pragma unroll
                for (int j = FR - 1; j > 0; --j) L[j] = L[j - 1];
                L[0] = rw[((FR - 1 - k) % FR) * PL + ob - m - 1];      // row[i0 - (n + 1)]
            }
        }
        for (int m = 0; m <= mR; ++m) {
            const float4 ta = *reinterpret_cast<const float4*>(tp + FR * m), tb = *reinterpret_cast<const float4*>(tp + FR * m + 4);
            const float t[FR] = {ta.x, ta.y, ta.z, ta.w, tb.x, tb.y, tb.z, tb.w};
#pragma unroll
            for (int k = 0; k < FR; ++k) {
                if (!ODD || (k & 1)) {
#pragma unroll
                    for (int j = 0; j < FR; ++j) acc[j] = fmaf(t[k], R[j], acc[j]);
                }
#pragma unroll
                for (int j = 0; j < FR - 1; ++j) R[j] = R[j + 1];
                R[FR - 1] = rw[k * PL + ob + m + 1];                     // row[i0 + FR - 1 + (n + 1)]
            }
        }
#pragma unroll
        for (int j = 0; j < FR; ++j)
            if (i0 + j < nu) q[base + i0 + j] = acc[j] * itau;
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

// taps for tau = 1 (the kernel scales by 1/tau: h ~ 1/tau^2, times the tau of the quadrature)
void fdk_filter_taps(int nu, int filter, std::vector<double>& g) {
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
int launch_fdk_filter_taps(const float* b, const Grid& g, const double* d_dsd, const double* d_dso, int nViews, const float* d_taps,
                           const float* d_colw, float* q, cudaStream_t st, bool odd_only) {
    ProfScope ps(PK_EW, st);
    const int nuC = (g.nu + FR - 1) / FR * FR;
    const int PAD = nuC + 2 * FR;                   // zero padding on each side (multiple of FR)
    int PL = (nuC + 2 * PAD) / FR;                  // words per plane
    PL += (PL % 32 == 1) ? 0 : ((33 - PL % 32) % 32);   // = 1 mod 32: the fill of the planes is then conflict-free as well
    const int NT = nuC + 2 * FR;                    // taps incl. the overshoot of the last block, multiple of 4
    const size_t smem = ((size_t)NT + (size_t)FR * PL) * sizeof(float);
    if (smem > 200 * 1024) return TIGRE_ERR_ARG;
    auto kern = odd_only ? fdk_conv_kernel<true> : fdk_conv_kernel<false>;
    if (smem > 48 * 1024) TG_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dim3 grid(g.nv, nViews);
    kern<<<grid, 128, smem, st>>>(b, g.nu, g.nv, (float)g.du, (float)g.dv, d_dsd, d_dso, d_taps, d_colw, q, PAD, PL, NT);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg
