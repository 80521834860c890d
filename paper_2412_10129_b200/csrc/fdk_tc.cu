// fdk_tc.cu — the FDK pre-filter (readings P12, P26, P34) on the 5th-generation
// tensor cores: the one dense contraction of the path.
//
// The row filter q[row][n] = (1/tau) sum_k p1[row][k] g[|n - k|] is the GEMM  Q = P1 . T  with T the symmetric Toeplitz matrix
// of the taps (nu x nu), M = nViews * nv detector rows, N = K = nu.  fp32 exactness (filter parity 1e-5 under the ramp
// filter's cancellation) rules out a single tf32 pass, so every product is split:  a = a_hi + a_lo,  b = b_hi + b_lo  with
// a_hi = rn_tf32(a), a_lo = rn_tf32(a - a_hi) (11 + 11 significant bits, the remainder below 2^-24 |a|) and
//   a b  ~  a_hi b_hi + a_hi b_lo + a_lo b_hi       (the dropped a_lo b_lo is below 2^-24 |a b|)
// three kind::tf32 tcgen05.mma per K step into ONE fp32 accumulator in tensor memory.
//
// One CTA per SM, persistent over tiles of 128 detector rows; per tile four passes of 256 output columns; per pass a ring of
// K blocks of 32 (one 128-byte swizzle row of tf32):
//   warp 8 (one lane)   TMA producer: A = 128 raw detector rows x 32 columns into a 4-stage ring, and the 32 new rows of the
//                       Toeplitz operand's row ring (see FT_RING_ROWS), 128-byte swizzled
//   warps 0-7           transform: two threads per row of the A tile; they multiply the raw values by the cosine pre-weight
//                       (and the Parker / Wang column weight), round to a_hi in place and write a_lo beside it (the swizzle
//                       only permutes 16-byte chunks inside the row's own 128 bytes), then fence the async proxy
//   warp 9 (one lane)   issues the tcgen05.mma of the K block (4 K steps of 8 x 3 products, M 128 x N 256 in two column
//                       segments around the ring's wrap), commits the stage back to the producer and, after the last K
//                       block, the accumulator to the epilogue
//   warps 0-7 again     epilogue: tcgen05.ld of the thread's half of its accumulator row, times 1/tau of its view, stored to q
// Detector widths that are not a multiple of 4 (TMA row pitch) and drivers without the tensor-map encoder keep fdk.cu's kernel.
#include <cuda.h>
#include <algorithm>
#include <cmath>
#include <vector>
#include "common.cuh"
#include "tma.cuh"

namespace tg {

namespace {

constexpr int FT_M = 128, FT_N = 256, FT_K = 32, FT_STAGES = 4;
constexpr int FT_TW = 8;   // transform / epilogue warps: two threads per row of the A tile (warp w: rows 32 (w & 3).., column half w >> 2)
constexpr int FT_A_BYTES = FT_M * FT_K * 4;                          // 16 KB
constexpr int FT_B_BYTES = FT_N * FT_K * 4;                          // 32 KB
constexpr int FT_STAGE_BYTES = 2 * FT_A_BYTES;                       // A (-> a_hi), a_lo = 32 KB per stage
// The Toeplitz operand is a RING of rows in shared memory.  B_kb[n][k] = g[|(n0 + n) - (32 kb + k)|] = H[n0 + n - 32 kb][k] with
// H[m][k] = g[|m - k|]: the 256 x 32 tiles of consecutive K blocks are the SAME rows of H shifted by 32, so a K block brings 32 new
// rows (2 x 4 KB) instead of a whole tile (2 x 32 KB).  288 = 256 + 32 rows: the new rows of K block kb take the slots that left the
// window after K block kb - 2, the very tensor-core reads whose completion frees A's stage; the window wraps around the ring, so the
// N = 256 product is issued as two tcgen05.mma (N1 and 256 - N1 columns of the accumulator).  With S stages of A in flight the
// producer runs up to S K blocks ahead of the tensor core, so the ring holds 256 + 32 (S - 1) rows; at the start of a pass the
// whole window is reloaded, after the previous pass's products have finished (one pipeline drain per 32 K blocks).
constexpr int FT_RING_ROWS = FT_N + FT_K * (FT_STAGES - 1);          // 352 rows of 128 bytes = 44 swizzle atoms
constexpr int FT_RING_BYTES = FT_RING_ROWS * 128;                    // 44 KB
constexpr int FT_RINGS_OFF = FT_STAGES * FT_STAGE_BYTES;             // [A stages][ring: hi, lo]
constexpr int FT_BAR_OFF = FT_RINGS_OFF + 2 * FT_RING_BYTES;
constexpr int FT_SMEM = FT_BAR_OFF + 1024 /* alignment */ + 256 /* barriers, tmem slot */;
constexpr int FT_THREADS = 32 * (FT_TW + 2);   // + the TMA warp and the MMA warp

__device__ __forceinline__ float rn_tf32(float x) {
    uint32_t r;
    asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x));
    return __uint_as_float(r);
}
__device__ __forceinline__ void tma_load_2d(void* dst, const CUtensorMap* map, int c0, int c1, uint64_t* bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(smem_u32(dst)),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(c0), "r"(c1), "r"(smem_u32(bar))
        : "memory");
}
// K-major operand tile, 128-byte swizzle: rows of 128 bytes, 8-row atoms 1024 bytes apart (cute::UMMA::SmemDescriptor: start
// address >> 4 in bits 0-13, leading byte offset (unused here) 16-29, stride byte offset >> 4 in 32-45, version 1 in 46-47,
// layout type SWIZZLE_128B = 2 in 61-63)
__device__ __forceinline__ uint64_t umma_desc_k128(uint32_t smem_addr) {
    return (uint64_t)((smem_addr & 0x3FFFFu) >> 4) | (1ull << 16) | ((uint64_t)(1024 >> 4) << 32) | (1ull << 46) | (2ull << 61);
}
// kind::tf32, fp32 accumulator, both operands K-major, M 128, N columns (cute::UMMA::InstrDescriptor)
__device__ __forceinline__ constexpr uint32_t ft_idesc(int n) {
    return (1u << 4) | (2u << 7) | (2u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(FT_M >> 4) << 24);
}

__device__ __forceinline__ void umma_tf32(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t"
        ".reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::tf32 [%0], %1, %2, %3, p;\n\t"
        "}\n" ::"r"(tmem_d),
        "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
        : "memory");
}
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

struct FtRow {       // per-view quantities the transform and the epilogue need (device table, one per view)
    float dsd, itau, offu, offv;
};

// H_hi / H_lo [rowsH][32]: H[j][k] = g[|j - shift - k|] (0 beyond the taps), split into two tf32 parts; shift = 32 nKb
__global__ void __launch_bounds__(256) ft_toeplitz_kernel(const float* __restrict__ taps, int nu, int rowsH, int shift, float* __restrict__ hhi,
                                                          float* __restrict__ hlo) {
    const int total = rowsH * FT_K;
    for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < total; i += gridDim.x * blockDim.x) {
        const int j = i / FT_K, k = i - j * FT_K;
        const int m = abs(j - shift - k);
        const float t = m < nu ? __ldg(taps + m) : 0.f;
        const float hi = rn_tf32(t);
        hhi[i] = hi;
        hlo[i] = rn_tf32(t - hi);
    }
}

__global__ void __launch_bounds__(FT_THREADS, 1)
fdk_tc_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapBh, const __grid_constant__ CUtensorMap mapBl,
              const FtRow* __restrict__ rows, const float* __restrict__ colw, float* __restrict__ q, int nu, int nv, long long mTotal,
              float du, float dv, int nTiles) {
    extern __shared__ unsigned char smem_raw[];
    unsigned char* sm = reinterpret_cast<unsigned char*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~(uintptr_t)1023);
    uint64_t* bars = reinterpret_cast<uint64_t*>(sm + FT_BAR_OFF);
    uint64_t *full = bars, *ready = bars + FT_STAGES, *empty = bars + 2 * FT_STAGES, *accfull = bars + 3 * FT_STAGES,
             *accempty = bars + 3 * FT_STAGES + 1;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 3 * FT_STAGES + 2);
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

    if (threadIdx.x == 0) {
        for (int s = 0; s < FT_STAGES; ++s) {
            mbar_init(full + s, 1);
            mbar_init(ready + s, 32 * FT_TW);
            mbar_init(empty + s, 1);
        }
        mbar_init(accfull, 1);
        mbar_init(accempty, 32 * FT_TW);
        mbar_fence_init();
    }
    if (warp == FT_TW) {   // one warp allocates (and later frees) the accumulator's 256 columns of tensor memory
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(tmem_slot)), "r"(FT_N) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tmem = *tmem_slot;

    const int nPass = (nu + FT_N - 1) / FT_N, nKb = (nu + FT_K - 1) / FT_K;

    if (warp == FT_TW) {
        // ------------------------------------------------------------ TMA producer
        if (lane == 0) {
            uint32_t it = 0, pc = 0;
            for (int tile = blockIdx.x; tile < nTiles; tile += gridDim.x)
                for (int ps = 0; ps < nPass; ++ps, ++pc)
                    for (int kb = 0; kb < nKb; ++kb, ++it) {
                        const int s = it % FT_STAGES;
                        mbar_wait(empty + s, ((it / FT_STAGES) & 1) ^ 1);
                        unsigned char* st = sm + s * FT_STAGE_BYTES;
                        // rows of H this K block adds to the ring (all 256 + nothing at the start of a pass: 8 boxes of 32 rows)
                        unsigned char* ring = sm + FT_RINGS_OFF;
                        const int nbox = kb == 0 ? FT_N / FT_K : 1;
                        if (kb == 0 && pc > 0) mbar_wait(accfull, (pc - 1) & 1);   // the previous pass's products no longer read the ring
                        mbar_arrive_expect_tx(full + s, FT_A_BYTES + 2 * nbox * FT_K * 128);
                        tma_load_2d(st, &mapA, kb * FT_K, tile * FT_M, full + s);
                        for (int bx = 0; bx < nbox; ++bx) {
                            const int slot = kb == 0 ? bx * FT_K : (FT_RING_ROWS - (FT_K * kb) % FT_RING_ROWS) % FT_RING_ROWS;   // ring row
                            const int j = ps * FT_N + FT_K * (nKb - kb) + bx * FT_K;                                                // row of H
                            tma_load_2d(ring + slot * 128, &mapBh, 0, j, full + s);
                            tma_load_2d(ring + FT_RING_BYTES + slot * 128, &mapBl, 0, j, full + s);
                        }
                    }
        }
    } else if (warp == FT_TW + 1) {
        // ------------------------------------------------------------ MMA issuer
        if (lane == 0) {
            uint32_t it = 0, pc = 0;
            for (int tile = blockIdx.x; tile < nTiles; tile += gridDim.x)
                for (int ps = 0; ps < nPass; ++ps, ++pc) {
                    mbar_wait(accempty, (pc & 1) ^ 1);   // the epilogue has drained the accumulator of the previous pass
                    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                    for (int kb = 0; kb < nKb; ++kb, ++it) {
                        const int s = it % FT_STAGES;
                        mbar_wait(ready + s, (it / FT_STAGES) & 1);
                        asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                        const uint32_t a0 = smem_u32(sm + s * FT_STAGE_BYTES);
                        const uint64_t dAh = umma_desc_k128(a0), dAl = umma_desc_k128(a0 + FT_A_BYTES);
                        // the window of this K block starts at ring row P and wraps: columns [0, N1) from rows [P, 288), the rest from row 0
                        const uint32_t ring = smem_u32(sm + FT_RINGS_OFF);
                        const int P = (FT_RING_ROWS - (FT_K * kb) % FT_RING_ROWS) % FT_RING_ROWS;
                        const int N1 = min(FT_N, FT_RING_ROWS - P), N2 = FT_N - N1;
                        const uint64_t dBh1 = umma_desc_k128(ring + P * 128), dBl1 = umma_desc_k128(ring + FT_RING_BYTES + P * 128);
                        const uint64_t dBh2 = umma_desc_k128(ring), dBl2 = umma_desc_k128(ring + FT_RING_BYTES);
                        const uint32_t id1 = ft_idesc(N1), id2 = ft_idesc(N2);
#pragma unroll
                        for (int kk = 0; kk < FT_K / 8; ++kk) {   // K step of 8 tf32 = 32 bytes inside the swizzle row: +2 in 16-byte units
                            const uint64_t o = (uint64_t)(kk * 2);
                            const uint32_t acc = (kb | kk) != 0;
                            umma_tf32(tmem, dAh + o, dBh1 + o, id1, acc);
                            umma_tf32(tmem, dAh + o, dBl1 + o, id1, 1);
                            umma_tf32(tmem, dAl + o, dBh1 + o, id1, 1);
                            if (N2 > 0) {
                                umma_tf32(tmem + (uint32_t)N1, dAh + o, dBh2 + o, id2, acc);
                                umma_tf32(tmem + (uint32_t)N1, dAh + o, dBl2 + o, id2, 1);
                                umma_tf32(tmem + (uint32_t)N1, dAl + o, dBh2 + o, id2, 1);
                            }
                        }
                        umma_commit(empty + s);            // the stage is free once these have read it
                    }
                    umma_commit(accfull);                  // the accumulator is complete once everything issued so far has finished
                }
        }
    } else {
        // ------------------------------------------------------------ transform + epilogue (8 warps: two threads per row of the tile,
        // each half of its chunks and, in the epilogue, half of its columns)
        const int t = threadIdx.x & 127, half = threadIdx.x >> 7;
        uint32_t it = 0, pc = 0;
        for (int tile = blockIdx.x; tile < nTiles; tile += gridDim.x) {
            const long long gr = (long long)tile * FT_M + t;     // global detector row (view * nv + iv)
            const bool rowok = gr < mTotal;
            const int ia = rowok ? (int)(gr / nv) : 0, iv = rowok ? (int)(gr - (long long)ia * nv) : 0;
            const FtRow rw = rows[ia];
            const float v = ((float)iv + 0.5f) * dv - 0.5f * (float)nv * dv + rw.offv;
            const float crow = fmaf(rw.dsd, rw.dsd, v * v);
            const float u0 = 0.5f * du - 0.5f * (float)nu * du + rw.offu;   // u of column 0
            const float* cw = colw ? colw + (size_t)ia * nu : nullptr;
            for (int ps = 0; ps < nPass; ++ps, ++pc) {
                for (int kb = 0; kb < nKb; ++kb, ++it) {
                    const int s = it % FT_STAGES;
                    mbar_wait(full + s, (it / FT_STAGES) & 1);
                    unsigned char* rowA = sm + s * FT_STAGE_BYTES + t * 128;
#pragma unroll
                    for (int cc = 0; cc < 4; ++cc) {
                        const int c = 4 * half + cc;
                        const int p = (c + t) & 7;                 // physical 16-byte chunk (rotated per lane: no bank conflicts)
                        const int k = kb * FT_K + 4 * (p ^ (t & 7));   // logical column of its first element (128-byte swizzle)
                        float4 a = *reinterpret_cast<float4*>(rowA + p * 16);
                        // cosine pre-weight DSD / sqrt(DSD^2 + u^2 + v^2) (readings P12, P34) and the optional column weight
                        const float ua = fmaf((float)k, du, u0), ub = ua + du, uc = ub + du, ud = uc + du;
                        float4 w = make_float4(rw.dsd * rsqrtf(fmaf(ua, ua, crow)), rw.dsd * rsqrtf(fmaf(ub, ub, crow)),
                                               rw.dsd * rsqrtf(fmaf(uc, uc, crow)), rw.dsd * rsqrtf(fmaf(ud, ud, crow)));
                        if (cw && k < nu) {
                            const float4 c4 = __ldg(reinterpret_cast<const float4*>(cw + k));
                            w.x *= c4.x, w.y *= c4.y, w.z *= c4.z, w.w *= c4.w;
                        }
                        a.x *= w.x, a.y *= w.y, a.z *= w.z, a.w *= w.w;
                        float4 hi = make_float4(rn_tf32(a.x), rn_tf32(a.y), rn_tf32(a.z), rn_tf32(a.w));
                        float4 lo = make_float4(rn_tf32(a.x - hi.x), rn_tf32(a.y - hi.y), rn_tf32(a.z - hi.z), rn_tf32(a.w - hi.w));
                        *reinterpret_cast<float4*>(rowA + p * 16) = hi;
                        *reinterpret_cast<float4*>(rowA + FT_A_BYTES + p * 16) = lo;
                    }
                    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // generic-proxy writes -> visible to the tensor core's reads
                    mbar_arrive(ready + s);
                }
                // ---- epilogue of this pass
                mbar_wait(accfull, pc & 1);
                asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
                const uint32_t trow = tmem + ((uint32_t)((warp & 3) * 32) << 16);
                float* qrow = q + (size_t)(rowok ? gr : 0) * nu + (size_t)ps * FT_N;
#pragma unroll 1
                for (int c0 = half * (FT_N / 2); c0 < (half + 1) * (FT_N / 2); c0 += 32) {
                    uint32_t r[32];
                    asm volatile(
                        "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, "
                        "%19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
                        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
                          "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
                          "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]),
                          "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
                        : "r"(trow + (uint32_t)c0));
                    asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
                    if (rowok) {
#pragma unroll
                        for (int j = 0; j < 32; j += 4) {
                            const int n = ps * FT_N + c0 + j;
                            if (n < nu)   // nu is a multiple of 4
                                *reinterpret_cast<float4*>(qrow + c0 + j) =
                                    make_float4(__uint_as_float(r[j]) * rw.itau, __uint_as_float(r[j + 1]) * rw.itau,
                                                __uint_as_float(r[j + 2]) * rw.itau, __uint_as_float(r[j + 3]) * rw.itau);
                        }
                    }
                }
                asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
                mbar_arrive(accempty);
            }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    __syncwarp();
    if (warp == FT_TW) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(FT_N) : "memory");
}

bool encode_2d_sw128(CUtensorMap* map, const void* base, uint64_t cols, uint64_t rowsN, uint32_t boxRows) {
    TensorMapEncodeTiledFn enc = tensor_map_encoder();
    if (!enc) return false;
    const cuuint64_t dims[2] = {cols, rowsN};
    const cuuint64_t strides[1] = {cols * sizeof(float)};
    const cuuint32_t box[2] = {(cuuint32_t)FT_K, boxRows};
    const cuuint32_t estr[2] = {1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, const_cast<void*>(base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
               CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

int g_fdk_path = 0;   // 0 = tensor-core filter when the problem qualifies, 1 = the CUDA-core kernel of fdk.cu only (tigre_set_fdk_path)

// Returns TIGRE_OK if the tensor-core filter ran, 1 if this problem does not qualify (the caller runs fdk.cu's kernel), a negative
// status on an error.  h_taps: nu taps for tau = 1 (tap 0 included); dsd / dso / offd: per-view host values.
int launch_fdk_filter_tc(const float* b, const Grid& g, const std::vector<double>& dsd, const std::vector<double>& dso,
                         const std::vector<double>& offd, int nViews, const std::vector<float>& h_taps, const float* d_colw, float* q,
                         cudaStream_t st) {
    if (g_fdk_path == 1 || !tensor_map_encoder()) return 1;
    const int nu = g.nu, nv = g.nv;
    if ((nu & 3) || nu < FT_K || (reinterpret_cast<uintptr_t>(b) & 15) || (reinterpret_cast<uintptr_t>(q) & 15) || b == q) return 1;
    int dev = 0, cc = 0, sms = 148;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&cc, cudaDevAttrComputeCapabilityMajor, dev);
    cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    if (cc < 10) return 1;
    const long long mTotal = (long long)nViews * nv;
    const int nTiles = (int)((mTotal + FT_M - 1) / FT_M);
    TempBuf taps, thi, tlo, rows;
    TG_TRY(upload(taps, h_taps.data(), sizeof(float) * nu, st));
    const int nPass = (nu + FT_N - 1) / FT_N, nKb = (nu + FT_K - 1) / FT_K;
    const int rowsH = FT_K * nKb + FT_N * nPass;   // rows of H any (pass, K block) can ask for
    TG_TRY(thi.alloc(sizeof(float) * (size_t)rowsH * FT_K, st));
    TG_TRY(tlo.alloc(sizeof(float) * (size_t)rowsH * FT_K, st));
    std::vector<FtRow> hr(nViews);
    for (int a = 0; a < nViews; ++a) {
        hr[a].dsd = (float)dsd[a];
        hr[a].itau = (float)(dsd[a] / (g.du * dso[a]));
        hr[a].offu = (float)offd[2 * a], hr[a].offv = (float)offd[2 * a + 1];
    }
    TG_TRY(upload(rows, hr.data(), sizeof(FtRow) * nViews, st));
    ProfScope ps(PK_EW, st, 2);
    ft_toeplitz_kernel<<<std::min(sms * 4, (rowsH * FT_K + 255) / 256), 256, 0, st>>>(taps.as<float>(), nu, rowsH, FT_K * nKb, thi.as<float>(), tlo.as<float>());
    CUtensorMap mA, mBh, mBl;
    if (!encode_2d_sw128(&mA, b, (uint64_t)nu, (uint64_t)mTotal, FT_M) || !encode_2d_sw128(&mBh, thi.p, (uint64_t)FT_K, (uint64_t)rowsH, FT_K) ||
        !encode_2d_sw128(&mBl, tlo.p, (uint64_t)FT_K, (uint64_t)rowsH, FT_K))
        return 1;
    TG_CUDA(cudaFuncSetAttribute(fdk_tc_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, FT_SMEM));
    fdk_tc_kernel<<<std::min(sms, nTiles), FT_THREADS, FT_SMEM, st>>>(mA, mBh, mBl, rows.as<FtRow>(), d_colw, q, nu, nv, mTotal, (float)g.du,
                                                                         (float)g.dv, nTiles);
    TG_CUDA(cudaGetLastError());
    return TIGRE_OK;
}

}  // namespace tg

extern "C" int tigre_set_fdk_path(int path) {
    if (path != 0 && path != 1) return TIGRE_ERR_ARG;
    tg::g_fdk_path = path;
    return TIGRE_OK;
}
