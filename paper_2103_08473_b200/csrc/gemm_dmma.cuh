// Complex128 GEMM on the FP64 tensor-core path of sm_100a.
//
//   C[m*csm + n*csn] (+)= alpha * sum_k A[m*lda + k] * B[n*ldb + k]          (complex, interleaved re/im)
//
// sm_100a has exactly one FP64 MMA: DMMA.8x8x4 (mma.sync.m8n8k4.f64); tcgen05/TMEM have no f64 kind.
// Complex arithmetic is mapped onto it with the 4M real embedding, with NO planar split of the operands:
//   * lane (g = lane/4, q = lane%4) loads ONE complex A element A[m0+g][k0+q] and ONE complex B element
//     B[n0+g/2][k0+q] (16-byte LDS each) for a group of 4 complex k;
//   * DMMA #1 takes a = Re A and b = (g odd ? Im B : Re B);  DMMA #2 takes a = Im A and b = (g odd ? Re B : -Im B);
//   * in the m8n8 accumulator fragment lane (g,q) then owns columns 2q (=Re) and 2q+1 (=Im) of row g, i.e. exactly
//     the complex element C[m0+g][n0+q]: the epilogue stores double2 directly.
//   Two DMMAs = 8 rows x 4 complex columns x 4 complex k = 128 complex MACs = 512 real FMAs: no wasted lanes.
//
// Data movement: operands are staged by TMA (cp.async.bulk.tensor) into a 4-stage shared-memory ring guarded by
// full/empty mbarriers; one producer warp issues the copies, eight consumer warps issue DMMA.  The shared-memory
// layout is [k-group of 4 complex][row][64 bytes]: the 16-byte fragment loads of a quarter-warp cover one contiguous
// 128-byte line, so they are bank-conflict free without swizzling; each TMA box is {4 complex} x {rows}.
// Out-of-range rows / k are zero-filled by TMA, so ragged M, N, K need no special code in the main loop.
#pragma once
#include <cuda.h>
#include "gemm_simple.cuh"

constexpr int DMMA_BM = 128;        // CTA tile rows (A operand)
constexpr int DMMA_BKG = 4;         // k-groups (of 4 complex) per pipeline stage -> BK = 16 complex
constexpr int DMMA_STAGES = 4;
constexpr int DMMA_CONSUMER_WARPS = 8;
constexpr int DMMA_THREADS = (DMMA_CONSUMER_WARPS + 1) * 32;

struct DmmaArgs {
    int64_t M, N, K;
    c128* C; int64_t csm, csn, bsC;
    c128 alpha; int accumulate;
    int batchA, batchB;   // 1 if the operand is indexed by the batch coordinate, 0 if broadcast
    int ksplit; int64_t kchunk;
    c128* partial;
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE;\n"
        "bra WAIT_LOOP;\n"
        "DONE:\n"
        "}\n" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}

template <int NI>
__global__ void __launch_bounds__(DMMA_THREADS, 1)
gemm_dmma_kernel(const __grid_constant__ CUtensorMap mapA, const __grid_constant__ CUtensorMap mapB, DmmaArgs p)
{
    constexpr int BN = 8 * NI;
    constexpr int A_KG = DMMA_BM * 64, B_KG = BN * 64;                 // bytes per k-group
    constexpr int A_STAGE = DMMA_BKG * A_KG, B_STAGE = DMMA_BKG * B_KG;
    constexpr int STAGE = A_STAGE + B_STAGE;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + DMMA_STAGES * STAGE);
    uint64_t* empty = full + DMMA_STAGES;

    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int bz = blockIdx.z / p.ksplit, split = blockIdx.z % p.ksplit;
    const int64_t m0 = (int64_t)blockIdx.y * DMMA_BM, n0 = (int64_t)blockIdx.x * BN;
    const int64_t kbeg = (int64_t)split * p.kchunk;
    const int64_t kend = (kbeg + p.kchunk < p.K) ? kbeg + p.kchunk : p.K;
    const int kt = (int)((kend - kbeg + 4 * DMMA_BKG - 1) / (4 * DMMA_BKG));

    if (threadIdx.x == 0) {
        for (int s = 0; s < DMMA_STAGES; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], DMMA_CONSUMER_WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();

    if (warp == DMMA_CONSUMER_WARPS) {
        // ===== TMA producer =====
        if (lane == 0) {
            const int cA = p.batchA ? bz : 0, cB = p.batchB ? bz : 0;
            for (int it = 0; it < kt; it++) {
                const int s = it % DMMA_STAGES;
                if (it >= DMMA_STAGES) mbar_wait(&empty[s], ((it / DMMA_STAGES) & 1) ^ 1);
                mbar_expect_tx(&full[s], STAGE);
                unsigned char* sa = smem + s * STAGE;
                unsigned char* sb = sa + A_STAGE;
                const int64_t k0 = kbeg + (int64_t)it * 4 * DMMA_BKG;
#pragma unroll
                for (int kg = 0; kg < DMMA_BKG; kg++) {
                    const int cd = (int)((k0 + 4 * kg) * 2);   // coordinate in doubles
                    tma_load_3d(sa + kg * A_KG, &mapA, cd, (int)m0, cA, &full[s]);
                    tma_load_3d(sb + kg * B_KG, &mapB, cd, (int)n0, cB, &full[s]);
                }
            }
        }
        return;
    }

    // ===== DMMA consumers: warp tile 32 rows x 4*NI complex columns =====
    const int g = lane >> 2, q = lane & 3;
    const int wm = warp & 3, wn = warp >> 2;
    const bool odd = g & 1;
    double acc[4][NI][2];
#pragma unroll
    for (int mi = 0; mi < 4; mi++)
#pragma unroll
        for (int nj = 0; nj < NI; nj++) { acc[mi][nj][0] = 0.0; acc[mi][nj][1] = 0.0; }

    const int a_off = (wm * 32 + g) * 64 + q * 16;
    const int b_off = (wn * 4 * NI + (g >> 1)) * 64 + q * 16;

    for (int it = 0; it < kt; it++) {
        const int s = it % DMMA_STAGES;
        mbar_wait(&full[s], (it / DMMA_STAGES) & 1);
        const unsigned char* sa = smem + s * STAGE + a_off;
        const unsigned char* sb = smem + s * STAGE + A_STAGE + b_off;
#pragma unroll
        for (int kg = 0; kg < DMMA_BKG; kg++) {
            double2 a[4];
#pragma unroll
            for (int mi = 0; mi < 4; mi++) a[mi] = *reinterpret_cast<const double2*>(sa + kg * A_KG + mi * 8 * 64);
#pragma unroll
            for (int nj = 0; nj < NI; nj++) {
                const double2 b = *reinterpret_cast<const double2*>(sb + kg * B_KG + nj * 4 * 64);
                const double b1 = odd ? b.y : b.x;
                const double b2 = odd ? b.x : -b.y;
#pragma unroll
                for (int mi = 0; mi < 4; mi++) dmma884(acc[mi][nj][0], acc[mi][nj][1], a[mi].x, b1);
#pragma unroll
                for (int mi = 0; mi < 4; mi++) dmma884(acc[mi][nj][0], acc[mi][nj][1], a[mi].y, b2);
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

    // ===== epilogue: lane (g,q) owns C[m][n] = (acc[..][0], acc[..][1]) =====
#pragma unroll
    for (int mi = 0; mi < 4; mi++) {
        const int64_t m = m0 + wm * 32 + mi * 8 + g;
        if (m >= p.M) continue;
#pragma unroll
        for (int nj = 0; nj < NI; nj++) {
            const int64_t n = n0 + wn * 4 * NI + nj * 4 + q;
            if (n >= p.N) continue;
            c128 r = mk(acc[mi][nj][0], acc[mi][nj][1]);
            if (p.ksplit > 1) {
                p.partial[((int64_t)blockIdx.z * p.M + m) * p.N + n] = r;
            } else {
                c128* c = p.C + (int64_t)bz * p.bsC + m * p.csm + n * p.csn;
                r = cmul(p.alpha, r);
                *c = p.accumulate ? cadd(*c, r) : r;
            }
        }
    }
}

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
typedef CUresult (*PFN_encodeTiled)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                    const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                    CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static PFN_encodeTiled get_encode_fn()
{
    static PFN_encodeTiled fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* ptr = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<PFN_encodeTiled>(ptr);
    }
    return fn;
}

// rows x K complex matrix with leading dimension ld (elements), nb batches with stride bs (elements)
static int make_operand_map(CUtensorMap* map, const c128* base, int64_t rows, int64_t K, int64_t ld, int nb, int64_t bs,
                            int box_rows)
{
    PFN_encodeTiled enc = get_encode_fn();
    if (!enc) { snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled unavailable"); return CCSD_ECUDA; }
    cuuint64_t dims[3] = {(cuuint64_t)(2 * K), (cuuint64_t)rows, (cuuint64_t)(nb > 0 ? nb : 1)};
    cuuint64_t strides[2] = {(cuuint64_t)(ld * 16), (cuuint64_t)((nb > 1 && bs > 0) ? bs * 16 : ld * 16)};
    cuuint32_t box[3] = {8, (cuuint32_t)box_rows, 1};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<c128*>(base), dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled failed (%d): rows=%lld K=%lld ld=%lld nb=%d", (int)r,
                 (long long)rows, (long long)K, (long long)ld, nb);
        return CCSD_ECUDA;
    }
    return CCSD_OK;
}

static inline bool dmma_supported(const GemmParams& p)
{
    if (p.sak != 1 || p.sbk != 1) return false;
    if (p.M < 1 || p.N < 1 || p.K < 1) return false;
    if (p.sam < p.K || p.sbn < p.K) return false;                  // rows must not overlap (TMA stride >= extent)
    if (p.K > (1LL << 30) || p.M > (1LL << 31) - 256 || p.N > (1LL << 31) - 256) return false;
    if (p.sam * 16 >= (1LL << 40) || p.sbn * 16 >= (1LL << 40)) return false;
    if (p.batch > 1 && ((p.bsA != 0 && p.bsA * 16 >= (1LL << 40)) || (p.bsB != 0 && p.bsB * 16 >= (1LL << 40)))) return false;
    if ((reinterpret_cast<uintptr_t>(p.A) | reinterpret_cast<uintptr_t>(p.B)) & 15) return false;
    if ((p.M + DMMA_BM - 1) / DMMA_BM > 65535) return false;
    if ((int64_t)p.batch * 64 > 65535) return false;
    return true;
}
static inline bool dmma_worthwhile(const GemmParams& p)
{
    return (double)p.M * (double)p.N * (double)p.K * p.batch >= 2.0e5;
}
// column-tile width (complex) in {32,40,48,56,64} that wastes the fewest padded columns; ties -> wider
static inline int dmma_bn_for(int64_t N)
{
    int best = 64;
    int64_t bestpad = ((N + 63) / 64) * 64;
    for (int bn = 56; bn >= 32; bn -= 8) {
        int64_t pad = ((N + bn - 1) / bn) * bn;
        if (pad < bestpad) { bestpad = pad; best = bn; }
    }
    return best;
}

template <int NI>
static int launch_dmma_t(cudaStream_t st, const CUtensorMap& mA, const CUtensorMap& mB, const DmmaArgs& a, dim3 grid)
{
    constexpr int BN = 8 * NI;
    constexpr int smem = DMMA_STAGES * DMMA_BKG * (DMMA_BM + BN) * 64 + 2 * DMMA_STAGES * 8;
    static bool configured = false;
    if (!configured) {
        CCSD_CUDA_TRY(cudaFuncSetAttribute(gemm_dmma_kernel<NI>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
        configured = true;
    }
    gemm_dmma_kernel<NI><<<grid, DMMA_THREADS, smem, st>>>(mA, mB, a);
    g_launches++;
    return CCSD_OK;
}

static int launch_gemm_dmma(cudaStream_t st, const GemmParams& p)
{
    const int bn = dmma_bn_for(p.N);
    CUtensorMap mA, mB;
    CCSD_TRY(make_operand_map(&mA, p.A, p.M, p.K, p.sam, p.batch, p.bsA, DMMA_BM));
    CCSD_TRY(make_operand_map(&mB, p.B, p.N, p.K, p.sbn, p.batch, p.bsB, bn));
    DmmaArgs a;
    a.M = p.M; a.N = p.N; a.K = p.K;
    a.C = p.C; a.csm = p.csm; a.csn = p.csn; a.bsC = p.bsC;
    a.alpha = p.alpha; a.accumulate = p.accumulate;
    a.batchA = (p.batch > 1 && p.bsA != 0) ? 1 : 0;
    a.batchB = (p.batch > 1 && p.bsB != 0) ? 1 : 0;
    a.ksplit = p.ksplit; a.kchunk = p.kchunk; a.partial = p.partial;
    dim3 grid((unsigned)((p.N + bn - 1) / bn), (unsigned)((p.M + DMMA_BM - 1) / DMMA_BM), (unsigned)(p.batch * p.ksplit));
    switch (bn) {
    case 32: return launch_dmma_t<4>(st, mA, mB, a, grid);
    case 40: return launch_dmma_t<5>(st, mA, mB, a, grid);
    case 48: return launch_dmma_t<6>(st, mA, mB, a, grid);
    case 56: return launch_dmma_t<7>(st, mA, mB, a, grid);
    default: return launch_dmma_t<8>(st, mA, mB, a, grid);
    }
}
