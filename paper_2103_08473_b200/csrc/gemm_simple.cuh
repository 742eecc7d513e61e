// Simple FP64-FMA complex GEMM / GEMV kernels with fully general strides.
// They are the on-device debugging reference (ccsd_options.gemm_mode = 1) and serve the shapes the DMMA
// tensor-core kernel (gemm_dmma.cuh) does not take (K not a multiple of 4, non-unit K strides, tiny operands).
#pragma once
#include "common.cuh"

struct GemmParams {
    int64_t M, N, K;
    const c128* A; int64_t sam, sak;   // A[m*sam + k*sak]
    const c128* B; int64_t sbn, sbk;   // B[n*sbn + k*sbk]
    c128* C; int64_t csm, csn;         // C[m*csm + n*csn]
    c128 alpha; int accumulate;        // C = alpha*A*B^T (+ C)
    int batch; int64_t bsA, bsB, bsC;  // batch strides (elements)
    int ksplit; int64_t kchunk;        // split-K: slice s covers k in [s*kchunk, min(K,(s+1)*kchunk))
    c128* partial;                     // ksplit > 1: partial[(b*ksplit + s)][m][n] (dense M x N), reduced afterwards
    const double *As, *Bs;             // optional 3M sum planes  As[m*sam + k] = Re A + Im A  (DMMA kernel only)
};

constexpr int SG_BM = 64, SG_BN = 64, SG_BK = 8, SG_T = 16;

__global__ void __launch_bounds__(SG_T* SG_T) gemm_simple_kernel(GemmParams p)
{
    __shared__ c128 As[SG_BK][SG_BM + 1];
    __shared__ c128 Bs[SG_BK][SG_BN + 1];
    const int tx = threadIdx.x % SG_T, ty = threadIdx.x / SG_T;
    const int b = blockIdx.z / p.ksplit, s = blockIdx.z % p.ksplit;
    const int64_t m0 = (int64_t)blockIdx.y * SG_BM, n0 = (int64_t)blockIdx.x * SG_BN;
    const int64_t kbeg = (int64_t)s * p.kchunk;
    const int64_t kend = (kbeg + p.kchunk < p.K) ? kbeg + p.kchunk : p.K;
    const c128* A = p.A + (int64_t)b * p.bsA;
    const c128* B = p.B + (int64_t)b * p.bsB;
    c128 acc[4][4];
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) acc[i][j] = mk(0.0, 0.0);

    for (int64_t k0 = kbeg; k0 < kend; k0 += SG_BK) {
        // 64 x 8 elements per operand, 256 threads -> 2 each.  k fastest across threads.
#pragma unroll
        for (int r = 0; r < 2; r++) {
            int e = threadIdx.x + r * 256;
            int kk = e % SG_BK, mm = e / SG_BK;
            int64_t k = k0 + kk;
            int64_t m = m0 + mm, n = n0 + mm;
            As[kk][mm] = (m < p.M && k < kend) ? A[m * p.sam + k * p.sak] : mk(0.0, 0.0);
            Bs[kk][mm] = (n < p.N && k < kend) ? B[n * p.sbn + k * p.sbk] : mk(0.0, 0.0);
        }
        __syncthreads();
#pragma unroll
        for (int kk = 0; kk < SG_BK; kk++) {
            c128 a[4], bb[4];
#pragma unroll
            for (int i = 0; i < 4; i++) a[i] = As[kk][ty + i * SG_T];
#pragma unroll
            for (int j = 0; j < 4; j++) bb[j] = Bs[kk][tx + j * SG_T];
#pragma unroll
            for (int i = 0; i < 4; i++)
#pragma unroll
                for (int j = 0; j < 4; j++) cfma(acc[i][j], a[i], bb[j]);
        }
        __syncthreads();
    }
#pragma unroll
    for (int i = 0; i < 4; i++)
#pragma unroll
        for (int j = 0; j < 4; j++) {
            int64_t m = m0 + ty + i * SG_T, n = n0 + tx + j * SG_T;
            if (m >= p.M || n >= p.N) continue;
            if (p.ksplit > 1) {
                p.partial[((int64_t)blockIdx.z * p.M + m) * p.N + n] = acc[i][j];
            } else {
                c128* c = p.C + (int64_t)b * p.bsC + m * p.csm + n * p.csn;
                c128 r = cmul(p.alpha, acc[i][j]);
                *c = p.accumulate ? cadd(*c, r) : r;
            }
        }
}

// C = alpha * sum_s partial[s] (+ C)
__global__ void splitk_reduce_kernel(GemmParams p)
{
    int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    int64_t per = p.M * p.N;
    if (idx >= per * p.batch) return;
    int64_t b = idx / per, r = idx % per, m = r / p.N, n = r % p.N;
    c128 s = mk(0.0, 0.0);
    for (int q = 0; q < p.ksplit; q++) s = cadd(s, p.partial[(b * p.ksplit + q) * per + r]);
    c128* c = p.C + b * p.bsC + m * p.csm + n * p.csn;
    c128 val = cmul(p.alpha, s);
    *c = p.accumulate ? cadd(*c, val) : val;
}

// y[m*sy] (+)= alpha * sum_k A[m*lda + k] * x[k]        one warp per row
__global__ void gemv_kernel(int64_t M, int64_t K, const c128* __restrict__ A, int64_t lda, const c128* __restrict__ x,
                            c128* __restrict__ y, int64_t sy, c128 alpha, int accumulate)
{
    int64_t row = (int64_t)blockIdx.x * (blockDim.x / 32) + threadIdx.x / 32;
    int lane = threadIdx.x % 32;
    if (row >= M) return;
    const c128* a = A + row * lda;
    c128 acc = mk(0.0, 0.0);
    for (int64_t k = lane; k < K; k += 32) cfma(acc, a[k], x[k]);
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        acc.x += __shfl_xor_sync(0xffffffffu, acc.x, off);
        acc.y += __shfl_xor_sync(0xffffffffu, acc.y, off);
    }
    if (lane == 0) {
        c128 r = cmul(alpha, acc);
        y[row * sy] = accumulate ? cadd(y[row * sy], r) : r;
    }
}
