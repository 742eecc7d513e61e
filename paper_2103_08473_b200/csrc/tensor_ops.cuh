// Generic dense tensor contraction  C[c-indices] (+)= alpha * sum_k A[a-indices] B[b-indices]  for tensors of rank <= 4,
// written with index strings like the contraction strings of the paper ("S(a,b,i,j)+=V(a,b,c,d)*T(c,d,i,j)",
// permuted adds "A(a,c,b,d)+=B(a,b,c,d)").  Both operands are permuted into [free][contracted] matrices (skipped when they
// already are), multiplied by the NT DMMA GEMM of gemm_dmma.cuh, and the result is added into C under one or several index
// orders with signs (the P- operators of the working equations).  Used by the Lambda equations (lambda.cuh), whose ~40
// terms are written one call per printed term; the three big GEMM families of the CCSD iteration keep their
// own pre-laid-out operands.
#pragma once
#include <cstring>
#include "common.cuh"

struct TView {
    const c128* p;
    int rank;
    int64_t dim[4];
    char idx[5];
};
static inline TView tview(const c128* p, const char* idx, int64_t d0, int64_t d1 = 1, int64_t d2 = 1, int64_t d3 = 1)
{
    TView t;
    t.p = p;
    t.rank = (int)strlen(idx);
    t.dim[0] = d0; t.dim[1] = d1; t.dim[2] = d2; t.dim[3] = d3;
    memset(t.idx, 0, sizeof(t.idx));
    strncpy(t.idx, idx, 4);
    return t;
}

struct PermArgs {
    int rank;
    int64_t od[4];        // output extents (row-major, od[rank-1] fastest)
    int64_t is[4];        // input stride of every OUTPUT dimension
    int64_t total;
};
// out[linear] (+)= alpha * in[gathered]; conj: conjugate the input element
__global__ void __launch_bounds__(256) permute_kernel(c128* __restrict__ out, const c128* __restrict__ in, PermArgs a, double alpha,
                                                      int add, int conj)
{
    for (int64_t e = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; e < a.total; e += (int64_t)gridDim.x * blockDim.x) {
        int64_t r = e, off = 0;
#pragma unroll
        for (int q = 3; q >= 0; q--) {
            if (q < a.rank) {
                const int64_t x = r % a.od[q];
                r /= a.od[q];
                off += x * a.is[q];
            }
        }
        c128 v = in[off];
        if (conj) v.y = -v.y;
        v = cscale(alpha, v);
        out[e] = add ? cadd(out[e], v) : v;
    }
}

// out (dense, index order oidx) (+)= alpha * in (dense, index order in.idx); the two strings are permutations of each other
static int permute_into(cudaStream_t st, c128* out, const char* oidx, const TView& in, double alpha, int add, int conj = 0)
{
    PermArgs a;
    a.rank = in.rank;
    if ((int)strlen(oidx) != in.rank) return CCSD_EINVAL;
    int64_t istride[4];
    istride[in.rank - 1] = 1;
    for (int q = in.rank - 2; q >= 0; q--) istride[q] = istride[q + 1] * in.dim[q + 1];
    a.total = 1;
    for (int q = 0; q < in.rank; q++) {
        const char* pos = strchr(in.idx, oidx[q]);
        if (!pos) return CCSD_EINVAL;
        const int k = (int)(pos - in.idx);
        a.od[q] = in.dim[k];
        a.is[q] = istride[k];
        a.total *= in.dim[k];
    }
    for (int q = in.rank; q < 4; q++) { a.od[q] = 1; a.is[q] = 0; }
    if (a.total == 0) return CCSD_OK;
    int64_t blocks = (a.total + 255) / 256;
    if (blocks > 148 * 32) blocks = 148 * 32;
    permute_kernel<<<(unsigned)blocks, 256, 0, st>>>(out, in.p, a, alpha, add, conj);
    count_launches(1);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

struct TcScratch {
    c128 *a, *b, *c;      // permuted operands and the raw GEMM result
    int64_t elems;        // capacity of each
    double *as, *bs;      // 3M sum planes of the operands of the large products (null: the kernel forms the sums itself)
    int64_t plane_elems;  // capacity of each plane
};
struct TcOut {
    const char* idx;      // index order under which the result is added into C
    double sign;
};
