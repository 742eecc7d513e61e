// Bandwidth-bound tensor transposition kernels ("A(a,c,b,d) += B(a,b,c,d)").
// complex128 elements are 16 bytes: every global access is one 16-byte vector load/store per thread, a warp
// covers 512 contiguous bytes on both the read and the write side; the 32x32 tile goes through padded shared
// memory so that neither side is strided in HBM.
#pragma once
#include "common.cuh"

constexpr int TR_TILE = 32;

// General 4-index permutation.  Input extents d[4] (row-major, d[3] fastest).  x runs over input dim 3, y over the
// input dim p that becomes the fastest output dim; r1, r2 are the two remaining input dims.
struct Tr4 {
    int64_t nx, ny, n1, n2;        // extents: x = in dim 3, y = in dim p, r1, r2
    int64_t iy, i1, i2;            // input strides of y, r1, r2 (x has stride 1)
    int64_t ox, o1, o2;            // output strides of x, r1, r2 (y has stride 1)
    int conj;
};

__global__ void __launch_bounds__(256) transpose4_kernel(const c128* __restrict__ in, c128* __restrict__ out, Tr4 t)
{
    __shared__ c128 tile[TR_TILE][TR_TILE + 1];
    const int64_t tx_n = (t.nx + TR_TILE - 1) / TR_TILE, ty_n = (t.ny + TR_TILE - 1) / TR_TILE;
    int64_t b = blockIdx.x;
    const int64_t bx = b % tx_n; b /= tx_n;
    const int64_t by = b % ty_n; b /= ty_n;
    const int64_t r1 = b % t.n1, r2 = b / t.n1;
    const c128* src = in + r1 * t.i1 + r2 * t.i2;
    c128* dst = out + r1 * t.o1 + r2 * t.o2;
    const int lx = threadIdx.x % TR_TILE, ly = threadIdx.x / TR_TILE;   // 32 x 8
#pragma unroll
    for (int k = 0; k < TR_TILE; k += 8) {
        int64_t x = bx * TR_TILE + lx, y = by * TR_TILE + ly + k;
        if (x < t.nx && y < t.ny) {
            c128 val = src[y * t.iy + x];
            if (t.conj) val.y = -val.y;
            tile[ly + k][lx] = val;
        }
    }
    __syncthreads();
#pragma unroll
    for (int k = 0; k < TR_TILE; k += 8) {
        int64_t y = by * TR_TILE + lx, x = bx * TR_TILE + ly + k;
        if (x < t.nx && y < t.ny) dst[x * t.ox + y] = tile[lx][ly + k];
    }
}

// Fastest index preserved: plain strided row copy.  rows enumerate the three slow input dims.
struct Cp4 {
    int64_t nx, n0, n1, n2;
    int64_t i0, i1, i2, o0, o1, o2;
    int conj;
};
__global__ void __launch_bounds__(256) copy4_kernel(const c128* __restrict__ in, c128* __restrict__ out, Cp4 t)
{
    int64_t row = (int64_t)blockIdx.x * blockDim.y + threadIdx.y;
    if (row >= t.n0 * t.n1 * t.n2) return;
    int64_t a2 = row % t.n2, a1 = (row / t.n2) % t.n1, a0 = row / (t.n2 * t.n1);
    const c128* src = in + a0 * t.i0 + a1 * t.i1 + a2 * t.i2;
    c128* dst = out + a0 * t.o0 + a1 * t.o1 + a2 * t.o2;
    for (int64_t x = (int64_t)blockIdx.y * blockDim.x + threadIdx.x; x < t.nx; x += (int64_t)gridDim.y * blockDim.x) {
        c128 val = src[x];
        if (t.conj) val.y = -val.y;
        dst[x] = val;
    }
}

// out[c*ld_out + r] = in[r*ld_in + c]
static inline int launch_transpose2d_ld(cudaStream_t st, const c128* in, int64_t ld_in, c128* out, int64_t ld_out,
                                        int64_t rows, int64_t cols, int conj)
{
    if (rows <= 0 || cols <= 0) return CCSD_OK;
    Tr4 t;
    t.nx = cols; t.ny = rows; t.n1 = 1; t.n2 = 1;
    t.iy = ld_in; t.i1 = 0; t.i2 = 0;
    t.ox = ld_out; t.o1 = 0; t.o2 = 0;
    t.conj = conj;
    int64_t blocks = ((cols + TR_TILE - 1) / TR_TILE) * ((rows + TR_TILE - 1) / TR_TILE);
    if (blocks > 0x7fffffffLL) return CCSD_EINVAL;
    transpose4_kernel<<<(unsigned)blocks, 256, 0, st>>>(in, out, t);
    g_launches++;
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}
static inline int launch_transpose2d(cudaStream_t st, const c128* in, c128* out, int64_t rows, int64_t cols, int conj)
{
    return launch_transpose2d_ld(st, in, cols, out, rows, rows, cols, conj);
}

// out dimension q is input dimension perm[q]
static inline int launch_transpose4d(cudaStream_t st, const c128* in, c128* out, const int64_t d[4], const int perm[4], int conj)
{
    int seen[4] = {0, 0, 0, 0};
    for (int q = 0; q < 4; q++) {
        if (perm[q] < 0 || perm[q] > 3 || seen[perm[q]]) return CCSD_EINVAL;
        seen[perm[q]] = 1;
        if (d[q] < 0) return CCSD_EINVAL;
    }
    if (d[0] * d[1] * d[2] * d[3] == 0) return CCSD_OK;
    int64_t is[4] = {d[1] * d[2] * d[3], d[2] * d[3], d[3], 1};
    int64_t od[4], os[4], os_of_in[4];
    for (int q = 0; q < 4; q++) od[q] = d[perm[q]];
    os[3] = 1; os[2] = od[3]; os[1] = od[2] * od[3]; os[0] = od[1] * od[2] * od[3];
    for (int q = 0; q < 4; q++) os_of_in[perm[q]] = os[q];
    if (perm[3] == 3) {
        Cp4 t;
        t.nx = d[3]; t.n0 = d[0]; t.n1 = d[1]; t.n2 = d[2];
        t.i0 = is[0]; t.i1 = is[1]; t.i2 = is[2];
        t.o0 = os_of_in[0]; t.o1 = os_of_in[1]; t.o2 = os_of_in[2];
        t.conj = conj;
        int bx = 1;
        while (bx < 256 && bx < d[3]) bx <<= 1;
        int by = 256 / bx;
        int64_t rows = d[0] * d[1] * d[2];
        int64_t gy = (d[3] + bx - 1) / bx;
        if (gy > 64) gy = 64;
        dim3 grid((unsigned)((rows + by - 1) / by), (unsigned)gy), block(bx, by);
        copy4_kernel<<<grid, block, 0, st>>>(in, out, t);
    } else {
        int p = perm[3];           // input dim that becomes fastest in the output
        int r[2], nr = 0;
        for (int q = 0; q < 3; q++)
            if (q != p) r[nr++] = q;
        Tr4 t;
        t.nx = d[3]; t.ny = d[p]; t.n1 = d[r[0]]; t.n2 = d[r[1]];
        t.iy = is[p]; t.i1 = is[r[0]]; t.i2 = is[r[1]];
        t.ox = os_of_in[3]; t.o1 = os_of_in[r[0]]; t.o2 = os_of_in[r[1]];
        t.conj = conj;
        int64_t blocks = ((t.nx + TR_TILE - 1) / TR_TILE) * ((t.ny + TR_TILE - 1) / TR_TILE) * t.n1 * t.n2;
        if (blocks > 0x7fffffffLL) return CCSD_EINVAL;
        transpose4_kernel<<<(unsigned)blocks, 256, 0, st>>>(in, out, t);
    }
    g_launches++;
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}
