// Generic "one functor per output layout" fill kernel: out[row*ld + col] (+)= f(row, col).
// Every permutation / (un)packing / antisymmetrisation / elementwise step of the path that is not a GEMM is
// expressed through it (writes are coalesced along col; reads are gathers through L2).  The bandwidth-critical
// plain 4-index transposition has its own shared-memory tiled kernel in transpose.cuh.
#pragma once
#include "common.cuh"

template <class F>
__global__ void __launch_bounds__(256) fill_kernel(c128* __restrict__ out, int64_t rows, int64_t cols, int64_t ld, int add, F f)
{
    const int64_t row = (int64_t)blockIdx.x * blockDim.y + threadIdx.y;
    if (row >= rows) return;
    const int64_t c0 = (int64_t)blockIdx.y * (blockDim.x * 4) + threadIdx.x;
#pragma unroll
    for (int r = 0; r < 4; r++) {
        int64_t col = c0 + (int64_t)r * blockDim.x;
        if (col < cols) {
            c128 val = f(row, col);
            c128* p = out + row * ld + col;
            *p = add ? cadd(*p, val) : val;
        }
    }
}

template <class F>
static inline void launch_fill(cudaStream_t st, c128* out, int64_t rows, int64_t cols, int64_t ld, int add, F f)
{
    if (rows <= 0 || cols <= 0) return;
    int bx = 1;
    while (bx < 256 && bx < cols) bx <<= 1;
    int by = 256 / bx;
    dim3 block(bx, by);
    dim3 grid((unsigned)((rows + by - 1) / by), (unsigned)((cols + (int64_t)bx * 4 - 1) / ((int64_t)bx * 4)));
    fill_kernel<<<grid, block, 0, st>>>(out, rows, cols, ld, add, f);
    count_launches(1);
}

// 3M "sum plane" of a complex buffer: out[i] = Re in[i] + Im in[i]  (gemm_dmma.cuh, DmmaCfg::PL).  Streaming:
// 32 bytes read + 16 bytes written per thread and step.
__global__ void __launch_bounds__(256) sum_plane_kernel(const c128* __restrict__ in, double* __restrict__ out, int64_t n, int pairs)
{
    const int64_t stride = (int64_t)gridDim.x * blockDim.x * 2;
    for (int64_t i = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) * 2; i < n; i += stride) {
        if (i + 1 < n && !pairs) {      // out is only 8-byte aligned (a slab that starts at an odd element)
            const c128 x = in[i], y = in[i + 1];
            out[i] = x.x + x.y;
            out[i + 1] = y.x + y.y;
        } else if (i + 1 < n) {
            const c128 x = in[i], y = in[i + 1];
            *reinterpret_cast<double2*>(out + i) = make_double2(x.x + x.y, y.x + y.y);
        } else {
            const c128 x = in[i];
            out[i] = x.x + x.y;
        }
    }
}
static inline void launch_sum_plane(cudaStream_t st, const c128* in, double* out, int64_t n)
{
    if (n <= 0) return;
    int64_t blocks = (n / 2 + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    if (blocks < 1) blocks = 1;
    sum_plane_kernel<<<(unsigned)blocks, 256, 0, st>>>(in, out, n, (reinterpret_cast<uintptr_t>(out) & 15) == 0 ? 1 : 0);
    count_launches(1);
}

// pair table: tab[p] = (x, y) with x<y, p = pair_idx(x, y, m)
__global__ void pair_table_kernel(int2* tab, int m)
{
    int64_t total = (int64_t)m * (m - 1) / 2;
    int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= total) return;
    // largest x with x*m - x(x+1)/2 <= p
    double mm = (double)m - 0.5;
    int x = (int)floor(mm - sqrt(mm * mm - 2.0 * (double)p));
    if (x < 0) x = 0;
    while (x > 0 && (int64_t)x * m - (int64_t)x * (x + 1) / 2 > p) x--;
    while ((int64_t)(x + 1) * m - (int64_t)(x + 1) * (x + 2) / 2 <= p) x++;
    int y = (int)(p - ((int64_t)x * m - (int64_t)x * (x + 1) / 2)) + x + 1;
    tab[p] = make_int2(x, y);
}
