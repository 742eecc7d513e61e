// Deterministic two-stage reductions (energy, DIIS Gram entries) and the DIIS linear combination.
#pragma once
#include "common.cuh"

constexpr int RED_BLOCKS = 592;  // 4 x 148 SMs
constexpr int RED_THREADS = 256;
__device__ double g_red_partials[2 * RED_BLOCKS];   // stage-1 partials (one stream at a time per process)

__device__ __forceinline__ double2 block_sum2(double2 v)
{
    __shared__ double2 sh[RED_THREADS / 32];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, off);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, off);
    }
    if (threadIdx.x % 32 == 0) sh[threadIdx.x / 32] = v;
    __syncthreads();
    double2 r = make_double2(0.0, 0.0);
    if (threadIdx.x < 32) {
        if (threadIdx.x < RED_THREADS / 32) r = sh[threadIdx.x];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            r.x += __shfl_xor_sync(0xffffffffu, r.x, off);
            r.y += __shfl_xor_sync(0xffffffffu, r.y, off);
        }
    }
    return r;
}

template <class F>
__global__ void __launch_bounds__(RED_THREADS) reduce_stage1(int64_t count, F f)
{
    double2 acc = make_double2(0.0, 0.0);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x) {
        double2 t = f(i);
        acc.x += t.x;
        acc.y += t.y;
    }
    double2 r = block_sum2(acc);
    if (threadIdx.x == 0) {
        g_red_partials[2 * blockIdx.x] = r.x;
        g_red_partials[2 * blockIdx.x + 1] = r.y;
    }
}
// out[0] += sum of .x partials, out[1] += sum of .y partials (if two)
__global__ void __launch_bounds__(RED_THREADS) reduce_stage2(int nblocks, double* out, int two)
{
    double2 acc = make_double2(0.0, 0.0);
    for (int i = threadIdx.x; i < nblocks; i += blockDim.x) {
        acc.x += g_red_partials[2 * i];
        acc.y += g_red_partials[2 * i + 1];
    }
    double2 r = block_sum2(acc);
    if (threadIdx.x == 0) {
        out[0] += r.x;
        if (two) out[1] += r.y;
    }
}

template <class F>
static inline void launch_reduce(cudaStream_t st, int64_t count, double* out, int two, F f)
{
    if (count <= 0) return;
    int blocks = (int)((count + RED_THREADS - 1) / RED_THREADS);
    if (blocks > RED_BLOCKS) blocks = RED_BLOCKS;
    reduce_stage1<<<blocks, RED_THREADS, 0, st>>>(count, f);
    reduce_stage2<<<1, RED_THREADS, 0, st>>>(blocks, out, two);
    g_launches += 2;
}

// out[0..1] += sum_ia f[i][o+a] t1[i][a] + sum_x V[x] tau[x]     (complex; warp-shuffle reduced)
static inline void launch_energy(cudaStream_t st, const c128* f, int n, int o, int v, const c128* t1, const c128* V,
                                 const c128* taup, int64_t count2, double* out)
{
    launch_reduce(st, (int64_t)o * v, out, 1, [=] __device__(int64_t x) {
        int64_t i = x / v, a = x % v;
        return cmul(f[i * n + o + a], t1[x]);
    });
    launch_reduce(st, count2, out, 1, [=] __device__(int64_t x) { return cmul(V[x], taup[x]); });
}

// out[0] += Re sum conj(x) y
static inline void launch_redot(cudaStream_t st, const c128* x, const c128* y, int64_t count, double* out)
{
    launch_reduce(st, count, out, 0, [=] __device__(int64_t i) {
        c128 a = x[i], b = y[i];
        return make_double2(fma(a.x, b.x, a.y * b.y), 0.0);
    });
}

struct DiisCombo {
    int m;
    double c[12];
    const c128* u[12];
};
__global__ void __launch_bounds__(256) combine_kernel(DiisCombo cb, c128* __restrict__ t1, c128* __restrict__ t2p, int64_t n1, int64_t nvec)
{
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (int64_t)gridDim.x * blockDim.x) {
        c128 s = mk(0.0, 0.0);
        for (int k = 0; k < cb.m; k++) {
            c128 x = cb.u[k][i];
            s.x = fma(cb.c[k], x.x, s.x);
            s.y = fma(cb.c[k], x.y, s.y);
        }
        if (i < n1) t1[i] = s; else t2p[i - n1] = s;
    }
}
static inline void launch_combine(cudaStream_t st, const DiisCombo& cb, c128* t1, c128* t2p, int64_t n1, int64_t nvec)
{
    int64_t blocks = (nvec + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    combine_kernel<<<(unsigned)blocks, 256, 0, st>>>(cb, t1, t2p, n1, nvec);
    g_launches++;
}
