// Shared device/host helpers of the CCSD library (product code; shares nothing with oracle/).
#pragma once
#include <cuda_runtime.h>
#include <atomic>
#include <cstdint>
#include <cstdio>

constexpr int CCSD_MAX_DEVICES = 64;   // per-device caches of function attributes

typedef double2 c128;  // (re, im) == ccsd_c128 == torch.complex128

extern thread_local char g_cuda_err[256];
extern std::atomic<long long> g_launches;   // kernels launched by this library (all contexts, all host threads)
extern thread_local long long t_launch_tally;   // ... by this host thread (counts the kernel nodes of a stream capture)
static inline void count_launches(long long n)
{
    g_launches.fetch_add(n, std::memory_order_relaxed);
    t_launch_tally += n;
}

#define CCSD_CUDA_TRY(expr)                                                                      \
    do {                                                                                         \
        cudaError_t _e = (expr);                                                                 \
        if (_e != cudaSuccess) {                                                                 \
            snprintf(g_cuda_err, sizeof(g_cuda_err), "%s at %s:%d", cudaGetErrorString(_e), __FILE__, __LINE__); \
            return CCSD_ECUDA;                                                                   \
        }                                                                                        \
    } while (0)

#define CCSD_TRY(expr)                \
    do {                              \
        int _s = (expr);              \
        if (_s != CCSD_OK) return _s; \
    } while (0)

__host__ __device__ __forceinline__ c128 mk(double re, double im) { return make_double2(re, im); }
__host__ __device__ __forceinline__ c128 cadd(c128 a, c128 b) { return mk(a.x + b.x, a.y + b.y); }
__host__ __device__ __forceinline__ c128 csub(c128 a, c128 b) { return mk(a.x - b.x, a.y - b.y); }
__host__ __device__ __forceinline__ c128 cneg(c128 a) { return mk(-a.x, -a.y); }
__host__ __device__ __forceinline__ c128 cconj(c128 a) { return mk(a.x, -a.y); }
__host__ __device__ __forceinline__ c128 cscale(double s, c128 a) { return mk(s * a.x, s * a.y); }
__host__ __device__ __forceinline__ c128 cmul(c128 a, c128 b) { return mk(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
// acc += a*b
__device__ __forceinline__ void cfma(c128& acc, c128 a, c128 b)
{
    acc.x = fma(a.x, b.x, acc.x);
    acc.x = fma(-a.y, b.y, acc.x);
    acc.y = fma(a.x, b.y, acc.y);
    acc.y = fma(a.y, b.x, acc.y);
}

// packed index of x<y in a dimension of size m (row-major strict upper triangle)
__host__ __device__ __forceinline__ int64_t pair_idx(int x, int y, int m)
{
    return (int64_t)x * m - (int64_t)x * (x + 1) / 2 + (y - x - 1);
}

// signed lookup into a row-major matrix whose COLUMN index is an antisymmetric pair of size m:
//   value(row, x, y) with value(row, y, x) = -value(row, x, y), zero on the diagonal
__device__ __forceinline__ c128 asym_col(const c128* __restrict__ p, int64_t row, int64_t ld, int x, int y, int m)
{
    if (x == y) return mk(0.0, 0.0);
    if (x < y) return p[row * ld + pair_idx(x, y, m)];
    return cneg(p[row * ld + pair_idx(y, x, m)]);
}

// signed lookup into packed amplitudes t2p[(i<j)][(a<b)]
__device__ __forceinline__ c128 t2_at(const c128* __restrict__ t2p, int i, int j, int a, int b, int o, int v, int64_t vv)
{
    if (i == j || a == b) return mk(0.0, 0.0);
    double sgn = 1.0;
    if (i > j) { int t = i; i = j; j = t; sgn = -sgn; }
    if (a > b) { int t = a; a = b; b = t; sgn = -sgn; }
    c128 x = t2p[pair_idx(i, j, o) * vv + pair_idx(a, b, v)];
    return mk(sgn * x.x, sgn * x.y);
}

static inline int64_t round_up(int64_t x, int64_t m) { return (x + m - 1) / m * m; }
