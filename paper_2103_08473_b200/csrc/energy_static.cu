// ccsd_energy_static: the correlation energy of eq 9 (tau of eq 23; reading G11) for callers that
// cannot allocate -- code under stream capture, tight serving loops, harnesses that forbid cudaMalloc.  It is the
// energy_tau_kernel / reduce_stage2 pair of reduce.cuh (the path behind ccsd_contract(CCSD_TERM_ENERGY)) in its "energy
// only" form, with everything that path takes from a caller workspace -- the two pair tables and the per-block partial
// sums -- in ONE file-scope device array of fixed size instead.  Same tile -> block assignment, same shuffle trees, same
// fixed-order second stage: the result has the bits of the workspace path.
//
// A translation unit of its own: the array, the set-up that resolves its device address and the kernels that use it sit
// in this file; nothing here is called by, or changes, the other entry points.
#include "../../include/ccsd.h"
#include "common.cuh"

namespace {

constexpr int ES_BLOCKS = 592;                 // 4 x 148 SMs, as RED_BLOCKS of reduce.cuh
constexpr int ES_THREADS = 256;
constexpr int ES_TILE_COLS = ES_THREADS * 4;   // a tile = one row x 1024 columns of the packed amplitudes
constexpr int64_t ES_MAX_OO = (int64_t)CCSD_ENERGY_STATIC_MAX_NOCC * (CCSD_ENERGY_STATIC_MAX_NOCC - 1) / 2;
constexpr int64_t ES_MAX_VV = (int64_t)CCSD_ENERGY_STATIC_MAX_NVIR * (CCSD_ENERGY_STATIC_MAX_NVIR - 1) / 2;
// layout of the scratch, in 8-byte words: [partials: 2 per block][po: one int2 per (i<j)][pv: one int2 per (a<b)]
constexpr int64_t ES_OFF_PO = 2 * ES_BLOCKS;
constexpr int64_t ES_OFF_PV = ES_OFF_PO + ES_MAX_OO;
constexpr int64_t ES_WORDS = ES_OFF_PV + ES_MAX_VV;
static_assert(ES_WORDS * 8 == CCSD_ENERGY_STATIC_SCRATCH_BYTES, "include/ccsd.h states the size of the static scratch");
static_assert(sizeof(int2) == 8 && sizeof(double) == 8, "one word per table entry");

// The scratch.  Every GPU that loads the library holds these 1.07 MiB until the process exits.  In HOST code this name is
// a host-side stand-in for the symbol, not a device address: only es_scratch() below may be handed to a kernel.
static __device__ __align__(256) unsigned long long g_energy_scratch[ES_WORDS];

struct EsTiles {
    int o, v;
    int64_t oo, vv;
    int chunks2, chunks1;
    int64_t ntiles;
};

__device__ __forceinline__ double2 es_block_sum2(double2 v)
{
    __shared__ double2 sh[ES_THREADS / 32];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, off);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, off);
    }
    __syncthreads();
    if (threadIdx.x % 32 == 0) sh[threadIdx.x / 32] = v;
    __syncthreads();
    double2 r = make_double2(0.0, 0.0);
    if (threadIdx.x < 32) {
        if (threadIdx.x < ES_THREADS / 32) r = sh[threadIdx.x];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) {
            r.x += __shfl_xor_sync(0xffffffffu, r.x, off);
            r.y += __shfl_xor_sync(0xffffffffu, r.y, off);
        }
    }
    return r;
}

// tab[p] = (x, y) of the packed pair p = x m - x (x + 1) / 2 + (y - x - 1), x < y < m
__global__ void es_pair_table_kernel(int2* tab, int m)
{
    const int64_t total = (int64_t)m * (m - 1) / 2;
    const int64_t p = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= total) return;
    const double mm = (double)m - 0.5;
    int x = (int)floor(mm - sqrt(mm * mm - 2.0 * (double)p));
    if (x < 0) x = 0;
    while (x > 0 && (int64_t)x * m - (int64_t)x * (x + 1) / 2 > p) x--;
    while ((int64_t)(x + 1) * m - (int64_t)(x + 1) * (x + 2) / 2 <= p) x++;
    const int y = (int)(p - ((int64_t)x * m - (int64_t)x * (x + 1) / 2)) + x + 1;
    tab[p] = make_int2(x, y);
}

// partial sums of  sum_ia f[i][o+a] t1[i][a]  +  sum_{i<j,a<b} <ij||ab> (t2 + P-(t1 t1))^{ab}_{ij};  one (re, im) per block
__global__ void __launch_bounds__(ES_THREADS)
es_energy_kernel(EsTiles T, const c128* __restrict__ f, int n, const c128* __restrict__ t1, const c128* __restrict__ t2p,
                 const c128* __restrict__ V, const int2* __restrict__ po, const int2* __restrict__ pv, double* __restrict__ partials)
{
    const int o = T.o, v = T.v;
    const int64_t doubles_tiles = T.oo * T.chunks2;
    c128 acc = mk(0.0, 0.0);
    for (int64_t tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        const bool dbl = tile < doubles_tiles;
        const int64_t row = dbl ? tile / T.chunks2 : (tile - doubles_tiles) / T.chunks1;
        const int chunk = (int)(dbl ? tile % T.chunks2 : (tile - doubles_tiles) % T.chunks1);
        if (dbl) {
            const int2 ij = po[row];
            const c128 *ti = t1 + (int64_t)ij.x * v, *tj = t1 + (int64_t)ij.y * v;
#pragma unroll
            for (int r = 0; r < 4; r++) {
                const int64_t col = (int64_t)chunk * ES_TILE_COLS + r * ES_THREADS + threadIdx.x;
                if (col >= T.vv) continue;
                const int2 ab = pv[col];
                c128 x = t2p[row * T.vv + col];
                cfma(x, ti[ab.x], tj[ab.y]);
                x = csub(x, cmul(tj[ab.x], ti[ab.y]));
                cfma(acc, V[row * T.vv + col], x);
            }
        } else {
#pragma unroll
            for (int r = 0; r < 4; r++) {
                const int64_t col = (int64_t)chunk * ES_TILE_COLS + r * ES_THREADS + threadIdx.x;
                if (col >= v) continue;
                cfma(acc, f[row * n + o + col], t1[row * v + col]);
            }
        }
    }
    const double2 r = es_block_sum2(acc);
    if (threadIdx.x == 0) {     // every launched block writes its two words: nothing in the scratch has to start at zero
        partials[2 * blockIdx.x] = r.x;
        partials[2 * blockIdx.x + 1] = r.y;
    }
}

// out[0..1] = the partials summed in a fixed order (0 + sum, as the workspace path forms it)
__global__ void __launch_bounds__(ES_THREADS) es_stage2_kernel(const double* __restrict__ partials, int nblocks, double* out)
{
    double2 acc = make_double2(0.0, 0.0);
    for (int i = threadIdx.x; i < nblocks; i += blockDim.x) {
        acc.x += partials[2 * i];
        acc.y += partials[2 * i + 1];
    }
    const double2 r = es_block_sum2(acc);
    if (threadIdx.x == 0) {
        out[0] = 0.0 + r.x;
        out[1] = 0.0 + r.y;
    }
}

// Device address of g_energy_scratch on the CURRENT device, resolved once per device (idempotent; racing host threads store
// the same value).  cudaGetSymbolAddress allocates nothing: the array is part of the module image.
std::atomic<unsigned long long*> g_scratch_addr[CCSD_MAX_DEVICES];

int es_scratch(unsigned long long** ptr)
{
    int dev = -1;
    CCSD_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= CCSD_MAX_DEVICES) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "ccsd_energy_static: device ordinal %d beyond %d", dev, CCSD_MAX_DEVICES - 1);
        return CCSD_ECUDA;
    }
    unsigned long long* p = g_scratch_addr[dev].load(std::memory_order_acquire);
    if (!p) {
        CCSD_CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_energy_scratch));
        if (!p || reinterpret_cast<uintptr_t>(p) % 256) {
            snprintf(g_cuda_err, sizeof(g_cuda_err), "ccsd_energy_static: bad address %p for the static scratch", (void*)p);
            return CCSD_ECUDA;
        }
        g_scratch_addr[dev].store(p, std::memory_order_release);
    }
    *ptr = p;
    return CCSD_OK;
}

}  // namespace

extern "C" int ccsd_energy_static(int nocc, int nvir, const ccsd_c128* f_, const ccsd_c128* oovv_, const ccsd_c128* t1_,
                                  const ccsd_c128* t2p_, ccsd_c128* e_out, void* cuda_stream)
{
    if (!f_ || !oovv_ || !t1_ || !t2p_ || !e_out || nocc < 2 || nvir < 2) return CCSD_EINVAL;
    if (nocc > CCSD_ENERGY_STATIC_MAX_NOCC || nvir > CCSD_ENERGY_STATIC_MAX_NVIR) {
        snprintf(g_cuda_err, sizeof(g_cuda_err),
                 "ccsd_energy_static: nocc = %d, nvir = %d beyond the static scratch (nocc <= %d, nvir <= %d); use "
                 "ccsd_contract(CCSD_TERM_ENERGY) with a caller workspace", nocc, nvir, CCSD_ENERGY_STATIC_MAX_NOCC,
                 CCSD_ENERGY_STATIC_MAX_NVIR);
        return CCSD_EINVAL;
    }
    unsigned long long* base = nullptr;
    CCSD_TRY(es_scratch(&base));
    double* partials = reinterpret_cast<double*>(base);
    int2* po = reinterpret_cast<int2*>(base + ES_OFF_PO);
    int2* pv = reinterpret_cast<int2*>(base + ES_OFF_PV);

    EsTiles T;
    T.o = nocc; T.v = nvir;
    T.oo = (int64_t)nocc * (nocc - 1) / 2; T.vv = (int64_t)nvir * (nvir - 1) / 2;
    T.chunks2 = (int)((T.vv + ES_TILE_COLS - 1) / ES_TILE_COLS);
    T.chunks1 = (nvir + ES_TILE_COLS - 1) / ES_TILE_COLS;
    T.ntiles = T.oo * T.chunks2 + (int64_t)nocc * T.chunks1;
    const int blocks = (int)(T.ntiles < ES_BLOCKS ? T.ntiles : ES_BLOCKS);

    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    es_pair_table_kernel<<<(unsigned)((T.oo + 255) / 256), 256, 0, st>>>(po, nocc);
    es_pair_table_kernel<<<(unsigned)((T.vv + 255) / 256), 256, 0, st>>>(pv, nvir);
    es_energy_kernel<<<blocks, ES_THREADS, 0, st>>>(T, reinterpret_cast<const c128*>(f_), nocc + nvir, reinterpret_cast<const c128*>(t1_),
                                                    reinterpret_cast<const c128*>(t2p_), reinterpret_cast<const c128*>(oovv_), po, pv,
                                                    partials);
    es_stage2_kernel<<<1, ES_THREADS, 0, st>>>(partials, blocks, reinterpret_cast<double*>(e_out));
    count_launches(4);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}
