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
// A second scheme, 3M (Karatsuba: three real products per complex product, DmmaCfg::M3), is the default; its operand
// sums Re + Im come from TMA-staged "sum planes" where the caller provides them (DmmaCfg::PL).
//
// Data movement: operands are staged by TMA (cp.async.bulk.tensor) into a 3-6 stage shared-memory ring (DmmaCfg::STAGES,
// as many 16-complex-k stages as fit 220 KB) guarded by full/empty mbarriers.  There is NO producer warp: all eight warps
// issue DMMA, and the TMA issue for k-iteration it + STAGES - 2 is done by lane 0 of warp it % 8 (a ninth warp would cap
// the register budget at 168 per thread and spill the 3M tiles).  The shared-memory layout is
// [k-group of 4 complex][row][64 bytes]: the 16-byte fragment loads of a quarter-warp cover one contiguous 128-byte
// line, so they are bank-conflict free without swizzling; each TMA box is {4 complex} x {rows} (or, with the 4-d
// "wide" maps, one box per operand and stage).  Out-of-range rows / k are zero-filled by TMA, so ragged M, N, K need
// no special code in the main loop.
#pragma once
#include <cuda.h>
#include "gemm_simple.cuh"

constexpr int DMMA_BKG = 4;         // k-groups (of 4 complex) per pipeline stage -> BK = 16 complex

// Tile configuration.  NWM x NWN warps, all of them DMMA consumers (no dedicated producer warp: with 8 warps = 2 per
// SM sub-partition every thread may use 255 registers; a ninth warp would cap them at 168).  Every warp owns MI x NJ
// fragment pairs.  An A fragment is 8 rows x 4 complex k; a B fragment is 4 complex columns (4M: 8 real columns =
// re/im interleaved) or 8 complex columns (3M).
// PL (3M only): the sums Ar + Ai / Br + Bi come from precomputed real "sum planes" (TMA-staged beside the complex
// tiles) instead of DADDs in the main loop: DADD shares the FP64 pipe with DMMA and every DADD between DMMAs costs
// far more than its two issue cycles (measured: 5 % of the kernel).
// PF: fragment loads run one k-group ahead of the DMMAs (two register copies of every fragment).  The 128 x 56 tiles have no
// registers left for that (84 FP64 accumulators x 2 + 9 fragments + planes): they load just in time and rely on the second
// warp of the SM sub-partition to cover the shared-memory latency.
template <int NWM_, int NWN_, int MI_, int NJ_, bool M3_, bool PL_ = false, bool PF_ = true>
struct DmmaCfg {
    static constexpr int NWM = NWM_, NWN = NWN_, MI = MI_, NJ = NJ_;
    static constexpr bool M3 = M3_, PL = PL_, PF = PF_;
    static_assert(!PL_ || M3_, "sum planes belong to the 3M scheme");
    static constexpr int NB = M3_ ? 8 : 4;                       // complex columns per B fragment
    static constexpr int BM = NWM_ * MI_ * 8, BN = NWN_ * NJ_ * NB;
    static constexpr int WARPS = NWM_ * NWN_, THREADS = WARPS * 32;
    static constexpr int A_KG = BM * 64, B_KG = BN * 64;           // bytes per k-group (complex tiles)
    static constexpr int AS_KG = BM * 32, BS_KG = BN * 32;         // bytes per k-group (sum planes)
    static constexpr int A_STAGE = DMMA_BKG * A_KG, B_STAGE = DMMA_BKG * B_KG;
    static constexpr int P_STAGE = PL_ ? DMMA_BKG * (AS_KG + BS_KG) : 0;
    static constexpr int STAGE = A_STAGE + B_STAGE + P_STAGE;
    static constexpr int STAGES = (220 * 1024 / STAGE) > 6 ? 6 : (220 * 1024 / STAGE);
    static constexpr int SMEM = STAGES * STAGE + 2 * STAGES * 8;
    static_assert(BM <= 256 && BN <= 256, "TMA box dimension limit");
    static_assert(STAGES >= 3, "pipeline needs >= 3 stages");
    static_assert(SMEM <= 227 * 1024, "shared memory");
};

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
__device__ __forceinline__ void tma_load_4d(void* dst, const CUtensorMap* map, int c0, int c1, int c2, int c3, uint64_t* bar)
{
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(smem_u32(dst)), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ void dmma884(double& c0, double& c1, double a, double b)
{
    asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                 : "+d"(c0), "+d"(c1) : "d"(a), "d"(b));
}
// x with its sign bit XORed by `mask` (0 or 0x80000000): a negation on the integer pipe, so that the FP64 pipe
// (shared by DMMA and DADD) sees nothing but DMMAs
__device__ __forceinline__ double dsignflip(double x, unsigned mask)
{
    return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}

// Operand loaders: what one k-iteration (16 complex k) of one CTA stages into shared memory.  The loader is a
// __grid_constant__ kernel parameter (the tensor maps must live in parameter space for TMA).
//   setup(p, bz, split, st) -> number of k-iterations of this CTA;   load<Cfg>(st, L, stage, bar, m0, n0) issues the
//   TMA copies of k-iteration L (exactly Cfg::STAGE bytes; out-of-range rows / k are zero-filled by TMA).
struct PlainLoader {   // C = A B^T with both operands K-contiguous, optional batch coordinate, split-K
    CUtensorMap mapA, mapB, mapAs, mapBs;
    // wide = 1: the maps are 4-d views {4 complex k, row, k-group, batch} (k-group stride 64 bytes), so that ONE copy per
    // operand fills a whole stage in the [k-group][row][64 B] layout (4 instead of 16 TMA instructions per k-iteration:
    // the issuing warp issues no DMMA meanwhile, and that time is lost to its SM sub-partition).  Needs K % 4 == 0,
    // because a partial last k-group cannot be zero-filled through the bounds of such a view; wide = 0: 3-d maps
    // {k, row, batch} with one copy per k-group.
    int wide;
    struct State { int64_t kbeg; int cA, cB; };
    __device__ __forceinline__ int setup(const DmmaArgs& p, int bz, int split, State& st) const
    {
        st.kbeg = (int64_t)split * p.kchunk;
        const int64_t kend = (st.kbeg + p.kchunk < p.K) ? st.kbeg + p.kchunk : p.K;
        st.cA = p.batchA ? bz : 0;
        st.cB = p.batchB ? bz : 0;
        return (int)((kend - st.kbeg + 4 * DMMA_BKG - 1) / (4 * DMMA_BKG));
    }
    template <class Cfg>
    __device__ __forceinline__ void load(const State& st, int L, unsigned char* sa, uint64_t* bar, int m0, int n0) const
    {
        unsigned char* sb = sa + Cfg::A_STAGE;
        const int64_t k0 = st.kbeg + (int64_t)L * 4 * DMMA_BKG;
        if (wide) {
            const int gk = (int)(k0 / 4);
            tma_load_4d(sa, &mapA, 0, m0, gk, st.cA, bar);
            tma_load_4d(sb, &mapB, 0, n0, gk, st.cB, bar);
            if constexpr (Cfg::PL) {
                unsigned char* sp = sb + Cfg::B_STAGE;
                tma_load_4d(sp, &mapAs, 0, m0, gk, st.cA, bar);
                tma_load_4d(sp + DMMA_BKG * Cfg::AS_KG, &mapBs, 0, n0, gk, st.cB, bar);
            }
            return;
        }
#pragma unroll
        for (int kg = 0; kg < DMMA_BKG; kg++) {
            const int cd = (int)((k0 + 4 * kg) * 2);   // coordinate in doubles
            tma_load_3d(sa + kg * Cfg::A_KG, &mapA, cd, m0, st.cA, bar);
            tma_load_3d(sb + kg * Cfg::B_KG, &mapB, cd, n0, st.cB, bar);
            if constexpr (Cfg::PL) {
                unsigned char* sp = sb + Cfg::B_STAGE;
                tma_load_3d(sp + kg * Cfg::AS_KG, &mapAs, cd / 2, m0, st.cA, bar);
                tma_load_3d(sp + DMMA_BKG * Cfg::AS_KG + kg * Cfg::BS_KG, &mapBs, cd / 2, n0, st.cB, bar);
            }
        }
    }
};

template <class Cfg, class Loader>
__global__ void __launch_bounds__(Cfg::THREADS, 1)
gemm_dmma_kernel(const __grid_constant__ Loader ld, DmmaArgs p)
{
    constexpr int MI = Cfg::MI, NJ = Cfg::NJ, S = Cfg::STAGES, D = Cfg::STAGES - 2;
    constexpr int A_KG = Cfg::A_KG, B_KG = Cfg::B_KG, A_STAGE = Cfg::A_STAGE, STAGE = Cfg::STAGE;
    extern __shared__ __align__(128) unsigned char smem[];
    uint64_t* full = reinterpret_cast<uint64_t*>(smem + S * STAGE);
    uint64_t* empty = full + S;

    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    const int bz = blockIdx.z / p.ksplit, split = blockIdx.z % p.ksplit;
    const int64_t m0 = (int64_t)blockIdx.y * Cfg::BM, n0 = (int64_t)blockIdx.x * Cfg::BN;
    typename Loader::State lst;
    const int kt = ld.setup(p, bz, split, lst);

    // TMA for k-iteration L into stage L % S (one elected lane).  It is issued D = S - 2 iterations ahead, so the
    // stage it overwrites was released by every warp at least one whole iteration ago: the wait never spins long.
    auto issue = [&](int L) {
        const int s = L % S;
        if (L >= S) mbar_wait(&empty[s], ((L / S) & 1) ^ 1);
        mbar_expect_tx(&full[s], STAGE);
        ld.template load<Cfg>(lst, L, smem + s * STAGE, &full[s], (int)m0, (int)n0);
    };

    if (threadIdx.x == 0) {
        for (int s = 0; s < S; s++) {
            mbar_init(&full[s], 1);
            mbar_init(&empty[s], Cfg::WARPS);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0)
        for (int L = 0; L < D && L < kt; L++) issue(L);

    // warp tile (8 MI) rows x (NB NJ) complex columns; lane (g,q) loads ONE complex A element per A fragment and ONE
    // complex B element per B fragment and k-group.  Fragment loads run one k-group ahead of the DMMAs (also across
    // stage boundaries), so neither the shared-memory latency nor the barrier wait is exposed.
    const int g = lane >> 2, q = lane & 3;
    const int wm = warp % Cfg::NWM, wn = warp / Cfg::NWM;
    const int a_off = (wm * MI * 8 + g) * 64 + q * 16;
    const int b_off = Cfg::M3 ? (wn * NJ * 8 + g) * 64 + q * 16 : (wn * NJ * 4 + (g >> 1)) * 64 + q * 16;
    constexpr int B_ROWS = Cfg::M3 ? 8 : 4;   // rows of the B tile per B fragment

    double2 an[MI], bn[NJ];
    double asn[Cfg::PL ? MI : 1], bsn[Cfg::PL ? NJ : 1];
    const int as_off = (wm * MI * 8 + g) * 32 + q * 8, bs_off = (wn * NJ * 8 + g) * 32 + q * 8;
    auto load_frags = [&](int s, int kg) {
        const unsigned char* sa = smem + s * STAGE + a_off + kg * A_KG;
        const unsigned char* sb = smem + s * STAGE + A_STAGE + b_off + kg * B_KG;
#pragma unroll
        for (int mi = 0; mi < MI; mi++) an[mi] = *reinterpret_cast<const double2*>(sa + mi * 8 * 64);
#pragma unroll
        for (int nj = 0; nj < NJ; nj++) bn[nj] = *reinterpret_cast<const double2*>(sb + nj * B_ROWS * 64);
        if constexpr (Cfg::PL) {
            const unsigned char* sp = smem + s * STAGE + A_STAGE + Cfg::B_STAGE;
            const unsigned char* sas = sp + as_off + kg * Cfg::AS_KG;
            const unsigned char* sbs = sp + DMMA_BKG * Cfg::AS_KG + bs_off + kg * Cfg::BS_KG;
#pragma unroll
            for (int mi = 0; mi < MI; mi++) asn[mi] = *reinterpret_cast<const double*>(sas + mi * 8 * 32);
#pragma unroll
            for (int nj = 0; nj < NJ; nj++) bsn[nj] = *reinterpret_cast<const double*>(sbs + nj * 8 * 32);
        }
    };

    // accumulate: the lines of C this thread will read-modify-write are pulled into L2 now, so that the epilogue's
    // loads do not pay a DRAM latency each (it matters for the short-K products, whose main loop is a few microseconds)
    if (p.accumulate && p.ksplit <= 1) {
#pragma unroll
        for (int mi = 0; mi < MI; mi++) {
            const int64_t m = m0 + wm * MI * 8 + mi * 8 + g;
#pragma unroll
            for (int nj = 0; nj < NJ; nj++) {
                const int64_t n = Cfg::M3 ? n0 + wn * NJ * 8 + nj * 8 + 2 * q : n0 + wn * NJ * 4 + nj * 4 + q;
                if (m < p.M && n < p.N)
                    asm volatile("prefetch.global.L2 [%0];" ::"l"(p.C + (int64_t)bz * p.bsC + m * p.csm + n * p.csn));
            }
        }
    }

    // accumulators: 4M: (Re, Im) of C[row g][col q] per fragment pair;  3M: P1, P2, P3 of C[row g][cols 2q, 2q+1]
    constexpr int NACC = Cfg::M3 ? 3 : 1;
    double acc[NACC][MI][NJ][2];
#pragma unroll
    for (int t = 0; t < NACC; t++)
#pragma unroll
        for (int mi = 0; mi < MI; mi++)
#pragma unroll
            for (int nj = 0; nj < NJ; nj++) { acc[t][mi][nj][0] = 0.0; acc[t][mi][nj][1] = 0.0; }
    const bool odd = g & 1;
    const unsigned negmask = odd ? 0u : 0x80000000u;

    if (Cfg::PF && kt > 0) {
        mbar_wait(&full[0], 0);
        load_frags(0, 0);
    }
    for (int it = 0; it < kt; it++) {
        const int s = it % S;
        if (it + D < kt && warp == it % Cfg::WARPS) {      // producer duty rotates over the warps
            if (lane == 0) issue(it + D);
            __syncwarp();
        }
#pragma unroll
        for (int kg = 0; kg < DMMA_BKG; kg++) {
            double2 a[MI], b[NJ];
            double as[MI], bs[NJ];
            if constexpr (!Cfg::PF) {
                if (kg == 0) mbar_wait(&full[s], (it / S) & 1);
                load_frags(s, kg);
            }
#pragma unroll
            for (int mi = 0; mi < MI; mi++) { a[mi] = an[mi]; if constexpr (Cfg::PL) as[mi] = asn[mi]; }
#pragma unroll
            for (int nj = 0; nj < NJ; nj++) { b[nj] = bn[nj]; if constexpr (Cfg::PL) bs[nj] = bsn[nj]; }
            if constexpr (Cfg::PF) {
                if (kg + 1 < DMMA_BKG) {
                    load_frags(s, kg + 1);
                } else if (it + 1 < kt) {
                    mbar_wait(&full[(it + 1) % S], ((it + 1) / S) & 1);
                    load_frags((it + 1) % S, 0);
                }
            }
            if constexpr (!Cfg::M3) {
                // 4M: DMMA #1 (Re A) x (Re column: Re B | Im column: Im B); DMMA #2 (Im A) x (-Im B | Re B)
#pragma unroll
                for (int nj = 0; nj < NJ; nj++) {
                    const double b1 = odd ? b[nj].y : b[nj].x;
                    const double b2 = dsignflip(odd ? b[nj].x : b[nj].y, negmask);
#pragma unroll
                    for (int mi = 0; mi < MI; mi++) dmma884(acc[0][mi][nj][0], acc[0][mi][nj][1], a[mi].x, b1);
#pragma unroll
                    for (int mi = 0; mi < MI; mi++) dmma884(acc[0][mi][nj][0], acc[0][mi][nj][1], a[mi].y, b2);
                }
            } else {
                // 3M (Karatsuba): P1 = Ar Br, P2 = Ai Bi, P3 = (Ar + Ai)(Br + Bi); Re = P1 - P2, Im = P3 - P1 - P2
                if constexpr (!Cfg::PL) {
#pragma unroll
                    for (int mi = 0; mi < MI; mi++) as[mi] = a[mi].x + a[mi].y;
#pragma unroll
                    for (int nj = 0; nj < NJ; nj++) bs[nj] = b[nj].x + b[nj].y;
                }
#pragma unroll
                for (int nj = 0; nj < NJ; nj++) {
#pragma unroll
                    for (int mi = 0; mi < MI; mi++) dmma884(acc[0][mi][nj][0], acc[0][mi][nj][1], a[mi].x, b[nj].x);
#pragma unroll
                    for (int mi = 0; mi < MI; mi++) dmma884(acc[1][mi][nj][0], acc[1][mi][nj][1], a[mi].y, b[nj].y);
#pragma unroll
                    for (int mi = 0; mi < MI; mi++) dmma884(acc[2][mi][nj][0], acc[2][mi][nj][1], as[mi], bs[nj]);
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(&empty[s]);
    }

    // ===== epilogue =====
    constexpr int NE = Cfg::M3 ? 2 : 1;
#pragma unroll
    for (int mi = 0; mi < MI; mi++) {
        const int64_t m = m0 + wm * MI * 8 + mi * 8 + g;
        if (m >= p.M) continue;
        // accumulate: all the old values of this fragment row are loaded first (NJ x NE independent loads in flight); one
        // load-add-store after the other costs a DRAM latency each, 20 us per CTA for the short-K products of the iteration
        c128 prev[NJ][NE];
        const bool rmw = p.accumulate && p.ksplit <= 1;
        if (rmw) {
#pragma unroll
            for (int nj = 0; nj < NJ; nj++)
#pragma unroll
                for (int e = 0; e < NE; e++) {
                    const int64_t n = Cfg::M3 ? n0 + wn * NJ * 8 + nj * 8 + 2 * q + e : n0 + wn * NJ * 4 + nj * 4 + q;
                    prev[nj][e] = n < p.N ? p.C[(int64_t)bz * p.bsC + m * p.csm + n * p.csn] : mk(0.0, 0.0);
                }
        }
#pragma unroll
        for (int nj = 0; nj < NJ; nj++)
#pragma unroll
            for (int e = 0; e < NE; e++) {
                int64_t n;
                c128 r;
                if constexpr (Cfg::M3) {
                    n = n0 + wn * NJ * 8 + nj * 8 + 2 * q + e;
                    r = mk(acc[0][mi][nj][e] - acc[NACC - 2][mi][nj][e],
                           acc[NACC - 1][mi][nj][e] - acc[0][mi][nj][e] - acc[NACC - 2][mi][nj][e]);
                } else {
                    n = n0 + wn * NJ * 4 + nj * 4 + q;
                    r = mk(acc[0][mi][nj][0], acc[0][mi][nj][1]);
                }
                if (n >= p.N) continue;
                if (p.ksplit > 1) {
                    p.partial[((int64_t)blockIdx.z * p.M + m) * p.N + n] = r;
                } else {
                    c128* c = p.C + (int64_t)bz * p.bsC + m * p.csm + n * p.csn;
                    r = cmul(p.alpha, r);
                    *c = rmw ? cadd(prev[nj][e], r) : r;
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

// 4-d "wide" view of the same operand: {4 complex k (8 doubles), rows, K/4 k-groups, batches}; a box {8, box_rows, 4, 1}
// lands in shared memory as [k-group][row][64 B].  elem_doubles = 2 (complex operand) or 1 (real sum plane, box {4,..}).
static int make_wide_map(CUtensorMap* map, const void* base, int64_t rows, int64_t K, int64_t ld, int nb, int64_t bs, int box_rows,
                         int elem_doubles)
{
    PFN_encodeTiled enc = get_encode_fn();
    if (!enc) { snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled unavailable"); return CCSD_ECUDA; }
    const cuuint64_t eb = 8ull * elem_doubles;   // bytes per element
    cuuint64_t dims[4] = {(cuuint64_t)(4 * elem_doubles), (cuuint64_t)rows, (cuuint64_t)(K / 4), (cuuint64_t)(nb > 0 ? nb : 1)};
    cuuint64_t strides[3] = {(cuuint64_t)ld * eb, 4 * eb, (cuuint64_t)((nb > 1 && bs > 0) ? bs : ld) * eb};
    cuuint32_t box[4] = {(cuuint32_t)(4 * elem_doubles), (cuuint32_t)box_rows, DMMA_BKG, 1};
    cuuint32_t es[4] = {1, 1, 1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled (wide) failed (%d): rows=%lld K=%lld ld=%lld nb=%d", (int)r,
                 (long long)rows, (long long)K, (long long)ld, nb);
        return CCSD_ECUDA;
    }
    return CCSD_OK;
}

// rows x K real sum plane (same leading dimension / batch stride, in elements, as the complex operand it belongs to)
static int make_plane_map(CUtensorMap* map, const double* base, int64_t rows, int64_t K, int64_t ld, int nb, int64_t bs,
                          int box_rows)
{
    PFN_encodeTiled enc = get_encode_fn();
    if (!enc) { snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled unavailable"); return CCSD_ECUDA; }
    cuuint64_t dims[3] = {(cuuint64_t)K, (cuuint64_t)rows, (cuuint64_t)(nb > 0 ? nb : 1)};
    cuuint64_t strides[2] = {(cuuint64_t)(ld * 8), (cuuint64_t)((nb > 1 && bs > 0) ? bs * 8 : ld * 8)};
    cuuint32_t box[3] = {4, (cuuint32_t)box_rows, 1};
    cuuint32_t es[3] = {1, 1, 1};
    CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, const_cast<double*>(base), dims, strides, box, es,
                     CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                     CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "cuTensorMapEncodeTiled (plane) failed (%d): rows=%lld K=%lld ld=%lld", (int)r,
                 (long long)rows, (long long)K, (long long)ld);
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
    if ((p.M + 127) / 128 > 65535) return false;
    if ((int64_t)p.batch * 64 > 65535) return false;
    return true;
}
static inline bool dmma_worthwhile(const GemmParams& p)
{
    return (double)p.M * (double)p.N * (double)p.K * p.batch >= 2.0e5;
}

template <class Cfg>
static int launch_dmma_cfg(cudaStream_t st, const CUtensorMap& mA, const CUtensorMap& mB, const CUtensorMap& mAs,
                           const CUtensorMap& mBs, int wide, const DmmaArgs& a, dim3 grid)
{
    // the dynamic shared-memory limit is a per-device attribute of the function: set once per device
    static std::atomic<bool> configured[CCSD_MAX_DEVICES];
    int dev = 0;
    CCSD_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= CCSD_MAX_DEVICES || !configured[dev].load(std::memory_order_acquire)) {
        CCSD_CUDA_TRY(cudaFuncSetAttribute(gemm_dmma_kernel<Cfg, PlainLoader>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM));
        if (dev >= 0 && dev < CCSD_MAX_DEVICES) configured[dev].store(true, std::memory_order_release);
    }
    PlainLoader ld;
    ld.mapA = mA; ld.mapB = mB; ld.mapAs = mAs; ld.mapBs = mBs;
    ld.wide = wide;
    gemm_dmma_kernel<Cfg, PlainLoader><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(ld, a);
    count_launches(1);
    return CCSD_OK;
}

// The kernel variants that are compiled.  Families: "4M" (variants 0-4) and "3M" (variants 5-7) are the two shipping
// families, column-tile width chosen per launch; the rest are tuning variants reachable through gemm_mode >= 100.
struct DmmaVariant {
    int bm, bn;
    bool m3, planes;
    int (*launch)(cudaStream_t, const CUtensorMap&, const CUtensorMap&, const CUtensorMap&, const CUtensorMap&, int,
                  const DmmaArgs&, dim3);
};
#define DMMA_V(nwm, nwn, mi, nj, m3, ...) \
    {DmmaCfg<nwm, nwn, mi, nj, m3, ##__VA_ARGS__>::BM, DmmaCfg<nwm, nwn, mi, nj, m3, ##__VA_ARGS__>::BN, m3, \
     DmmaCfg<nwm, nwn, mi, nj, m3, ##__VA_ARGS__>::PL, &launch_dmma_cfg<DmmaCfg<nwm, nwn, mi, nj, m3, ##__VA_ARGS__>>}
static const DmmaVariant k_dmma_variants[] = {
    DMMA_V(4, 2, 4, 4, false), DMMA_V(4, 2, 4, 5, false), DMMA_V(4, 2, 4, 6, false), DMMA_V(4, 2, 4, 7, false),
    DMMA_V(4, 2, 4, 8, false),                                       // 0-4: 4M, 128 x {32,40,48,56,64}, 8 warps
    DMMA_V(4, 2, 4, 2, true), DMMA_V(4, 2, 4, 3, true), DMMA_V(4, 2, 4, 4, true),   // 5-7: 3M, 128 x {32,48,64}, 8 warps
    DMMA_V(4, 4, 4, 4, false),                                       // 8: 4M 128 x 64, 16 warps
    DMMA_V(4, 3, 4, 2, true),                                        // 9: 3M 128 x 48, 12 warps
    DMMA_V(4, 3, 4, 5, false),                                       // 10: 4M 128 x 60, 12 warps
    DMMA_V(4, 2, 4, 2, true, true), DMMA_V(4, 2, 4, 3, true, true),  // 11-12: 3M with sum planes, 128 x {32,48}
    DMMA_V(8, 1, 2, 5, true),                                        // 13: 3M 128 x 40, 8 warps in a column (N = nocc products)
    DMMA_V(8, 1, 2, 7, true, false, false), DMMA_V(8, 1, 2, 7, true, true, false),   // 14-15: 3M 128 x 56 (+ planes), one column of warps
};
#undef DMMA_V
constexpr int DMMA_NVARIANTS = (int)(sizeof(k_dmma_variants) / sizeof(k_dmma_variants[0]));
#ifndef CCSD_DEFAULT_3M
#define CCSD_DEFAULT_3M 1
#endif

// Tile variant AND split-K depth of a launch, chosen together against wave quantisation on the SMs: a launch costs
//     waves(tiles x splits) x (k per split + pipeline overhead) x columns of the tile x relative cost per column
// (every CTA tile is 128 rows).  The relative cost per column is measured: narrow tiles re-read the A tile more often and,
// for 3M without planes, spend a larger share of the FP64 pipe on the sums (cfg3 (ov)^3 GEMM: 128x32 vs 128x48 = 1.037
// without planes, 1.026 with; 128x40 = 1.05; 128x56 = 1.00: 74.66 vs 74.63 ms).  For many waves this is "padded columns x
// relative cost" (cfg3: N = 561 -> 12 x 48, N = nvir = 224 -> 4 x 56, N = nocc = 34 -> 40); for the smaller configurations
// the waves decide (cfg2 pp-ladder: 6 x 100 tiles of 48 columns are 4.05 waves, 5 x 100 of 56 columns 3.4).
struct DmmaPlan { int variant, ksplit; int64_t kchunk; double cost; };
static inline DmmaPlan dmma_plan(int64_t M, int64_t N, int64_t K, int64_t batch, bool m3, bool planes, bool may_split, int64_t partial_elems,
                                 int only_variant = -1)
{
    static const int fam_4m[] = {4, 3, 2, 1, 0}, fam_3m[] = {6, 5, 13, 14}, fam_pl[] = {12, 11, 15};
    const int* fam = planes ? fam_pl : (m3 ? fam_3m : fam_4m);
    const int nfam = planes ? 3 : (m3 ? 4 : 5);
    const double overhead = 96.0;   // pipeline fill + epilogue, in units of k
    DmmaPlan best{-1, 1, K, 0.0};
    for (int q = 0; q < (only_variant >= 0 ? 1 : nfam); q++) {
        const int v = only_variant >= 0 ? only_variant : fam[q];
        const int bm = k_dmma_variants[v].bm, bn = k_dmma_variants[v].bn;
        const double rel = !k_dmma_variants[v].m3 ? 1.0 + 0.01 * (64 - bn) / 8.0
                           : bn == 32 ? (k_dmma_variants[v].planes ? 1.026 : 1.037) : bn == 40 ? 1.05 : 1.0;
        const int64_t tiles = ((M + bm - 1) / bm) * ((N + bn - 1) / bn) * batch;
        const int64_t cap = may_split && K >= 512 ? partial_elems / (M * N * batch) : 1;
        for (int ks = 1; ks <= 592 && (ks == 1 || (ks <= cap && K / ks >= 256)); ks++) {
            if (ks > 16 && tiles * ks > 2 * 592) break;   // deep splits only for skinny outputs
            const int64_t chunk = ks == 1 ? K : round_up((K + ks - 1) / ks, 16);
            const int64_t nsplit = (K + chunk - 1) / chunk;
            const int64_t waves = (tiles * nsplit + 147) / 148;
            const double cost = (double)waves * ((double)chunk + overhead) * (ks > 1 ? 1.02 : 1.0) * bn * rel;
            if (best.variant < 0 || cost < best.cost * (ks > 1 ? 0.97 : 0.999)) {   // a split has to pay for its reduction pass
                best.variant = v; best.cost = cost;
                best.ksplit = (int)nsplit; best.kchunk = nsplit > 1 ? chunk : K;
            }
        }
    }
    return best;
}

static int launch_gemm_dmma(cudaStream_t st, const GemmParams& p, int variant)
{
    if (variant < 0 || variant >= DMMA_NVARIANTS) return CCSD_EINVAL;
    const DmmaVariant& V = k_dmma_variants[variant];
    CUtensorMap mA, mB;
    // measured: the wide maps help the 48-column tiles (pp-ladder 0.928 -> 0.935 of peak) but cost the 32-column ones, which
    // move more bytes per flop, 10-15 % (config-4 sweep at nocc = 40: 0.90 -> 0.78; triples GEMM 5.06 -> 5.36 s)
    const int wide = (p.K % 4 == 0 && p.K >= 4 && V.bn >= 48) ? 1 : 0;
    if (V.planes && (!p.As || !p.Bs)) return CCSD_EINVAL;
    CUtensorMap mAs, mBs;
    if (wide) {
        CCSD_TRY(make_wide_map(&mA, p.A, p.M, p.K, p.sam, p.batch, p.bsA, V.bm, 2));
        CCSD_TRY(make_wide_map(&mB, p.B, p.N, p.K, p.sbn, p.batch, p.bsB, V.bn, 2));
        mAs = mA; mBs = mB;           // unused unless the variant stages sum planes
        if (V.planes) {
            CCSD_TRY(make_wide_map(&mAs, p.As, p.M, p.K, p.sam, p.batch, p.bsA, V.bm, 1));
            CCSD_TRY(make_wide_map(&mBs, p.Bs, p.N, p.K, p.sbn, p.batch, p.bsB, V.bn, 1));
        }
    } else {
        CCSD_TRY(make_operand_map(&mA, p.A, p.M, p.K, p.sam, p.batch, p.bsA, V.bm));
        CCSD_TRY(make_operand_map(&mB, p.B, p.N, p.K, p.sbn, p.batch, p.bsB, V.bn));
        mAs = mA; mBs = mB;
        if (V.planes) {
            CCSD_TRY(make_plane_map(&mAs, p.As, p.M, p.K, p.sam, p.batch, p.bsA, V.bm));
            CCSD_TRY(make_plane_map(&mBs, p.Bs, p.N, p.K, p.sbn, p.batch, p.bsB, V.bn));
        }
    }
    DmmaArgs a;
    a.M = p.M; a.N = p.N; a.K = p.K;
    a.C = p.C; a.csm = p.csm; a.csn = p.csn; a.bsC = p.bsC;
    a.alpha = p.alpha; a.accumulate = p.accumulate;
    a.batchA = (p.batch > 1 && p.bsA != 0) ? 1 : 0;
    a.batchB = (p.batch > 1 && p.bsB != 0) ? 1 : 0;
    a.ksplit = p.ksplit; a.kchunk = p.kchunk; a.partial = p.partial;
    dim3 grid((unsigned)((p.N + V.bn - 1) / V.bn), (unsigned)((p.M + V.bm - 1) / V.bm), (unsigned)(p.batch * p.ksplit));
    return V.launch(st, mA, mB, mAs, mBs, wide, a, grid);
}
