// Perturbative triples +T, (T), -T (arXiv 2103.08473 Appendix 7.3, eqs 39-44).
//
// For every unique occupied triple i<j<k the connected driver of eq 40 is ONE complex GEMM on the DMMA kernel of
// gemm_dmma.cuh with a segmented K dimension (TripLoader):
//     Mt[(a<b)][c] = sum_e ( <ab||ie> t2[j,k,e,c] + <ab||je> t2[k,i,e,c] + <ab||ke> t2[i,j,e,c] )          3 x v
//                  + sum_m ( <cm||ij> t2[k,m,a,b] + <cm||jk> t2[i,m,a,b] + <cm||ki> t2[j,m,a,b] )          3 x o
// (the hole terms of eq 40, sum_m <am||ij> t2[k,m,b,c], are antisymmetric in (b,c) instead of (a,b); stored with
// their lone index last they share the layout of the particle terms), so that for a<b<c
//     Wbar[a,b,c] = W^abc + W^bca + W^cab = Mt[(ab)][c] + Mt[(bc)][a] - Mt[(ac)][b]      (Mt is stored transposed).
// Zbar (eq 42) and Ybar (eq 44) have the same cyclic structure with rank-3 "matrices" formed on the fly.  A batch of
// triples is one launch (grid.z); the three energies are reduced deterministically (per-block partials, fixed order).
// The paper blocks the occupied space to bound the n_red^3 v^3 working set; here the batch of triples
// per launch plays that role (Mt: vv x v per triple).
// Reading G22: brackets of eq 40 are V^{ab}_{ie}, V^{am}_{ij}; left factors are conjugated; D < 0.
#pragma once
#include "gemm_dmma.cuh"
#include "fill.cuh"

// K-segmented operand loader: k-iteration L belongs to one of six segments (three particle, three hole); each segment
// is a (batch coordinate of A, batch coordinate of B) pair derived from the CTA's (i,j,k).
struct TripLoader {
    CUtensorMap PA, PB, PAs, PBs;   // particle: A = -<ab||xe> [x][(a<b)][e],  B = t2[z,y,e,c] as [(z,y)][c][e]
    CUtensorMap HA, HB, HAs, HBs;   // hole:     A = t2[z,m,a,b] [z][(a<b)][m],  B = <cm||xy> as [(x,y)][c][m]
    const int4* ijk;
    int o, op;
    int tp;                         // k-iterations per particle segment (16 e each)
    int ngh, th;                    // hole part: k-GROUPS (4 m each) per segment; k-iterations of the three segments together
    struct State { int i, j, k; };
    __device__ __forceinline__ int setup(const DmmaArgs&, int bz, int, State& st) const
    {
        const int4 t = ijk[bz];
        st.i = t.x; st.j = t.y; st.k = t.z;
        return 3 * tp + th;
    }
    // (x,y,z) = (i,j,k), (j,k,i), (k,i,j)
    __device__ __forceinline__ void cyc(const State& st, int seg, int& x, int& y, int& z) const
    {
        x = seg == 0 ? st.i : (seg == 1 ? st.j : st.k);
        y = seg == 0 ? st.j : (seg == 1 ? st.k : st.i);
        z = seg == 0 ? st.k : (seg == 1 ? st.i : st.j);
    }
    template <class Cfg>
    __device__ __forceinline__ void load(const State& st, int L, unsigned char* sa, uint64_t* bar, int m0, int n0) const
    {
        unsigned char* sb = sa + Cfg::A_STAGE;
        unsigned char* sp = sb + Cfg::B_STAGE;
        if (L < 3 * tp) {   // particle segments: whole k-iterations
            const int seg = L / tp, kk = (L - seg * tp) * 4 * DMMA_BKG;
            int x, y, z;
            cyc(st, seg, x, y, z);
            const int cA = x, cB = z * o + y;
#pragma unroll
            for (int kg = 0; kg < DMMA_BKG; kg++) {
                const int cd = (kk + 4 * kg) * 2;
                tma_load_3d(sa + kg * Cfg::A_KG, &PA, cd, m0, cA, bar);
                tma_load_3d(sb + kg * Cfg::B_KG, &PB, cd, n0, cB, bar);
                if constexpr (Cfg::PL) {
                    tma_load_3d(sp + kg * Cfg::AS_KG, &PAs, cd / 2, m0, cA, bar);
                    tma_load_3d(sp + DMMA_BKG * Cfg::AS_KG + kg * Cfg::BS_KG, &PBs, cd / 2, n0, cB, bar);
                }
            }
            return;
        }
        // hole segments: nocc is small (34 at cfg3), so they are packed at k-GROUP granularity -- the three segments follow
        // each other without rounding each up to a whole k-iteration (3 x 34 -> 7 instead of 9 iterations of 16).  A k-group
        // is its own TMA copy anyway; k-groups beyond the last segment read out of range and are zero-filled.
        const int g0 = (L - 3 * tp) * DMMA_BKG;
#pragma unroll
        for (int kg = 0; kg < DMMA_BKG; kg++) {
            const int G = g0 + kg;
            const int seg = (G >= ngh) + (G >= 2 * ngh);
            int x, y, z;
            cyc(st, seg, x, y, z);
            const int cA = z, cB = x * o + y;
            const int cd = G >= 3 * ngh ? 2 * op : (G - seg * ngh) * 8;      // doubles; 2 op = out of range -> zeros
            tma_load_3d(sa + kg * Cfg::A_KG, &HA, cd, m0, cA, bar);
            tma_load_3d(sb + kg * Cfg::B_KG, &HB, cd, n0, cB, bar);
            if constexpr (Cfg::PL) {
                tma_load_3d(sp + kg * Cfg::AS_KG, &HAs, cd / 2, m0, cA, bar);
                tma_load_3d(sp + DMMA_BKG * Cfg::AS_KG + kg * Cfg::BS_KG, &HBs, cd / 2, n0, cB, bar);
            }
        }
    }
};

template <class Cfg>
static int launch_trip_cfg(cudaStream_t st, const TripLoader& ld, const DmmaArgs& a, dim3 grid)
{
    static std::atomic<bool> configured[CCSD_MAX_DEVICES];   // per device, as in launch_dmma_cfg
    int dev = 0;
    CCSD_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= CCSD_MAX_DEVICES || !configured[dev].load(std::memory_order_acquire)) {
        CCSD_CUDA_TRY(cudaFuncSetAttribute(gemm_dmma_kernel<Cfg, TripLoader>, cudaFuncAttributeMaxDynamicSharedMemorySize, Cfg::SMEM));
        if (dev >= 0 && dev < CCSD_MAX_DEVICES) configured[dev].store(true, std::memory_order_release);
    }
    gemm_dmma_kernel<Cfg, TripLoader><<<grid, Cfg::THREADS, Cfg::SMEM, st>>>(ld, a);
    count_launches(1);
    return CCSD_OK;
}

struct TripVariant {
    int bm, bn;
    bool planes;
    int (*launch)(cudaStream_t, const TripLoader&, const DmmaArgs&, dim3);
};
static const TripVariant k_trip_variants[] = {
    {128, 32, false, &launch_trip_cfg<DmmaCfg<4, 2, 4, 2, true>>},
    {128, 48, false, &launch_trip_cfg<DmmaCfg<4, 2, 4, 3, true>>},
    {128, 32, true, &launch_trip_cfg<DmmaCfg<4, 2, 4, 2, true, true>>},
    {128, 48, true, &launch_trip_cfg<DmmaCfg<4, 2, 4, 3, true, true>>},
    {128, 56, false, &launch_trip_cfg<DmmaCfg<8, 1, 2, 7, true, false, false>>},
    {128, 56, true, &launch_trip_cfg<DmmaCfg<8, 1, 2, 7, true, true, false>>},
};

// ---- what the energy kernel needs of one triple --------------------------------------------------------------------
struct TripData {
    const c128* t1;        // [o][v]
    const c128* t2p;       // [(i<j)][(a<b)]
    const c128* Voovv_p;   // <ij||ab> [(i<j)][(a<b)]
    const c128* f;         // [n][n]
    const double* eps;
    int o, v, n;
    int64_t vv;
};

// the three occupied pairs (ij), (jk), (ki) = -(ik) of a triple with their lone indices k, i, j
struct TripPairs {
    int64_t p[3];   // packed occupied-pair rows
    double sg[3];
    int s[3];
};
__device__ __forceinline__ TripPairs trip_pairs(int i, int j, int k, int o)
{
    TripPairs t;
    t.p[0] = pair_idx(i, j, o); t.sg[0] = 1.0; t.s[0] = k;
    t.p[1] = pair_idx(j, k, o); t.sg[1] = 1.0; t.s[1] = i;
    t.p[2] = pair_idx(i, k, o); t.sg[2] = -1.0; t.s[2] = j;
    return t;
}
// Zt[(xy)][z] = sum_r <xy||p_r> t1[s_r, z] + t2[p_r, (xy)] conj(f[s_r, z])  (eq 42; <xy||ij> = conj <ij||xy>)
// Yt[(xy)][z] = sum_r t2[p_r, (xy)] t1[s_r, z]                                (eq 44, the t2 t1 part)
__device__ __forceinline__ void trip_zy(const TripData& d, const TripPairs& tp, int64_t XY, int z, c128& Z, c128& Y)
{
#pragma unroll
    for (int r = 0; r < 3; r++) {
        const c128 V = cconj(d.Voovv_p[tp.p[r] * d.vv + XY]);
        const c128 T = d.t2p[tp.p[r] * d.vv + XY];
        const c128 t = cscale(tp.sg[r], d.t1[tp.s[r] * d.v + z]);
        const c128 fc = cscale(tp.sg[r], cconj(d.f[(int64_t)tp.s[r] * d.n + d.o + z]));
        cfma(Z, V, t);
        cfma(Z, T, fc);
        cfma(Y, T, t);
    }
}
// Wbar, Zbar, Ybar of one (i<j<k, a<b<c).  The GEMM writes its result transposed, Mc[c][(a<b)] = Mt[(a<b)][c], so that
// for consecutive (b<c) pairs at fixed a two of the three reads (and every read of the pair-indexed tensors) are
// contiguous; a second, row-major copy for the third read costs more in the GEMM epilogue than it saves here.
__device__ __forceinline__ void trip_element(const TripData& d, const TripPairs& tp,
                                             const c128* __restrict__ Mc, int i, int j, int k, int a, int b, int c,
                                             int64_t AB, int64_t BC, c128& W, c128& Z, c128& Y)
{
    const int v = d.v;
    const int64_t AC = pair_idx(a, c, v);
    W = csub(cadd(Mc[c * d.vv + AB], Mc[a * d.vv + BC]), Mc[b * d.vv + AC]);
    c128 z1 = mk(0, 0), y1 = mk(0, 0), z2 = mk(0, 0), y2 = mk(0, 0), z3 = mk(0, 0), y3 = mk(0, 0);
    trip_zy(d, tp, AB, c, z1, y1);
    trip_zy(d, tp, BC, a, z2, y2);
    trip_zy(d, tp, AC, b, z3, y3);
    Z = csub(cadd(z1, z2), z3);
    Y = csub(cadd(y1, y2), y3);
    // t1^3 part of eq 44: the cyclic sum of its 6 terms / 3 is the determinant of t1[{i,j,k}][{a,b,c}]
    const c128 ia = d.t1[i * v + a], ib = d.t1[i * v + b], ic = d.t1[i * v + c];
    const c128 ja = d.t1[j * v + a], jb = d.t1[j * v + b], jc = d.t1[j * v + c];
    const c128 ka = d.t1[k * v + a], kb = d.t1[k * v + b], kc = d.t1[k * v + c];
    c128 det = cmul(ia, csub(cmul(jb, kc), cmul(kb, jc)));
    det = csub(det, cmul(ja, csub(cmul(ib, kc), cmul(kb, ic))));
    det = cadd(det, cmul(ka, csub(cmul(ib, jc), cmul(jb, ic))));
    Y = cadd(Y, det);
}

constexpr int TRIP_THREADS = 256;
// grid (v - 2, nb): block (a, batch entry); the threads walk the packed pairs (b<c) with b > a, which are the
// contiguous tail [pair_idx(a+1, a+2), vv) of the pair table.  partials[(bz*gridDim.x + a)*5 + {0..4}] = sums of
//   |Wbar|^2/D, Re/Im conj(Zbar) Wbar / D, Re/Im conj(Ybar) Wbar        (eqs 39, 41, 43 over a<b<c)
__global__ void __launch_bounds__(TRIP_THREADS) trip_energy_kernel(TripData d, const c128* __restrict__ Mcbuf, int64_t bsM,
                                                                   const int4* __restrict__ ijk, const int2* __restrict__ pv,
                                                                   double* __restrict__ partials)
{
    const int a = blockIdx.x, bz = blockIdx.y, v = d.v, o = d.o;
    const int4 t = ijk[bz];
    const int i = t.x, j = t.y, k = t.z;
    const c128* Mc = Mcbuf + (int64_t)bz * bsM;
    const TripPairs tp = trip_pairs(i, j, k, o);
    const double eoa = d.eps[i] + d.eps[j] + d.eps[k] - d.eps[o + a];
    double acc[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (int64_t BC = pair_idx(a + 1, a + 2, v) + threadIdx.x; BC < d.vv; BC += TRIP_THREADS) {
        const int2 bc = pv[BC];
        c128 W, Z, Y;
        trip_element(d, tp, Mc, i, j, k, a, bc.x, bc.y, pair_idx(a, bc.x, v), BC, W, Z, Y);
        const double rD = 1.0 / (eoa - d.eps[o + bc.x] - d.eps[o + bc.y]);
        acc[0] += (W.x * W.x + W.y * W.y) * rD;
        acc[1] += (Z.x * W.x + Z.y * W.y) * rD;     // Re conj(Z) W
        acc[2] += (Z.x * W.y - Z.y * W.x) * rD;     // Im conj(Z) W
        acc[3] += Y.x * W.x + Y.y * W.y;
        acc[4] += Y.x * W.y - Y.y * W.x;
    }
    __shared__ double sh[TRIP_THREADS / 32][5];
#pragma unroll
    for (int q = 0; q < 5; q++) {
        double x = acc[q];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x += __shfl_xor_sync(0xffffffffu, x, off);
        if (threadIdx.x % 32 == 0) sh[threadIdx.x / 32][q] = x;
    }
    __syncthreads();
    if (threadIdx.x < 5) {
        double x = 0.0;
        for (int w = 0; w < TRIP_THREADS / 32; w++) x += sh[w][threadIdx.x];
        partials[((int64_t)bz * gridDim.x + a) * 5 + threadIdx.x] = x;
    }
}
// acc[q] += sum over `count` blocks of partials[.][q], in a fixed order (one block, deterministic)
__global__ void __launch_bounds__(256) trip_reduce_kernel(const double* __restrict__ partials, int64_t count, double* __restrict__ acc)
{
    __shared__ double sh[8][5];
    double s[5] = {0.0, 0.0, 0.0, 0.0, 0.0};
    for (int64_t x = threadIdx.x; x < count; x += 256)
#pragma unroll
        for (int q = 0; q < 5; q++) s[q] += partials[x * 5 + q];
#pragma unroll
    for (int q = 0; q < 5; q++) {
        double x = s[q];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) x += __shfl_xor_sync(0xffffffffu, x, off);
        if (threadIdx.x % 32 == 0) sh[threadIdx.x / 32][q] = x;
    }
    __syncthreads();
    if (threadIdx.x < 5) {
        double x = 0.0;
        for (int w = 0; w < 8; w++) x += sh[w][threadIdx.x];
        acc[threadIdx.x] += x;
    }
}

// parity hook: dense, fully antisymmetric Wbar/Zbar/Ybar[a][b][c] of ONE triple (buffers zeroed by the caller)
__global__ void __launch_bounds__(TRIP_THREADS) trip_dense_kernel(TripData d, const c128* __restrict__ Mc,
                                                                  const int2* __restrict__ pv, int i, int j, int k,
                                                                  c128* __restrict__ Wd, c128* __restrict__ Zd, c128* __restrict__ Yd)
{
    const int a = blockIdx.x, v = d.v;
    const TripPairs tp = trip_pairs(i, j, k, d.o);
    for (int64_t BC = pair_idx(a + 1, a + 2, v) + threadIdx.x; BC < d.vv; BC += TRIP_THREADS) {
        const int b = pv[BC].x, c = pv[BC].y;
        c128 W, Z, Y;
        trip_element(d, tp, Mc, i, j, k, a, b, c, pair_idx(a, b, v), BC, W, Z, Y);
        const int64_t idx[6] = {((int64_t)a * v + b) * v + c, ((int64_t)b * v + c) * v + a, ((int64_t)c * v + a) * v + b,
                                ((int64_t)b * v + a) * v + c, ((int64_t)a * v + c) * v + b, ((int64_t)c * v + b) * v + a};
#pragma unroll
        for (int q = 0; q < 6; q++) {
            const double sg = q < 3 ? 1.0 : -1.0;
            if (Wd) Wd[idx[q]] = cscale(sg, W);
            if (Zd) Zd[idx[q]] = cscale(sg, Z);
            if (Yd) Yd[idx[q]] = cscale(sg, Y);
        }
    }
}
