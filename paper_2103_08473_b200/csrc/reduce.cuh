// Deterministic two-stage reductions and the fused streaming kernels of the amplitude update:
//   * jacobi_multidot_kernel: Jacobi step e = S/D, u = t + e (reading G12) FUSED with the Gram row
//     Re<e_new|e_l> of DIIS (reading G13): S, t and the m-1 stored error vectors are streamed once, e and u written once;
//   * diis_solve_kernel: second stage of that reduction + the bordered Pulay system (<= 13 x 13) on the device, so that
//     an iteration has no mid-iteration host synchronisation;
//   * combine_kernel: t = sum_l c_l u_l with the coefficients read from device memory;
//   * energy_tau_kernel: tau = t2 + P-(t1 t1) (eq 23) with its 3M sum plane, FUSED with the energy
//     reduction (eq 9; reading G11): the tau it leaves behind is the next iteration's GEMM operand.
// Stage-1 partials live in a scratch buffer of the caller's context (RED_SCRATCH_DOUBLES doubles): two contexts on two
// streams never share reduction scratch.  Every sum is formed in a fixed order (fixed tile -> block assignment, fixed
// shuffle trees, stage 2 in one block), so results are bit-reproducible from run to run.
#pragma once
#include "common.cuh"

constexpr int RED_BLOCKS = 592;  // 4 x 148 SMs
constexpr int RED_THREADS = 256;
constexpr int DIIS_MAX = 12;     // ndiis is clamped to this
constexpr int RED_SCRATCH_DOUBLES = RED_BLOCKS * 16;   // stage-1 partials: up to DIIS_MAX (+ padding) per block
constexpr int TILE_COLS = RED_THREADS * 4;             // one tile = one row x 1024 columns of a packed vector

__device__ __forceinline__ double2 block_sum2(double2 v)
{
    __shared__ double2 sh[RED_THREADS / 32];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        v.x += __shfl_xor_sync(0xffffffffu, v.x, off);
        v.y += __shfl_xor_sync(0xffffffffu, v.y, off);
    }
    __syncthreads();   // sh may still be read by a previous call
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
__global__ void __launch_bounds__(RED_THREADS) reduce_stage1(int64_t count, F f, double* __restrict__ partials)
{
    double2 acc = make_double2(0.0, 0.0);
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < count; i += (int64_t)gridDim.x * blockDim.x) {
        double2 t = f(i);
        acc.x += t.x;
        acc.y += t.y;
    }
    double2 r = block_sum2(acc);
    if (threadIdx.x == 0) {
        partials[2 * blockIdx.x] = r.x;
        partials[2 * blockIdx.x + 1] = r.y;
    }
}
// out[0] += sum of .x partials, out[1] += sum of .y partials (if two)
__global__ void __launch_bounds__(RED_THREADS) reduce_stage2(const double* __restrict__ partials, int nblocks, double* out, int two)
{
    double2 acc = make_double2(0.0, 0.0);
    for (int i = threadIdx.x; i < nblocks; i += blockDim.x) {
        acc.x += partials[2 * i];
        acc.y += partials[2 * i + 1];
    }
    double2 r = block_sum2(acc);
    if (threadIdx.x == 0) {
        out[0] += r.x;
        if (two) out[1] += r.y;
    }
}

// out[0..1] += sum_{i < count} f(i)     (scratch: RED_SCRATCH_DOUBLES doubles owned by the caller's context)
template <class F>
static inline void launch_reduce(cudaStream_t st, double* scratch, int64_t count, double* out, int two, F f)
{
    if (count <= 0) return;
    int blocks = (int)((count + RED_THREADS - 1) / RED_THREADS);
    if (blocks > RED_BLOCKS) blocks = RED_BLOCKS;
    reduce_stage1<<<blocks, RED_THREADS, 0, st>>>(count, f, scratch);
    reduce_stage2<<<1, RED_THREADS, 0, st>>>(scratch, blocks, out, two);
    count_launches(2);
}

// out[0] += Re sum conj(x) y
static inline void launch_redot(cudaStream_t st, double* scratch, const c128* x, const c128* y, int64_t count, double* out)
{
    launch_reduce(st, scratch, count, out, 0, [=] __device__(int64_t i) {
        c128 a = x[i], b = y[i];
        return make_double2(fma(a.x, b.x, a.y * b.y), 0.0);
    });
}

// ---------------------------------------------------------------------------------------------------------------
// tiles of a packed amplitude vector [t1 (o x v) | t2p (oo x vv)]: rows [0, oo) are doubles rows (vv columns), rows
// [oo, oo + o) singles rows (v columns); a tile is one row x TILE_COLS columns.  Tiles are dealt to blocks round robin.
// ---------------------------------------------------------------------------------------------------------------
struct VecTiles {
    int o, v;
    int64_t oo, vv, ov;
    int chunks2, chunks1;     // tiles per doubles / singles row
    int64_t ntiles;
};
static inline VecTiles vec_tiles(int o, int v)
{
    VecTiles t;
    t.o = o; t.v = v;
    t.oo = (int64_t)o * (o - 1) / 2; t.vv = (int64_t)v * (v - 1) / 2; t.ov = (int64_t)o * v;
    t.chunks2 = (int)((t.vv + TILE_COLS - 1) / TILE_COLS);
    t.chunks1 = (v + TILE_COLS - 1) / TILE_COLS;
    t.ntiles = t.oo * t.chunks2 + (int64_t)o * t.chunks1;
    return t;
}
static inline int tile_blocks(const VecTiles& t) { return (int)(t.ntiles < RED_BLOCKS ? (t.ntiles > 0 ? t.ntiles : 1) : RED_BLOCKS); }

struct JacobiArgs {
    VecTiles T;
    const c128 *S1, *S2, *t1, *t2p;      // residuals and current amplitudes ([o][v], [(i<j)][(a<b)])
    c128 *E, *U;                          // new error / update vectors, each [ov + oo vv]
    const c128* Eold[DIIS_MAX];           // the m - 1 stored error vectors the new one is dotted with (positions 0..m-2)
    int m;                                // Gram row length; position m - 1 is <e_new|e_new>
    const double* eps;                    // spinor energies used in D (level shift included)
    const int2 *po, *pv;
    int ccd;                              // 1: singles frozen at zero
    double* partials;                     // [gridDim.x][DIIS_MAX]
};

__global__ void __launch_bounds__(RED_THREADS) jacobi_multidot_kernel(const __grid_constant__ JacobiArgs a)
{
    const VecTiles& T = a.T;
    double acc[DIIS_MAX];
#pragma unroll
    for (int k = 0; k < DIIS_MAX; k++) acc[k] = 0.0;
    const int o = T.o, v = T.v;
    const int64_t doubles_tiles = T.oo * T.chunks2;
    for (int64_t tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        const bool dbl = tile < doubles_tiles;
        const int64_t row = dbl ? tile / T.chunks2 : (tile - doubles_tiles) / T.chunks1;
        const int chunk = (int)(dbl ? tile % T.chunks2 : (tile - doubles_tiles) % T.chunks1);
        const int64_t ncols = dbl ? T.vv : v;
        const int64_t base = dbl ? T.ov + row * T.vv : row * v;       // offset of the row in the packed vector
        const c128* S = dbl ? a.S2 + row * T.vv : a.S1 + row * v;
        const c128* t = dbl ? a.t2p + row * T.vv : a.t1 + row * v;
        double erow;
        if (dbl) { const int2 ij = a.po[row]; erow = a.eps[ij.x] + a.eps[ij.y]; } else erow = a.eps[row];
#pragma unroll
        for (int r = 0; r < 4; r++) {
            const int64_t col = (int64_t)chunk * TILE_COLS + r * RED_THREADS + threadIdx.x;
            if (col >= ncols) continue;
            double d;
            if (dbl) { const int2 ab = a.pv[col]; d = erow - a.eps[o + ab.x] - a.eps[o + ab.y]; } else d = erow - a.eps[o + col];
            c128 e, u;
            if (!dbl && a.ccd) {
                e = mk(0.0, 0.0); u = mk(0.0, 0.0);
            } else {
                const c128 s = S[col];
                e = mk(s.x / d, s.y / d);
                u = cadd(t[col], e);
            }
            a.E[base + col] = e;
            a.U[base + col] = u;
#pragma unroll
            for (int k = 0; k < DIIS_MAX - 1; k++)
                if (k < a.m - 1) {
                    const c128 y = a.Eold[k][base + col];
                    acc[k] += fma(e.x, y.x, e.y * y.y);
                }
            const double self = fma(e.x, e.x, e.y * e.y);
#pragma unroll
            for (int k = 0; k < DIIS_MAX; k++)
                if (k == a.m - 1) acc[k] += self;
        }
    }
    // block reduction of the m sums, two at a time
#pragma unroll
    for (int k = 0; k < DIIS_MAX; k += 2) {
        if (k >= a.m) break;
        const double2 r = block_sum2(make_double2(acc[k], acc[k + 1 < DIIS_MAX ? k + 1 : k]));
        if (threadIdx.x == 0) {
            a.partials[(int64_t)blockIdx.x * DIIS_MAX + k] = r.x;
            if (k + 1 < DIIS_MAX) a.partials[(int64_t)blockIdx.x * DIIS_MAX + k + 1] = r.y;
        }
    }
}

// Gaussian elimination with partial pivoting, in place; returns non-zero if singular.  A is dim x dim with row stride 14.
__device__ inline int solve_bordered(double (*A)[14], double* b, int dim)
{
    for (int col = 0; col < dim; col++) {
        int piv = col;
        for (int r = col + 1; r < dim; r++)
            if (fabs(A[r][col]) > fabs(A[piv][col])) piv = r;
        if (!(fabs(A[piv][col]) >= 1e-300) || !isfinite(A[piv][col])) return 1;
        if (piv != col) {
            for (int k = 0; k < dim; k++) { const double t = A[col][k]; A[col][k] = A[piv][k]; A[piv][k] = t; }
            const double t = b[col]; b[col] = b[piv]; b[piv] = t;
        }
        for (int r = col + 1; r < dim; r++) {
            const double fct = A[r][col] / A[col][col];
            for (int k = col; k < dim; k++) A[r][k] -= fct * A[col][k];
            b[r] -= fct * b[col];
        }
    }
    for (int r = dim - 1; r >= 0; r--) {
        double s = b[r];
        for (int k = r + 1; k < dim; k++) s -= A[r][k] * b[k];
        b[r] = s / A[r][r];
        if (!isfinite(b[r])) return 1;
    }
    return 0;
}

struct DiisSolveArgs {
    const double* partials;   // [nblocks][DIIS_MAX]
    int nblocks, m, slot, extrapolate;
    int order[DIIS_MAX + 1];  // slots, oldest first; order[m-1] == slot
    double* gram;             // device, [13][13] by slot
    double* coef;             // device out: coef[k] multiplies u[order[k]]
    double* info;             // device out: info[0] = <e_new|e_new>, info[1] = 1 if every subspace was singular
};
// Second stage of the Gram row, update of the Gram matrix, bordered Pulay system [[B,-1],[-1^T,0]] [c;lambda] = [0;-1] on
// the last mm <= m pairs; a singular system drops the oldest vector and retries (reading G13).
__global__ void __launch_bounds__(RED_THREADS) diis_solve_kernel(const __grid_constant__ DiisSolveArgs a)
{
    __shared__ double dot[DIIS_MAX];
    const int warp = threadIdx.x / 32, lane = threadIdx.x % 32;
    for (int k = warp; k < a.m; k += RED_THREADS / 32) {
        double s = 0.0;
        for (int b = lane; b < a.nblocks; b += 32) s += a.partials[(int64_t)b * DIIS_MAX + k];
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
        if (lane == 0) dot[k] = s;
    }
    __syncthreads();
    if (threadIdx.x != 0) return;
    const int m = a.m;
    for (int k = 0; k < m; k++) {
        a.gram[a.slot * 13 + a.order[k]] = dot[k];
        a.gram[a.order[k] * 13 + a.slot] = dot[k];
    }
    a.info[0] = dot[m - 1];
    a.info[1] = 0.0;
    for (int k = 0; k < DIIS_MAX; k++) a.coef[k] = 0.0;
    if (!a.extrapolate || m < 2) { a.coef[m - 1] = 1.0; return; }
    double A[14][14], rhs[14];
    for (int mm = m; ; mm--) {
        if (mm < 1) { a.info[1] = 1.0; for (int k = 0; k < m; k++) a.coef[k] = 0.0; a.coef[m - 1] = 1.0; return; }
        const int dim = mm + 1;
        for (int r = 0; r < mm; r++)
            for (int q = 0; q < mm; q++) A[r][q] = a.gram[a.order[m - mm + r] * 13 + a.order[m - mm + q]];
        for (int r = 0; r < mm; r++) { A[r][mm] = -1.0; A[mm][r] = -1.0; rhs[r] = 0.0; }
        A[mm][mm] = 0.0;
        rhs[mm] = -1.0;
        if (solve_bordered(A, rhs, dim) == 0) {
            for (int r = 0; r < mm; r++) a.coef[m - mm + r] = rhs[r];
            return;
        }
    }
}

struct DiisCombo {
    int m;
    const double* coef;       // device, DIIS_MAX entries
    const c128* u[DIIS_MAX];
};
__global__ void __launch_bounds__(256) combine_kernel(const __grid_constant__ DiisCombo cb, c128* __restrict__ t1, c128* __restrict__ t2p,
                                                      int64_t n1, int64_t nvec)
{
    double c[DIIS_MAX];
#pragma unroll
    for (int k = 0; k < DIIS_MAX; k++) c[k] = k < cb.m ? cb.coef[k] : 0.0;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < nvec; i += (int64_t)gridDim.x * blockDim.x) {
        c128 s = mk(0.0, 0.0);
#pragma unroll
        for (int k = 0; k < DIIS_MAX; k++)
            if (k < cb.m) {
                const c128 x = cb.u[k][i];
                s.x = fma(c[k], x.x, s.x);
                s.y = fma(c[k], x.y, s.y);
            }
        if (i < n1) t1[i] = s; else t2p[i - n1] = s;
    }
}
static inline void launch_combine(cudaStream_t st, const DiisCombo& cb, c128* t1, c128* t2p, int64_t n1, int64_t nvec)
{
    int64_t blocks = (nvec + 255) / 256;
    if (blocks > 148 * 16) blocks = 148 * 16;
    combine_kernel<<<(unsigned)blocks, 256, 0, st>>>(cb, t1, t2p, n1, nvec);
    count_launches(1);
}

// Host-side bookkeeping of a DIIS subspace (which slot is overwritten next, the age order of the slots) plus the device
// buffers of the solve.  The order never depends on data, so the host needs no read-back to advance it.
struct DiisRing {
    int nd, count, next, norder;
    int order[DIIS_MAX + 1];
    c128 *u, *e;              // [max(nd,1)][nvec]
    double *gram, *coef, *info, *scratch;   // device: 13 x 13, DIIS_MAX, 4, RED_SCRATCH_DOUBLES
    void reset() { count = next = norder = 0; }
};

// One Jacobi + DIIS update of (t1, t2p) from the residuals (S1, S2): 3 launches, no host synchronisation.
// After the call ring.info[0] holds ||S/D||^2 and ring.info[1] the singular flag (device memory).
static inline void launch_jacobi_diis(cudaStream_t st, DiisRing& R, int o, int v, const c128* S1, const c128* S2, c128* t1, c128* t2p,
                                      const double* eps, const int2* po, const int2* pv, int ccd)
{
    const VecTiles T = vec_tiles(o, v);
    const int64_t nvec = T.ov + T.oo * T.vv;
    const int slot = R.nd > 0 ? R.next : 0;
    int order[DIIS_MAX + 1], m = 0;
    if (R.nd > 0) {
        for (int k = 0; k < R.norder; k++)
            if (R.order[k] != slot) order[m++] = R.order[k];   // the slot being overwritten leaves the subspace
        order[m++] = slot;
    } else {
        order[m++] = 0;
    }
    JacobiArgs ja;
    ja.T = T;
    ja.S1 = S1; ja.S2 = S2; ja.t1 = t1; ja.t2p = t2p;
    ja.E = R.e + (int64_t)slot * nvec;
    ja.U = R.u + (int64_t)slot * nvec;
    for (int k = 0; k < DIIS_MAX; k++) ja.Eold[k] = k < m - 1 ? R.e + (int64_t)order[k] * nvec : nullptr;
    ja.m = m;
    ja.eps = eps; ja.po = po; ja.pv = pv; ja.ccd = ccd;
    ja.partials = R.scratch;
    const int blocks = tile_blocks(T);
    jacobi_multidot_kernel<<<blocks, RED_THREADS, 0, st>>>(ja);
    DiisSolveArgs sa;
    sa.partials = R.scratch; sa.nblocks = blocks; sa.m = m; sa.slot = slot; sa.extrapolate = R.nd > 0 ? 1 : 0;
    for (int k = 0; k <= DIIS_MAX; k++) sa.order[k] = k < m ? order[k] : 0;
    sa.gram = R.gram; sa.coef = R.coef; sa.info = R.info;
    diis_solve_kernel<<<1, RED_THREADS, 0, st>>>(sa);
    DiisCombo cb;
    cb.m = m; cb.coef = R.coef;
    for (int k = 0; k < DIIS_MAX; k++) cb.u[k] = k < m ? R.u + (int64_t)order[k] * nvec : nullptr;
    launch_combine(st, cb, t1, t2p, T.ov, nvec);
    count_launches(2);
    if (R.nd > 0) {
        for (int k = 0; k < m; k++) R.order[k] = order[k];
        R.norder = m;
        R.next = (slot + 1) % R.nd;
        if (R.count < R.nd) R.count++;
    }
}

// ---------------------------------------------------------------------------------------------------------------
// tau (eq 23) + its 3M sum plane + the correlation energy (eq 9; reading G11) in one pass over the packed amplitudes:
//   partial sums of  sum_ia f[i][o+a] t1[i][a]  +  sum_{i<j,a<b} <ij||ab> tau^{ab}_{ij}      (complex)
// ---------------------------------------------------------------------------------------------------------------
struct EnergyArgs {
    VecTiles T;
    const c128 *f, *t1, *t2p, *V;         // Fock [n][n], amplitudes, <ij||ab> [(i<j)][(a<b)]
    c128* taup;                           // out: tau [(i<j)][(a<b)]  (may be null: energy only)
    double* plane;                        // out: Re + Im of tau (may be null)
    const int2 *po, *pv;
    int n;
    double* partials;                     // [gridDim.x][2]
};
__global__ void __launch_bounds__(RED_THREADS) energy_tau_kernel(const __grid_constant__ EnergyArgs a)
{
    const VecTiles& T = a.T;
    const int o = T.o, v = T.v;
    const int64_t doubles_tiles = T.oo * T.chunks2;
    c128 acc = mk(0.0, 0.0);
    for (int64_t tile = blockIdx.x; tile < T.ntiles; tile += gridDim.x) {
        const bool dbl = tile < doubles_tiles;
        const int64_t row = dbl ? tile / T.chunks2 : (tile - doubles_tiles) / T.chunks1;
        const int chunk = (int)(dbl ? tile % T.chunks2 : (tile - doubles_tiles) % T.chunks1);
        if (dbl) {
            const int2 ij = a.po[row];
            const c128 *ti = a.t1 + (int64_t)ij.x * v, *tj = a.t1 + (int64_t)ij.y * v;
#pragma unroll
            for (int r = 0; r < 4; r++) {
                const int64_t col = (int64_t)chunk * TILE_COLS + r * RED_THREADS + threadIdx.x;
                if (col >= T.vv) continue;
                const int2 ab = a.pv[col];
                c128 x = a.t2p[row * T.vv + col];
                cfma(x, ti[ab.x], tj[ab.y]);
                x = csub(x, cmul(tj[ab.x], ti[ab.y]));
                if (a.taup) a.taup[row * T.vv + col] = x;
                if (a.plane) a.plane[row * T.vv + col] = x.x + x.y;
                cfma(acc, a.V[row * T.vv + col], x);
            }
        } else {
#pragma unroll
            for (int r = 0; r < 4; r++) {
                const int64_t col = (int64_t)chunk * TILE_COLS + r * RED_THREADS + threadIdx.x;
                if (col >= v) continue;
                cfma(acc, a.f[row * a.n + o + col], a.t1[row * v + col]);
            }
        }
    }
    const double2 r = block_sum2(acc);
    if (threadIdx.x == 0) {
        a.partials[2 * blockIdx.x] = r.x;
        a.partials[2 * blockIdx.x + 1] = r.y;
    }
}
// out[0..1] = E_corr (overwritten, not accumulated)
static inline void launch_energy_tau(cudaStream_t st, double* scratch, const c128* f, int n, int o, int v, const c128* t1,
                                     const c128* t2p, const c128* V, c128* taup, double* plane, const int2* po, const int2* pv,
                                     double* out)
{
    EnergyArgs ea;
    ea.T = vec_tiles(o, v);
    ea.f = f; ea.t1 = t1; ea.t2p = t2p; ea.V = V; ea.taup = taup; ea.plane = plane; ea.po = po; ea.pv = pv; ea.n = n;
    ea.partials = scratch;
    const int blocks = tile_blocks(ea.T);
    cudaMemsetAsync(out, 0, 2 * sizeof(double), st);
    energy_tau_kernel<<<blocks, RED_THREADS, 0, st>>>(ea);
    reduce_stage2<<<1, RED_THREADS, 0, st>>>(scratch, blocks, out, 1);
    count_launches(2);
}
