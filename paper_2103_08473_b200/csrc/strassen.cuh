// One or two levels of Strassen's algorithm around the DMMA GEMM (gemm_dmma.cuh) for the large contractions of eq 32 / eqs 29-30
// (PAPER.md:594-606): C = A B^T with every dimension halved is 7 half-size products instead of 8, i.e. 7/8 of the FP64
// tensor-pipe work (49 quarter-size products for 64 with two levels: 0.766), for three streaming passes (operand sums,
// result sums).  All arithmetic stays FP64; the result differs from the plain product by rounding only (measured max error
// 2e-15 - 1.2e-14 of the largest element against 1-7e-15 for the plain 3M product; the parity bound
// is 1e-12).
//
// "NT" convention of the library: C[m][n] = sum_k A[m][k] B[n][k].  Quadrants by halves (Mh, Nh, Kh = ceil of half the
// extent, Kh rounded up to even so that plane rows stay 16-byte aligned; what lies beyond the extent reads as zero):
//     A = [A11 A12; A21 A22]  (row half, k half),   B = [B11 B12; B21 B22]  (row half n, k half)
//     P1 = (A11 + A22)(B11 + B22)^T   P2 = (A21 + A22) B11^T      P3 = A11 (B21 - B22)^T     P4 = A22 (B12 - B11)^T
//     P5 = (A11 + A12) B22^T          P6 = (A21 - A11)(B11 + B21)^T                          P7 = (A12 - A22)(B12 + B22)^T
//     C11 = P1 + P4 - P5 + P7         C12 = P3 + P5               C21 = P2 + P4              C22 = P1 - P2 + P3 + P6
// (Strassen 1969 with X = B^T, X_kl = B_lk^T.)  The seven left and the seven right operands are written as two STACKS
// S[q][row][k], q < 7, together with their 3M sum planes, so that the seven products are ONE batched launch of the GEMM
// (uniform batch strides; 7 x the tiles of a half-size product fill the 148 SMs where a single one would leave a ragged last
// wave).  The stack of an operand that does not change between iterations (<ab||cd>, <bk||cd>, <kl||cd>) is built once.
#pragma once
#include "common.cuh"

struct StrassenStack {      // the operand combinations of one side: 7 (one level) or 7 x 7 (two levels) matrices
    c128* S;                // [7^levels][Rh][Kh]; two levels: index q1 * 7 + q2 (q1 outer level, q2 inner)
    double* Sp;             // their sum planes Re + Im, same layout
    int64_t R, K, Rh, Kh;   // extents of the operand it was made from, and of one stacked matrix
    int levels;
};

static inline int64_t strassen_half(int64_t x) { return (x + 1) / 2; }
static inline int64_t strassen_khalf(int64_t K) { return round_up((K + 1) / 2, 2); }
static inline int64_t strassen_rows(int64_t R, int levels) { return levels == 2 ? strassen_half(strassen_half(R)) : strassen_half(R); }
static inline int64_t strassen_cols(int64_t K, int levels) { return levels == 2 ? strassen_khalf(strassen_khalf(K)) : strassen_khalf(K); }
static inline int64_t strassen_stack_elems(int64_t R, int64_t K, int levels = 1)
{
    return (levels == 2 ? 49 : 7) * strassen_rows(R, levels) * strassen_cols(K, levels);
}
static inline StrassenStack strassen_stack(c128* S, double* Sp, int64_t R, int64_t K, int levels = 1)
{
    StrassenStack s;
    s.S = S; s.Sp = Sp; s.R = R; s.K = K; s.Rh = strassen_rows(R, levels); s.Kh = strassen_cols(K, levels); s.levels = levels;
    return s;
}

constexpr int STR_THREADS = 256;

// Read access to the operand a LEFT stack was made from: the quadrants are x11 = s[2], x22 = s[3], x12 = s[4] - s[2],
// x21 = s[5] + s[2] (one subtraction: exact up to one rounding of the larger term); with two levels the same rule is applied to the
// quadrants of the stacked half-size matrices.  Lets the packed <ab||cd> be dropped once its stack exists: the few readers that
// want single elements (ccsd_get_tensor, the one-time unpacking in the Lambda set-up) pay up to four loads per element.
struct StrassenView {
    const c128* S;
    int64_t R1, K1, Rq, Kq;   // extents of a half; of a quarter (two levels)
    int levels;
};
static inline StrassenView strassen_view(const StrassenStack& s)
{
    StrassenView v;
    v.S = s.S; v.levels = s.levels;
    v.R1 = strassen_half(s.R); v.K1 = strassen_khalf(s.K);
    v.Rq = s.levels == 2 ? s.Rh : 0; v.Kq = s.levels == 2 ? s.Kh : 0;
    return v;
}
// value of quadrant (u, v) from the seven combinations, given a reader of combination q at the position in question
template <class F>
__device__ __forceinline__ c128 strassen_left_quadrant(int u, int v, F comb)
{
    if (u == 0 && v == 0) return comb(2);
    if (u == 1 && v == 1) return comb(3);
    if (u == 0) return csub(comb(4), comb(2));
    return cadd(comb(5), comb(2));
}
__device__ __forceinline__ c128 strassen_left_at(const StrassenView& w, int64_t r, int64_t k)
{
    const int u1 = r >= w.R1, v1 = k >= w.K1;
    const int64_t rr = r - u1 * w.R1, kk = k - v1 * w.K1;
    if (w.levels == 1) {
        const int64_t plane = w.R1 * w.K1, at = rr * w.K1 + kk;
        return strassen_left_quadrant(u1, v1, [&](int q) { return w.S[q * plane + at]; });
    }
    const int u2 = rr >= w.Rq, v2 = kk >= w.Kq;
    const int64_t plane = w.Rq * w.Kq, at = (rr - u2 * w.Rq) * w.Kq + (kk - v2 * w.Kq);
    return strassen_left_quadrant(u1, v1, [&](int q1) {
        return strassen_left_quadrant(u2, v2, [&](int q2) { return w.S[(q1 * 7 + q2) * plane + at]; });
    });
}

// the seven operand combinations of one side (SIDE 0: left operand A, SIDE 1: right operand B) from its four quadrants
template <int SIDE>
__device__ __forceinline__ void strassen_combos(c128 x11, c128 x12, c128 x21, c128 x22, c128 s[7])
{
    if (SIDE == 0) {
        s[0] = cadd(x11, x22); s[1] = cadd(x21, x22); s[2] = x11; s[3] = x22;
        s[4] = cadd(x11, x12); s[5] = csub(x21, x11); s[6] = csub(x12, x22);
    } else {
        s[0] = cadd(x11, x22); s[1] = x11; s[2] = csub(x21, x22); s[3] = csub(x12, x11);
        s[4] = x22; s[5] = cadd(x11, x21); s[6] = cadd(x12, x22);
    }
}
// the four quadrants of C from the seven products
__device__ __forceinline__ void strassen_quadrants(const c128 p[7], c128& c11, c128& c12, c128& c21, c128& c22)
{
    c11 = cadd(csub(cadd(p[0], p[3]), p[4]), p[6]);
    c12 = cadd(p[2], p[4]);
    c21 = cadd(p[1], p[3]);
    c22 = cadd(cadd(csub(p[0], p[1]), p[2]), p[5]);
}

// SIDE 0: left operand A [R = M][K];  SIDE 1: right operand B [R = N][K] (both k-contiguous, leading dimension ld)
template <int SIDE>
__global__ void __launch_bounds__(STR_THREADS)
strassen_prep_kernel(const c128* __restrict__ in, int64_t ld, int64_t R, int64_t K, int64_t Rh, int64_t Kh,
                     c128* __restrict__ S, double* __restrict__ Sp)
{
    const int64_t k = (int64_t)blockIdx.x * STR_THREADS + threadIdx.x;
    if (k >= Kh) return;
    const int64_t plane = Rh * Kh;
    const c128 zero = mk(0.0, 0.0);
    for (int64_t r = blockIdx.y; r < Rh; r += gridDim.y) {
        const bool k2 = k + Kh < K, r2 = r + Rh < R, k1 = k < K;
        const c128 x11 = k1 ? in[r * ld + k] : zero;
        const c128 x12 = k2 ? in[r * ld + k + Kh] : zero;
        const c128 x21 = (r2 && k1) ? in[(r + Rh) * ld + k] : zero;
        const c128 x22 = (r2 && k2) ? in[(r + Rh) * ld + k + Kh] : zero;
        c128 s[7];
        strassen_combos<SIDE>(x11, x12, x21, x22, s);
        const int64_t at = r * Kh + k;
#pragma unroll
        for (int q = 0; q < 7; q++) {
            S[q * plane + at] = s[q];
            Sp[q * plane + at] = s[q].x + s[q].y;
        }
    }
}

// Two levels in one pass: the 49 combinations S[q1 * 7 + q2] = combos(combos(quadrants)[q1] quadrants)[q2] of an operand, from
// its 4 x 4 blocks (R1, K1: extents of a half, Rq, Kq: of a quarter).  Same additions in the same order as two passes of
// strassen_prep_kernel, without writing and re-reading the seven half-size matrices.
template <int SIDE>
__global__ void __launch_bounds__(STR_THREADS)
strassen_prep2_kernel(const c128* __restrict__ in, int64_t ld, int64_t R, int64_t K, int64_t R1, int64_t K1, int64_t Rq, int64_t Kq,
                      c128* __restrict__ S, double* __restrict__ Sp)
{
    const int64_t k = (int64_t)blockIdx.x * STR_THREADS + threadIdx.x;
    if (k >= Kq) return;
    const int64_t plane = Rq * Kq;
    const c128 zero = mk(0.0, 0.0);
    for (int64_t r = blockIdx.y; r < Rq; r += gridDim.y) {
        c128 s1[2][2][7];      // [inner row half][inner k half][q1]: the outer combinations at the four inner block positions
#pragma unroll
        for (int u2 = 0; u2 < 2; u2++)
#pragma unroll
            for (int v2 = 0; v2 < 2; v2++) {
                const int64_t rr = r + u2 * Rq, kk = k + v2 * Kq;       // position inside a half
                const bool in_half = rr < R1 && kk < K1;
                c128 x[2][2];
#pragma unroll
                for (int u1 = 0; u1 < 2; u1++)
#pragma unroll
                    for (int v1 = 0; v1 < 2; v1++) {
                        const int64_t row = rr + u1 * R1, col = kk + v1 * K1;
                        x[u1][v1] = (in_half && row < R && col < K) ? in[row * ld + col] : zero;
                    }
                strassen_combos<SIDE>(x[0][0], x[0][1], x[1][0], x[1][1], s1[u2][v2]);
            }
        const int64_t at = r * Kq + k;
#pragma unroll
        for (int q1 = 0; q1 < 7; q1++) {
            c128 s2[7];
            strassen_combos<SIDE>(s1[0][0][q1], s1[0][1][q1], s1[1][0][q1], s1[1][1][q1], s2);
#pragma unroll
            for (int q2 = 0; q2 < 7; q2++) {
                S[(q1 * 7 + q2) * plane + at] = s2[q2];
                Sp[(q1 * 7 + q2) * plane + at] = s2[q2].x + s2[q2].y;
            }
        }
    }
}

static inline void launch_strassen_prep(cudaStream_t st, int side, const c128* in, int64_t ld, const StrassenStack& s)
{
    if (s.Rh <= 0 || s.Kh <= 0) return;
    dim3 grid((unsigned)((s.Kh + STR_THREADS - 1) / STR_THREADS), (unsigned)(s.Rh < 32768 ? s.Rh : 32768));
    if (s.levels == 2) {
        const int64_t R1 = strassen_half(s.R), K1 = strassen_khalf(s.K);
        if (side == 0) strassen_prep2_kernel<0><<<grid, STR_THREADS, 0, st>>>(in, ld, s.R, s.K, R1, K1, s.Rh, s.Kh, s.S, s.Sp);
        else strassen_prep2_kernel<1><<<grid, STR_THREADS, 0, st>>>(in, ld, s.R, s.K, R1, K1, s.Rh, s.Kh, s.S, s.Sp);
    } else {
        if (side == 0) strassen_prep_kernel<0><<<grid, STR_THREADS, 0, st>>>(in, ld, s.R, s.K, s.Rh, s.Kh, s.S, s.Sp);
        else strassen_prep_kernel<1><<<grid, STR_THREADS, 0, st>>>(in, ld, s.R, s.K, s.Rh, s.Kh, s.S, s.Sp);
    }
    count_launches(1);
}

// C (+)= alpha * (the four quadrants from the seven products).  The products are stored with the unit-stride index of C as
// their fast index: P[q][slow][fast], (fast, slow) = (m, n) halves if csm == 1 ("transposed" C), else (n, m).
__global__ void __launch_bounds__(STR_THREADS)
strassen_combine_kernel(const c128* __restrict__ P, int64_t Fh, int64_t Sh, int64_t F, int64_t Sx, c128* __restrict__ C,
                        int64_t stride_f, int64_t stride_s, int fast_is_m, c128 alpha, int accumulate)
{
    const int64_t f = (int64_t)blockIdx.x * STR_THREADS + threadIdx.x;
    if (f >= Fh) return;
    const int64_t plane = Fh * Sh;
    for (int64_t s = blockIdx.y; s < Sh; s += gridDim.y) {
        const int64_t at = s * Fh + f;
        c128 p[7], c11, c12, c21, c22;
#pragma unroll
        for (int q = 0; q < 7; q++) p[q] = P[q * plane + at];
        strassen_quadrants(p, c11, c12, c21, c22);
        // quadrant (row half of m, row half of n): c12 is (m low, n high).  In (fast, slow) terms:
        const c128 q_fs[2][2] = {{c11, fast_is_m ? c12 : c21}, {fast_is_m ? c21 : c12, c22}};   // [fast half][slow half]
        c128 old[2][2];        // all reads of C before the first write: the loads are independent of the stores
#pragma unroll
        for (int hf = 0; hf < 2; hf++)
#pragma unroll
            for (int hs = 0; hs < 2; hs++) {
                const int64_t ff = f + hf * Fh, ss = s + hs * Sh;
                old[hf][hs] = (accumulate && ff < F && ss < Sx) ? C[ff * stride_f + ss * stride_s] : mk(0.0, 0.0);
            }
#pragma unroll
        for (int hf = 0; hf < 2; hf++)
#pragma unroll
            for (int hs = 0; hs < 2; hs++) {
                const int64_t ff = f + hf * Fh, ss = s + hs * Sh;
                if (ff >= F || ss >= Sx) continue;
                C[ff * stride_f + ss * stride_s] = cadd(cmul(alpha, q_fs[hf][hs]), old[hf][hs]);
            }
    }
}

// Two levels in one pass: the 49 quarter-size products P[q1 * 7 + q2][slow][fast] -> the seven half-size products (in
// registers, at the four inner positions) -> the 16 blocks of C.  (Fh, Sh: extents of a half, Fq, Sq: of a quarter.)
__global__ void __launch_bounds__(STR_THREADS)   // 255 registers: every load of a thread in flight at once (a 128-register cap is 35 % slower)
strassen_combine2_kernel(const c128* __restrict__ P, int64_t Fq, int64_t Sq, int64_t Fh, int64_t Sh, int64_t F, int64_t Sx,
                         c128* __restrict__ C, int64_t stride_f, int64_t stride_s, int fast_is_m, c128 alpha, int accumulate)
{
    const int64_t f = (int64_t)blockIdx.x * STR_THREADS + threadIdx.x;
    if (f >= Fq) return;
    const int64_t plane = Fq * Sq;
    for (int64_t s = blockIdx.y; s < Sq; s += gridDim.y) {
        const int64_t at = s * Fq + f;
        // out[inner position][outer quadrant], quadrants in the order (c11, c12, c21, c22).  The half-size products P1[q1] are
        // never held together: each is formed at the four inner positions from its seven quarter-size products and added
        // straight into the outer quadrants it belongs to -- in the order q1 = 0..6, which is the order of
        // strassen_quadrants (c11 = ((P1 + P4) - P5) + P7, ...), so the sums have the bits of two separate passes.
        c128 out[4][4];
#pragma unroll
        for (int q1 = 0; q1 < 7; q1++) {
            c128 p[7], sub[4];
#pragma unroll
            for (int q2 = 0; q2 < 7; q2++) p[q2] = P[(q1 * 7 + q2) * plane + at];
            strassen_quadrants(p, sub[0], sub[1], sub[2], sub[3]);
#pragma unroll
            for (int u = 0; u < 4; u++) {
                const c128 x = sub[u];
                if (q1 == 0) { out[u][0] = x; out[u][3] = x; }
                if (q1 == 1) { out[u][2] = x; out[u][3] = csub(out[u][3], x); }
                if (q1 == 2) { out[u][1] = x; out[u][3] = cadd(out[u][3], x); }
                if (q1 == 3) { out[u][0] = cadd(out[u][0], x); out[u][2] = cadd(out[u][2], x); }
                if (q1 == 4) { out[u][0] = csub(out[u][0], x); out[u][1] = cadd(out[u][1], x); }
                if (q1 == 5) { out[u][3] = cadd(out[u][3], x); }
                if (q1 == 6) { out[u][0] = cadd(out[u][0], x); }
            }
        }
        // quadrant index (c11, c12, c21, c22) -> (fast half, slow half): c12 is (m low, n high).  One inner position at a time:
        // its four reads of C are issued together, before its four writes.
#pragma unroll
        for (int u = 0; u < 4; u++) {
            const int f2 = fast_is_m ? (u >> 1) : (u & 1), s2 = fast_is_m ? (u & 1) : (u >> 1);
            const int64_t fi = f + f2 * Fq, si = s + s2 * Sq;
            if (fi >= Fh || si >= Sh) continue;
            c128 old[4];
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const int hf = fast_is_m ? (q >> 1) : (q & 1), hs = fast_is_m ? (q & 1) : (q >> 1);
                const int64_t ff = fi + hf * Fh, ss = si + hs * Sh;
                old[q] = (accumulate && ff < F && ss < Sx) ? C[ff * stride_f + ss * stride_s] : mk(0.0, 0.0);
            }
#pragma unroll
            for (int q = 0; q < 4; q++) {
                const int hf = fast_is_m ? (q >> 1) : (q & 1), hs = fast_is_m ? (q & 1) : (q >> 1);
                const int64_t ff = fi + hf * Fh, ss = si + hs * Sh;
                if (ff < F && ss < Sx) C[ff * stride_f + ss * stride_s] = cadd(cmul(alpha, out[u][q]), old[q]);
            }
        }
    }
}

// P: products [7^levels][S][F] (S, F: the slow / fast extent of one product) of a C with extents M x N and strides (csm, csn)
static inline void launch_strassen_combine(cudaStream_t st, const c128* P, int64_t M, int64_t N, c128* C, int64_t csm, int64_t csn,
                                           c128 alpha, int accumulate, int levels = 1)
{
    const int fast_is_m = csm == 1;
    const int64_t F = fast_is_m ? M : N, Sx = fast_is_m ? N : M;
    const int64_t Fh = strassen_half(F), Sh = strassen_half(Sx);
    if (Fh <= 0 || Sh <= 0) return;
    if (levels == 2) {
        const int64_t Fq = strassen_half(Fh), Sq = strassen_half(Sh);
        dim3 grid((unsigned)((Fq + STR_THREADS - 1) / STR_THREADS), (unsigned)(Sq < 32768 ? Sq : 32768));
        strassen_combine2_kernel<<<grid, STR_THREADS, 0, st>>>(P, Fq, Sq, Fh, Sh, F, Sx, C, fast_is_m ? csm : csn,
                                                               fast_is_m ? csn : csm, fast_is_m, alpha, accumulate);
    } else {
        dim3 grid((unsigned)((Fh + STR_THREADS - 1) / STR_THREADS), (unsigned)(Sh < 32768 ? Sh : 32768));
        strassen_combine_kernel<<<grid, STR_THREADS, 0, st>>>(P, Fh, Sh, F, Sx, C, fast_is_m ? csm : csn, fast_is_m ? csn : csm,
                                                              fast_is_m, alpha, accumulate);
    }
    count_launches(1);
}
