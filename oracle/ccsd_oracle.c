/*
 * ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, explicit-loop CPU implementation of the complex spinor-basis CCSD amplitude equations of
 * arXiv 2103.08473 (Appendix 7.1, eqs 22-33), the Fock build (eq 5
 * PAPER.md:67), the antisymmetrised integrals (eq 6 PAPER.md:71 in reading G1 of DESIGN.md) and
 * the correlation energy (eq 9; contraction string PAPER.md:178-182).  It is the reference the CUDA
 * library is compared with.  It shares no code, header, table or helper with paper_2103_08473_b200/ and only
 * tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Every tensor is a dense, UNPACKED, row-major array of C99 `double _Complex` (== numpy complex128):
 *     f[p][q]                      Fock matrix, n = o + v, occupied spinors first
 *     t1[i][a]  t2[i][j][a][b]  tau[i][j][a][b]
 *     oooo[k][l][i][j] = <kl||ij>    ooov[k][l][i][c] = <kl||ic>    oovv[k][l][c][d] = <kl||cd>
 *     vovo[a][k][c][i] = <ak||ci>    vovv[a][k][c][d] = <ak||cd>    vvvv[a][b][c][d] = <ab||cd>
 *     Hvv,Gvv[a][c]  Hoo,Goo[k][i]  Hov[k][c]  Hvovo[a][k][c][i]  C[k][b][i][j]  A[k][l][i][j]
 * Reading of the paper's notation: V^{pq}_{rs} = <pq||rs>;
 * F^p_q = f_pq including the diagonal; "dagger" = swap upper/lower index pairs and complex-conjugate;
 * S = the full residual <Phi_mu| exp(-T) H exp(T) |Phi_0>.
 *
 * `restricted` = 0: every sum runs over the full index ranges with the paper's factors 1/2 (the definition).
 * `restricted` = 1: sums over an antisymmetric index pair run over x<y without the 1/2, and 4-index antisymmetric
 *                   outputs are evaluated for i<j, a<b and filled by antisymmetry.  Same numbers up to rounding
 *                   order (tests/test_oracle_pins.py::test_restricted_equals_full); used for the larger shapes.
 *
 * Parity pins (tests/test_oracle_pins.py, all independent of this file's formulas): determinant-space
 * <Phi_mu|exp(-T)Hexp(T)|Phi_0> brute force; CCSD = FCI for two electrons; closed-form MP2; antisymmetry of every
 * term; real energy under Kramers symmetry.  "parity unpinned": nothing here (the DIIS convention lives in
 * ccsd_oracle.py and is unpinned by the paper; the converged energy does not depend on it).
 *
 * Build: gcc -O2 -fopenmp -fcx-limited-range -shared -fPIC (no -ffast-math); see oracle/build.py.
 */
#include <complex.h>
#include <stddef.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex zc;

typedef struct {
    int o, v, restricted;
    const zc *f;
    const zc *oooo, *ooov, *oovv, *vovo, *vovv, *vvvv;
} oracle_sys;

typedef struct {
    zc *tau;             /* [o][o][v][v] */
    zc *Hvv, *Gvv;       /* [v][v]  (a,c) */
    zc *Hoo, *Goo;       /* [o][o]  (k,i) */
    zc *Hov;             /* [o][v]  (k,c) */
    zc *Hvovo;           /* [v][o][v][o] (a,k,c,i) */
    zc *C;               /* [o][v][o][o] (k,b,i,j) */
    zc *A;               /* [o][o][o][o] (k,l,i,j) */
} oracle_inter;

#define IDX2(p, q, nq) ((size_t)(p) * (nq) + (q))
#define IDX4(p, q, r, s, nq, nr, ns) ((((size_t)(p) * (nq) + (q)) * (nr) + (r)) * (ns) + (s))

#define F_(p, q) f[IDX2(p, q, n)]
#define T1(i, a) t1[IDX2(i, a, v)]
#define T2(i, j, a, b) t2[IDX4(i, j, a, b, o, v, v)]
#define TAU(i, j, a, b) tau[IDX4(i, j, a, b, o, v, v)]
#define OOOO(k, l, i, j) oooo[IDX4(k, l, i, j, o, o, o)]
#define OOOV(k, l, i, c) ooov[IDX4(k, l, i, c, o, o, v)]
#define OOVV(k, l, c, d) oovv[IDX4(k, l, c, d, o, v, v)]
#define VOVO(a, k, c, i) vovo[IDX4(a, k, c, i, o, v, o)]
#define VOVV(a, k, c, d) vovv[IDX4(a, k, c, d, o, v, v)]
#define VVVV(a, b, c, d) vvvv[IDX4(a, b, c, d, v, v, v)]
#define HVOVO(a, k, c, i) Hvovo[IDX4(a, k, c, i, o, v, o)]
#define CI(k, b, i, j) Cint[IDX4(k, b, i, j, v, o, o)]
#define AI(k, l, i, j) Aint[IDX4(k, l, i, j, o, o, o)]

#define UNPACK_SYS                                                                                             \
    const int o = sys->o, v = sys->v, n = o + v, R = sys->restricted;                                          \
    const zc *f = sys->f, *oooo = sys->oooo, *ooov = sys->ooov, *oovv = sys->oovv, *vovo = sys->vovo,          \
             *vovv = sys->vovv, *vvvv = sys->vvvv;                                                             \
    (void)n; (void)R; (void)f; (void)oooo; (void)ooov; (void)oovv; (void)vovo; (void)vovv; (void)vvvv;

/* ------------------------------------------------------------------------------------------------------------
 * Fock matrix, PAPER.md:208, 244 ("KU Fock matrix"), from eq 5 with the reference determinant:
 *   f[p][q] = h[p][q] + sum_{i<o} <pi||qi>,  <pq||rs> = (pr|qs) - (ps|qr),  (pq|rs) = sum_L B[L][p][q] B[L][r][s]
 * ---------------------------------------------------------------------------------------------------------- */
void oracle_fock(int n, int o, int naux, const zc *h, const zc *B, zc *f)
{
#pragma omp parallel for schedule(static)
    for (int p = 0; p < n; p++)
        for (int q = 0; q < n; q++) {
            zc s = h[IDX2(p, q, n)];
            for (int i = 0; i < o; i++)
                for (int L = 0; L < naux; L++) {
                    const zc *BL = B + (size_t)L * n * n;
                    s += BL[IDX2(p, q, n)] * BL[IDX2(i, i, n)] - BL[IDX2(p, i, n)] * BL[IDX2(i, q, n)];
                }
            f[IDX2(p, q, n)] = s;
        }
}

/* One antisymmetrised integral <pq||rs> = (pr|qs) - (ps|qr)  (eq 6, reading G1).
 * Bt is B re-indexed as Bt[p][q][L] (a plain copy so that the L-sum is contiguous). */
static inline zc g_elem(const zc *Bt, int n, int naux, int p, int q, int r, int s)
{
    const zc *pr = Bt + IDX2(p, r, n) * naux, *qs = Bt + IDX2(q, s, n) * naux;
    const zc *ps = Bt + IDX2(p, s, n) * naux, *qr = Bt + IDX2(q, r, n) * naux;
    zc acc = 0.0;
    for (int L = 0; L < naux; L++) acc += pr[L] * qs[L] - ps[L] * qr[L];
    return acc;
}

/* Bt[p][q][L] = B[L][p][q] */
void oracle_transpose_B(int n, int naux, const zc *B, zc *Bt)
{
#pragma omp parallel for schedule(static)
    for (int p = 0; p < n; p++)
        for (int q = 0; q < n; q++)
            for (int L = 0; L < naux; L++) Bt[IDX2(p, q, n) * naux + L] = B[(size_t)L * n * n + IDX2(p, q, n)];
}

/* A block of <pq||rs>: p in [p0,p0+np), q in [q0,q0+nq), r in [r0,..), s in [s0,..) -> out[np][nq][nr][ns].
 * antisym_pq / antisym_rs = 1 (only legal when the two ranges coincide): evaluate x<y only and fill by antisymmetry. */
void oracle_g_block(int n, int naux, const zc *Bt, int p0, int np, int q0, int nq, int r0, int nr, int s0, int ns,
                    int antisym_pq, int antisym_rs, zc *out)
{
#pragma omp parallel for schedule(dynamic) collapse(2)
    for (int p = 0; p < np; p++)
        for (int q = 0; q < nq; q++) {
            if (antisym_pq && q < p) continue;
            for (int r = 0; r < nr; r++)
                for (int s = 0; s < ns; s++) {
                    if (antisym_rs && s < r) continue;
                    zc val = g_elem(Bt, n, naux, p0 + p, q0 + q, r0 + r, s0 + s);
                    out[IDX4(p, q, r, s, nq, nr, ns)] = val;
                    if (antisym_rs) out[IDX4(p, q, s, r, nq, nr, ns)] = -val;
                    if (antisym_pq) {
                        out[IDX4(q, p, r, s, nq, nr, ns)] = -val;
                        if (antisym_rs) out[IDX4(q, p, s, r, nq, nr, ns)] = val;
                    }
                }
        }
}

/* A single element, for sampled checks at sizes where whole blocks are not affordable. */
void oracle_g_element(int n, int naux, const zc *Bt, int p, int q, int r, int s, zc *out)
{
    *out = g_elem(Bt, n, naux, p, q, r, s);
}

/* eq 23:  tau[i,j,a,b] = t2[i,j,a,b] + t1[i,a] t1[j,b] - t1[j,a] t1[i,b] */
void oracle_tau(int o, int v, const zc *t1, const zc *t2, zc *tau)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int i = 0; i < o; i++)
        for (int j = 0; j < o; j++)
            for (int a = 0; a < v; a++)
                for (int b = 0; b < v; b++)
                    TAU(i, j, a, b) = T2(i, j, a, b) + T1(i, a) * T1(j, b) - T1(j, a) * T1(i, b);
}

/* ------------------------------------------------------------------------------------------------------------
 * Intermediates, eqs 24-31.  `in->tau` must already hold eq 23.
 * oracle_intermediates_part evaluates ONE group of equations (`which`: 0 = eqs 24-25, 1 = eqs 26-27, 2 = eq 28,
 * 3 = eq 29, 4 = eq 30, 5 = eq 31; -1 = all) for the outermost output index in [lo, hi) (ignored for which = -1):
 * the same loop nests, so that bench.py can time a slab of a BASELINE-size term without running all of it.
 * oracle_intermediates is the whole thing.
 * ---------------------------------------------------------------------------------------------------------- */
void oracle_intermediates_part(const oracle_sys *sys, const zc *t1, const zc *t2, oracle_inter *in, int which, int lo, int hi)
{
    UNPACK_SYS
    const zc *tau = in->tau;
    zc *Hvv = in->Hvv, *Gvv = in->Gvv, *Hoo = in->Hoo, *Goo = in->Goo, *Hov = in->Hov, *Hvovo = in->Hvovo,
       *Cint = in->C, *Aint = in->A;
    const double half = R ? 1.0 : 0.5;
#define PART(k) (which < 0 || which == (k))
#define LO(k) (which == (k) ? lo : 0)
#define HI(k, full) (which == (k) ? hi : (full))

    /* eq 24: Hvv[a,c] = f[a,c] + 1/2 sum_{k,l,d} <kl||cd> tau[k,l,d,a]
     * eq 25: Gvv[a,c] = Hvv[a,c] + sum_{k,d} <ak||cd> t1[k,d] - sum_k f[k,c] t1[k,a] */
    if (PART(0))
#pragma omp parallel for schedule(static) collapse(2)
    for (int a = LO(0); a < HI(0, v); a++)
        for (int c = 0; c < v; c++) {
            zc s = 0.0;
            for (int k = 0; k < o; k++)
                for (int l = R ? k + 1 : 0; l < o; l++)
                    for (int d = 0; d < v; d++) s += OOVV(k, l, c, d) * TAU(k, l, d, a);
            zc hv = F_(o + a, o + c) + half * s;
            zc gsum = hv;
            for (int k = 0; k < o; k++) {
                for (int d = 0; d < v; d++) gsum += VOVV(a, k, c, d) * T1(k, d);
                gsum -= F_(k, o + c) * T1(k, a);
            }
            Hvv[IDX2(a, c, v)] = hv;
            Gvv[IDX2(a, c, v)] = gsum;
        }

    /* eq 26: Hoo[k,i] = -f[k,i] + 1/2 sum_{l,c,d} <kl||cd> tau[l,i,c,d]
     * eq 27: Goo[k,i] = Hoo[k,i] - sum_{l,c} <kl||ic> t1[l,c] - sum_c f[k,c] t1[i,c] */
    if (PART(1))
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = LO(1); k < HI(1, o); k++)
        for (int i = 0; i < o; i++) {
            zc s = 0.0;
            for (int l = 0; l < o; l++)
                for (int c = 0; c < v; c++)
                    for (int d = R ? c + 1 : 0; d < v; d++) s += OOVV(k, l, c, d) * TAU(l, i, c, d);
            zc ho = -F_(k, i) + half * s;
            zc gsum = ho;
            for (int c = 0; c < v; c++) {
                for (int l = 0; l < o; l++) gsum -= OOOV(k, l, i, c) * T1(l, c);
                gsum -= F_(k, o + c) * T1(i, c);
            }
            Hoo[IDX2(k, i, o)] = ho;
            Goo[IDX2(k, i, o)] = gsum;
        }

    /* eq 28: Hov[k,c] = f[k,c] + sum_{l,d} <kl||cd> t1[l,d] */
    if (PART(2))
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = LO(2); k < HI(2, o); k++)
        for (int c = 0; c < v; c++) {
            zc s = F_(k, o + c);
            for (int l = 0; l < o; l++)
                for (int d = 0; d < v; d++) s += OOVV(k, l, c, d) * T1(l, d);
            Hov[IDX2(k, c, v)] = s;
        }

    /* eq 29: Hvovo[a,k,c,i] = <ak||ci> + sum_d <ak||cd> t1[i,d] - sum_l <kl||ic> t1[l,a]
     *                         + sum_{l,d} <kl||cd> ( 1/2 t2[l,i,a,d] + t1[l,a] t1[i,d] ) */
    if (PART(3))
#pragma omp parallel for schedule(static) collapse(2)
    for (int a = LO(3); a < HI(3, v); a++)
        for (int k = 0; k < o; k++)
            for (int c = 0; c < v; c++)
                for (int i = 0; i < o; i++) {
                    zc s = VOVO(a, k, c, i);
                    for (int d = 0; d < v; d++) s += VOVV(a, k, c, d) * T1(i, d);
                    for (int l = 0; l < o; l++) s -= OOOV(k, l, i, c) * T1(l, a);
                    for (int l = 0; l < o; l++)
                        for (int d = 0; d < v; d++)
                            s += OOVV(k, l, c, d) * (0.5 * T2(l, i, a, d) + T1(l, a) * T1(i, d));
                    HVOVO(a, k, c, i) = s;
                }

    /* eq 30: C[k,b,i,j] = conj(<ij||kb>) + sum_c ( <bk||ci> t1[j,c] - <bk||cj> t1[i,c] )
     *                     - 1/2 sum_{c,d} <bk||cd> tau[i,j,c,d] */
    if (PART(4))
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = LO(4); k < HI(4, o); k++)
        for (int b = 0; b < v; b++)
            for (int i = 0; i < o; i++)
                for (int j = R ? i + 1 : 0; j < o; j++) {
                    zc s = conj(OOOV(i, j, k, b));
                    for (int c = 0; c < v; c++) s += VOVO(b, k, c, i) * T1(j, c) - VOVO(b, k, c, j) * T1(i, c);
                    zc q = 0.0;
                    for (int c = 0; c < v; c++)
                        for (int d = R ? c + 1 : 0; d < v; d++) q += VOVV(b, k, c, d) * TAU(i, j, c, d);
                    s -= half * q;
                    CI(k, b, i, j) = s;
                    if (R) CI(k, b, j, i) = -s;
                }
    if (R && PART(4))
        for (int k = LO(4); k < HI(4, o); k++)
            for (int b = 0; b < v; b++)
                for (int i = 0; i < o; i++) CI(k, b, i, i) = 0.0;

    /* eq 31: A[k,l,i,j] = <kl||ij> + sum_c ( <kl||ic> t1[j,c] - <kl||jc> t1[i,c] ) + 1/2 sum_{c,d} <kl||cd> tau[i,j,c,d] */
    if (PART(5))
#pragma omp parallel for schedule(static) collapse(2)
    for (int k = LO(5); k < HI(5, o); k++)
        for (int l = 0; l < o; l++)
            for (int i = 0; i < o; i++)
                for (int j = 0; j < o; j++) {
                    zc s = OOOO(k, l, i, j);
                    for (int c = 0; c < v; c++) s += OOOV(k, l, i, c) * T1(j, c) - OOOV(k, l, j, c) * T1(i, c);
                    zc q = 0.0;
                    for (int c = 0; c < v; c++)
                        for (int d = R ? c + 1 : 0; d < v; d++) q += OOVV(k, l, c, d) * TAU(i, j, c, d);
                    AI(k, l, i, j) = s + half * q;
                }
#undef PART
#undef LO
#undef HI
}

void oracle_intermediates(const oracle_sys *sys, const zc *t1, const zc *t2, oracle_inter *in)
{
    oracle_intermediates_part(sys, t1, t2, in, -1, 0, 0);
}

/* ------------------------------------------------------------------------------------------------------------
 * eq 32, one term at a time.  out[i][j][a][b] is OVERWRITTEN with term `term`:
 *   0 ring      P-_ij P-_ab sum_{k,c} Hvovo[a,k,c,i] t2[j,k,c,b]
 *   1 Goo       sum_k ( Goo[k,j] t2[i,k,a,b] - Goo[k,i] t2[j,k,a,b] )            (P-_ji, reading G7)
 *   2 V^dag t1  sum_c ( conj(<cj||ab>) t1[i,c] - conj(<ci||ab>) t1[j,c] )
 *   3 Gvv       sum_c ( Gvv[a,c] t2[i,j,c,b] - Gvv[b,c] t2[i,j,c,a] )
 *   4 C t1      sum_k ( C[k,a,i,j] t1[k,b] - C[k,b,i,j] t1[k,a] )
 *   5 hh-ladder 1/2 sum_{k,l} A[k,l,i,j] tau[k,l,a,b]
 *   6 pp-ladder 1/2 sum_{c,d} <ab||cd> tau[i,j,c,d]
 *   7 driver    conj(<ij||ab>)
 * oracle_s2_term_range restricts the outermost output index i to [i_lo, i_hi) and the virtual output index a to
 * [a_lo, a_hi) (the same loop nests; the antisymmetric images of those elements are filled as usual, the rest of out is
 * left untouched): bench.py times slabs of the BASELINE-size terms with it.  For the a-range only the rows
 * vvvv[a_lo .. a_hi) of <ab||cd> are read by the pp-ladder, so sys->vvvv may point a_lo * v^3 elements BEFORE a buffer
 * that holds just those rows.  oracle_s2_term is the full range.
 * ---------------------------------------------------------------------------------------------------------- */
void oracle_s2_term_range(const oracle_sys *sys, const zc *t1, const zc *t2, const oracle_inter *in, int term, int i_lo,
                          int i_hi, int a_lo, int a_hi, zc *out)
{
    UNPACK_SYS
    const zc *tau = in->tau, *Gvv = in->Gvv, *Goo = in->Goo, *Hvovo = in->Hvovo, *Cint = in->C, *Aint = in->A;
    const double half = R ? 1.0 : 0.5;
#define OUT(i, j, a, b) out[IDX4(i, j, a, b, o, v, v)]

    if (term == 0) {
        /* X[i,j,a,b] = sum_{k,c} Hvovo[a,k,c,i] t2[j,k,c,b], all i,j,a,b; then antisymmetrise. */
        zc *X = out; /* build X in place in a scratch copy: need all four permutations, so use a second pass */
        size_t tot = (size_t)o * o * v * v;
        zc *tmp = (zc *)malloc(tot * sizeof(zc));
        if (i_lo > 0 || i_hi < o || a_lo > 0 || a_hi < v) memset(tmp, 0, tot * sizeof(zc));
#pragma omp parallel for schedule(static) collapse(2)
        for (int i = i_lo; i < i_hi; i++)
            for (int j = 0; j < o; j++)
                for (int a = a_lo; a < a_hi; a++)
                    for (int b = 0; b < v; b++) {
                        zc s = 0.0;
                        for (int k = 0; k < o; k++)
                            for (int c = 0; c < v; c++) s += HVOVO(a, k, c, i) * T2(j, k, c, b);
                        tmp[IDX4(i, j, a, b, o, v, v)] = s;
                    }
#define XX(i, j, a, b) tmp[IDX4(i, j, a, b, o, v, v)]
#pragma omp parallel for schedule(static) collapse(2)
        for (int i = 0; i < o; i++)
            for (int j = 0; j < o; j++)
                for (int a = 0; a < v; a++)
                    for (int b = 0; b < v; b++)
                        X[IDX4(i, j, a, b, o, v, v)] = XX(i, j, a, b) - XX(j, i, a, b) - XX(i, j, b, a) + XX(j, i, b, a);
#undef XX
        free(tmp);
        return;
    }

#pragma omp parallel for schedule(dynamic) collapse(2)
    for (int i = i_lo; i < i_hi; i++)
        for (int j = 0; j < o; j++) {
            if (R && j <= i) continue;
            for (int a = a_lo; a < a_hi; a++)
                for (int b = R ? a + 1 : 0; b < v; b++) {
                    zc s = 0.0;
                    switch (term) {
                    case 1:
                        for (int k = 0; k < o; k++)
                            s += Goo[IDX2(k, j, o)] * T2(i, k, a, b) - Goo[IDX2(k, i, o)] * T2(j, k, a, b);
                        break;
                    case 2:
                        for (int c = 0; c < v; c++)
                            s += conj(VOVV(c, j, a, b)) * T1(i, c) - conj(VOVV(c, i, a, b)) * T1(j, c);
                        break;
                    case 3:
                        for (int c = 0; c < v; c++)
                            s += Gvv[IDX2(a, c, v)] * T2(i, j, c, b) - Gvv[IDX2(b, c, v)] * T2(i, j, c, a);
                        break;
                    case 4:
                        for (int k = 0; k < o; k++) s += CI(k, a, i, j) * T1(k, b) - CI(k, b, i, j) * T1(k, a);
                        break;
                    case 5:
                        for (int k = 0; k < o; k++)
                            for (int l = R ? k + 1 : 0; l < o; l++) s += AI(k, l, i, j) * TAU(k, l, a, b);
                        s *= half;
                        break;
                    case 6:
                        for (int c = 0; c < v; c++)
                            for (int d = R ? c + 1 : 0; d < v; d++) s += VVVV(a, b, c, d) * TAU(i, j, c, d);
                        s *= half;
                        break;
                    case 7:
                        s = conj(OOVV(i, j, a, b));
                        break;
                    default:
                        break;
                    }
                    OUT(i, j, a, b) = s;
                    if (R) {
                        OUT(j, i, a, b) = -s;
                        OUT(i, j, b, a) = -s;
                        OUT(j, i, b, a) = s;
                    }
                }
        }
    if (R && i_lo == 0 && i_hi == o && a_lo == 0 && a_hi == v) {
        for (int i = 0; i < o; i++)
            for (int j = 0; j < o; j++)
                for (int a = 0; a < v; a++)
                    for (int b = 0; b < v; b++)
                        if (i == j || a == b) OUT(i, j, a, b) = 0.0;
    }
#undef OUT
}

void oracle_s2_term(const oracle_sys *sys, const zc *t1, const zc *t2, const oracle_inter *in, int term, zc *out)
{
    oracle_s2_term_range(sys, t1, t2, in, term, 0, sys->o, 0, sys->v, out);
}

/* eq 32: S2 = sum of the eight terms above.  scratch[o][o][v][v]. */
void oracle_s2(const oracle_sys *sys, const zc *t1, const zc *t2, const oracle_inter *in, zc *S2, zc *scratch)
{
    size_t tot = (size_t)sys->o * sys->o * sys->v * sys->v;
    memset(S2, 0, tot * sizeof(zc));
    for (int term = 0; term < 8; term++) {
        oracle_s2_term(sys, t1, t2, in, term, scratch);
        for (size_t x = 0; x < tot; x++) S2[x] += scratch[x];
    }
}

/* eq 33:
 * S1[i,a] = conj(f[i,a]) + sum_c Hvv[a,c] t1[i,c] + sum_k Hoo[k,i] t1[k,a] + sum_{k,c} Hov[k,c] t2[i,k,a,c]
 *         + sum_k ( sum_c (Hov[k,c] - 2 f[k,c]) t1[i,c] ) t1[k,a]
 *         + 1/2 sum_{k,c,d} <ak||cd> tau[i,k,c,d] + 1/2 sum_{k,l,c} <kl||ic> tau[k,l,c,a] - sum_{k,c} <ak||ci> t1[k,c] */
void oracle_s1_range(const oracle_sys *sys, const zc *t1, const zc *t2, const oracle_inter *in, int i_lo, int i_hi, zc *S1)
{   /* rows i in [i_lo, i_hi) of S1 (the same loop nest; bench.py times a slab of it) */
    UNPACK_SYS
    const zc *tau = in->tau, *Hvv = in->Hvv, *Hoo = in->Hoo, *Hov = in->Hov;
    const double half = R ? 1.0 : 0.5;
#pragma omp parallel for schedule(static) collapse(2)
    for (int i = i_lo; i < i_hi; i++)
        for (int a = 0; a < v; a++) {
            zc s = conj(F_(i, o + a));
            for (int c = 0; c < v; c++) s += Hvv[IDX2(a, c, v)] * T1(i, c);
            for (int k = 0; k < o; k++) s += Hoo[IDX2(k, i, o)] * T1(k, a);
            for (int k = 0; k < o; k++)
                for (int c = 0; c < v; c++) s += Hov[IDX2(k, c, v)] * T2(i, k, a, c);
            for (int k = 0; k < o; k++) {
                zc inner = 0.0;
                for (int c = 0; c < v; c++) inner += (Hov[IDX2(k, c, v)] - 2.0 * F_(k, o + c)) * T1(i, c);
                s += inner * T1(k, a);
            }
            zc q = 0.0;
            for (int k = 0; k < o; k++)
                for (int c = 0; c < v; c++)
                    for (int d = R ? c + 1 : 0; d < v; d++) q += VOVV(a, k, c, d) * TAU(i, k, c, d);
            s += half * q;
            q = 0.0;
            for (int k = 0; k < o; k++)
                for (int l = R ? k + 1 : 0; l < o; l++)
                    for (int c = 0; c < v; c++) q += OOOV(k, l, i, c) * TAU(k, l, c, a);
            s += half * q;
            for (int k = 0; k < o; k++)
                for (int c = 0; c < v; c++) s -= VOVO(a, k, c, i) * T1(k, c);
            S1[IDX2(i, a, v)] = s;
        }
}

void oracle_s1(const oracle_sys *sys, const zc *t1, const zc *t2, const oracle_inter *in, zc *S1)
{
    oracle_s1_range(sys, t1, t2, in, 0, sys->o, S1);
}

/* Correlation energy (eq 9 PAPER.md:97 evaluated for CCSD; string form PAPER.md:178-182; reading G11):
 *   E = sum_{i,a} f[i,a] t1[i,a] + 1/4 sum_{i,j,a,b} <ij||ab> tau[i,j,a,b]            (complex) */
void oracle_energy(const oracle_sys *sys, const zc *t1, const zc *tau, zc *E)
{
    UNPACK_SYS
    double ere = 0.0, eim = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : ere, eim)
    for (int i = 0; i < o; i++) {
        zc s = 0.0;
        for (int a = 0; a < v; a++) s += F_(i, o + a) * T1(i, a);
        zc q = 0.0;
        for (int j = R ? i + 1 : 0; j < o; j++)
            for (int a = 0; a < v; a++)
                for (int b = R ? a + 1 : 0; b < v; b++) q += OOVV(i, j, a, b) * TAU(i, j, a, b);
        s += (R ? 1.0 : 0.25) * q;
        ere += creal(s);
        eim += cimag(s);
    }
    *E = ere + eim * I;
}

/* ------------------------------------------------------------------------------------------------------------
 * Single-element evaluators for sampled parity checks at full BASELINE sizes (no whole-tensor oracle run needed).
 * Inputs are PACKED row-major arrays exactly as they cross the library's C ABI.
 * pp-ladder element (eq 32): R[(i<j)][(a<b)] = sum_{c<d} W[(a<b)][(c<d)] tau[(i<j)][(c<d)]
 * ---------------------------------------------------------------------------------------------------------- */
void oracle_pp_ladder_samples(long oo, long vv, const zc *taup, const zc *W, int nsamp, const long *ij, const long *ab,
                              zc *out)
{
    (void)oo;
#pragma omp parallel for schedule(dynamic)
    for (int s = 0; s < nsamp; s++) {
        const zc *wr = W + (size_t)ab[s] * vv, *tr = taup + (size_t)ij[s] * vv;
        zc acc = 0.0;
        for (long cd = 0; cd < vv; cd++) acc += wr[cd] * tr[cd];
        out[s] = acc;
    }
}

/* Plain matrix-product samples C[m][n] = sum_k A[m][k] * B[n][k] (optionally conj(B)): the common shape of every
 * GEMM-view contraction in DESIGN.md's term table, used to spot-check them at full size. */
void oracle_nt_samples(long K, const zc *A, long lda, const zc *B, long ldb, int conjB, int nsamp, const long *ms,
                       const long *ns, zc *out)
{
#pragma omp parallel for schedule(dynamic)
    for (int s = 0; s < nsamp; s++) {
        const zc *ar = A + (size_t)ms[s] * lda, *br = B + (size_t)ns[s] * ldb;
        zc acc = 0.0;
        for (long k = 0; k < K; k++) acc += ar[k] * (conjB ? conj(br[k]) : br[k]);
        out[s] = acc;
    }
}

int oracle_num_threads(void)
{
    int nt = 1;
#ifdef _OPENMP
#pragma omp parallel
    {
#pragma omp master
        nt = omp_get_num_threads();
    }
#endif
    return nt;
}
