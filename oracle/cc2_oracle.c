/*
 * ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain explicit-loop CPU implementation of the CC2 doubles equations of arXiv 2103.08473, Appendix 7.2
 * (eqs 34-38).  "In the CC2 method the T1 amplitude equations in 7.1 are unchanged":
 * the singles residual is eq 33 of ccsd_oracle.c; this file holds only what 7.2 adds.
 *
 * Arrays (dense, unpacked, row-major C99 double _Complex == numpy complex128), as in ccsd_oracle.c:
 *     f[p][q]  t1[i][a]  t2[i][j][a][b]
 *     oooo[m][n][i][j] = <mn||ij>   ooov[m][n][i][e] = <mn||ie>   oovv[m][n][e][f] = <mn||ef>
 *     vovo[a][m][e][i] = <am||ei>   vovv[a][m][e][f] = <am||ef>   vvvv[a][b][e][f] = <ab||ef>
 * Reading of the notation (G1/G4/G5 carried over to 7.2 as G21):
 *     V^{pq}_{rs} = <pq||rs>  (upper = bra pair, lower = ket pair), so
 *     V^{ab}_{ij} = <ab||ij> = conj <ij||ab>,   V^{ab}_{ej} = <ab||ej> = conj <ej||ab>,
 *     V^{mb}_{ij} = <mb||ij> = conj <ij||mb>,   V^{mb}_{ej} = <mb||ej> = - <bm||ej>,
 *     f^p_q = f[p][q] including the diagonal, so that S is the full residual
 *         <Phi_ij^ab| exp(-T1) H exp(T1) + [F, T2] |Phi_0>           (F = the Fock operator sum_pq f_pq a+_p a_q).
 * Pins (tests/test_cc2_pins.py): that determinant-space definition, brute force over all Slater determinants;
 * CC2 doubles == CCSD doubles at t2 = 0 plus the two Fock terms; antisymmetry.
 *
 * Shares no code with paper_2103_08473_b200/.  Build: gcc -O2 -fopenmp -fcx-limited-range -shared -fPIC.
 */
#include <complex.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef double _Complex zc;

#define IDX2(p, q, nq) ((size_t)(p) * (nq) + (q))
#define IDX4(p, q, r, s, nq, nr, ns) ((((size_t)(p) * (nq) + (q)) * (nr) + (r)) * (ns) + (s))
#define F_(p, q) f[IDX2(p, q, n)]
#define T1(i, a) t1[IDX2(i, a, v)]
#define T2(i, j, a, b) t2[IDX4(i, j, a, b, o, v, v)]
#define OOOO(k, l, i, j) oooo[IDX4(k, l, i, j, o, o, o)]
#define OOOV(k, l, i, c) ooov[IDX4(k, l, i, c, o, o, v)]
#define OOVV(k, l, c, d) oovv[IDX4(k, l, c, d, o, v, v)]
#define VOVO(a, k, c, i) vovo[IDX4(a, k, c, i, o, v, o)]
#define VOVV(a, k, c, d) vovv[IDX4(a, k, c, d, o, v, v)]
#define VVVV(a, b, c, d) vvvv[IDX4(a, b, c, d, v, v, v)]
#define WOOOO(m, nn, i, j) Woooo[IDX4(m, nn, i, j, o, o, o)]
#define WVVVV(a, b, e, ff) Wvvvv[IDX4(a, b, e, ff, v, v, v)]
#define WVVVO(a, b, e, j) Wvvvo[IDX4(a, b, e, j, v, v, o)]
#define WOVOO(m, b, i, j) Wovoo[IDX4(m, b, i, j, v, o, o)]

/* <mb||ej> = -<bm||ej>  (antisymmetry of the bra pair) from the stored class <am||ei> */
#define OVVO(m, b, e, j) (-VOVO(b, m, e, j))

/* eq 35:  W^{mn}_{ij} = V^{mn}_{ij} + sum_e P-_ij t^e_j V^{mn}_{ie} + 1/4 sum_ef P-_ij t^e_i t^f_j V^{mn}_{ef} */
void oracle_cc2_Woooo(int o, int v, const zc *t1, const zc *oooo, const zc *ooov, const zc *oovv, zc *Woooo)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int m = 0; m < o; m++)
        for (int nn = 0; nn < o; nn++)
            for (int i = 0; i < o; i++)
                for (int j = 0; j < o; j++) {
                    zc s = OOOO(m, nn, i, j);
                    for (int e = 0; e < v; e++) s += T1(j, e) * OOOV(m, nn, i, e) - T1(i, e) * OOOV(m, nn, j, e);
                    zc q = 0.0;
                    for (int e = 0; e < v; e++)
                        for (int ff = 0; ff < v; ff++)
                            q += (T1(i, e) * T1(j, ff) - T1(j, e) * T1(i, ff)) * OOVV(m, nn, e, ff);
                    WOOOO(m, nn, i, j) = s + 0.25 * q;
                }
}

/* eq 36:  W^{ab}_{ef} = V^{ab}_{ef} - sum_m P-_ab t^b_m V^{am}_{ef} + 1/4 sum_mn P-_ab t^a_m t^b_n V^{mn}_{ef} */
void oracle_cc2_Wvvvv(int o, int v, const zc *t1, const zc *vvvv, const zc *vovv, const zc *oovv, zc *Wvvvv)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int a = 0; a < v; a++)
        for (int b = 0; b < v; b++)
            for (int e = 0; e < v; e++)
                for (int ff = 0; ff < v; ff++) {
                    zc s = VVVV(a, b, e, ff);
                    for (int m = 0; m < o; m++) s -= T1(m, b) * VOVV(a, m, e, ff) - T1(m, a) * VOVV(b, m, e, ff);
                    zc q = 0.0;
                    for (int m = 0; m < o; m++)
                        for (int nn = 0; nn < o; nn++)
                            q += (T1(m, a) * T1(nn, b) - T1(m, b) * T1(nn, a)) * OOVV(m, nn, e, ff);
                    WVVVV(a, b, e, ff) = s + 0.25 * q;
                }
}

/* eq 37:  W^{ab}_{ej} = V^{ab}_{ej} - 1/2 sum_m P-_ab t^a_m V^{mb}_{ej},   V^{ab}_{ej} = conj <ej||ab> */
void oracle_cc2_Wvvvo(int o, int v, const zc *t1, const zc *vovv, const zc *vovo, zc *Wvvvo)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int a = 0; a < v; a++)
        for (int b = 0; b < v; b++)
            for (int e = 0; e < v; e++)
                for (int j = 0; j < o; j++) {
                    zc s = conj(VOVV(e, j, a, b));
                    zc q = 0.0;
                    for (int m = 0; m < o; m++) q += T1(m, a) * OVVO(m, b, e, j) - T1(m, b) * OVVO(m, a, e, j);
                    WVVVO(a, b, e, j) = s - 0.5 * q;
                }
}

/* eq 38:  W^{mb}_{ij} = V^{mb}_{ij} + 1/2 sum_e P-_ij t^e_i V^{mb}_{ej},   V^{mb}_{ij} = conj <ij||mb> */
void oracle_cc2_Wovoo(int o, int v, const zc *t1, const zc *ooov, const zc *vovo, zc *Wovoo)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int m = 0; m < o; m++)
        for (int b = 0; b < v; b++)
            for (int i = 0; i < o; i++)
                for (int j = 0; j < o; j++) {
                    zc s = conj(OOOV(i, j, m, b));
                    zc q = 0.0;
                    for (int e = 0; e < v; e++) q += T1(i, e) * OVVO(m, b, e, j) - T1(j, e) * OVVO(m, b, e, i);
                    WOVOO(m, b, i, j) = s + 0.5 * q;
                }
}

/*
 * eq 34:
 *   S[i,j,a,b] = V^{ab}_{ij} + sum_e P-_ij t^e_i W^{ab}_{ej} - sum_m P-_ab t^a_m W^{mb}_{ij}
 *              + sum_{m<n} P-_ab t^a_m t^b_n W^{mn}_{ij} + sum_{e<f} P-_ij t^e_i t^f_j W^{ab}_{ef}
 *              + sum_e P-_ab f^b_e t^{ae}_{ij} - sum_m P-_ij f^m_j t^{ab}_{im}
 * term: -1 = all seven; 0..6 = that term alone, in the order written (per-term parity).
 */
void oracle_cc2_s2(int o, int v, const zc *f, const zc *t1, const zc *t2, const zc *oovv, const zc *Woooo,
                   const zc *Wvvvv, const zc *Wvvvo, const zc *Wovoo, int term, zc *S2)
{
    const int n = o + v;
#pragma omp parallel for schedule(static) collapse(2)
    for (int i = 0; i < o; i++)
        for (int j = 0; j < o; j++)
            for (int a = 0; a < v; a++)
                for (int b = 0; b < v; b++) {
                    zc s = 0.0;
                    if (term < 0 || term == 0) s += conj(OOVV(i, j, a, b));
                    if (term < 0 || term == 1)
                        for (int e = 0; e < v; e++) s += T1(i, e) * WVVVO(a, b, e, j) - T1(j, e) * WVVVO(a, b, e, i);
                    if (term < 0 || term == 2)
                        for (int m = 0; m < o; m++) s -= T1(m, a) * WOVOO(m, b, i, j) - T1(m, b) * WOVOO(m, a, i, j);
                    if (term < 0 || term == 3)
                        for (int m = 0; m < o; m++)
                            for (int nn = m + 1; nn < o; nn++)
                                s += (T1(m, a) * T1(nn, b) - T1(m, b) * T1(nn, a)) * WOOOO(m, nn, i, j);
                    if (term < 0 || term == 4)
                        for (int e = 0; e < v; e++)
                            for (int ff = e + 1; ff < v; ff++)
                                s += (T1(i, e) * T1(j, ff) - T1(j, e) * T1(i, ff)) * WVVVV(a, b, e, ff);
                    if (term < 0 || term == 5)
                        for (int e = 0; e < v; e++)
                            s += F_(o + b, o + e) * T2(i, j, a, e) - F_(o + a, o + e) * T2(i, j, b, e);
                    if (term < 0 || term == 6)
                        for (int m = 0; m < o; m++) s -= F_(m, j) * T2(i, m, a, b) - F_(m, i) * T2(j, m, a, b);
                    S2[IDX4(i, j, a, b, o, v, v)] = s;
                }
}
