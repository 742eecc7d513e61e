/*
 * ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain explicit-loop CPU implementation of the perturbative triples corrections +T, (T), -T of arXiv 2103.08473,
 * Appendix 7.3 (eqs 39-44; "three nested loops over occupied sub-blocks").
 *
 * Arrays (dense, unpacked, row-major C99 double _Complex == numpy complex128):
 *     fov[k][c] = f_kc        eps[p]  spinor energies (Re f_pp), occupied first
 *     t1[i][a]   t2[i][j][a][b]
 *     vvov[a][b][i][e] = <ab||ie>     vooo[a][m][i][j] = <am||ij>     vvoo[a][b][i][j] = <ab||ij>
 *
 * Reading G22 of DESIGN.md (the printed equations cannot all be taken literally for complex amplitudes: eq 39 has
 * no complex conjugate at all, eq 42 conjugates <ij||ab> in one term and t2 in the other; tests/test_triples_pins.py
 * checks every statement below against the determinant-space definitions of the fourth- and fifth-order energies):
 *   - W of eq 40 is the connected triples driver <Phi_ijk^abc| V_N T2 |Phi_0>; this fixes the brackets of eq 40 as
 *     "<ie||ab>" = V^{ab}_{ie} = <ab||ie> and "<ij||am>" = V^{am}_{ij} = <am||ij> (upper = bra, as in G1):
 *         W[i,j,k,a,b,c] = sum_e ( <ab||ie> t2[j,k,e,c] + <ab||je> t2[k,i,e,c] + <ab||ke> t2[i,j,e,c] )
 *                        + sum_m ( <am||ij> t2[k,m,b,c] + <am||jk> t2[i,m,b,c] + <am||ki> t2[j,m,b,c] )
 *     Wbar = W^abc + W^bca + W^cab   (fully antisymmetric in ijk and in abc).
 *   - Z of eq 42 is the disconnected driver <Phi_ijk^abc| V_N T1 + f_N T2 |Phi_0>:
 *         Z[i,j,k,a,b,c] = <ab||ij> t1[k,c] + t2[i,j,a,b] f_ck + (jk,i) + (ki,j),   f_ck = conj f_kc
 *     ( = "<ij||ab>^* t^c_k" as printed; the star of the second term sits on f, not on t2).
 *   - Y of eq 44 as printed (the disconnected triples amplitude <Phi_ijk^abc| T1 T2 + T1^3/6 |Phi_0>).
 *   - D^{abc}_{ijk} = eps_i + eps_j + eps_k - eps_a - eps_b - eps_c  (< 0, the sign convention of the CCSD denominators, G12);
 *     the left factor of every product is complex conjugated:
 *         E(+T)  = sum conj(Wbar) Wbar / (36 D)                      (eq 39; = "-sum .../36D" with the positive D)
 *         E((T)) = E(+T) + sum conj(Zbar) Wbar / (36 D)              (eq 41)
 *         E(-T)  = E(+T) + sum conj(Ybar) Wbar / 36                  (eq 43)
 *     These are <0|T2+ V_N R3 V_N T2|0>, <0|(T1+ V_N + T2+ f_N) R3 V_N T2|0> and <0|(T1 T2 + T1^3/6)+ P3 V_N T2|0>.
 *     (Conjugating the other factor instead gives the complex conjugate: same real parts.)
 *
 * restricted = 0: the sums run over ALL i,j,k,a,b,c with the factor 1/36 ("the full term is used, not only the upper
 *                 triangle").   restricted = 1: i<j<k only with the factor 1/6 (a,b,c still full).
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
#define IDX3(p, q, r, nq, nr) (((size_t)(p) * (nq) + (q)) * (nr) + (r))
#define IDX4(p, q, r, s, nq, nr, ns) ((((size_t)(p) * (nq) + (q)) * (nr) + (r)) * (ns) + (s))
#define T1(i, a) t1[IDX2(i, a, v)]
#define T2(i, j, a, b) t2[IDX4(i, j, a, b, o, v, v)]
#define VVOV(a, b, i, e) vvov[IDX4(a, b, i, e, v, o, v)]
#define VOOO(a, m, i, j) vooo[IDX4(a, m, i, j, o, o, o)]
#define VVOO(a, b, i, j) vvoo[IDX4(a, b, i, j, v, o, o)]
#define FOV(k, c) fov[IDX2(k, c, v)]

/* eq 40 for one (i,j,k): W[a][b][c] */
void oracle_triples_W(int o, int v, const zc *t2, const zc *vvov, const zc *vooo, int i, int j, int k, zc *W)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int a = 0; a < v; a++)
        for (int b = 0; b < v; b++)
            for (int c = 0; c < v; c++) {
                zc s = 0.0;
                for (int e = 0; e < v; e++)
                    s += VVOV(a, b, i, e) * T2(j, k, e, c) + VVOV(a, b, j, e) * T2(k, i, e, c) +
                         VVOV(a, b, k, e) * T2(i, j, e, c);
                for (int m = 0; m < o; m++)
                    s += VOOO(a, m, i, j) * T2(k, m, b, c) + VOOO(a, m, j, k) * T2(i, m, b, c) +
                         VOOO(a, m, k, i) * T2(j, m, b, c);
                W[IDX3(a, b, c, v, v)] = s;
            }
}

/* eq 42 for one (i,j,k): Z[a][b][c] */
void oracle_triples_Z(int o, int v, const zc *fov, const zc *t1, const zc *t2, const zc *vvoo, int i, int j, int k,
                      zc *Z)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int a = 0; a < v; a++)
        for (int b = 0; b < v; b++)
            for (int c = 0; c < v; c++)
                Z[IDX3(a, b, c, v, v)] = VVOO(a, b, i, j) * T1(k, c) + T2(i, j, a, b) * conj(FOV(k, c)) +
                                         VVOO(a, b, j, k) * T1(i, c) + T2(j, k, a, b) * conj(FOV(i, c)) +
                                         VVOO(a, b, k, i) * T1(j, c) + T2(k, i, a, b) * conj(FOV(j, c));
}

/* eq 44 for one (i,j,k): Y[a][b][c] */
void oracle_triples_Y(int o, int v, const zc *t1, const zc *t2, int i, int j, int k, zc *Y)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int a = 0; a < v; a++)
        for (int b = 0; b < v; b++)
            for (int c = 0; c < v; c++)
                Y[IDX3(a, b, c, v, v)] =
                    (T1(i, a) * T1(j, b) * T1(k, c) - T1(j, a) * T1(i, b) * T1(k, c) + T1(j, a) * T1(k, b) * T1(i, c) -
                     T1(k, a) * T1(j, b) * T1(i, c) + T1(k, a) * T1(i, b) * T1(j, c) - T1(i, a) * T1(k, b) * T1(j, c)) / 3.0 +
                    T2(i, j, a, b) * T1(k, c) + T2(j, k, a, b) * T1(i, c) + T2(k, i, a, b) * T1(j, c);
}

/* Q^abc + Q^bca + Q^cab (eqs 39, 41, 43 write the cyclic sum in this or the reverse order; the two coincide) */
void oracle_triples_cyclic(int v, const zc *Q, zc *Qbar)
{
#pragma omp parallel for schedule(static) collapse(2)
    for (int a = 0; a < v; a++)
        for (int b = 0; b < v; b++)
            for (int c = 0; c < v; c++)
                Qbar[IDX3(a, b, c, v, v)] = Q[IDX3(a, b, c, v, v)] + Q[IDX3(b, c, a, v, v)] + Q[IDX3(c, a, b, v, v)];
}

/*
 * eqs 39, 41, 43.  out[0] = E(+T), out[1] = E((T)) - E(+T), out[2] = E(-T) - E(+T)   (complex).
 * work: 6 * v^3 elements.
 */
void oracle_triples_energies(int o, int v, int restricted, const double *eps, const zc *fov, const zc *t1,
                             const zc *t2, const zc *vvov, const zc *vooo, const zc *vvoo, zc *work, zc *out)
{
    const size_t v3 = (size_t)v * v * v;
    zc *W = work, *Wb = work + v3, *Z = work + 2 * v3, *Zb = work + 3 * v3, *Y = work + 4 * v3, *Yb = work + 5 * v3;
    zc e4 = 0.0, e5 = 0.0, ey = 0.0;
    for (int i = 0; i < o; i++)
        for (int j = restricted ? i + 1 : 0; j < o; j++)
            for (int k = restricted ? j + 1 : 0; k < o; k++) {
                oracle_triples_W(o, v, t2, vvov, vooo, i, j, k, W);
                oracle_triples_cyclic(v, W, Wb);
                oracle_triples_Z(o, v, fov, t1, t2, vvoo, i, j, k, Z);
                oracle_triples_cyclic(v, Z, Zb);
                oracle_triples_Y(o, v, t1, t2, i, j, k, Y);
                oracle_triples_cyclic(v, Y, Yb);
                double r4 = 0, i4 = 0, r5 = 0, i5 = 0, ry = 0, iy = 0;
#pragma omp parallel for schedule(static) reduction(+ : r4, i4, r5, i5, ry, iy)
                for (int a = 0; a < v; a++)
                    for (int b = 0; b < v; b++)
                        for (int c = 0; c < v; c++) {
                            const double D = eps[i] + eps[j] + eps[k] - eps[o + a] - eps[o + b] - eps[o + c];
                            const zc w = Wb[IDX3(a, b, c, v, v)];
                            const zc x4 = conj(w) * w / D, x5 = conj(Zb[IDX3(a, b, c, v, v)]) * w / D,
                                     xy = conj(Yb[IDX3(a, b, c, v, v)]) * w;
                            r4 += creal(x4); i4 += cimag(x4);
                            r5 += creal(x5); i5 += cimag(x5);
                            ry += creal(xy); iy += cimag(xy);
                        }
                e4 += r4 + I * i4; e5 += r5 + I * i5; ey += ry + I * iy;
            }
    const double w = restricted ? 1.0 / 6.0 : 1.0 / 36.0;
    out[0] = w * e4; out[1] = w * e5; out[2] = w * ey;
}

/*
 * The same sums restricted to a LIST of unique occupied triples i<j<k (ijk: ntrip x 3 ints): the partial sums of the
 * restricted form of eqs 39, 41, 43 (weight 1/6 over a<b<c-unrestricted virtual sums), i.e. what one rank of a
 * multi-GPU split evaluates ("only the unique blocks").  Over the full list this is
 * oracle_triples_energies(restricted = 1).  out as there.  work: 6 * v^3 elements.
 */
void oracle_triples_energies_list(int o, int v, int ntrip, const int *ijk, const double *eps, const zc *fov, const zc *t1,
                                  const zc *t2, const zc *vvov, const zc *vooo, const zc *vvoo, zc *work, zc *out)
{
    const size_t v3 = (size_t)v * v * v;
    zc *W = work, *Wb = work + v3, *Z = work + 2 * v3, *Zb = work + 3 * v3, *Y = work + 4 * v3, *Yb = work + 5 * v3;
    zc e4 = 0.0, e5 = 0.0, ey = 0.0;
    for (int q = 0; q < ntrip; q++) {
        const int i = ijk[3 * q], j = ijk[3 * q + 1], k = ijk[3 * q + 2];
        oracle_triples_W(o, v, t2, vvov, vooo, i, j, k, W);
        oracle_triples_cyclic(v, W, Wb);
        oracle_triples_Z(o, v, fov, t1, t2, vvoo, i, j, k, Z);
        oracle_triples_cyclic(v, Z, Zb);
        oracle_triples_Y(o, v, t1, t2, i, j, k, Y);
        oracle_triples_cyclic(v, Y, Yb);
        for (int a = 0; a < v; a++)
            for (int b = 0; b < v; b++)
                for (int c = 0; c < v; c++) {
                    const double D = eps[i] + eps[j] + eps[k] - eps[o + a] - eps[o + b] - eps[o + c];
                    const zc w = Wb[IDX3(a, b, c, v, v)];
                    e4 += conj(w) * w / D;
                    e5 += conj(Zb[IDX3(a, b, c, v, v)]) * w / D;
                    ey += conj(Yb[IDX3(a, b, c, v, v)]) * w;
                }
    }
    out[0] = e4 / 6.0; out[1] = e5 / 6.0; out[2] = ey / 6.0;
}
