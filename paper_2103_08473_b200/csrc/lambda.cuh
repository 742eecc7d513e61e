// CCSD Lambda equations and one-body density (arXiv 2103.08473 Appendix 7.4-7.5, eqs 45-61).
// Included by ccsd_lib.cu after the iteration driver.  First CUDA path of this row: every term of the working equations
// (reading G23 of DESIGN.md) is one tensor_contract call on dense unpacked tensors, the GEMM of each
// call running on the DMMA kernel; the elements of Hbar are built once per solve, an iteration contracts the multipliers
// with them.  The pp-ladder term runs on the packed, dressed <ef||ab> with the DMMA ladder launch of the CCSD iteration.
#pragma once
#include "tensor_ops.cuh"

// C[out index orders] += sign * alpha * sum_k A B   (see tensor_ops.cuh).  Extents are taken from the operands.
static int tensor_contract(const Env& env, const TcScratch& sc, double alpha, const TView& A, const TView& B, c128* C, int nout,
                           const TcOut* outs, bool may_swap = true)
{
    char K[5] = {0}, MA[5] = {0}, NB[5] = {0};
    int64_t dimOf[128];
    for (int q = 0; q < A.rank; q++) dimOf[(int)A.idx[q]] = A.dim[q];
    for (int q = 0; q < B.rank; q++) {
        if (strchr(A.idx, B.idx[q]) && dimOf[(int)B.idx[q]] != B.dim[q]) return CCSD_EINVAL;
        dimOf[(int)B.idx[q]] = B.dim[q];
    }
    int nk = 0, nm = 0, nn = 0;
    for (int q = 0; q < A.rank; q++) {
        if (strchr(B.idx, A.idx[q])) K[nk++] = A.idx[q]; else MA[nm++] = A.idx[q];
    }
    for (int q = 0; q < B.rank; q++)
        if (!strchr(A.idx, B.idx[q])) NB[nn++] = B.idx[q];
    if (nm + nn > 4 || nm + nn != (int)strlen(outs[0].idx)) return CCSD_EINVAL;
    int64_t M = 1, N = 1, Kk = 1;
    for (int q = 0; q < nm; q++) M *= dimOf[(int)MA[q]];
    for (int q = 0; q < nn; q++) N *= dimOf[(int)NB[q]];
    for (int q = 0; q < nk; q++) Kk *= dimOf[(int)K[q]];
    if (M * Kk > sc.elems || N * Kk > sc.elems || M * N > sc.elems) return CCSD_EINVAL;
    if (M == 0 || N == 0) return CCSD_OK;
    // the DMMA tiles are 128 rows x 48 columns: put the operand whose free extent pads less into the row position
    if (may_swap && N > 1 && (M == 1 || round_up(N, 128) * round_up(M, 48) < round_up(M, 128) * round_up(N, 48)))
        return tensor_contract(env, sc, alpha, B, A, C, nout, outs, false);
    char ap[9] = {0}, bp[9] = {0}, cp[9] = {0};
    strcpy(ap, MA); strcat(ap, K);
    strcpy(bp, NB); strcat(bp, K);
    strcpy(cp, MA); strcat(cp, NB);
    const c128 *Ap = A.p, *Bp = B.p;
    if (strcmp(ap, A.idx) != 0) { CCSD_TRY(permute_into(env.st, sc.a, ap, A, 1.0, 0)); Ap = sc.a; }
    if (strcmp(bp, B.idx) != 0) { CCSD_TRY(permute_into(env.st, sc.b, bp, B, 1.0, 0)); Bp = sc.b; }
    if (N == 1) {   // matrix-vector product: one pass over the matrix at HBM speed
        CCSD_TRY(run_gemv(env, M, Kk, Ap, Kk, Bp, sc.c, 1, 1.0, 0));
    } else {
        GemmParams g = gp(M, N, Kk, Ap, Kk, Bp, Kk, sc.c, N, 1, 1.0, 0);
        if (sc.as && (double)M * (double)N * (double)Kk >= 2.0e10 && M * Kk <= sc.plane_elems && N * Kk <= sc.plane_elems &&
            Kk % 2 == 0) {   // large product: stage the 3M sums through planes (gemm_dmma.cuh), two streaming passes
            launch_sum_plane(env.st, Ap, sc.as, M * Kk);
            launch_sum_plane(env.st, Bp, sc.bs, N * Kk);
            g = with_planes(g, sc.as, sc.bs);
        }
        CCSD_TRY(run_gemm(env, g));
    }
    TView R;
    R.p = sc.c; R.rank = nm + nn;
    memset(R.idx, 0, sizeof(R.idx));
    strcpy(R.idx, cp);
    for (int q = 0; q < 4; q++) R.dim[q] = q < R.rank ? dimOf[(int)cp[q]] : 1;
    for (int k = 0; k < nout; k++) CCSD_TRY(permute_into(env.st, C, outs[k].idx, R, alpha * outs[k].sign, 1));
    return CCSD_OK;
}
// the common output patterns
static int tc1(const Env& env, const TcScratch& sc, double alpha, const TView& A, const TView& B, c128* C, const char* o0)
{
    const TcOut outs[1] = {{o0, 1.0}};
    return tensor_contract(env, sc, alpha, A, B, C, 1, outs);
}
// C += alpha (X - X with two labels exchanged): o0 and its exchanged twin o1
static int tc2(const Env& env, const TcScratch& sc, double alpha, const TView& A, const TView& B, c128* C, const char* o0,
               const char* o1)
{
    const TcOut outs[2] = {{o0, 1.0}, {o1, -1.0}};
    return tensor_contract(env, sc, alpha, A, B, C, 2, outs);
}
static int tc4(const Env& env, const TcScratch& sc, double alpha, const TView& A, const TView& B, c128* C, const char* o0,
               const char* o1, const char* o2, const char* o3)
{   // P-(ij) P-(ab): + o0 - o1 - o2 + o3
    const TcOut outs[4] = {{o0, 1.0}, {o1, -1.0}, {o2, -1.0}, {o3, 1.0}};
    return tensor_contract(env, sc, alpha, A, B, C, 4, outs);
}

// ---- state of one Lambda solve (all pointers into the caller's Lambda workspace) --------------------------------------
struct LambdaState {
    bool ready;
    TcScratch sc;
    // unpacked copies of what the CCSD context holds packed
    c128 *T1, *T2, *TAU, *OOVV, *OOOV, *WOOOO;     // [i][a] (copy: the solve stays consistent if the amplitudes move), [i][j][a][b], [m][n][e][f], [m][n][i][e], [m][n][i][j]
    // elements of Hbar (constant during the solve)
    c128 *Fov, *Foo, *Fvv;                         // [m][e], [m][i], [a][e]
    c128 *Wvovv, *Wooov, *Wovvo, *Wovoo, *Wvvvo;   // [a][m][e][f], [m][n][i][e], [m][b][e][j], [m][b][i][j], [a][b][e][i]
    c128 *inner, *X3, *Ypk;                        // build temporaries
    c128 *Wvovv_iaef, *Wvvvo_amef;                 // o v^3 elements in the operand layout of the iteration / of the build
    c128 *Wjp, *Wq;                                // W^{ej}_{ab} as [j][(a<b)][e] and W^{ef}_{am} as [a][m][(e<f)]: the packed pair halves the product
    c128 *FvvT, *OOVVhu;                           // Fbar^e_b as [b][e]; <ij||ae> as [(i<j)][a][e]
    c128* Wr;                                      // W^{je}_{bm} as [(j,b)][(m,e)]: operand of the ring-like term
    c128 *Wovoo_r, *OOVVr, *Wooov_r, *GooT, *l1T;  // W^{ie}_{mn} as [i][(m<n)][e]; <im||ab> as [(a<b)][i][m]; W^{ij}_{mb} as [(i<j)][b][m]; transposes
    double* Wrs;                                   // ... and its 3M sum plane
    // multipliers, residuals, per-iteration temporaries
    c128 *l1, *l2p, *L2, *R1, *R2, *R2p, *Gvv, *Goo, *Lt, *LT, *cl2p, *P2;
    // packed (i<j, a<b) route of the terms whose output is antisymmetric and whose contraction runs over a packable pair
    c128 *Pacc, *l2pT, *LTp, *L2hu, *Ltp, *Amc, *TAUp, *VoovvT, *VT2;
    c128 *T2huT, *T2ou;                            // t2 as [e][(m<n)][f] and [m][n][(e<f)]: eqs 50-51 over the packed pair
    double *VT2s, *Ltps;                           // sum planes of the (vv x oo x ov) product's operands
    double* cl2s;                                  // 3M sum plane of conj(l2p)
    // DIIS (as for the amplitudes: reading G13)
    DiisRing diis;
};

static void lambda_carve(const ccsd_ctx* c, char* base, LambdaState* L, size_t* total)
{
    Carver w{base, 0};
    const int64_t o = c->o, v = c->v, oo = c->oo, vv = c->vv, ov = c->ov;
    const int64_t o2v2 = o * o * v * v, ov3 = o * v * v * v, o3v = o * o * o * v;
    L->sc.elems = ov3 > o2v2 ? ov3 : o2v2;                       // largest operand / result of any product: o v^3, o^2 v^2,
    if (L->sc.elems < o3v) L->sc.elems = o3v;                     // o^3 v or (more occupied than virtual spinors) o^4
    if (L->sc.elems < o * o * o * o) L->sc.elems = o * o * o * o;
    L->sc.a = w.take<c128>(L->sc.elems);
    L->sc.b = w.take<c128>(L->sc.elems);
    L->sc.c = w.take<c128>(L->sc.elems);
    L->sc.plane_elems = o2v2;
    L->sc.as = c->planes ? w.take<double>(o2v2) : nullptr;
    L->sc.bs = c->planes ? w.take<double>(o2v2) : nullptr;
    L->T1 = w.take<c128>(ov); L->T2 = w.take<c128>(o2v2); L->TAU = w.take<c128>(o2v2); L->OOVV = w.take<c128>(o2v2);
    L->OOOV = w.take<c128>(o3v); L->WOOOO = w.take<c128>(o * o * o * o);
    L->Fov = w.take<c128>(ov); L->Foo = w.take<c128>(o * o); L->Fvv = w.take<c128>(v * v);
    L->Wvovv = w.take<c128>(ov3); L->Wooov = w.take<c128>(o3v); L->Wovvo = w.take<c128>(o2v2);
    L->Wovoo = w.take<c128>(o3v);
    L->Wvvvo = L->Wvovv;   // build order: W^{am}_{ef} is re-laid-out and dead before W^{ab}_{ei} is assembled in the same buffer
    L->Wvovv_iaef = w.take<c128>(ov3);
    L->Wjp = w.take<c128>(o * vv * v); L->Wq = w.take<c128>(v * o * vv);
    L->FvvT = w.take<c128>(v * v); L->OOVVhu = w.take<c128>(oo * v * v);
    L->Wr = w.take<c128>(o2v2);
    L->Wovoo_r = w.take<c128>(o * oo * v); L->OOVVr = w.take<c128>(vv * o * o); L->Wooov_r = w.take<c128>(oo * v * o);
    L->GooT = w.take<c128>(o * o); L->l1T = w.take<c128>(ov);
    L->Wrs = c->planes ? w.take<double>(o2v2) : nullptr;
    L->inner = w.take<c128>(o2v2); L->X3 = w.take<c128>(ov3 > o3v ? ov3 : o3v);
    L->Wvvvo_amef = L->X3;   // the build temporary is free when the finished W^{ab}_{ei} is re-laid-out into it
    L->Ypk = w.take<c128>(vv * v * o);
    L->l1 = w.take<c128>(ov); L->l2p = w.take<c128>(oo * vv); L->L2 = w.take<c128>(o2v2);
    L->R1 = w.take<c128>(ov); L->R2 = w.take<c128>(o2v2); L->R2p = w.take<c128>(oo * vv);
    L->Gvv = w.take<c128>(v * v); L->Goo = w.take<c128>(o * o);
    L->Lt = w.take<c128>(o3v); L->LT = w.take<c128>(o * o * o * o);
    L->cl2p = w.take<c128>(oo * vv); L->P2 = w.take<c128>(oo * vv);
    L->cl2s = w.take<double>(oo * vv);
    L->Pacc = w.take<c128>(oo * vv); L->l2pT = w.take<c128>(vv * oo); L->LTp = w.take<c128>(oo * oo);
    L->L2hu = w.take<c128>(oo * v * v); L->Ltp = w.take<c128>(oo * ov); L->Amc = w.take<c128>(oo * oo);
    L->TAUp = w.take<c128>(oo * vv); L->VoovvT = w.take<c128>(vv * oo); L->VT2 = w.take<c128>(vv * ov);
    L->T2huT = w.take<c128>(v * oo * v); L->T2ou = w.take<c128>(o * o * vv);
    L->VT2s = c->planes ? w.take<double>(vv * ov) : nullptr;
    L->Ltps = c->planes ? w.take<double>(oo * ov) : nullptr;
    L->diis.nd = c->opt.ndiis;
    const int nd = L->diis.nd > 0 ? L->diis.nd : 1;
    L->diis.u = w.take<c128>((int64_t)nd * c->nvec);
    L->diis.e = w.take<c128>((int64_t)nd * c->nvec);
    L->diis.gram = w.take<double>(13 * 13);
    L->diis.coef = w.take<double>(16);
    L->diis.info = w.take<double>(4);
    L->diis.scratch = w.take<double>(RED_SCRATCH_DOUBLES);
    *total = w.off;
}

// dense [x][y][p][q] from a tensor packed in its first pair (x<y, extent m1; pk1 = 0: that pair is stored unpacked) and
// in its second pair (p<q, extent m2; pk2 = 0: unpacked): antisymmetric fill
static void unpack_pairs(cudaStream_t st, c128* out, const c128* in, int m1, int pk1, int m2, int pk2, int64_t ncols = 0)
{   // ncols: number of (opaque) columns when the second pair is not packed and is not an m2 x m2 pair
    const int64_t n1 = (int64_t)m1 * m1, n2 = (!pk2 && ncols > 0) ? ncols : (int64_t)m2 * m2;
    const int64_t ld = pk2 ? (int64_t)m2 * (m2 - 1) / 2 : n2;
    const int m2d = m2 > 0 ? m2 : 1;
    launch_fill(st, out, n1, n2, n2, 0, [=] __device__(int64_t xy, int64_t pq) {
        int x = (int)(xy / m1), y = (int)(xy % m1), p = (int)(pq / m2d), q = (int)(pq % m2d);
        double sg = 1.0;
        int64_t row = xy, col = pq;
        if (pk1) {
            if (x == y) return mk(0.0, 0.0);
            if (x > y) { int t = x; x = y; y = t; sg = -sg; }
            row = pair_idx(x, y, m1);
        }
        if (pk2) {
            if (p == q) return mk(0.0, 0.0);
            if (p > q) { int t = p; p = q; q = t; sg = -sg; }
            col = pair_idx(p, q, m2);
        }
        return cscale(sg, in[row * ld + col]);
    });
}

#define LV(ptr, idx, ...) tview(ptr, idx, __VA_ARGS__)

// Elements of Hbar (eqs 45-49, 57 and the list of the paper's ref. 39; reading G23), once per solve.  Needs the
// intermediates of a CCSD residual evaluation at the current amplitudes (tau, H^k_c, G^a_c, G^k_i, A^{kl}_{ij}).
static int lambda_build_hbar(ccsd_ctx* c, LambdaState* L)
{
    cudaStream_t st = c->st;
    const Env& env = c->env;
    const TcScratch& sc = L->sc;
    const int o = c->o, v = c->v;
    const int64_t O = o, V = v, vv = c->vv;
    CCSD_TRY(residual_any(c));                                // tau, Hov, Gvv, Goo, Am of eqs 23-31 at the current (t1, t2)
    dcopy(st, L->T1, c->t1, O * V);
    unpack_pairs(st, L->T2, c->t2p, o, 1, v, 1);
    unpack_pairs(st, L->TAU, c->taup, o, 1, v, 1);
    unpack_pairs(st, L->OOVV, c->Voovv_p, o, 1, v, 1);
    unpack_pairs(st, L->OOOV, c->Vooov_p, o, 1, 0, 0, O * V);
    unpack_pairs(st, L->WOOOO, c->Am, o, 1, o, 1);             // eq 45 = eq 31
    {   // t2 in the two half-packed operand layouts of eqs 50-51
        const c128* t2p = c->t2p;
        const int64_t oo = c->oo;
        launch_fill(st, L->T2huT, V, oo * V, oo * V, 0, [=] __device__(int64_t e, int64_t col) {
            return asym_col(t2p, col / v, vv, (int)e, (int)(col % v), v);
        });
        unpack_pairs(st, L->T2ou, c->t2p, o, 1, 0, 0, vv);
    }
    // Fbar^m_e = H^k_c (eq 28), Fbar^a_e = G^a_c (eq 57 = eq 25), Fbar^m_i = -G^k_i (eq 27)
    dcopy(st, L->Fov, c->Hov, O * V);
    dcopy(st, L->Fvv, c->Gvv, V * V);
    CCSD_TRY(permute_into(st, L->Foo, "mi", LV(c->Goo, "mi", O, O), -1.0, 0));
    const c128 *T1 = L->T1, *VOVV = c->Vvovv_u /* <ak||cd> stored [a][c][k][d] */, *VOVO = c->Vvovo_m /* <ak||ci> [a][i][c][k] */;
    // W^{am}_{ef} = <am||ef> - t^a_n <nm||ef>
    CCSD_TRY(permute_into(st, L->Wvovv, "amef", LV(VOVV, "aemf", V, V, O, V), 1.0, 0));
    CCSD_TRY(tc1(env, sc, -1.0, LV(T1, "na", O, V), LV(L->OOVV, "nmef", O, O, V, V), L->Wvovv, "amef"));
    //   ... kept only in the two [free][contracted] layouts the iteration contracts it in
    CCSD_TRY(permute_into(st, L->Wvovv_iaef, "iaef", LV(L->Wvovv, "eifa", V, O, V, V), 1.0, 0));
    {   // [j][(a<b)][e] = W^{ej}_{ab} (antisymmetric in ab); Fbar^e_b transposed; <ij||ae> with the occupied pair packed
        const c128 *Wv = L->Wvovv, *Voovv = c->Voovv_p;
        const int2* pv = c->pv;
        launch_fill(st, L->Wjp, O * vv, V, V, 0, [=] __device__(int64_t row, int64_t e) {
            const int64_t j = row / vv;
            const int2 ab = pv[row % vv];
            return Wv[((e * o + j) * v + ab.x) * v + ab.y];
        });
        CCSD_TRY(permute_into(st, L->FvvT, "be", LV(L->Fvv, "eb", V, V), 1.0, 0));
        launch_fill(st, L->OOVVhu, c->oo * V, V, V, 0, [=] __device__(int64_t row, int64_t e) {
            return asym_col(Voovv, row / v, vv, (int)(row % v), (int)e, v);
        });
    }
    // W^{mn}_{ie} = <mn||ie> + t^f_i <mn||fe>
    dcopy(st, L->Wooov, L->OOOV, O * O * O * V);
    CCSD_TRY(tc1(env, sc, 1.0, LV(T1, "if", O, V), LV(L->OOVV, "mnfe", O, O, V, V), L->Wooov, "mnie"));
    // eqs 46-47: W^{mb}_{ej} = <mb||ej> + t^f_j <mb||ef> - t^b_n <mn||ej> - (t^{fb}_{jn} + t^f_j t^b_n) <mn||ef>
    CCSD_TRY(permute_into(st, L->Wovvo, "mbej", LV(VOVO, "bjem", V, O, V, O), -1.0, 0));                 // <mb||ej> = -<bm||ej>
    dcopy(st, L->inner, L->Wovvo, O * O * V * V);
    CCSD_TRY(tc1(env, sc, -1.0, LV(T1, "jf", O, V), LV(VOVV, "bemf", V, V, O, V), L->Wovvo, "mbej"));      // <mb||ef> = -<bm||ef>
    CCSD_TRY(tc1(env, sc, 1.0, LV(T1, "nb", O, V), LV(L->OOOV, "mnje", O, O, O, V), L->Wovvo, "mbej"));    // <mn||ej> = -<mn||je>
    CCSD_TRY(tc1(env, sc, -1.0, LV(L->T2, "jnfb", O, O, V, V), LV(L->OOVV, "mnef", O, O, V, V), L->Wovvo, "mbej"));
    CCSD_CUDA_TRY(cudaMemsetAsync(L->X3, 0, (size_t)(O * O * O * V) * sizeof(c128), st));
    CCSD_TRY(tc1(env, sc, 1.0, LV(T1, "jf", O, V), LV(L->OOVV, "mnef", O, O, V, V), L->X3, "jmne"));
    CCSD_TRY(tc1(env, sc, -1.0, LV(T1, "nb", O, V), LV(L->X3, "jmne", O, O, O, V), L->Wovvo, "mbej"));
    // inner^{mb}_{ej} = <mb||ej> - t^{bf}_{nj} <mn||ef>
    CCSD_TRY(tc1(env, sc, -1.0, LV(L->T2, "njbf", O, O, V, V), LV(L->OOVV, "mnef", O, O, V, V), L->inner, "mbej"));
    // W^{mb}_{ij}
    CCSD_TRY(permute_into(st, L->Wovoo, "mbij", LV(L->OOOV, "ijmb", O, O, O, V), 1.0, 0, 1));               // conj <ij||mb>
    CCSD_TRY(tc1(env, sc, -1.0, LV(L->Fov, "me", O, V), LV(L->T2, "ijbe", O, O, V, V), L->Wovoo, "mbij"));
    CCSD_TRY(tc1(env, sc, -1.0, LV(T1, "nb", O, V), LV(L->WOOOO, "mnij", O, O, O, O), L->Wovoo, "mbij"));
    CCSD_TRY(tc1(env, sc, -0.5, LV(L->TAU, "ijef", O, O, V, V), LV(VOVV, "bemf", V, V, O, V), L->Wovoo, "mbij"));
    CCSD_TRY(tc2(env, sc, 1.0, LV(L->T2, "jnbe", O, O, V, V), LV(L->OOOV, "mnie", O, O, O, V), L->Wovoo, "mbij", "mbji"));
    CCSD_TRY(tc2(env, sc, 1.0, LV(T1, "ie", O, V), LV(L->inner, "mbej", O, V, V, O), L->Wovoo, "mbij", "mbji"));
    // eqs 48-49: W^{ab}_{ei}
    CCSD_TRY(permute_into(st, L->Wvvvo, "abei", LV(VOVV, "eaib", V, V, O, V), 1.0, 0, 1));                  // conj <ei||ab>
    CCSD_TRY(tc1(env, sc, -1.0, LV(L->Fov, "me", O, V), LV(L->T2, "miab", O, O, V, V), L->Wvvvo, "abei"));
    CCSD_TRY(tc1(env, sc, -0.5, LV(L->TAU, "mnab", O, O, V, V), LV(L->OOOV, "mnie", O, O, O, V), L->Wvvvo, "abei"));
    CCSD_TRY(tc2(env, sc, 1.0, LV(L->T2, "miaf", O, O, V, V), LV(VOVV, "bemf", V, V, O, V), L->Wvvvo, "abei", "baei"));
    CCSD_TRY(tc2(env, sc, -1.0, LV(T1, "ma", O, V), LV(L->inner, "mbei", O, V, V, O), L->Wvvvo, "abei", "baei"));
    // + t^f_i W^{ab}_{ef}, W^{ab}_{ef} = <ab||ef> - P(ab) t^b_m <am||ef> + 1/2 tau^{ab}_{mn} <mn||ef>, never stored:
    //   (ii) -P(ab) t^b_m ( sum_f <am||ef> t^f_i )        (iii) 1/2 tau^{ab}_{mn} ( sum_f <mn||ef> t^f_i )
    CCSD_CUDA_TRY(cudaMemsetAsync(L->X3, 0, (size_t)(O * O * V * V) * sizeof(c128), st));
    CCSD_TRY(tc1(env, sc, 1.0, LV(VOVV, "aemf", V, V, O, V), LV(T1, "if", O, V), L->X3, "amei"));
    CCSD_TRY(tc2(env, sc, -1.0, LV(T1, "mb", O, V), LV(L->X3, "amei", V, O, V, O), L->Wvvvo, "abei", "baei"));
    CCSD_CUDA_TRY(cudaMemsetAsync(L->X3, 0, (size_t)(O * O * O * V) * sizeof(c128), st));
    CCSD_TRY(tc1(env, sc, 1.0, LV(L->OOVV, "mnef", O, O, V, V), LV(T1, "if", O, V), L->X3, "mnei"));
    CCSD_TRY(tc1(env, sc, 0.5, LV(L->TAU, "mnab", O, O, V, V), LV(L->X3, "mnei", O, O, V, O), L->Wvvvo, "abei"));
    //   (i) sum_f <ab||ef> t^f_i from the packed <ab||cd>: rows (a<b) in slabs, unpacked in (e,f), times t1
    {
        const c128* W = c->W;
        const StrassenView wv = strassen_view(c->sW);      // where <ab||cd> is kept as the ladder's operand stack only (c->W null)
        const int64_t slab_rows = (sc.elems / (V * V)) > 0 ? (sc.elems / (V * V)) : 1;
        for (int64_t r0 = 0; r0 < vv; r0 += slab_rows) {
            const int64_t nr = (vv - r0 < slab_rows) ? vv - r0 : slab_rows;
            launch_fill(st, sc.a, nr * V, V, V, 0, [=] __device__(int64_t row, int64_t ff) {
                const int64_t AB = r0 + row / v;
                const int e = (int)(row % v);
                if (W) return asym_col(W, AB, vv, e, (int)ff, v);
                if (e == (int)ff) return mk(0.0, 0.0);
                return e < (int)ff ? strassen_left_at(wv, AB, pair_idx(e, (int)ff, v)) : cneg(strassen_left_at(wv, AB, pair_idx((int)ff, e, v)));
            });
            // Ypk[(a<b)][e][i] = sum_f U[(ab),e][f] t1[i][f]
            CCSD_TRY(run_gemm(env, gp(nr * V, O, V, sc.a, V, T1, V, L->Ypk + r0 * V * O, O, 1, 1.0, 0)));
        }
        const c128* Y = L->Ypk;
        c128* Wv = L->Wvvvo;
        launch_fill(st, Wv, V * V, V * O, V * O, 1, [=] __device__(int64_t ab, int64_t ei) {
            const int a = (int)(ab / v), b = (int)(ab % v);
            if (a == b) return mk(0.0, 0.0);
            return a < b ? Y[pair_idx(a, b, v) * ((int64_t)v * o) + ei] : cneg(Y[pair_idx(b, a, v) * ((int64_t)v * o) + ei]);
        });
    }
    // W^{ab}_{ei} in the [free][contracted] layout the iteration contracts it in (into the build temporary, now free)
    CCSD_TRY(permute_into(st, L->Wvvvo_amef, "amef", LV(L->Wvvvo, "efam", V, V, V, O), 1.0, 0));
    {   // operands of the o^3 v^2-class terms with the pair they leave alone packed: W^{ie}_{mn}, <im||ab>, W^{ij}_{mb}
        const c128 *Wovoo = L->Wovoo, *Voovv = c->Voovv_p, *Wooov = L->Wooov;
        const int2 *po = c->po;
        const int64_t oo = c->oo;
        launch_fill(st, L->Wovoo_r, O, oo * V, oo * V, 0, [=] __device__(int64_t i, int64_t col) {   // [i][(m<n)][e] = W[i][e][m][n]
            const int2 mn = po[col / v];
            return Wovoo[((i * v + col % v) * o + mn.x) * o + mn.y];
        });
        launch_fill(st, L->OOVVr, vv, O * O, O * O, 0, [=] __device__(int64_t AB, int64_t im) {      // [(a<b)][i][m] = <im||ab>
            const int i = (int)(im / o), m = (int)(im % o);
            if (i == m) return mk(0.0, 0.0);
            return i < m ? Voovv[pair_idx(i, m, o) * vv + AB] : cneg(Voovv[pair_idx(m, i, o) * vv + AB]);
        });
        launch_fill(st, L->Wooov_r, oo * V, O, O, 0, [=] __device__(int64_t row, int64_t m) {        // [(i<j)][b][m] = W[i][j][m][b]
            const int2 ij = po[row / v];
            return Wooov[(((int64_t)ij.x * o + ij.y) * o + m) * v + row % v];
        });
    }
    // W^{je}_{bm} (finished above) in the [free][contracted] layout of the ring-like term, with its sum plane
    CCSD_TRY(permute_into(st, L->Wr, "jbme", LV(L->Wovvo, "jebm", O, V, V, O), 1.0, 0));
    if (L->Wrs) launch_sum_plane(st, L->Wr, L->Wrs, O * V * O * V);
    {   // ... and packed in its antisymmetric pair: [a][m][(e<f)]
        const c128* Wam = L->Wvvvo_amef;
        const int2* pv = c->pv;
        launch_fill(st, L->Wq, V * O, vv, vv, 0, [=] __device__(int64_t am, int64_t EF) {
            const int2 ef = pv[EF];
            return Wam[(am * v + ef.x) * v + ef.y];
        });
    }
    // packed operands of the iteration: A^{kl}_{ij} and tau as they are now, <mn||ab> and <em||ab> with the (a<b) pair as row
    dcopy(st, L->Amc, c->Am, c->oo * c->oo);
    dcopy(st, L->TAUp, c->taup, c->oo * vv);
    CCSD_TRY(launch_transpose2d(st, c->Voovv_p, L->VoovvT, c->oo, vv, 0));
    CCSD_TRY(launch_transpose2d(st, c->Vvovv_p, L->VT2, c->ov, vv, 0));
    if (L->VT2s) launch_sum_plane(st, L->VT2, L->VT2s, vv * c->ov);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

// Right-hand sides of eqs 52-56 at the current multipliers: R1[i][a], R2p[(i<j)][(a<b)].
static int lambda_residual(ccsd_ctx* c, LambdaState* L)
{
    cudaStream_t st = c->st;
    const Env& env = c->env;
    const TcScratch& sc = L->sc;
    const int o = c->o, v = c->v;
    const int64_t O = o, V = v, oo = c->oo, vv = c->vv;
    // eqs 50-51 over the packed pair of each product (both factors are antisymmetric in it, so the full sum is twice the
    // packed one):  G^a_e = -1/2 sum_{mnf} t^{ef}_{mn} lambda^{mn}_{af} = -sum_{m<n,f};  G^m_i = 1/2 sum_{nef} t^{ef}_{mn}
    // lambda^{in}_{ef} = sum_{n,e<f}.  The lambda operands go to the contraction scratch, the t operands were laid out once.
    {
        const c128* l2p = L->l2p;
        launch_fill(st, sc.a, V, oo * V, oo * V, 0, [=] __device__(int64_t a, int64_t col) {   // [a][(m<n)][f]
            return asym_col(l2p, col / v, vv, (int)a, (int)(col % v), v);
        });
        CCSD_TRY(run_gemm(env, gp(V, V, oo * V, sc.a, oo * V, L->T2huT, oo * V, L->Gvv, V, 1, -1.0, 0)));
        unpack_pairs(st, sc.b, L->l2p, o, 1, 0, 0, vv);                                        // [i][n][(e<f)]
        CCSD_TRY(run_gemm(env, gp(O, O, O * vv, L->T2ou, O * vv, sc.b, O * vv, L->Goo, O, 1, 1.0, 0)));
        // eqs 55-56 start here, while [i][m][(e<f)] is in the scratch: 1/2 sum_{mef} lambda^{im}_{ef} W^{ef}_{am} = sum_{m,e<f}
        dcopy(st, L->R1, L->Fov, O * V);
        CCSD_TRY(run_gemm(env, gp(V, O, O * vv, L->Wq, O * vv, sc.b, O * vv, L->R1, 1, V, 1.0, 1)));
        // ... and -1/2 sum_{mne} lambda^{mn}_{ae} W^{ie}_{mn} = -sum_{m<n,e}, with [a][(m<n)][e] still in the scratch
        CCSD_TRY(run_gemm(env, gp(V, O, oo * V, sc.a, oo * V, L->Wovoo_r, oo * V, L->R1, 1, V, -1.0, 1)));
    }
    CCSD_TRY(tc1(env, sc, 1.0, LV(L->l1, "ie", O, V), LV(L->Fvv, "ea", V, V), L->R1, "ia"));
    CCSD_TRY(tc1(env, sc, -1.0, LV(L->l1, "ma", O, V), LV(L->Foo, "im", O, O), L->R1, "ia"));
    CCSD_TRY(tc1(env, sc, -1.0, LV(L->Goo, "mn", O, O), LV(L->Wooov, "mina", O, O, O, V), L->R1, "ia"));
    CCSD_TRY(tc1(env, sc, -1.0, LV(L->Gvv, "ef", V, V), LV(L->Wvovv_iaef, "iaef", O, V, V, V), L->R1, "ia"));
    CCSD_TRY(tc1(env, sc, 1.0, LV(L->l1, "me", O, V), LV(L->Wovvo, "ieam", O, V, V, O), L->R1, "ia"));
    // eqs 52-54: every term goes into the packed accumulator Pacc[(i<j)][(a<b)] (the driver <ij||ab> is added by the final fill).
    // The terms with an antisymmetric (i<j, a<b) output and a pair-wise contraction run packed, into Pacc[(i<j)][(a<b)]:
    //   sum_{m<n} lambda^{mn}_{ab} W^{ij}_{mn}   (W^{ij}_{mn} = A^{kl}_{ij} of eq 31, packed in both pairs)
    CCSD_TRY(launch_transpose2d(st, L->l2p, L->l2pT, oo, vv, 0));
    CCSD_TRY(run_gemm(env, gp(vv, oo, oo, L->l2pT, oo, L->Amc, oo, L->Pacc, 1, vv, 1.0, 0)));
    // 1/2 lambda^{ij}_{ef} W^{ef}_{ab}, W^{ef}_{ab} = <ef||ab> - P(ef) t^f_m <em||ab> + 1/2 tau^{ef}_{mn} <mn||ab>, never stored:
    //   (iii) sum_{m<n} ( sum_{e<f} lambda^{ij}_{ef} tau^{ef}_{mn} ) <mn||ab>
    CCSD_TRY(run_gemm(env, gp(oo, oo, vv, L->l2p, vv, L->TAUp, vv, L->LTp, oo, 1, 1.0, 0)));
    CCSD_TRY(run_gemm(env, gp(vv, oo, oo, L->VoovvT, oo, L->LTp, oo, L->Pacc, 1, vv, 1.0, 1)));
    //   (ii) - sum_{em} ( sum_f lambda^{ij}_{ef} t^f_m ) <em||ab>
    {
        const c128* l2p = L->l2p;
        launch_fill(st, L->L2hu, oo * V, V, V, 0, [=] __device__(int64_t row, int64_t ff) {
            return asym_col(l2p, row / v, vv, (int)(row % v), (int)ff, v);
        });
        CCSD_TRY(run_gemm(env, gp(oo * V, O, V, L->L2hu, V, L->T1, V, L->Ltp, O, 1, 1.0, 0)));
        if (L->Ltps) launch_sum_plane(st, L->Ltp, L->Ltps, oo * c->ov);
        CCSD_TRY(run_gemm(env, with_planes(gp(vv, oo, c->ov, L->VT2, c->ov, L->Ltp, c->ov, L->Pacc, 1, vv, -1.0, 1), L->VT2s, L->Ltps)));
    }
    // P-_ij P-_ab ( sum_{me} lambda^{im}_{ae} W^{je}_{bm} + lambda^i_a Fbar^j_b ): the (ov)^3 GEMM as the ring of the CCSD iteration
    // runs it (operand laid out from the packed multipliers with its sum plane, the constant operand and plane laid out
    // once), both P- applied when the result is added into Pacc
    {
        const c128 *l2p = L->l2p, *l1 = L->l1, *Fov = L->Fov;
        const int64_t ov = c->ov;
        c128 *L2r = sc.a, *X = sc.c;
        double* L2rs = L->Wrs ? sc.as : nullptr;
        launch_fill(st, L2r, ov, ov, ov, 0, [=] __device__(int64_t ia, int64_t me) {      // [(i,a)][(m,e)] = lambda^{im}_{ae}
            const c128 x = t2_at(l2p, (int)(ia / v), (int)(me / v), (int)(ia % v), (int)(me % v), o, v, vv);
            if (L2rs) L2rs[ia * ov + me] = x.x + x.y;
            return x;
        });
        if (c->strassen)      // the Strassen levels of the CCSD iteration's (ov)^3 products, in the same scratch (strassen.cuh)
            CCSD_TRY(strassen_gemm(env, gp(ov, ov, ov, L2r, ov, L->Wr, ov, X, ov, 1, 1.0, 0), nullptr, nullptr, c->str_ring,
                                   c->strassen_levels));
        else
            CCSD_TRY(run_gemm(env, with_planes(gp(ov, ov, ov, L2r, ov, L->Wr, ov, X, ov, 1, 1.0, 0), L2rs, L->Wrs)));
        const int2 *po = c->po, *pv = c->pv;
        launch_fill(st, L->Pacc, oo, vv, vv, 1, [=] __device__(int64_t IJ, int64_t AB) {
            const int2 ij = po[IJ], ab = pv[AB];
            const int64_t i = ij.x, j = ij.y, a = ab.x, b = ab.y;
            c128 r = X[((i * v + a) * o + j) * v + b];
            r = csub(r, X[((j * v + a) * o + i) * v + b]);
            r = csub(r, X[((i * v + b) * o + j) * v + a]);
            r = cadd(r, X[((j * v + b) * o + i) * v + a]);
            cfma(r, l1[i * v + a], Fov[j * v + b]);
            cfma(r, cneg(l1[j * v + a]), Fov[i * v + b]);
            cfma(r, cneg(l1[i * v + b]), Fov[j * v + a]);
            cfma(r, l1[j * v + b], Fov[i * v + a]);
            return r;
        });
    }
    // -P-_ij sum_m ( lambda^{im}_{ab} Fbar^j_m + <im||ab> G^m_j ) on (a<b) rows and -P-_ab sum_m lambda^m_a W^{ij}_{mb} on (i<j) rows
    {
        const c128 *l2pT = L->l2pT;
        c128 *L2r2 = sc.b, *U = sc.a, *Vb = sc.c;        // [(a<b)][i][m], U[(a<b)][i][j], Vb[(i<j)][b][a]
        launch_fill(st, L2r2, vv, O * O, O * O, 0, [=] __device__(int64_t AB, int64_t im) {
            const int i = (int)(im / o), m = (int)(im % o);
            if (i == m) return mk(0.0, 0.0);
            return i < m ? l2pT[AB * oo + pair_idx(i, m, o)] : cneg(l2pT[AB * oo + pair_idx(m, i, o)]);
        });
        CCSD_TRY(permute_into(st, L->GooT, "jm", LV(L->Goo, "mj", O, O), 1.0, 0));
        CCSD_TRY(permute_into(st, L->l1T, "am", LV(L->l1, "ma", O, V), 1.0, 0));
        CCSD_TRY(run_gemm(env, gp(vv * O, O, O, L2r2, O, L->Foo, O, U, O, 1, 1.0, 0)));
        CCSD_TRY(run_gemm(env, gp(vv * O, O, O, L->OOVVr, O, L->GooT, O, U, O, 1, 1.0, 1)));
        CCSD_TRY(run_gemm(env, gp(oo * V, V, O, L->Wooov_r, O, L->l1T, O, Vb, V, 1, 1.0, 0)));
        const int2 *po = c->po, *pv = c->pv;
        launch_fill(st, L->Pacc, oo, vv, vv, 1, [=] __device__(int64_t IJ, int64_t AB) {
            const int2 ij = po[IJ], ab = pv[AB];
            const c128 u = csub(U[(AB * o + ij.y) * o + ij.x], U[(AB * o + ij.x) * o + ij.y]);
            const c128 w = csub(Vb[(IJ * v + ab.x) * v + ab.y], Vb[(IJ * v + ab.y) * v + ab.x]);
            return cadd(u, w);
        });
    }
    // P-_ab sum_e ( lambda^{ij}_{ae} Fbar^e_b + <ij||ae> G^b_e ) and P-_ij sum_e lambda^i_e W^{ej}_{ab}: the products run over the
    // packed output pair ((i<j) rows, resp. (a<b) rows), the P- of the other pair is applied when they are added into Pacc
    {
        c128 *Y = sc.c, *Z = sc.a;                       // Y[(i<j)][a][b], Z[j][(a<b)][i]
        CCSD_TRY(run_gemm(env, gp(oo * V, V, V, L->L2hu, V, L->FvvT, V, Y, V, 1, 1.0, 0)));
        CCSD_TRY(run_gemm(env, gp(oo * V, V, V, L->OOVVhu, V, L->Gvv, V, Y, V, 1, 1.0, 1)));
        CCSD_TRY(run_gemm(env, gp(O * vv, O, V, L->Wjp, V, L->l1, V, Z, O, 1, 1.0, 0)));
        const int2 *po = c->po, *pv = c->pv;
        launch_fill(st, L->Pacc, oo, vv, vv, 1, [=] __device__(int64_t IJ, int64_t AB) {
            const int2 ij = po[IJ], ab = pv[AB];
            const c128 y = csub(Y[(IJ * v + ab.x) * v + ab.y], Y[(IJ * v + ab.y) * v + ab.x]);
            const c128 z = csub(Z[((int64_t)ij.y * vv + AB) * o + ij.x], Z[((int64_t)ij.x * vv + AB) * o + ij.y]);
            return cadd(y, z);
        });
    }
    //   (i) sum_{e<f} lambda^{ij}_{ef} <ef||ab> = conj( sum_{e<f} conj(lambda) <ab||ef> ): the pp-ladder launch of the CCSD
    //       iteration (packed, Hermitian <ab||cd>, 3M with sum planes) on the conjugated multipliers
    {
        const c128* l2p = L->l2p;
        double* plane = c->planes ? L->cl2s : nullptr;
        launch_fill(st, L->cl2p, oo, vv, vv, 0, [=] __device__(int64_t IJ, int64_t EF) {
            c128 x = cconj(l2p[IJ * vv + EF]);
            if (plane) plane[IJ * vv + EF] = x.x + x.y;
            return x;
        });
        const int lvL = c->strassen_levels_L;
        if (c->strassen && c->sW.S && strassen_stack_elems(oo, vv, lvL) <= c->str_ring.b_elems) {
            // one Strassen level with the stack of <ab||cd> ccsd_init made; conj(lambda) is stacked in the scratch of the (ov)^3
            // products (idle here; tau's own stack stays valid for the CCSD residual's per-term hooks)
            StrassenStack sl = strassen_stack(c->str_ring.SB, c->str_ring.SBp, oo, vv, lvL);
            launch_strassen_prep(st, 1, L->cl2p, vv, sl);
            CCSD_TRY(strassen_gemm(env, gp(vv, oo, vv, c->W, vv, L->cl2p, vv, L->P2, 1, vv, 1.0, 0), &c->sW, &sl, c->str_L, lvL));
        } else {
            if (!c->W) return CCSD_ESTATE;
            CCSD_TRY(run_gemm(env, with_planes(gp(vv, oo, vv, c->W, vv, L->cl2p, vv, L->P2, 1, vv, 1.0, 0), c->Ws, plane)));
        }
    }
    {   // R2p[(i<j)][(a<b)] = <ij||ab> + conj(P2) + Pacc
        const c128 *Voovv = c->Voovv_p, *P2 = L->P2, *Pacc = L->Pacc;
        launch_fill(st, L->R2p, oo, vv, vv, 0, [=] __device__(int64_t IJ, int64_t AB) {
            return cadd(cadd(Voovv[IJ * vv + AB], cconj(P2[IJ * vv + AB])), Pacc[IJ * vv + AB]);
        });
    }
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

// One Lambda iteration: residual, Jacobi step lambda <- lambda + R/D with the CCSD denominators, DIIS as for the
// amplitudes (readings G12, G13, G23).  Returns ||R/D||_2 over the unique multipliers through *step_norm (host).
static int lambda_iterate(ccsd_ctx* c, LambdaState* L, double* step_norm)
{
    CCSD_TRY(lambda_residual(c, L));
    cudaStream_t st = c->st;
    // CCD: the Lagrangian has no singles constraint, lambda^i_a stays zero (the ccd flag of the update kernel)
    launch_jacobi_diis(st, L->diis, c->o, c->v, L->R1, L->R2p, L->l1, L->l2p, c->eps, c->po, c->pv, c->opt.ccd);
    CCSD_CUDA_TRY(cudaMemcpyAsync(c->red_host + 36, L->diis.info, 2 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CCSD_CUDA_TRY(cudaStreamSynchronize(st));
    if (step_norm) *step_norm = sqrt(c->red_host[36] > 0 ? c->red_host[36] : 0.0);
    CCSD_CUDA_TRY(cudaGetLastError());
    return c->red_host[37] != 0.0 ? CCSD_ESINGULAR : CCSD_OK;
}

// eqs 58-61: D[p][q] = <0|(1+Lambda) exp(-T) a+_p a_q exp(T)|0> - delta_pq(occ), [n][n] (device), unsymmetrised (reading G24)
static int lambda_density(ccsd_ctx* c, LambdaState* L, c128* D)
{
    cudaStream_t st = c->st;
    const Env& env = c->env;
    const TcScratch& sc = L->sc;
    const int o = c->o, v = c->v, n = c->n;
    const int64_t O = o, V = v;
    unpack_pairs(st, L->L2, L->l2p, o, 1, v, 1);
    // temporaries: the residual buffers of the solver are free between iterations
    c128 *goo = L->Goo, *gab = L->Gvv, *gai = L->R1, *x_oo = L->LT, *x_ea = L->R2;
    CCSD_CUDA_TRY(cudaMemsetAsync(goo, 0, (size_t)(O * O) * sizeof(c128), st));
    CCSD_CUDA_TRY(cudaMemsetAsync(gab, 0, (size_t)(V * V) * sizeof(c128), st));
    // eq 58: gamma_ij = -1/2 t^{ef}_{im} lambda^{jm}_{ef} - t^e_i lambda^j_e
    CCSD_TRY(tc1(env, sc, -0.5, LV(L->T2, "imef", O, O, V, V), LV(L->L2, "jmef", O, O, V, V), goo, "ij"));
    CCSD_TRY(tc1(env, sc, -1.0, LV(L->T1, "ie", O, V), LV(L->l1, "je", O, V), goo, "ij"));
    // eq 61: gamma_ab = 1/2 t^{ae}_{mn} lambda^{mn}_{be} + t^a_m lambda^m_b
    CCSD_TRY(tc1(env, sc, 0.5, LV(L->T2, "mnae", O, O, V, V), LV(L->L2, "mnbe", O, O, V, V), gab, "ab"));
    CCSD_TRY(tc1(env, sc, 1.0, LV(L->T1, "ma", O, V), LV(L->l1, "mb", O, V), gab, "ab"));
    // eq 60 as [i][a]: t + lambda^m_e (t^{ae}_{im} - t^e_i t^a_m) - 1/2 lambda^{mn}_{ef} (t^{ef}_{in} t^a_m + t^e_i t^{af}_{mn})
    dcopy(st, gai, L->T1, O * V);
    CCSD_TRY(tc1(env, sc, 1.0, LV(L->l1, "me", O, V), LV(L->T2, "imae", O, O, V, V), gai, "ia"));
    //   - ( sum_e lambda^m_e t^e_i + 1/2 sum_nef lambda^{mn}_{ef} t^{ef}_{in} ) t^a_m
    CCSD_CUDA_TRY(cudaMemsetAsync(x_oo, 0, (size_t)(O * O) * sizeof(c128), st));
    CCSD_TRY(tc1(env, sc, 1.0, LV(L->l1, "me", O, V), LV(L->T1, "ie", O, V), x_oo, "mi"));
    CCSD_TRY(tc1(env, sc, 0.5, LV(L->L2, "mnef", O, O, V, V), LV(L->T2, "inef", O, O, V, V), x_oo, "mi"));
    CCSD_TRY(tc1(env, sc, -1.0, LV(x_oo, "mi", O, O), LV(L->T1, "ma", O, V), gai, "ia"));
    //   - 1/2 t^e_i ( sum_mnf lambda^{mn}_{ef} t^{af}_{mn} )
    CCSD_CUDA_TRY(cudaMemsetAsync(x_ea, 0, (size_t)(V * V) * sizeof(c128), st));
    CCSD_TRY(tc1(env, sc, 1.0, LV(L->L2, "mnef", O, O, V, V), LV(L->T2, "mnaf", O, O, V, V), x_ea, "ea"));
    CCSD_TRY(tc1(env, sc, -0.5, LV(L->T1, "ie", O, V), LV(x_ea, "ea", V, V), gai, "ia"));
    const c128* l1 = L->l1;
    launch_fill(st, D, n, n, n, 0, [=] __device__(int64_t p, int64_t q) {
        if (p < o && q < o) return goo[p * o + q];                       // gamma_ij = <a+_i a_j>
        if (p >= o && q >= o) return gab[(q - o) * v + (p - o)];         // gamma_ab = <a+_b a_a>
        if (p < o) return gai[p * v + (q - o)];                          // <a+_i a_a> = gamma_ai
        return l1[q * v + (p - o)];                                      // <a+_a a_i> = gamma_ia = lambda^i_a
    });
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}
#undef LV
