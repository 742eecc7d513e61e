// Standalone evaluation of the intermediates of Appendix 7.1 (eqs 24-31) on caller-supplied tensors in
// the canonical layouts of include/ccsd.h: the ccsd_contract terms F_OV, F_VV, F_OO, W_OOOO, W_OVVO, C_OVOO (the names of
// BASELINE.json north_star: F_me, F_ae, F_mi, W_mnij, W_mbej and the C intermediate; DESIGN.md relates them to the
// paper's H/G/A/C).  Per-term parity and timing hooks: written term by term with tensor_contract (tensor_ops.cuh,
// lambda.cuh) on unpacked copies of the inputs; ccsd_iterate evaluates the same equations on its resident,
// pre-laid-out operands (ccsd_lib.cu) and is what the per-term times of bench.py refer to.
#pragma once
#include "lambda.cuh"

struct TermWs {
    TcScratch sc;
    int2 *po, *pv;
    c128 *taup, *T2, *TAU, *OOVV, *OOOV, *VOVV, *OOOO, *X, *tmp, *Fov, *Fvv, *Foo;
};
static void term_carve(int o_, int v_, char* base, TermWs* W, size_t* total)
{
    Carver w{base, 0};
    const int64_t o = o_, v = v_, oo = o * (o - 1) / 2, vv = v * (v - 1) / 2;
    const int64_t o2v2 = o * o * v * v, ov3 = o * v * v * v, o3v = o * o * o * v;
    W->sc.elems = ov3 > o2v2 ? ov3 : o2v2;
    if (W->sc.elems < o3v) W->sc.elems = o3v;
    if (W->sc.elems < o * o * o * o) W->sc.elems = o * o * o * o;
    W->sc.a = w.take<c128>(W->sc.elems);
    W->sc.b = w.take<c128>(W->sc.elems);
    W->sc.c = w.take<c128>(W->sc.elems);
    W->sc.as = W->sc.bs = nullptr;
    W->sc.plane_elems = 0;
    W->po = w.take<int2>(oo);
    W->pv = w.take<int2>(vv);
    W->taup = w.take<c128>(oo * vv);
    W->T2 = w.take<c128>(o2v2); W->TAU = w.take<c128>(o2v2); W->OOVV = w.take<c128>(o2v2);
    W->OOOV = w.take<c128>(o3v); W->VOVV = w.take<c128>(ov3); W->OOOO = w.take<c128>(o * o * o * o);
    W->X = w.take<c128>(o2v2); W->tmp = w.take<c128>(o2v2 > o3v ? o2v2 : o3v);
    W->Fov = w.take<c128>(o * v); W->Fvv = w.take<c128>(v * v); W->Foo = w.take<c128>(o * o);
    *total = w.off;
}

#define TV(ptr, idx, ...) tview(ptr, idx, __VA_ARGS__)

static int contract_intermediate(int term, int o, int v, const c128* const* in, int nin, c128* out, const Env& env, char* workspace)
{
    cudaStream_t st = env.st;
    TermWs W;
    size_t total = 0;
    term_carve(o, v, workspace, &W, &total);
    const TcScratch& sc = W.sc;
    const int n = o + v;
    const int64_t O = o, V = v, oo = O * (O - 1) / 2, vv = V * (V - 1) / 2;
    if (oo > 0) { pair_table_kernel<<<(unsigned)((oo + 255) / 256), 256, 0, st>>>(W.po, o); count_launches(1); }
    if (vv > 0) { pair_table_kernel<<<(unsigned)((vv + 255) / 256), 256, 0, st>>>(W.pv, v); count_launches(1); }
    // which inputs are which (see include/ccsd.h)
    const c128 *f = nullptr, *oovv = nullptr, *vovv = nullptr, *ooov = nullptr, *oooo = nullptr, *vovo = nullptr, *t1 = nullptr, *t2p = nullptr;
    switch (term) {
    case CCSD_TERM_F_OV: if (nin < 3) return CCSD_EINVAL; f = in[0]; oovv = in[1]; t1 = in[2]; break;
    case CCSD_TERM_F_VV: if (nin < 5) return CCSD_EINVAL; f = in[0]; oovv = in[1]; vovv = in[2]; t1 = in[3]; t2p = in[4]; break;
    case CCSD_TERM_F_OO: if (nin < 5) return CCSD_EINVAL; f = in[0]; oovv = in[1]; ooov = in[2]; t1 = in[3]; t2p = in[4]; break;
    case CCSD_TERM_W_OOOO: if (nin < 5) return CCSD_EINVAL; oooo = in[0]; ooov = in[1]; oovv = in[2]; t1 = in[3]; t2p = in[4]; break;
    case CCSD_TERM_W_OVVO: if (nin < 6) return CCSD_EINVAL; vovo = in[0]; vovv = in[1]; ooov = in[2]; oovv = in[3]; t1 = in[4]; t2p = in[5]; break;
    case CCSD_TERM_C_OVOO: if (nin < 5) return CCSD_EINVAL; ooov = in[0]; vovo = in[1]; vovv = in[2]; t1 = in[3]; t2p = in[4]; break;
    default: return CCSD_EINVAL;
    }
    for (int q = 0; q < nin; q++)
        if (!in[q]) return CCSD_EINVAL;
    // unpacked copies of the packed inputs
    if (t2p) {
        build_tau(st, W.taup, t1, t2p, o, v, W.po, W.pv, nullptr);                 // eq 23
        unpack_pairs(st, W.T2, t2p, o, 1, v, 1);
        unpack_pairs(st, W.TAU, W.taup, o, 1, v, 1);
    }
    if (oovv) unpack_pairs(st, W.OOVV, oovv, o, 1, v, 1);
    if (ooov) unpack_pairs(st, W.OOOV, ooov, o, 1, 0, 0, O * V);
    if (oooo) unpack_pairs(st, W.OOOO, oooo, o, 1, o, 1);
    if (vovv) {   // [a][k][(c<d)] -> [a][k][c][d]
        c128* dst = W.VOVV;
        launch_fill(st, dst, V * O * V, V, V, 0, [=] __device__(int64_t row, int64_t d) {
            return asym_col(vovv, row / v, vv, (int)(row % v), (int)d, v);
        });
    }
    if (f) {
        launch_fill(st, W.Fov, O, V, V, 0, [=] __device__(int64_t k, int64_t c) { return f[k * n + o + c]; });
        launch_fill(st, W.Fvv, V, V, V, 0, [=] __device__(int64_t a, int64_t c) { return f[(o + a) * n + o + c]; });
        launch_fill(st, W.Foo, O, O, O, 0, [=] __device__(int64_t k, int64_t i) { return f[k * n + i]; });
    }
    switch (term) {
    case CCSD_TERM_F_OV:     // eq 28: H^k_c = f_kc + sum_ld <kl||cd> t^d_l
        dcopy(st, out, W.Fov, O * V);
        CCSD_TRY(tc1(env, sc, 1.0, TV(W.OOVV, "klcd", O, O, V, V), TV(t1, "ld", O, V), out, "kc"));
        break;
    case CCSD_TERM_F_VV:     // eqs 24-25: G^a_c = f_ac + 1/2 sum <kl||cd> tau^{da}_{kl} + sum <ak||cd> t^d_k - sum f_kc t^a_k
        dcopy(st, out, W.Fvv, V * V);
        CCSD_TRY(tc1(env, sc, 0.5, TV(W.OOVV, "klcd", O, O, V, V), TV(W.TAU, "klda", O, O, V, V), out, "ac"));
        CCSD_TRY(tc1(env, sc, 1.0, TV(W.VOVV, "akcd", V, O, V, V), TV(t1, "kd", O, V), out, "ac"));
        CCSD_TRY(tc1(env, sc, -1.0, TV(W.Fov, "kc", O, V), TV(t1, "ka", O, V), out, "ac"));
        break;
    case CCSD_TERM_F_OO:     // eqs 26-27: G^k_i = -f_ki + 1/2 sum <kl||cd> tau^{cd}_{li} - sum <kl||ic> t^c_l - sum f_kc t^c_i
        CCSD_TRY(permute_into(st, out, "ki", TV(W.Foo, "ki", O, O), -1.0, 0));
        CCSD_TRY(tc1(env, sc, 0.5, TV(W.OOVV, "klcd", O, O, V, V), TV(W.TAU, "licd", O, O, V, V), out, "ki"));
        CCSD_TRY(tc1(env, sc, -1.0, TV(W.OOOV, "klic", O, O, O, V), TV(t1, "lc", O, V), out, "ki"));
        CCSD_TRY(tc1(env, sc, -1.0, TV(W.Fov, "kc", O, V), TV(t1, "ic", O, V), out, "ki"));
        break;
    case CCSD_TERM_W_OOOO: { // eq 31: A^{kl}_{ij} = <kl||ij> + P-_ij sum_c <kl||ic> t^c_j + 1/2 sum_cd <kl||cd> tau^{cd}_{ij}
        c128* A = W.tmp;
        dcopy(st, A, W.OOOO, O * O * O * O);
        CCSD_TRY(tc2(env, sc, 1.0, TV(W.OOOV, "klic", O, O, O, V), TV(t1, "jc", O, V), A, "klij", "klji"));
        CCSD_TRY(tc1(env, sc, 0.5, TV(W.OOVV, "klcd", O, O, V, V), TV(W.TAU, "ijcd", O, O, V, V), A, "klij"));
        const int2* po = W.po;
        launch_fill(st, out, oo, oo, oo, 0, [=] __device__(int64_t KL, int64_t IJ) {
            const int2 kl = po[KL], ij = po[IJ];
            return A[(((int64_t)kl.x * o + kl.y) * o + ij.x) * o + ij.y];
        });
        break;
    }
    case CCSD_TERM_W_OVVO:   // eq 29: H^{ak}_{ci} = <ak||ci> + sum_d <ak||cd> t^d_i - sum_l <kl||ic> t^a_l + sum_ld <kl||cd> (t^{ad}_{li}/2 + t^a_l t^d_i)
        dcopy(st, out, vovo, V * O * V * O);
        CCSD_TRY(tc1(env, sc, 1.0, TV(W.VOVV, "akcd", V, O, V, V), TV(t1, "id", O, V), out, "akci"));
        CCSD_TRY(tc1(env, sc, -1.0, TV(W.OOOV, "klic", O, O, O, V), TV(t1, "la", O, V), out, "akci"));
        CCSD_TRY(permute_into(st, W.X, "liad", TV(W.T2, "liad", O, O, V, V), 0.5, 0));
        CCSD_TRY(tc1(env, sc, 1.0, TV(t1, "la", O, V), TV(t1, "id", O, V), W.X, "liad"));
        CCSD_TRY(tc1(env, sc, 1.0, TV(W.OOVV, "klcd", O, O, V, V), TV(W.X, "liad", O, O, V, V), out, "akci"));
        break;
    case CCSD_TERM_C_OVOO: { // eq 30: C^{kb}_{ij} = conj <ij||kb> + P-_ij sum_c <bk||ci> t^c_j - 1/2 sum_cd <bk||cd> tau^{cd}_{ij}
        c128* C = W.tmp;
        CCSD_TRY(permute_into(st, C, "kbij", TV(W.OOOV, "ijkb", O, O, O, V), 1.0, 0, 1));
        CCSD_TRY(tc2(env, sc, 1.0, TV(vovo, "bkci", V, O, V, O), TV(t1, "jc", O, V), C, "kbij", "kbji"));
        CCSD_TRY(tc1(env, sc, -0.5, TV(W.VOVV, "bkcd", V, O, V, V), TV(W.TAU, "ijcd", O, O, V, V), C, "kbij"));
        const int2* po = W.po;
        launch_fill(st, out, O * V, oo, oo, 0, [=] __device__(int64_t kb, int64_t IJ) {
            const int2 ij = po[IJ];
            return C[(kb * o + ij.x) * o + ij.y];
        });
        break;
    }
    default: return CCSD_EINVAL;
    }
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}
// ---------------------------------------------------------------------------------------------------------------
// The remaining rows of the iteration as standalone terms: S1_RESIDUAL (eq 33),
// S2_SMALL_TERMS (the G_oo, V^dagger t1, G_vv, C t1 and driver lines of eq 32), ENERGY (eq 9,
// PAPER.md:97) and JACOBI_UPDATE (reading G12).  Same per-term parity role as the intermediates above.
// ---------------------------------------------------------------------------------------------------------------
static int contract_residual_term(int term, int o, int v, const c128* const* in, int nin, c128* out, const Env& env, char* workspace)
{
    cudaStream_t st = env.st;
    TermWs W;
    size_t total = 0;
    term_carve(o, v, workspace, &W, &total);
    const TcScratch& sc = W.sc;
    const int n = o + v;
    const int64_t O = o, V = v, oo = O * (O - 1) / 2, vv = V * (V - 1) / 2;
    for (int q = 0; q < nin; q++)
        if (!in[q]) return CCSD_EINVAL;
    pair_table_kernel<<<(unsigned)((oo + 255) / 256), 256, 0, st>>>(W.po, o);
    pair_table_kernel<<<(unsigned)((vv + 255) / 256), 256, 0, st>>>(W.pv, v);
    count_launches(2);
    if (term == CCSD_TERM_S1_RESIDUAL) {
        const c128 *f = in[0], *Hvv = in[1], *Hoo = in[2], *Hov = in[3], *vovv = in[4], *ooov = in[5], *vovo = in[6], *t1 = in[7], *t2p = in[8];
        build_tau(st, W.taup, t1, t2p, o, v, W.po, W.pv, nullptr);                 // eq 23
        unpack_pairs(st, W.T2, t2p, o, 1, v, 1);
        unpack_pairs(st, W.TAU, W.taup, o, 1, v, 1);
        unpack_pairs(st, W.OOOV, ooov, o, 1, 0, 0, O * V);
        c128* VOVV = W.VOVV;
        launch_fill(st, VOVV, V * O * V, V, V, 0, [=] __device__(int64_t row, int64_t d) {
            return asym_col(vovv, row / v, vv, (int)(row % v), (int)d, v);
        });
        // conj f_ia (= f_ai) + sum_c H^a_c t^c_i + sum_k H^k_i t^a_k + sum_kc H^k_c t^{ac}_{ik}
        launch_fill(st, out, O, V, V, 0, [=] __device__(int64_t i, int64_t a) { return cconj(f[i * n + o + a]); });
        CCSD_TRY(tc1(env, sc, 1.0, TV(Hvv, "ac", V, V), TV(t1, "ic", O, V), out, "ia"));
        CCSD_TRY(tc1(env, sc, 1.0, TV(Hoo, "ki", O, O), TV(t1, "ka", O, V), out, "ia"));
        CCSD_TRY(tc1(env, sc, 1.0, TV(Hov, "kc", O, V), TV(W.T2, "ikac", O, O, V, V), out, "ia"));
        // sum_k ( sum_c (H^k_c - 2 f_kc) t^c_i ) t^a_k
        launch_fill(st, W.Fov, O, V, V, 0, [=] __device__(int64_t k, int64_t c) {
            return csub(Hov[k * v + c], cscale(2.0, f[k * n + o + c]));
        });
        CCSD_CUDA_TRY(cudaMemsetAsync(W.Foo, 0, (size_t)(O * O) * sizeof(c128), st));
        CCSD_TRY(tc1(env, sc, 1.0, TV(W.Fov, "kc", O, V), TV(t1, "ic", O, V), W.Foo, "ki"));
        CCSD_TRY(tc1(env, sc, 1.0, TV(W.Foo, "ki", O, O), TV(t1, "ka", O, V), out, "ia"));
        // 1/2 sum_kcd <ak||cd> tau^{cd}_{ik} + 1/2 sum_klc <kl||ic> tau^{ca}_{kl} - sum_kc <ak||ci> t^c_k
        CCSD_TRY(tc1(env, sc, 0.5, TV(W.VOVV, "akcd", V, O, V, V), TV(W.TAU, "ikcd", O, O, V, V), out, "ia"));
        CCSD_TRY(tc1(env, sc, 0.5, TV(W.OOOV, "klic", O, O, O, V), TV(W.TAU, "klca", O, O, V, V), out, "ia"));
        CCSD_TRY(tc1(env, sc, -1.0, TV(vovo, "akci", V, O, V, O), TV(t1, "kc", O, V), out, "ia"));
    } else if (term == CCSD_TERM_S2_SMALL_TERMS) {
        const c128 *Gvv = in[0], *Goo = in[1], *Cp = in[2], *vovv = in[3], *oovv = in[4], *t1 = in[5], *t2p = in[6];
        unpack_pairs(st, W.T2, t2p, o, 1, v, 1);
        c128* VOVVc = W.VOVV;                       // conj <cj||ab> as [c][j][a][b]
        launch_fill(st, VOVVc, V * O * V, V, V, 0, [=] __device__(int64_t row, int64_t b) {
            return cconj(asym_col(vovv, row / v, vv, (int)(row % v), (int)b, v));
        });
        c128* Cu = W.tmp;                           // C [k][a][i][j]
        launch_fill(st, Cu, O * V * O, O, O, 0, [=] __device__(int64_t row, int64_t j) {
            return asym_col(Cp, row / o, oo, (int)(row % o), (int)j, o);
        });
        c128* S = W.X;
        CCSD_CUDA_TRY(cudaMemsetAsync(S, 0, (size_t)(O * O * V * V) * sizeof(c128), st));
        CCSD_TRY(tc2(env, sc, 1.0, TV(Goo, "kj", O, O), TV(W.T2, "ikab", O, O, V, V), S, "ijab", "jiab"));     // P-_ji sum_k G^k_j t^{ab}_{ik}
        CCSD_TRY(tc2(env, sc, 1.0, TV(VOVVc, "cjab", V, O, V, V), TV(t1, "ic", O, V), S, "ijab", "jiab"));     // P-_ij sum_c conj<cj||ab> t^c_i
        CCSD_TRY(tc2(env, sc, 1.0, TV(Gvv, "ac", V, V), TV(W.T2, "ijcb", O, O, V, V), S, "ijab", "ijba"));     // P-_ab sum_c G^a_c t^{cb}_{ij}
        CCSD_TRY(tc2(env, sc, 1.0, TV(Cu, "kaij", O, V, O, O), TV(t1, "kb", O, V), S, "ijab", "ijba"));        // P-_ab sum_k C^{ka}_{ij} t^b_k
        const int2 *po = W.po, *pv = W.pv;
        launch_fill(st, out, oo, vv, vv, 0, [=] __device__(int64_t IJ, int64_t AB) {                           // + conj <ij||ab>, packed
            const int2 ij = po[IJ], ab = pv[AB];
            return cadd(S[(((int64_t)ij.x * o + ij.y) * v + ab.x) * v + ab.y], cconj(oovv[IJ * vv + AB]));
        });
    } else {
        return CCSD_EINVAL;
    }
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

// ENERGY and JACOBI_UPDATE stream over the packed amplitudes; their workspace is the pair tables, tau and eps only.
struct StreamWs {
    int2 *po, *pv;
    c128 *taup, *evec;
    double *eps, *scratch;
};
static void stream_carve(int o_, int v_, char* base, StreamWs* W, size_t* total)
{
    Carver w{base, 0};
    const int64_t o = o_, v = v_, oo = o * (o - 1) / 2, vv = v * (v - 1) / 2;
    W->po = w.take<int2>(oo);
    W->pv = w.take<int2>(vv);
    W->taup = w.take<c128>(oo * vv);
    W->evec = w.take<c128>(o * v + oo * vv);
    W->eps = w.take<double>(o + v);
    W->scratch = w.take<double>(RED_SCRATCH_DOUBLES);
    *total = w.off;
}
static int contract_stream_term(int term, int o, int v, const c128* const* in, int nin, c128* out, cudaStream_t st, char* workspace,
                                double level_shift, int ccd)
{
    StreamWs W;
    size_t total = 0;
    stream_carve(o, v, workspace, &W, &total);
    const int n = o + v;
    const int64_t O = o, V = v, oo = O * (O - 1) / 2, vv = V * (V - 1) / 2;
    for (int q = 0; q < nin; q++)
        if (!in[q]) return CCSD_EINVAL;
    pair_table_kernel<<<(unsigned)((oo + 255) / 256), 256, 0, st>>>(W.po, o);
    pair_table_kernel<<<(unsigned)((vv + 255) / 256), 256, 0, st>>>(W.pv, v);
    count_launches(2);
    if (term == CCSD_TERM_ENERGY) {          // E = sum_ia f_ia t^a_i + sum_{i<j,a<b} <ij||ab> tau^{ab}_{ij}: the kernel ccsd_iterate uses
        const c128 *f = in[0], *oovv = in[1], *t1 = in[2], *t2p = in[3];
        launch_energy_tau(st, W.scratch, f, n, o, v, t1, t2p, oovv, W.taup, nullptr, W.po, W.pv, reinterpret_cast<double*>(out));
    } else if (term == CCSD_TERM_JACOBI_UPDATE) {   // u = t + S / D, D from eps_p = Re f_pp (+ level shift on the virtuals):
        const c128 *f = in[0], *t1 = in[1], *t2p = in[2], *S1 = in[3], *S2 = in[4];     // the kernel ccsd_iterate uses, no DIIS
        eps_kernel<<<(n + 127) / 128, 128, 0, st>>>(f, W.eps, nullptr, n, o, level_shift);
        count_launches(1);
        const VecTiles T = vec_tiles(o, v);
        JacobiArgs ja;
        ja.T = T; ja.S1 = S1; ja.S2 = S2; ja.t1 = t1; ja.t2p = t2p; ja.E = W.evec; ja.U = out;
        for (int k = 0; k < DIIS_MAX; k++) ja.Eold[k] = nullptr;
        ja.m = 1; ja.eps = W.eps; ja.po = W.po; ja.pv = W.pv; ja.ccd = ccd; ja.partials = W.scratch;
        jacobi_multidot_kernel<<<tile_blocks(T), RED_THREADS, 0, st>>>(ja);
        count_launches(1);
    } else {
        return CCSD_EINVAL;
    }
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}
#undef TV
