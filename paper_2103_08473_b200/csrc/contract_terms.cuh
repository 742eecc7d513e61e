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
    if (oo > 0) { pair_table_kernel<<<(unsigned)((oo + 255) / 256), 256, 0, st>>>(W.po, o); g_launches++; }
    if (vv > 0) { pair_table_kernel<<<(unsigned)((vv + 255) / 256), 256, 0, st>>>(W.pv, v); g_launches++; }
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
#undef TV
