// B200-native complex spinor-basis CCSD hot path: C ABI + host-side iteration driver.
// Equations: arXiv 2103.08473 Appendix 7.1 (eqs 22-33) in the reading of DESIGN.md.
// Every step runs in CUDA kernels of this library; there is no CPU fallback and no code shared with oracle/.
//
// Design (DESIGN.md "Data layout" / "Kernels"): every contraction of eqs 24-33 is brought to ONE form,
//     C[m][n] (+)= alpha * sum_k A[m][k] * B[n][k]          ("NT": both operands K-contiguous)
// by keeping the constant integral classes resident in HBM in every operand layout they are needed in (180 GB
// part: redundancy is cheap) and by re-laying-out the amplitudes once per iteration with bandwidth-bound fill /
// transpose kernels.  The GEMM is the FP64 tensor-core (DMMA) kernel of gemm_dmma.cuh.
#include "../../include/ccsd.h"
#include "common.cuh"
#include "fill.cuh"
#include "gemm_simple.cuh"
#include "gemm_dmma.cuh"
#include "triples.cuh"
#include "transpose.cuh"
#include "reduce.cuh"
#include "strassen.cuh"
#include "peak.cuh"

#include <cmath>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

thread_local char g_cuda_err[256] = "";
std::atomic<long long> g_launches{0};
thread_local long long t_launch_tally = 0;

// ---------------------------------------------------------------------------------------------------------------
// GEMM front end
// ---------------------------------------------------------------------------------------------------------------
struct Env {
    cudaStream_t st;
    int gemm_mode;          // 0 auto, 1 simple only, 2 DMMA 4M, 3 DMMA 3M, 100+v explicit variant
    c128* partial;          // split-K scratch
    int64_t partial_elems;
};

static GemmParams gp(int64_t M, int64_t N, int64_t K, const c128* A, int64_t lda, const c128* B, int64_t ldb, c128* C,
                     int64_t csm, int64_t csn, double alpha, int acc)
{
    GemmParams p;
    memset(&p, 0, sizeof(p));
    p.M = M; p.N = N; p.K = K;
    p.A = A; p.sam = lda; p.sak = 1;
    p.B = B; p.sbn = ldb; p.sbk = 1;
    p.C = C; p.csm = csm; p.csn = csn;
    p.alpha = mk(alpha, 0.0); p.accumulate = acc;
    p.batch = 1; p.ksplit = 1; p.kchunk = K;
    return p;
}

static GemmParams with_planes(GemmParams p, const double* As, const double* Bs)
{
    p.As = As; p.Bs = Bs;
    return p;
}

static int run_gemm(const Env& env, GemmParams p)
{
    if (p.M <= 0 || p.N <= 0 || p.batch <= 0) return CCSD_OK;
    if (p.K <= 0) return p.accumulate ? CCSD_OK : CCSD_EINVAL;
    bool dmma_ok = dmma_supported(p);
    // gemm_mode: 0 auto, 1 simple FMA kernel, 2 DMMA 4M, 3 DMMA 3M, 100+v explicit DMMA variant v (tuning)
    // sum planes are staged by TMA: 16-byte aligned rows, i.e. even leading dimensions
    const bool planes_ok = p.As && p.Bs && p.sam % 2 == 0 && p.sbn % 2 == 0 && (p.batch == 1 || (p.bsA % 2 == 0 && p.bsB % 2 == 0)) &&
                           ((reinterpret_cast<uintptr_t>(p.As) | reinterpret_cast<uintptr_t>(p.Bs)) & 15) == 0;
    int family = -1;   // -1 simple kernel, 0 4M, 1 3M, 2 3M with planes, 3 one explicit variant
    if (env.gemm_mode >= 100) family = 3;
    else if (env.gemm_mode == 2) family = 0;
    else if (env.gemm_mode == 3) family = planes_ok ? 2 : 1;
    else if (env.gemm_mode == 0 && dmma_ok && dmma_worthwhile(p)) family = CCSD_DEFAULT_3M != 0 ? (planes_ok ? 2 : 1) : 0;
    if (family == 3 && env.gemm_mode - 100 >= DMMA_NVARIANTS) return CCSD_EINVAL;
    if (family >= 0 && !dmma_ok) {   // strided operands: an explicitly requested tile variant is an error, a forced family is not
        if (family == 3) return CCSD_EINVAL;
        family = -1;
    }
    const bool use_dmma = family >= 0;
    int variant = -1;
    p.ksplit = 1; p.kchunk = p.K; p.partial = nullptr;
    if (use_dmma) {   // tile variant and split-K depth together, against wave quantisation on the 148 SMs (dmma_plan)
        const DmmaPlan plan = dmma_plan(p.M, p.N, p.K, p.batch, family != 0, family == 2, env.partial != nullptr, env.partial_elems,
                                        family == 3 ? env.gemm_mode - 100 : -1);
        variant = plan.variant;
        if (plan.ksplit > 1) { p.ksplit = plan.ksplit; p.kchunk = plan.kchunk; p.partial = env.partial; }
    } else if (env.partial && p.K >= 512) {
        // simple kernel: split-K chosen against wave quantisation: minimise  waves(ks) * (K/ks + pipeline overhead)
        const int64_t tiles = ((p.M + SG_BM - 1) / SG_BM) * ((p.N + SG_BN - 1) / SG_BN) * p.batch;
        const int64_t cap = env.partial_elems / (p.M * p.N * p.batch);
        const double overhead = 96.0;   // pipeline fill + epilogue, in units of k
        double best = 1e300;
        int best_ks = 1;
        for (int ks = 1; ks <= 592 && ks <= cap && (ks == 1 || p.K / ks >= 256); ks++) {
            if (ks > 16 && tiles * ks > 2 * 592) break;   // deep splits only for skinny outputs
            const int64_t chunk = round_up((p.K + ks - 1) / ks, 16);
            const int64_t nsplit = (p.K + chunk - 1) / chunk;
            const int64_t waves = (tiles * nsplit + 147) / 148;
            double cost = (double)waves * ((double)chunk + overhead) * (ks > 1 ? 1.02 : 1.0);
            if (cost < best * 0.97) { best = cost; best_ks = ks; }
        }
        if (best_ks > 1) {
            const int64_t chunk = round_up((p.K + best_ks - 1) / best_ks, 16);
            p.ksplit = (int)((p.K + chunk - 1) / chunk);
            p.kchunk = chunk;
            p.partial = env.partial;
            if (p.ksplit <= 1) { p.ksplit = 1; p.kchunk = p.K; p.partial = nullptr; }
        }
    }
    if (use_dmma) {
        CCSD_TRY(launch_gemm_dmma(env.st, p, variant));
    } else {
        dim3 grid((unsigned)((p.N + SG_BN - 1) / SG_BN), (unsigned)((p.M + SG_BM - 1) / SG_BM), (unsigned)(p.batch * p.ksplit));
        gemm_simple_kernel<<<grid, SG_T * SG_T, 0, env.st>>>(p);
        count_launches(1);
    }
    if (p.ksplit > 1) {
        int64_t tot = p.M * p.N * p.batch;
        splitk_reduce_kernel<<<(unsigned)((tot + 255) / 256), 256, 0, env.st>>>(p);
        count_launches(1);
    }
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

// ---- one Strassen level around run_gemm (strassen.cuh) ---------------------------------------------------------------
struct StrassenScratch {
    c128 *SA, *SB, *P;        // stacks of the left / right operand made per call, the seven products
    double *SAp, *SBp;
    int64_t a_elems, b_elems, p_elems;
};

// Where a Strassen level pays: the seven half-size products must still be long-K, many-tile DMMA GEMMs and the three
// streaming passes must be small beside the eighth product they save (measured: 0.93 at 1536^3 down to 0.88 at 7616^3).
static inline bool strassen_worthwhile(int64_t M, int64_t N, int64_t K)
{
    return M >= 1024 && K >= 1024 && N >= 96 && (double)M * (double)N * (double)K >= 2.0e9;
}

// p: a plain (batch 1, k-contiguous) product C (+)= alpha A B^T.  preA / preB: ready-made stacks of operands that do not
// change between calls; an operand without one is stacked here into w.  The products go to w.P, then into C.
static int strassen_gemm(const Env& env, const GemmParams& p, const StrassenStack* preA, const StrassenStack* preB,
                         const StrassenScratch& w, int levels = 1)
{
    if (p.M <= 0 || p.N <= 0 || p.K <= 0) return CCSD_OK;
    if (p.batch != 1 || p.sak != 1 || p.sbk != 1 || levels < 1 || levels > 2) return CCSD_EINVAL;
    const int64_t Mh = strassen_rows(p.M, levels), Nh = strassen_rows(p.N, levels), Kh = strassen_cols(p.K, levels);
    const int nprod = levels == 2 ? 49 : 7;
    StrassenStack sa, sb;
    if (preA) {
        sa = *preA;
    } else {
        if (nprod * Mh * Kh > w.a_elems) return CCSD_EINVAL;
        sa = strassen_stack(w.SA, w.SAp, p.M, p.K, levels);
        launch_strassen_prep(env.st, 0, p.A, p.sam, sa);
    }
    if (preB) {
        sb = *preB;
    } else {
        if (nprod * Nh * Kh > w.b_elems) return CCSD_EINVAL;
        sb = strassen_stack(w.SB, w.SBp, p.N, p.K, levels);
        launch_strassen_prep(env.st, 1, p.B, p.sbn, sb);
    }
    if (sa.R != p.M || sa.K != p.K || sb.R != p.N || sb.K != p.K || sa.levels != levels || sb.levels != levels ||
        nprod * Mh * Nh > w.p_elems)
        return CCSD_EINVAL;
    const bool fast_m = p.csm == 1;    // the products take C's unit-stride index as their fast index
    GemmParams g = gp(Mh, Nh, Kh, sa.S, Kh, sb.S, Kh, w.P, fast_m ? 1 : Nh, fast_m ? Mh : 1, 1.0, 0);
    g.batch = nprod; g.bsA = Mh * Kh; g.bsB = Nh * Kh; g.bsC = Mh * Nh;
    g.As = sa.Sp; g.Bs = sb.Sp;
    CCSD_TRY(run_gemm(env, g));
    launch_strassen_combine(env.st, w.P, p.M, p.N, p.C, p.csm, p.csn, p.alpha, p.accumulate, levels);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

static int run_gemv(const Env& env, int64_t M, int64_t K, const c128* A, int64_t lda, const c128* x, c128* y, int64_t sy,
                    double alpha, int acc)
{
    if (M <= 0) return CCSD_OK;
    gemv_kernel<<<(unsigned)((M + 7) / 8), 256, 0, env.st>>>(M, K, A, lda, x, y, sy, mk(alpha, 0.0), acc);
    count_launches(1);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

static void dcopy(cudaStream_t st, c128* dst, const c128* src, int64_t elems)
{
    if (elems > 0) cudaMemcpyAsync(dst, src, (size_t)elems * sizeof(c128), cudaMemcpyDeviceToDevice, st);
}

// ---------------------------------------------------------------------------------------------------------------
// context
// ---------------------------------------------------------------------------------------------------------------
static const char* k_step_names[CCSD_NSTEPS] = {"prep_permute", "fock_like", "Hvovo_linear", "Hvovo_quad", "C_ovoo",
                                                "A_oooo", "pp_ladder", "hh_ladder+Goo", "ring_gemm", "ring_antisym",
                                                "Vdag_t1", "Gvv_t2", "C_t1", "S1", "update_diis", "energy"};

// Slab of the iteration this context evaluates (opts.shard_rank / shard_world, DESIGN "Multi-GPU"): every
// large contraction has disjoint output rows, so rank r computes
//   rows (a<b) in [w_lo, w_hi) of <ab||cd> x tau (pp-ladder), of the hh-ladder / G_oo term and of the V^dagger t1 term;
//   rows (a, .) with a in [a_lo, a_hi) of H^{ak}_{ci} (eq 29) and of the ring product (eq 32), of C (eq 30) and of C.t1;
//   rows (i<j) in [ij_lo, ij_hi) of the G_vv.t2 term and of the driver;
// and adds them into ITS S2 buffer, which is zero elsewhere: the sum over the ranks (one all-reduce of the packed S2, issued
// by the caller) is the S2 of eq 32.  S1, the small intermediates (Fock-like, A) and the update are replicated.
// Only the rows [w_lo, w_hi) of the packed <ab||cd> are built and stored.  world = 1: the full ranges.
struct Shard {
    int rank, world;
    int a_lo, a_hi;
    int wa_lo, wa_hi;          // first-virtual-index range whose pairs (a, b > a) are the packed rows [w_lo, w_hi)
    int64_t w_lo, w_hi, ij_lo, ij_hi;
};
static Shard make_shard(int rank, int world, int o, int v)
{
    Shard s;
    s.rank = rank; s.world = world;
    const int64_t oo = (int64_t)o * (o - 1) / 2, vv = (int64_t)v * (v - 1) / 2;
    auto split = [&](int64_t n, int r) { return n * r / world; };
    s.a_lo = (int)split(v, rank); s.a_hi = (int)split(v, rank + 1);
    s.ij_lo = split(oo, rank); s.ij_hi = split(oo, rank + 1);
    // boundary k: the smallest a whose pairs start at or beyond row vv k / world (pairs before a: a v - a (a + 1) / 2)
    auto bound = [&](int k) {
        if (k >= world) return v - 1 > 0 ? v - 1 : 0;
        const int64_t target = split(vv, k);
        int a = 0;
        while (a < v - 1 && (int64_t)a * v - (int64_t)a * (a + 1) / 2 < target) a++;
        return a;
    };
    s.wa_lo = bound(rank); s.wa_hi = bound(rank + 1);
    s.w_lo = (int64_t)s.wa_lo * v - (int64_t)s.wa_lo * (s.wa_lo + 1) / 2;
    s.w_hi = (int64_t)s.wa_hi * v - (int64_t)s.wa_hi * (s.wa_hi + 1) / 2;
    if (s.w_hi > vv) s.w_hi = vv;
    if (s.w_lo > s.w_hi) s.w_lo = s.w_hi;
    return s;
}

struct LambdaState;
struct ccsd_ctx {
    Shard sh;
    char* ws_base;          // the caller's workspace (ccsd_shard_info reports offsets into it)
    LambdaState* lam;       // Lambda solve in progress (ccsd_lambda_init), or null
    int o, v, n, L, Lp;
    int64_t oo, vv, ov, oop, nvec;
    ccsd_options opt;
    cudaStream_t st;
    Env env;
    // tables
    int2 *po, *pv;
    double* eps;            // Re f_pp + level shift on the virtuals: denominators of the Jacobi step and of the MP2 start
    double* eps0;           // Re f_pp: denominators of the perturbative triples (the shift is a convergence aid only)
    // constants
    c128 *f, *W, *Vvovv_p, *Vvovv_u, *VvovvT, *Voovv_p, *G1, *Voovv_c, *Voovv_ou, *Vvovo_m, *Vvovo_c, *Vooov_p,
        *Vooov_b, *Vooov_cc, *Vooov_d, *Vooov_e, *Voooo_p;
    // init temporaries
    c128 *Boo, *Bov, *Bvo, *Bvv, *Jovov, *Jvoov, *Jvvoo, *Jvvov, *Jooov, *Joooo, *Jslab, *JslabT;
    int na_slab;
    c128* Wslab;            // direct_ladder: rows of <ab||cd> of one slab of the first virtual index, rebuilt every iteration
    double* Wslabs;         // ... and their 3M sum plane
    c128* WslabT;           // direct_ladder, one GPU: conj-transpose of the slab's columns beyond the slab (Hermitian half, s2_pp_ladder)
    double* WslabTs;
    // amplitudes and per-iteration tensors
    c128 *t1, *t2p, *t1T, *S1, *S2p, *taup, *TT, *AG, *Xm, *T2r, *tauc, *tauou, *t2hu;
    c128 *Hvv, *Gvv, *Hoo, *Goo, *Hov, *HovT, *HF, *inner, *Hm, *Cm, *Cm2, *Am, *tmp_ov;
    c128 *Xr, *P, *Qm, *Rr, *Y, *Z;
    // The K = (c<d) product of C on its own, Cq[(b,k)][(i<j)] = -sum_{c<d} <bk||cd> tau^{cd}_{ij}: the <ak||cd> tau term of S1
    // (eq 33) is a partial trace of it, S1[i,a] += sum_k <ak||cd> tau[i,k,c,d] = -+ Cq[(a,k)][(i,k)], so that term needs no product
    // of its own (one GPU, not CC2: a sharded context holds only a slab of C, CC2 never forms this product)
    c128* Cq;
    bool s1_trace;
    // In the same way the <ak||cd> t1 term of G^a_c (eq 25) is a partial trace of the linear term of H^{ak}_{ci} (eq 29):
    // sum_{kd} <ak||cd> t1[k,d] = sum_k ( sum_d <ak||cd> t1[i,d] ) at i = k.  gvtr[a][c] holds it; it is added to Gvv once both the
    // Fock-like terms and that product are there (gvv_trace_add), before Gvv's first use (the G_vv t2 product).
    c128* gvtr;
    bool gv_trace;
    // ... and the <kl||cd> tau term of H^k_i (eq 26) is a partial trace of the quartic term of A (eq 31):
    // sum_{l, c<d} <kl||cd> tau[l,i,c,d] = sum_l +- Aq[(k,l)][(l,i)], Aq[(k<l)][(i<j)] = sum_{c<d} <kl||cd> tau^{cd}_{ij} (build_Aq)
    c128* Aq;
    bool hoo_trace;
    // CC2 only: B blocks with the contracted virtual index fastest and the t1-dressed factors X (cc2_dressed_factors)
    c128 *BvvT, *BovT, *Xv, *Xo;
    double* Xvs;
    double* Bvvs;           // 3M sum plane of Bvv (the <ab||cd> slab GEMM over the auxiliary index)
    c128* partial;
    int64_t partial_elems;
    c128* partial_extra;    // split-K scratch of branches 1..4 of the captured residual
    int64_t partial_extra_elems;
    // 3M sum planes (Re + Im) of the operands of the five large GEMMs; null when the 4M / simple kernels are forced
    bool planes;
    double *Ws, *Vvovv_ps, *Voovv_ps, *G1s, *taups, *Xms, *T2rs, *Hms;
    // One Strassen level on the four large contractions (strassen.cuh; opts.strassen, one GPU, 3M planes): operand stacks of
    // the constants <ab||cd> (left operand of the pp-ladder), <bk||cd> (left operand of C) and <kl||cd> (right operand of the
    // quadratic H^{ak}_{ci} term) built once by ccsd_init, the stack of tau (right operand of the pp-ladder and of C) built by
    // prep_operands, and per-branch scratch for the stacks of Xm, Hm, T2r and for the seven products.
    bool strassen;
    int strassen_levels;    // of the two (ov)^3 products: 1 or 2 (the pp-ladder always takes one)
    int strassen_levels_C;  // of the <bk||cd> tau part of C: 1 or 2
    bool W_dropped;         // the packed <ab||cd> is not kept beside its operand stack (c->W = null after ccsd_init)
    c128* W_init;           // where ccsd_init builds it meanwhile
    int strassen_levels_L;  // of the pp-ladder: 1, or 2 with opts.strassen = 4 (an 18 GiB larger stack of <ab||cd> at cfg3)
    StrassenStack sW, sVvovv, sG1, sTau, sTauC;   // sTauC: tau stacked for C when C takes two levels (else C shares sTau)
    StrassenScratch str_ring, str_C, str_L;
    // DIIS ring (reduce.cuh): stored pairs, device-side Gram matrix / coefficients / reduction scratch
    DiisRing diis;
    double* red;            // device reduction outputs (64 doubles)
    double* red_host;       // pinned host mirror
    bool tau_valid;         // taup (and its plane) belong to the current (t1, t2p)
    // the residual evaluation as a CUDA graph (captured on its second use; opts.graph, a capturable stream, timing off)
    cudaGraphExec_t res_graph;
    long long graph_kernels;   // kernel launches one replay stands for
    bool graph_warm, graph_failed;
    // ccsd_init's build of the packed <ab||cd> (the "transposes" metric): device ms of the slab GEMMs over the
    // auxiliary index, of the slab transpositions and of the antisymmetrise-and-pack fills, and the elements the last two moved
    double init_stats[CCSD_NINIT_STATS];
    std::vector<cudaEvent_t>* init_events;   // 4 per slab, alive only during ccsd_init
    // timing
    int timing;
    cudaEvent_t ev[CCSD_NSTEPS + 1];
    float step_ms[CCSD_NSTEPS];
    float trip_ms[2];
    bool have_residual;
};

struct Carver {
    char* base;
    size_t off;
    template <class T>
    T* take(int64_t elems)
    {
        size_t bytes = ((size_t)(elems > 0 ? elems : 1) * sizeof(T) + 255) & ~(size_t)255;
        T* p = base ? reinterpret_cast<T*>(base + off) : nullptr;
        off += bytes;
        return p;
    }
};

static void carve(ccsd_ctx* c, char* base, size_t* total, int degrade)
{
    Carver w{base, 0};
    const int64_t o = c->o, v = c->v, n = c->n, Lp = c->Lp, oo = c->oo, vv = c->vv, ov = c->ov, oop = c->oop;
    c->planes = (c->opt.gemm_mode == 0 && CCSD_DEFAULT_3M != 0) || c->opt.gemm_mode == 3;
    // Strassen levels (strassen.cuh) on the (ov)^3 products, the pp-ladder and the <bk||cd> tau part of C: one GPU, 3M planes.
    // opts.strassen: 1 = levels chosen by size, 2 = one level wherever it pays, 3 = two levels everywhere whatever the size (tests)
    // In a sharded context the left operands are this rank's row slabs (rov rows of the (ov)^3 products and of C, rw rows of
    // <ab||cd>); the right operands (G1, T2r, tau) are whole.
    const bool force = c->opt.strassen == 3;
    const int64_t rov = (int64_t)(c->sh.a_hi - c->sh.a_lo) * o, rw = c->sh.w_hi - c->sh.w_lo;
    c->strassen = c->opt.strassen != 0 && c->planes && !c->opt.cc2 && (force ? (o >= 2 && v >= 2) : strassen_worthwhile(rov, ov, ov));
    bool use_L = c->strassen && !c->opt.direct_ladder && (force || strassen_worthwhile(rw, oo, vv));
    bool use_C = c->strassen && (force || strassen_worthwhile(rov, oo, vv));
    // two levels on the (ov)^3 products where a quarter-size product is still a long-K, many-tile GEMM (measured: 0.80 of the
    // plain product at ov = 7616 against 0.89 for one level; 0.90 against 0.93 at ov = 3840; no gain at 1536)
    c->strassen_levels = force ? 2 : (c->opt.strassen == 2 ? 1 : (ov >= 3072 ? 2 : 1));
    // C and the ladder: a second level only where a quarter of their (i<j) extent still fills whole 48-column tiles (cfg3: 141 ->
    // 144; cfg2: 69 -> 96 does not)
    c->strassen_levels_C = force ? 2 : ((c->strassen_levels == 2 && strassen_half(strassen_half(oo)) >= 128) ? 2 : 1);
    c->strassen_levels_L = force ? 2 : ((c->strassen_levels_C == 2 && use_C && use_L) ? 2 : 1);
    // The operand stacks of the constants grow like v^4 (the two-level stack of <ab||cd> is 3 x the tensor with planes).  `degrade`
    // gives up levels one step at a time -- the ladder's first, then C's, then the (ov)^3 products' -- see carve_auto.
    for (int k = 0; k < degrade && c->strassen && !force; k++) {
        if (use_L && c->strassen_levels_L == 2) c->strassen_levels_L = 1;
        else if (use_L) use_L = false;
        else if (use_C && c->strassen_levels_C == 2) c->strassen_levels_C = 1;
        else if (use_C) use_C = false;
        else if (c->strassen_levels == 2) c->strassen_levels = 1;
        else c->strassen = false;
    }
    c->po = w.take<int2>(oo);
    c->pv = w.take<int2>(vv);
    c->eps = w.take<double>(n);
    c->eps0 = w.take<double>(n);
    c->f = w.take<c128>(n * n);
    // <ab||cd> is not stored in direct_ladder mode (rebuilt every iteration) nor in CC2 mode (its only use factorises)
    // With the Strassen ladder <ab||cd> lives on as its operand stack only (c->sW; single elements: strassen_left_at).  ccsd_init
    // builds the packed tensor in the memory of C's operand stack, stacks it, and only then fills C's stack (c->W_init).
    c->W_dropped = use_L && use_C && strassen_stack_elems(rov, vv, c->strassen_levels_C) * (int64_t)(sizeof(c128) + sizeof(double)) >=
                                         rw * vv * (int64_t)sizeof(c128) + 512;
    c->W_init = nullptr;
    c->W = (c->opt.direct_ladder || c->opt.cc2 || c->W_dropped) ? nullptr : w.take<c128>((c->sh.w_hi - c->sh.w_lo) * vv);   // this rank's rows
    c->Vvovv_p = w.take<c128>(v * o * vv);
    c->Vvovv_u = w.take<c128>(v * v * o * v);
    c->VvovvT = w.take<c128>(o * vv * v);
    c->Voovv_p = w.take<c128>(oo * vv);
    c->G1 = w.take<c128>(ov * ov);
    c->Voovv_c = w.take<c128>(v * oo * v);
    c->Voovv_ou = w.take<c128>(o * o * vv);
    c->Vvovo_m = w.take<c128>(ov * ov);
    c->Vvovo_c = w.take<c128>(ov * ov);
    c->Vooov_p = w.take<c128>(oo * ov);
    c->Vooov_b = w.take<c128>(o * ov * o);
    c->Vooov_cc = w.take<c128>(ov * oo);
    c->Vooov_d = w.take<c128>(o * o * ov);
    c->Vooov_e = w.take<c128>(o * oo * v);
    c->Voooo_p = w.take<c128>(oo * oo);
    // init temporaries
    c->Boo = w.take<c128>(o * o * Lp);
    c->Bov = w.take<c128>(ov * Lp);
    c->Bvo = w.take<c128>(ov * Lp);
    c->Bvv = w.take<c128>(v * v * Lp);
    const size_t j_begin = w.off;     // [Jovov, Joooo]: dead once ccsd_init has filled the integral classes (Strassen scratch below)
    c->Jovov = w.take<c128>(ov * ov);
    c->Jvoov = w.take<c128>(ov * ov);
    c->Jvvoo = w.take<c128>(v * v * o * o);
    c->Jvvov = w.take<c128>(v * v * ov);
    c->Jooov = w.take<c128>(o * o * ov);
    c->Joooo = w.take<c128>(o * o * o * o);
    const size_t j_end = w.off;
    {
        double per_a = (double)v * v * v * 16.0;
        // direct_ladder: slabs grow with the tensor they replace (a sixth of its bytes, 1.5 - 6 GB), so that the ladder GEMM
        // on one slab of rows fills several waves of the 148 SMs once the problem is large enough to need this mode
        double budget = 1.5e9;
        if (c->opt.direct_ladder) {
            budget = (double)vv * (double)vv * 16.0 / 6.0;
            if (budget < 1.5e9) budget = 1.5e9;
            if (budget > 6.0e9) budget = 6.0e9;
        }
        int na = (int)(budget / (per_a > 1 ? per_a : 1));
        if (na < 1) na = 1;
        if (na > v) na = (int)v;
        c->na_slab = na;
        c->Jslab = w.take<c128>((int64_t)na * v * v * v);
        c->JslabT = w.take<c128>((int64_t)na * v * v * v);
        c->Wslab = nullptr;
        c->Wslabs = nullptr;
        c->WslabT = nullptr;
        c->WslabTs = nullptr;
        if (c->opt.direct_ladder) {
            const int64_t max_rows = (int64_t)na * (v - 1);        // pairs (a,b), b > a, of na values of a: at most na (v-1)
            c->Wslab = w.take<c128>(max_rows * vv);
            c->Wslabs = w.take<double>(max_rows * vv);
            if (c->opt.shard_world <= 1) {
                c->WslabT = w.take<c128>(vv * round_up(max_rows, 2));
                c->WslabTs = w.take<double>(vv * round_up(max_rows, 2));
            }
        }
    }
    // amplitudes, residuals, operands
    c->t1 = w.take<c128>(ov);
    c->t2p = w.take<c128>(oo * vv);
    c->t1T = w.take<c128>(ov);
    c->S1 = w.take<c128>(ov);
    c->S2p = w.take<c128>(oo * vv);
    c->taup = w.take<c128>(oo * vv);
    c->TT = w.take<c128>(vv * 2 * oop);
    c->AG = w.take<c128>(oo * 2 * oop);
    c->Xm = w.take<c128>(ov * ov);
    c->T2r = w.take<c128>(ov * ov);
    c->tauc = w.take<c128>(v * oo * v);
    c->tauou = w.take<c128>(o * o * vv);
    c->t2hu = w.take<c128>(oo * v * v);
    c->Hvv = w.take<c128>(v * v);
    c->Gvv = w.take<c128>(v * v);
    c->Hoo = w.take<c128>(o * o);
    c->Goo = w.take<c128>(o * o);
    c->Hov = w.take<c128>(ov);
    c->HovT = w.take<c128>(ov);
    c->HF = w.take<c128>(ov);
    c->inner = w.take<c128>(o * o);
    c->Hm = w.take<c128>(ov * ov);
    c->Cm = w.take<c128>(ov * oo);
    c->Cm2 = w.take<c128>(ov * oo);
    c->Am = w.take<c128>(oo * oo);
    c->tmp_ov = w.take<c128>(ov);
    c->Xr = w.take<c128>(ov * ov);
    c->P = w.take<c128>(o * o * vv);
    c->Qm = w.take<c128>(oo * v * v);
    c->Rr = w.take<c128>(v * oo * v);
    c->Y = w.take<c128>(ov * o * o);
    c->Z = w.take<c128>(oo * o * o);
    c->s1_trace = !c->opt.cc2 && c->opt.shard_world <= 1;
    c->Cq = c->s1_trace ? w.take<c128>(ov * oo) : nullptr;
    c->gv_trace = c->s1_trace;
    c->gvtr = c->gv_trace ? w.take<c128>(v * v) : nullptr;
    c->hoo_trace = c->s1_trace;
    c->Aq = c->hoo_trace ? w.take<c128>(oo * oo) : nullptr;
    c->partial_elems = 16 * 1024 * 1024;  // split-K partials: >= 256 MB and >= 4 copies of the largest split-K output
    if (c->partial_elems < 4 * oo * vv) c->partial_elems = 4 * oo * vv;
    if (c->partial_elems < 4 * ov * ov) c->partial_elems = 4 * ov * ov;
    c->partial = w.take<c128>(c->partial_elems);
    // four more split-K slots, one per parallel branch of the captured residual (residual_forked): 32 Mi elements at most
    c->partial_extra_elems = c->partial_elems < 32 * 1024 * 1024 ? c->partial_elems : 32 * 1024 * 1024;
    c->partial_extra = (c->opt.graph && !c->opt.cc2) ? w.take<c128>(4 * c->partial_extra_elems) : nullptr;
    c->Ws = c->Vvovv_ps = c->Voovv_ps = c->G1s = c->taups = c->Xms = c->T2rs = c->Hms = nullptr;
    if (c->planes) {   // an operand whose product runs through Strassen stacks needs no plane of its own (the stacks carry theirs)
        c->Ws = (c->opt.direct_ladder || c->opt.cc2 || use_L) ? nullptr : w.take<double>((c->sh.w_hi - c->sh.w_lo) * vv);
        c->Vvovv_ps = use_C ? nullptr : w.take<double>(ov * vv);
        c->Voovv_ps = w.take<double>(oo * vv);
        c->taups = w.take<double>(oo * vv);
        if (!c->strassen) {
            c->G1s = w.take<double>(ov * ov);
            c->Xms = w.take<double>(ov * ov);
            c->T2rs = w.take<double>(ov * ov);
            c->Hms = w.take<double>(ov * ov);
        }
    }
    c->Bvvs = (c->planes && !c->opt.cc2) ? w.take<double>(v * v * Lp) : nullptr;
    c->BvvT = c->BovT = c->Xv = c->Xo = nullptr;
    c->Xvs = nullptr;
    if (c->opt.cc2) {
        c->BvvT = w.take<c128>(v * Lp * v);
        c->BovT = w.take<c128>(o * Lp * v);
        c->Xv = w.take<c128>(ov * Lp);
        c->Xo = w.take<c128>(o * o * Lp);
        c->Xvs = w.take<double>(ov * Lp);
    }
    memset(&c->sW, 0, sizeof(c->sW)); memset(&c->sVvovv, 0, sizeof(c->sVvovv)); memset(&c->sG1, 0, sizeof(c->sG1));
    memset(&c->sTau, 0, sizeof(c->sTau)); memset(&c->sTauC, 0, sizeof(c->sTauC));
    memset(&c->str_ring, 0, sizeof(c->str_ring)); memset(&c->str_C, 0, sizeof(c->str_C)); memset(&c->str_L, 0, sizeof(c->str_L));
    if (c->strassen) {
        const int lv = c->strassen_levels;
        // Per-iteration stacks and products go into the dead init temporaries [Jovov, Joooo] while they fit there (largest
        // first), the rest and the stacks of the constants are appended.
        Carver dead{base ? base + j_begin : nullptr, 0};
        const size_t dead_bytes = j_end - j_begin;
        auto place = [&](int64_t elems, size_t elem_bytes) -> Carver& {
            const size_t bytes = ((size_t)(elems > 0 ? elems : 1) * elem_bytes + 255) & ~(size_t)255;
            return dead.off + bytes <= dead_bytes ? dead : w;
        };
        auto stack = [&](bool scratch, int64_t R, int64_t K, int levels) {
            const int64_t e = strassen_stack_elems(R, K, levels);
            c128* S = (scratch ? place(e, sizeof(c128)) : w).take<c128>(e);
            double* Sp = (scratch ? place(e, sizeof(double)) : w).take<double>(e);
            return strassen_stack(S, Sp, R, K, levels);
        };
        const int lvL = c->strassen_levels_L;
        if (use_L) c->sW = stack(false, rw, vv, lvL);
        const int lvC = c->strassen_levels_C;
        if (use_C) c->sVvovv = stack(false, rov, vv, lvC);
        if (c->W_dropped) c->W_init = c->sVvovv.S;      // S and Sp are adjacent: together they hold the packed tensor
        c->sG1 = stack(false, ov, ov, lv);
        StrassenStack sa = stack(true, rov, ov, lv), sb = stack(true, ov, ov, lv);
        c->str_ring.SA = sa.S; c->str_ring.SAp = sa.Sp; c->str_ring.a_elems = strassen_stack_elems(rov, ov, lv);
        c->str_ring.SB = sb.S; c->str_ring.SBp = sb.Sp; c->str_ring.b_elems = strassen_stack_elems(ov, ov, lv);
        c->str_ring.p_elems = (lv == 2 ? 49 : 7) * strassen_rows(rov, lv) * strassen_rows(ov, lv);
        c->str_ring.P = place(c->str_ring.p_elems, sizeof(c128)).take<c128>(c->str_ring.p_elems);
        if ((use_L && lvL == 1) || (use_C && lvC == 1)) c->sTau = stack(true, oo, vv, 1);
        if ((use_L && lvL == 2) || (use_C && lvC == 2)) c->sTauC = stack(true, oo, vv, 2);
        if (use_L) {
            c->str_L.p_elems = (lvL == 2 ? 49 : 7) * strassen_rows(rw, lvL) * strassen_rows(oo, lvL);
            c->str_L.P = place(c->str_L.p_elems, sizeof(c128)).take<c128>(c->str_L.p_elems);
        }
        if (use_C) {
            c->str_C.p_elems = (lvC == 2 ? 49 : 7) * strassen_rows(rov, lvC) * strassen_rows(oo, lvC);
            c->str_C.P = place(c->str_C.p_elems, sizeof(c128)).take<c128>(c->str_C.p_elems);
        }
    }
    c->nvec = ov + oo * vv;
    int nd = c->opt.ndiis > 0 ? c->opt.ndiis : 1;
    c->diis.nd = c->opt.ndiis;
    c->diis.u = w.take<c128>((int64_t)nd * c->nvec);
    c->diis.e = w.take<c128>((int64_t)nd * c->nvec);
    c->diis.gram = w.take<double>(13 * 13);
    c->diis.coef = w.take<double>(16);
    c->diis.info = w.take<double>(4);
    c->diis.scratch = w.take<double>(RED_SCRATCH_DOUBLES);
    c->red = w.take<double>(64);
    *total = w.off;
}

// Workspace layout with as many Strassen levels as fit: a workspace beyond 128 GiB (of a 180 GB part; the Lambda and triples
// workspaces need room beside it) gives levels up step by step, down to plain products, instead of asking for memory no GPU has
// (cfg3: 107 GiB with everything; plain products need 60 GiB).  Host arithmetic only: ccsd_workspace_bytes and ccsd_init agree.
static void carve_auto(ccsd_ctx* c, char* base, size_t* total)
{
    int degrade = 0;
    for (; degrade < 6; degrade++) {
        size_t t = 0;
        carve(c, nullptr, &t, degrade);
        if (t <= ((size_t)128 << 30) || !c->strassen || c->opt.strassen == 3) break;
    }
    carve(c, base, total, degrade);
}

static int check_sizes(int nocc, int nvir, int naux)
{
    if (nocc < 2 || nvir < 2 || naux < 1) return CCSD_EINVAL;
    if (nocc > 4096 || nvir > 8192) return CCSD_EINVAL;
    return CCSD_OK;
}

static void setup_dims(ccsd_ctx* c, int nocc, int nvir, int naux, const ccsd_options* opts)
{
    c->o = nocc; c->v = nvir; c->n = nocc + nvir; c->L = naux; c->Lp = (int)round_up(naux, 4);
    c->oo = (int64_t)nocc * (nocc - 1) / 2;
    c->vv = (int64_t)nvir * (nvir - 1) / 2;
    c->ov = (int64_t)nocc * nvir;
    c->oop = round_up(c->oo > 0 ? c->oo : 1, 4);
    if (opts) c->opt = *opts; else ccsd_default_options(&c->opt);
    if (c->opt.ndiis < 0) c->opt.ndiis = 0;
    if (c->opt.ndiis > DIIS_MAX) c->opt.ndiis = DIIS_MAX;
    if (c->opt.shard_world < 1) { c->opt.shard_world = 1; c->opt.shard_rank = 0; }
    c->sh = make_shard(c->opt.shard_rank, c->opt.shard_world, nocc, nvir);
}

// ---------------------------------------------------------------------------------------------------------------
// integral-class functors over the chemists'-notation blocks J (eq 6 PAPER.md:71 reading G1):
//   <pq||rs> = (pr|qs) - (ps|qr)
// ---------------------------------------------------------------------------------------------------------------
struct GOovv {  // <kl||cd> = (kc|ld) - (kd|lc)
    const c128* J; int64_t o, v;
    __device__ c128 operator()(int k, int l, int c, int d) const
    {
        int64_t ov = o * v;
        return csub(J[(k * v + c) * ov + l * v + d], J[(k * v + d) * ov + l * v + c]);
    }
};
struct GVovo {  // <ak||ci> = (ac|ki) - (ai|kc)
    const c128 *Jvvoo, *Jvoov; int64_t o, v;
    __device__ c128 operator()(int a, int k, int c, int i) const
    {
        return csub(Jvvoo[(a * v + c) * o * o + k * o + i], Jvoov[(a * o + i) * o * v + k * v + c]);
    }
};
struct GVovv {  // <ak||cd> = (ac|kd) - (ad|kc)
    const c128* J; int64_t o, v;
    __device__ c128 operator()(int a, int k, int c, int d) const
    {
        int64_t ov = o * v;
        return csub(J[(a * v + c) * ov + k * v + d], J[(a * v + d) * ov + k * v + c]);
    }
};
struct GOoov {  // <kl||ic> = (ki|lc) - (kc|li)
    const c128* J; int64_t o, v;
    __device__ c128 operator()(int k, int l, int i, int c) const
    {
        int64_t ov = o * v;
        return csub(J[(k * o + i) * ov + l * v + c], J[(l * o + i) * ov + k * v + c]);
    }
};
struct GOooo {  // <kl||ij> = (ki|lj) - (kj|li)
    const c128* J; int64_t o;
    __device__ c128 operator()(int k, int l, int i, int j) const
    {
        int64_t o2 = o * o;
        return csub(J[(k * o + i) * o2 + l * o + j], J[(k * o + j) * o2 + l * o + i]);
    }
};

// eps[p] = Re f_pp (+ shift on the virtuals, .LSHIFT PAPER.md:1062); eps0[p] = Re f_pp (may be null)
__global__ void eps_kernel(const c128* f, double* eps, double* eps0, int n, int o, double shift)
{
    int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= n) return;
    const double e = f[(int64_t)p * n + p].x;
    eps[p] = e + (p >= o ? shift : 0.0);
    if (eps0) eps0[p] = e;
}

// Bxy[(p,q)][l] = B[l][p][q], auxiliary index fastest and zero-padded to Lp
static void bblock(cudaStream_t st, c128* out, const c128* B, int n, int L, int Lp, int p0, int np, int q0, int nq)
{
    launch_fill(st, out, (int64_t)np * nq, Lp, Lp, 0, [=] __device__(int64_t row, int64_t l) {
        if (l >= L) return mk(0.0, 0.0);
        int64_t p = p0 + row / nq, q = q0 + row % nq;
        return B[l * (int64_t)n * n + p * n + q];
    });
}

// Rows of the packed <ab||cd> = (ac|bd) - (ad|bc) owned by the slab a in [a0, a0 + na_slab) of the first virtual index
// (pairs (a,b), b > a: a contiguous range [r0, r0 + nrows) of packed rows), from the factor B; the v^4 staging tensor is
// never materialised:
//   Jslab[(a,c)][(b,d)] = (ac|bd), b > a0               (GEMM over the auxiliary index)
//   JslabT[(b,c)][(a,d)] = Jslab[(a,d)][(b,c)]         (tiled transposition, bandwidth bound)
//   W[(a<b)][(c<d)] = Jslab[(a,c)][(b,d)] - JslabT[(b,c)][(a,d)]     (both reads contiguous in d)
// absolute = true: dst is the whole matrix (row r0 of the slab goes to dst + r0 vv); false: dst holds the slab only.
// upper = true (integral-direct ladder on one GPU): only the columns (c<d) with c >= a0, i.e. the packed columns CD >= r0, are
// built (the rest follows from <ab||cd> = conj <cd||ab> and is never needed, s2_pp_ladder) -- half the flops of the slab GEMM
// summed over the slabs -- and the 3M sum plane is written along into `plane` (may be null).
static int build_W_slab(ccsd_ctx* c, int a0, int a_end, c128* dst, bool absolute, int64_t* r0_out, int64_t* nrows_out,
                        bool upper = false, double* plane = nullptr)
{
    cudaStream_t st = c->st;
    const int v = c->v, Lp = c->Lp;
    const int64_t vv = c->vv, v2 = (int64_t)v * v;
    const int2* pv = c->pv;
    const int na = (a0 + c->na_slab <= a_end) ? c->na_slab : a_end - a0;
    const int64_t rows = (int64_t)na * v;
    // only b > a is needed, i.e. the columns (b,d) with b >= a0 + 1 of the slab (half the columns on average)
    const int64_t col0 = (int64_t)(a0 + 1) * v, ncol = v2 - col0;
    auto mark = [&]() {
        if (!c->init_events) return;
        cudaEvent_t e = nullptr;
        if (cudaEventCreate(&e) == cudaSuccess) { cudaEventRecord(e, st); c->init_events->push_back(e); }
    };
    mark();
    const int cfrom = upper ? a0 : 0;          // rows (a, c) with c >= cfrom: one product per a when that is not all of them
    GemmParams g = gp(rows, ncol, Lp, c->Bvv + (int64_t)a0 * v * Lp, Lp, c->Bvv + col0 * Lp, Lp, c->Jslab + col0, v2, 1, 1.0, 0);
    if (c->Bvvs) g = with_planes(g, c->Bvvs + (int64_t)a0 * v * Lp, c->Bvvs + col0 * Lp);
    if (cfrom > 0) {
        // the restricted index goes into the COLUMN position of the product (tiles of 32-56 columns pad v - a0 <= nvir far less
        // than 128-row tiles would): Jslab^T, one product per a with the (b,d) operand shared, stored through csm = 1
        const int64_t off = ((int64_t)a0 * v + cfrom) * Lp;
        g = gp(ncol, v - cfrom, Lp, c->Bvv + col0 * Lp, Lp, c->Bvv + off, Lp, c->Jslab + (int64_t)cfrom * v2 + col0, 1, v2, 1.0, 0);
        g.batch = na; g.bsA = 0; g.bsB = (int64_t)v * Lp; g.bsC = (int64_t)v * v2;
        if (c->Bvvs) g = with_planes(g, c->Bvvs + col0 * Lp, c->Bvvs + off);
    }
    CCSD_TRY(run_gemm(c->env, g));
    mark();
    CCSD_TRY(launch_transpose2d_ld(st, c->Jslab + col0, v2, c->JslabT + col0 * rows, rows, rows, ncol, 0));
    mark();
    const int alast = (a0 + na - 1 < v - 2) ? a0 + na - 1 : v - 2;
    const int64_t r0 = pair_idx(a0, a0 + 1, v), r1 = pair_idx(alast, v - 1, v) + 1;
    const int64_t cd0 = upper ? r0 : 0;        // first packed column built
    const c128 *J = c->Jslab, *JT = c->JslabT;
    launch_fill(st, dst + (absolute ? r0 * vv : 0) + cd0, r1 - r0, vv - cd0, vv, 0, [=] __device__(int64_t r, int64_t col) {
        const int64_t CD = cd0 + col;
        int2 ab = pv[r0 + r], cd = pv[CD];
        int64_t al = ab.x - a0;
        c128 x = J[(al * v + cd.x) * v2 + (int64_t)ab.y * v + cd.y];
        c128 y = JT[((int64_t)ab.y * v + cd.x) * rows + al * v + cd.y];
        x = csub(x, y);
        if (plane) plane[r * vv + CD] = x.x + x.y;
        return x;
    });
    mark();
    if (c->init_events) {
        c->init_stats[3] += (double)rows * (double)ncol;       // elements transposed
        c->init_stats[4] += (double)(r1 - r0) * (double)vv;    // elements packed
    }
    *r0_out = r0;
    *nrows_out = r1 - r0;
    return CCSD_OK;
}

static int build_constants(ccsd_ctx* c, const c128* h, const c128* B)
{
    cudaStream_t st = c->st;
    const Env& env = c->env;
    const int o = c->o, v = c->v, n = c->n, L = c->L, Lp = c->Lp;
    const int64_t oo = c->oo, vv = c->vv, ov = c->ov;
    const int2 *po = c->po, *pv = c->pv;

    if (oo > 0) { pair_table_kernel<<<(unsigned)((oo + 255) / 256), 256, 0, st>>>(c->po, o); count_launches(1); }
    if (vv > 0) { pair_table_kernel<<<(unsigned)((vv + 255) / 256), 256, 0, st>>>(c->pv, v); count_launches(1); }

    // Fock matrix f = h + sum_i <pi||qi>
    launch_fill(st, c->f, n, n, n, 0, [=] __device__(int64_t p, int64_t q) {
        c128 s = h[p * n + q];
        for (int l = 0; l < L; l++) {
            const c128* Bl = B + (int64_t)l * n * n;
            c128 d = mk(0.0, 0.0), x = mk(0.0, 0.0);
            for (int i = 0; i < o; i++) {
                d = cadd(d, Bl[(int64_t)i * n + i]);
                cfma(x, Bl[p * n + i], Bl[(int64_t)i * n + q]);
            }
            cfma(s, Bl[p * n + q], d);
            s = csub(s, x);
        }
        return s;
    });
    eps_kernel<<<(n + 127) / 128, 128, 0, st>>>(c->f, c->eps, c->eps0, n, o, c->opt.level_shift);
    count_launches(1);

    // B blocks with the auxiliary index fastest (zero-padded to a multiple of 4): Bxy[(p,q)][l] = B[l][p][q]
    bblock(st, c->Boo, B, n, L, Lp, 0, o, 0, o);
    bblock(st, c->Bov, B, n, L, Lp, 0, o, o, v);
    bblock(st, c->Bvo, B, n, L, Lp, o, v, 0, o);
    bblock(st, c->Bvv, B, n, L, Lp, o, v, o, v);
    if (c->Bvvs) launch_sum_plane(st, c->Bvv, c->Bvvs, (int64_t)v * v * Lp);

    // chemists' blocks (pq|rs) = sum_L B[L,p,q] B[L,r,s]  as NT GEMMs over the auxiliary index
    CCSD_TRY(run_gemm(env, gp(ov, ov, Lp, c->Bov, Lp, c->Bov, Lp, c->Jovov, ov, 1, 1.0, 0)));
    CCSD_TRY(run_gemm(env, gp(ov, ov, Lp, c->Bvo, Lp, c->Bov, Lp, c->Jvoov, ov, 1, 1.0, 0)));
    CCSD_TRY(run_gemm(env, gp((int64_t)v * v, (int64_t)o * o, Lp, c->Bvv, Lp, c->Boo, Lp, c->Jvvoo, (int64_t)o * o, 1, 1.0, 0)));
    CCSD_TRY(run_gemm(env, gp((int64_t)v * v, ov, Lp, c->Bvv, Lp, c->Bov, Lp, c->Jvvov, ov, 1, 1.0, 0)));
    CCSD_TRY(run_gemm(env, gp((int64_t)o * o, ov, Lp, c->Boo, Lp, c->Bov, Lp, c->Jooov, ov, 1, 1.0, 0)));
    CCSD_TRY(run_gemm(env, gp((int64_t)o * o, (int64_t)o * o, Lp, c->Boo, Lp, c->Boo, Lp, c->Joooo, (int64_t)o * o, 1, 1.0, 0)));

    GOovv goovv{c->Jovov, o, v};
    GVovo gvovo{c->Jvvoo, c->Jvoov, o, v};
    GVovv gvovv{c->Jvvov, o, v};
    GOoov gooov{c->Jooov, o, v};
    GOooo goooo{c->Joooo, o};

    // <kl||cd> in four operand layouts
    launch_fill(st, c->Voovv_p, oo, vv, vv, 0, [=] __device__(int64_t KL, int64_t CD) {
        int2 kl = po[KL], cd = pv[CD];
        return goovv(kl.x, kl.y, cd.x, cd.y);
    });
    launch_fill(st, c->G1, ov, ov, ov, 0, [=] __device__(int64_t ck, int64_t ld) {
        int cc = ck / o, k = ck % o, l = ld / v, d = ld % v;
        return goovv(k, l, cc, d);
    });
    launch_fill(st, c->Voovv_c, v, oo * v, oo * v, 0, [=] __device__(int64_t cc, int64_t col) {
        int2 kl = po[col / v];
        int d = col % v;
        return goovv(kl.x, kl.y, (int)cc, d);
    });
    launch_fill(st, c->Voovv_ou, (int64_t)o * o, vv, vv, 0, [=] __device__(int64_t row, int64_t CD) {
        int2 cd = pv[CD];
        return goovv((int)(row / o), (int)(row % o), cd.x, cd.y);
    });
    // <ak||ci>
    launch_fill(st, c->Vvovo_m, ov, ov, ov, 0, [=] __device__(int64_t ai, int64_t ck) {
        int a = ai / o, i = ai % o, cc = ck / o, k = ck % o;
        return gvovo(a, k, cc, i);
    });
    launch_fill(st, c->Vvovo_c, ov * o, v, v, 0, [=] __device__(int64_t row, int64_t cc) {
        int i = row % o, k = (row / o) % o, b = row / ((int64_t)o * o);
        return gvovo(b, k, (int)cc, i);
    });
    // <ak||cd>
    launch_fill(st, c->Vvovv_p, ov, vv, vv, 0, [=] __device__(int64_t ak, int64_t CD) {
        int2 cd = pv[CD];
        return gvovv((int)(ak / o), (int)(ak % o), cd.x, cd.y);
    });
    launch_fill(st, c->Vvovv_u, (int64_t)v * v, ov, ov, 0, [=] __device__(int64_t ac, int64_t kd) {
        return gvovv((int)(ac / v), (int)(kd / v), (int)(ac % v), (int)(kd % v));
    });
    launch_fill(st, c->VvovvT, o * vv, v, v, 0, [=] __device__(int64_t row, int64_t cc) {
        int j = row / vv;
        int2 ab = pv[row % vv];
        return cconj(gvovv((int)cc, j, ab.x, ab.y));
    });
    // <kl||ic>
    launch_fill(st, c->Vooov_p, oo, ov, ov, 0, [=] __device__(int64_t KL, int64_t ic) {
        int2 kl = po[KL];
        return gooov(kl.x, kl.y, (int)(ic / v), (int)(ic % v));
    });
    launch_fill(st, c->Vooov_b, (int64_t)o * ov, o, o, 0, [=] __device__(int64_t row, int64_t l) {
        int k = row % o, cc = (row / o) % v, i = row / ((int64_t)o * v);
        return gooov(k, (int)l, i, cc);
    });
    launch_fill(st, c->Vooov_cc, ov, oo, oo, 0, [=] __device__(int64_t bk, int64_t IJ) {
        int2 ij = po[IJ];
        return cconj(gooov(ij.x, ij.y, (int)(bk % o), (int)(bk / o)));
    });
    launch_fill(st, c->Vooov_d, (int64_t)o * o, ov, ov, 0, [=] __device__(int64_t ki, int64_t lc) {
        return gooov((int)(ki / o), (int)(lc / v), (int)(ki % o), (int)(lc % v));
    });
    launch_fill(st, c->Vooov_e, o, oo * v, oo * v, 0, [=] __device__(int64_t i, int64_t col) {
        int2 kl = po[col / v];
        return gooov(kl.x, kl.y, (int)i, (int)(col % v));
    });
    // <kl||ij>
    launch_fill(st, c->Voooo_p, oo, oo, oo, 0, [=] __device__(int64_t KL, int64_t IJ) {
        int2 kl = po[KL], ij = po[IJ];
        return goooo(kl.x, kl.y, ij.x, ij.y);
    });

    // <ab||cd> = (ac|bd) - (ad|bc), packed, built in slabs of the first virtual index so that the v^4 staging
    // tensor is never materialised.  For a in [a0, a0+na):
    //   Jslab[(a,c)][(b,d)] = (ac|bd)                      (GEMM over the auxiliary index)
    //   JslabT[(b,c)][(a,d)] = Jslab[(a,d)][(b,c)]         (tiled transposition, bandwidth bound)
    //   W[(a<b)][(c<d)] = Jslab[(a,c)][(b,d)] - JslabT[(b,c)][(a,d)]     (both reads contiguous in d)
    c128* const Wdst = c->W ? c->W : c->W_init;
    if (Wdst) {
        std::vector<cudaEvent_t> events;
        c->init_events = &events;
        int s = CCSD_OK;
        for (int a0 = c->sh.wa_lo; a0 < c->sh.wa_hi && vv > 0 && s == CCSD_OK; a0 += c->na_slab) {
            int64_t r0 = 0, nrows = 0;      // "absolute" rows, relative to this rank's first row
            s = build_W_slab(c, a0, c->sh.wa_hi, Wdst - c->sh.w_lo * vv, true, &r0, &nrows);
        }
        c->init_events = nullptr;
        if (s == CCSD_OK && !events.empty() && cudaStreamSynchronize(st) == cudaSuccess) {
            for (size_t q = 0; q + 3 < events.size(); q += 4)
                for (int k = 0; k < 3; k++) {
                    float ms = 0.f;
                    if (cudaEventElapsedTime(&ms, events[q + k], events[q + k + 1]) == cudaSuccess) c->init_stats[k] += ms;
                }
        }
        for (cudaEvent_t e : events) cudaEventDestroy(e);
        CCSD_TRY(s);
    }
    if (c->planes) {   // sum planes of the constant operands of the large GEMMs (3M, gemm_dmma.cuh)
        if (c->W && c->Ws) launch_sum_plane(st, c->W, c->Ws, (c->sh.w_hi - c->sh.w_lo) * vv);
        if (c->Vvovv_ps) launch_sum_plane(st, c->Vvovv_p, c->Vvovv_ps, ov * vv);
        launch_sum_plane(st, c->Voovv_p, c->Voovv_ps, oo * vv);
        if (c->G1s) launch_sum_plane(st, c->G1, c->G1s, ov * ov);
    }
    if (c->opt.cc2) {   // BvvT[a][l][e] = B[l][a][e], BovT[k][l][d] = B[l][k][d]: K-contiguous operands of cc2_dressed_factors
        const int64_t dv[4] = {v, v, Lp, 1}, dk[4] = {o, v, Lp, 1};
        const int perm[4] = {0, 2, 1, 3};
        CCSD_TRY(launch_transpose4d(st, c->Bvv, c->BvvT, dv, perm, 0));
        CCSD_TRY(launch_transpose4d(st, c->Bov, c->BovT, dk, perm, 0));
    }
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

// MP2 start: t1 = f_ai / D^a_i, t2 = <ab||ij> / D^ab_ij
static void mp2_guess(ccsd_ctx* c)
{
    const int o = c->o, v = c->v, n = c->n;
    const int64_t vv = c->vv;
    const c128 *f = c->f, *V = c->Voovv_p;
    const double* eps = c->eps;
    const int2 *po = c->po, *pv = c->pv;
    const int ccd = c->opt.ccd;
    launch_fill(c->st, c->t1, o, v, v, 0, [=] __device__(int64_t i, int64_t a) {
        if (ccd) return mk(0.0, 0.0);
        double d = eps[i] - eps[o + a];
        c128 x = cconj(f[i * n + o + a]);
        return mk(x.x / d, x.y / d);
    });
    launch_fill(c->st, c->t2p, c->oo, vv, vv, 0, [=] __device__(int64_t IJ, int64_t AB) {
        int2 ij = po[IJ], ab = pv[AB];
        double d = eps[ij.x] + eps[ij.y] - eps[o + ab.x] - eps[o + ab.y];
        c128 x = cconj(V[IJ * vv + AB]);
        return mk(x.x / d, x.y / d);
    });
    c->diis.reset();
    c->have_residual = false;
    c->tau_valid = false;
}

// ---------------------------------------------------------------------------------------------------------------
// one residual evaluation, eqs 23-33
// ---------------------------------------------------------------------------------------------------------------
static void tick(ccsd_ctx* c, int k)
{
    if (c->timing) cudaEventRecord(c->ev[k], c->st);
}

// eq 23 on packed storage: tau = t2 + t1[i,a] t1[j,b] - t1[j,a] t1[i,b]
// (plane != null: also its 3M sum plane, so that the two can never be out of step; t2p == null: t2 = 0, the CC2 operand)
static void build_tau(cudaStream_t st, c128* taup, const c128* t1, const c128* t2p, int o, int v, const int2* po,
                      const int2* pv, double* plane)
{
    const int64_t oo = (int64_t)o * (o - 1) / 2, vv = (int64_t)v * (v - 1) / 2;
    launch_fill(st, taup, oo, vv, vv, 0, [=] __device__(int64_t IJ, int64_t AB) {
        int2 ij = po[IJ], ab = pv[AB];
        c128 x = t2p ? t2p[IJ * vv + AB] : mk(0.0, 0.0);
        cfma(x, t1[ij.x * v + ab.x], t1[ij.y * v + ab.y]);
        c128 y = cmul(t1[ij.y * v + ab.x], t1[ij.x * v + ab.y]);
        x = csub(x, y);
        if (plane) plane[IJ * vv + AB] = x.x + x.y;
        return x;
    });
}

// tau of the current amplitudes (eq 23) is usually there already: the energy kernel that closed the previous iteration
// built it (energy_async).  Kept out of the residual proper, so that the captured graph is the same every time.
static void ensure_tau(ccsd_ctx* c)
{
    if (!c->tau_valid) build_tau(c->st, c->taup, c->t1, c->t2p, c->o, c->v, c->po, c->pv, c->taups);
    c->tau_valid = true;
}

static int prep_operands(ccsd_ctx* c)
{
    cudaStream_t st = c->st;
    const int o = c->o, v = c->v;
    const int64_t oo = c->oo, vv = c->vv, ov = c->ov, oop = c->oop;
    const c128 *t1 = c->t1, *t2p = c->t2p, *taup = c->taup;
    double *Xms = c->strassen ? nullptr : c->Xms, *T2rs = c->strassen ? nullptr : c->T2rs;   // Strassen stacks carry their own planes
    if (c->sTau.S) launch_strassen_prep(st, 1, c->taup, vv, c->sTau);    // right operand of the pp-ladder and of C
    if (c->sTauC.S) launch_strassen_prep(st, 1, c->taup, vv, c->sTauC);  // ... of C with two levels
    launch_fill(st, c->t1T, v, o, o, 0, [=] __device__(int64_t a, int64_t i) { return t1[i * v + a]; });
    // TT[(a<b)][0:oo) = tau^T   (K-contiguous operand of the hh-ladder + Goo product; the second half of TT, t2^T, is the operand
    // of the Goo term on its own: fill_TT_t2, made where that form is used -- the per-term hook and CC2)
    CCSD_TRY(launch_transpose2d_ld(st, c->taup, vv, c->TT, 2 * oop, oo, vv, 0));
    // Xm[(a,i)][(l,d)] = 1/2 t2[l,i,a,d] + t1[l,a] t1[i,d]      (eq 29 operand)
    const int64_t xrow0 = (int64_t)c->sh.a_lo * o, xrows = (int64_t)(c->sh.a_hi - c->sh.a_lo) * o;   // this rank's rows (a, i)
    launch_fill(st, c->Xm + xrow0 * ov, xrows, ov, ov, 0, [=] __device__(int64_t row, int64_t ld) {
        const int64_t ai = xrow0 + row;
        int a = ai / o, i = ai % o, l = ld / v, d = ld % v;
        c128 x = cscale(0.5, t2_at(t2p, l, i, a, d, o, v, vv));
        cfma(x, t1[l * v + a], t1[i * v + d]);
        if (Xms) Xms[ai * ov + ld] = x.x + x.y;
        return x;
    });
    // T2r[(j,b)][(c,k)] = t2[j,k,c,b]                            (eq 32 ring operand)
    launch_fill(st, c->T2r, ov, ov, ov, 0, [=] __device__(int64_t jb, int64_t ck) {
        int j = jb / v, b = jb % v, cc = ck / o, k = ck % o;
        c128 x = t2_at(t2p, j, k, cc, b, o, v, vv);
        if (T2rs) T2rs[jb * ov + ck] = x.x + x.y;
        return x;
    });
    // tauc[a][(k<l, d)] = tau[k,l,d,a]
    launch_fill(st, c->tauc, v, oo * v, oo * v, 0, [=] __device__(int64_t a, int64_t col) {
        int64_t KL = col / v;
        int d = col % v;
        return asym_col(taup, KL, vv, d, (int)a, v);
    });
    // tauou[(i,l)][(c<d)] = tau[i,l,c,d]: operand of the quartic terms of H^k_i and S1 where those are products of their own
    if (!(c->hoo_trace && c->s1_trace))
    launch_fill(st, c->tauou, (int64_t)o * o, vv, vv, 0, [=] __device__(int64_t il, int64_t CD) {
        int i = il / o, l = il % o;
        if (i == l) return mk(0.0, 0.0);
        if (i < l) return taup[pair_idx(i, l, o) * vv + CD];
        return cneg(taup[pair_idx(l, i, o) * vv + CD]);
    });
    // t2hu[(i<j, b)][c] = t2[i,j,b,c]
    launch_fill(st, c->t2hu, oo * v, v, v, 0, [=] __device__(int64_t row, int64_t cc) {
        int64_t IJ = row / v;
        int b = row % v;
        return asym_col(t2p, IJ, vv, b, (int)cc, v);
    });
    return CCSD_OK;
}

// Aq[(k<l)][(i<j)] = sum_{c<d} <kl||cd> tau^{cd}_{ij}: the quartic term of A (eq 31), kept on its own because H^k_i (eq 26)
// reads its own quartic term off it (fock_like); build_A adds it into A.  Runs before fock_like.
static int build_Aq(ccsd_ctx* c)
{
    if (!c->hoo_trace) return CCSD_OK;
    return run_gemm(c->env, with_planes(gp(c->oo, c->oo, c->vv, c->Voovv_p, c->vv, c->taup, c->vv, c->Aq, c->oo, 1, 1.0, 0),
                                        c->Voovv_ps, c->taups));
}

static int fock_like(ccsd_ctx* c)
{
    cudaStream_t st = c->st;
    const Env& env = c->env;
    const int o = c->o, v = c->v, n = c->n;
    const int64_t oo = c->oo, vv = c->vv, ov = c->ov;
    const c128* f = c->f;
    // eq 28: Hov[k,c] = f[k,c] + sum_{ld} <kl||cd> t1[l,d]            (HovT[(c,k)])
    launch_fill(st, c->HovT, v, o, o, 0, [=] __device__(int64_t cc, int64_t k) { return f[k * n + o + cc]; });
    CCSD_TRY(run_gemv(env, ov, ov, c->G1, ov, c->t1, c->HovT, 1, 1.0, 1));
    const c128* HovT = c->HovT;
    launch_fill(st, c->Hov, o, v, v, 0, [=] __device__(int64_t k, int64_t cc) { return HovT[cc * o + k]; });
    // eq 24: Hvv[a,c] = f[a,c] + sum_{k<l,d} <kl||cd> tau[k,l,d,a]
    launch_fill(st, c->Hvv, v, v, v, 0, [=] __device__(int64_t a, int64_t cc) { return f[(o + a) * n + o + cc]; });
    CCSD_TRY(run_gemm(env, gp(v, v, oo * v, c->tauc, oo * v, c->Voovv_c, oo * v, c->Hvv, v, 1, 1.0, 1)));
    // eq 25: Gvv = Hvv + sum_{kd} <ak||cd> t1[k,d] - sum_k f[k,c] t1[k,a]
    dcopy(st, c->Gvv, c->Hvv, (int64_t)v * v);
    if (!c->gv_trace)     // else: read off the linear term of H^{ak}_{ci} (build_Hvovo, gvv_trace_add)
        CCSD_TRY(run_gemv(env, (int64_t)v * v, ov, c->Vvovv_u, ov, c->t1, c->Gvv, 1, 1.0, 1));
    {
        GemmParams p = gp(v, v, o, c->t1T, o, f + o, 1, c->Gvv, v, 1, -1.0, 1);
        p.sbn = 1; p.sbk = n;  // B[c][k] = f[k][o+c]
        CCSD_TRY(run_gemm(env, p));
    }
    // eq 26: Hoo[k,i] = -f[k,i] + sum_{l, c<d} <kl||cd> tau[l,i,c,d]   (tau[l,i] = -tauou[(i,l)])
    if (c->hoo_trace) {   // <kl||cd> = +-V[(k,l)], tau[l,i] = +-tau[(l,i)]: the sum over (c<d) is +-Aq[(k,l)][(l,i)]
        const c128* Aq = c->Aq;
        launch_fill(st, c->Hoo, o, o, o, 0, [=] __device__(int64_t k, int64_t i) {
            c128 s = cneg(f[k * n + i]);
            for (int l = 0; l < o; l++) {
                if (l == (int)k || l == (int)i) continue;
                const int64_t KL = (int)k < l ? pair_idx((int)k, l, o) : pair_idx(l, (int)k, o);
                const int64_t LI = l < (int)i ? pair_idx(l, (int)i, o) : pair_idx((int)i, l, o);
                const c128 x = Aq[KL * oo + LI];
                s = (((int)k < l) == (l < (int)i)) ? cadd(s, x) : csub(s, x);
            }
            return s;
        });
    } else {
        launch_fill(st, c->Hoo, o, o, o, 0, [=] __device__(int64_t k, int64_t i) { return cneg(f[k * n + i]); });
        CCSD_TRY(run_gemm(env, gp(o, o, o * vv, c->Voovv_ou, o * vv, c->tauou, o * vv, c->Hoo, o, 1, -1.0, 1)));
    }
    // eq 27: Goo = Hoo - sum_{lc} <kl||ic> t1[l,c] - sum_c f[k,c] t1[i,c]
    dcopy(st, c->Goo, c->Hoo, (int64_t)o * o);
    CCSD_TRY(run_gemv(env, (int64_t)o * o, ov, c->Vooov_d, ov, c->t1, c->Goo, 1, -1.0, 1));
    CCSD_TRY(run_gemm(env, gp(o, o, v, f + o, n, c->t1, v, c->Goo, o, 1, -1.0, 1)));
    return CCSD_OK;
}

static int build_Hvovo(ccsd_ctx* c)
{
    const Env& env = c->env;
    const int o = c->o, v = c->v;
    const int64_t ov = c->ov;
    // eq 29, stored as Hm[(a,i)][(c,k)]; this rank's rows: a in [a_lo, a_hi)
    const int a0 = c->sh.a_lo, na = c->sh.a_hi - c->sh.a_lo;
    const int64_t off = (int64_t)a0 * o * ov, rows = (int64_t)na * o;
    if (na <= 0) { tick(c, 3); return CCSD_OK; }
    dcopy(c->st, c->Hm + off, c->Vvovo_m + off, rows * ov);
    {   // + sum_d <ak||cd> t1[i,d]        batched over a: C_a[(c,k)][i]
        GemmParams p = gp(ov, o, v, c->Vvovv_u + (int64_t)a0 * ov * v, v, c->t1, v, c->Hm + off, 1, ov, 1.0, 1);
        p.batch = na; p.bsA = ov * v; p.bsB = 0; p.bsC = (int64_t)o * ov;
        CCSD_TRY(run_gemm(env, p));
    }
    if (c->gv_trace) {    // gvtr[a][c] = sum_k ( Hm - <ak||ci> )[(a,k)][(c,k)]: the product just added, at i = k
        const c128 *Hm = c->Hm, *V0 = c->Vvovo_m;
        launch_fill(c->st, c->gvtr, v, v, v, 0, [=] __device__(int64_t a, int64_t cc) {
            c128 s = mk(0.0, 0.0);
            for (int k = 0; k < o; k++) {
                const int64_t at = (a * o + k) * ov + cc * o + k;
                s = cadd(s, csub(Hm[at], V0[at]));
            }
            return s;
        });
    }
    // - sum_l <kl||ic> t1[l,a]            C[a][(i,c,k)]
    CCSD_TRY(run_gemm(env, gp(na, (int64_t)o * ov, o, c->t1T + (int64_t)a0 * o, o, c->Vooov_b, o, c->Hm + off, (int64_t)o * ov, 1, -1.0, 1)));
    tick(c, 3);
    // + sum_{ld} <kl||cd> (1/2 t2[l,i,a,d] + t1[l,a] t1[i,d])       (ov x ov x ov)
    if (c->strassen) {   // seven half-size products (strassen.cuh); the ring product stacks Hm itself, no plane of Hm needed
        return strassen_gemm(env, gp(rows, ov, ov, c->Xm + off, ov, c->G1, ov, c->Hm + off, ov, 1, 1.0, 1), nullptr, &c->sG1, c->str_ring,
                             c->strassen_levels);
    }
    CCSD_TRY(run_gemm(env, with_planes(gp(rows, ov, ov, c->Xm + off, ov, c->G1, ov, c->Hm + off, ov, 1, 1.0, 1),
                                       c->Xms ? c->Xms + off : nullptr, c->G1s)));
    if (c->Hms) launch_sum_plane(c->st, c->Hm + off, c->Hms + off, rows * ov);   // operand of the ring GEMM
    return CCSD_OK;
}

// CC2 only.  With t2 = 0 the two quadratic terms that need <ab||cd> and <bk||cd> factorise through the auxiliary index of
// (pq|rs) = sum_L B^L_pq B^L_rs (Cholesky vectors), with the t1-dressed factors
//     Xv[(a,i)][L] = sum_e B^L_ae t1[i,e],      Xo[(k,j)][L] = sum_d B^L_kd t1[j,d]:
//     sum_{e<f} <ab||ef> tau0^{ef}_{ij} = sum_ef <ab||ef> t_i^e t_j^f = sum_L ( Xv_ai Xv_bj - Xv_aj Xv_bi )        (K = L)
//     sum_{c<d} <bk||cd> tau0^{cd}_{ij}                               = sum_L ( Xv_bi Xo_kj - Xv_bj Xo_ki )
// i.e. (ov)^2 L and ov o^2 L work instead of oo vv^2 and ov oo vv: the doubles equations of CC2 drop from O(o^2 v^4) to
// O(o^2 v^2 L), which is what makes CC2 an N^5 method.
static int cc2_dressed_factors(ccsd_ctx* c)
{
    const int o = c->o, v = c->v, Lp = c->Lp;
    {
        GemmParams p = gp(Lp, o, v, c->BvvT, v, c->t1, v, c->Xv, 1, Lp, 1.0, 0);      // per a: C_a[L][i]
        p.batch = v; p.bsA = (int64_t)Lp * v; p.bsB = 0; p.bsC = (int64_t)o * Lp;
        CCSD_TRY(run_gemm(c->env, p));
    }
    {
        GemmParams p = gp(Lp, o, v, c->BovT, v, c->t1, v, c->Xo, 1, Lp, 1.0, 0);      // per k: C_k[L][j]
        p.batch = o; p.bsA = (int64_t)Lp * v; p.bsB = 0; p.bsC = (int64_t)o * Lp;
        CCSD_TRY(run_gemm(c->env, p));
    }
    if (c->planes) launch_sum_plane(c->st, c->Xv, c->Xvs, c->ov * Lp);
    return CCSD_OK;
}

static int build_C(ccsd_ctx* c)
{
    cudaStream_t st = c->st;
    const Env& env = c->env;
    const int o = c->o, v = c->v;
    const int64_t oo = c->oo, vv = c->vv;
    const int2* po = c->po;
    // eq 30, stored as Cm[(b,k)][(i<j)]; this rank's rows: b in [a_lo, a_hi)
    const int64_t row0 = (int64_t)c->sh.a_lo * o, rows = (int64_t)(c->sh.a_hi - c->sh.a_lo) * o;
    if (rows <= 0) return CCSD_OK;
    dcopy(st, c->Cm + row0 * oo, c->Vooov_cc + row0 * oo, rows * oo);
    CCSD_TRY(run_gemm(env, gp(rows * o, o, v, c->Vvovo_c + row0 * o * v, v, c->t1, v, c->Y + row0 * o * o, o, 1, 1.0, 0)));
    const c128* Y = c->Y;
    launch_fill(st, c->Cm + row0 * oo, rows, oo, oo, 1, [=] __device__(int64_t r, int64_t IJ) {
        const int64_t bk = row0 + r;
        int2 ij = po[IJ];
        return csub(Y[(bk * o + ij.x) * o + ij.y], Y[(bk * o + ij.y) * o + ij.x]);
    });
    if (c->opt.cc2) {   // - sum_L ( Xv_bi Xo_kj - Xv_bj Xo_ki ): Q[(b,i)][(k,j)] in the buffer the linear term just released
        c128* Q = c->Y;
        CCSD_TRY(run_gemm(env, gp(c->ov, (int64_t)o * o, c->Lp, c->Xv, c->Lp, c->Xo, c->Lp, Q, (int64_t)o * o, 1, 1.0, 0)));
        launch_fill(st, c->Cm, c->ov, oo, oo, 1, [=] __device__(int64_t bk, int64_t IJ) {
            int2 ij = po[IJ];
            const int64_t b = bk / o, k = bk % o;
            return csub(Q[((b * o + ij.y) * o + k) * o + ij.x], Q[((b * o + ij.x) * o + k) * o + ij.y]);
        });
        return CCSD_OK;
    }
    // - sum_{c<d} <bk||cd> tau^{cd}_{ij}: into Cq when S1 takes its <ak||cd> tau term from it (s1_c_trace), then added to Cm
    c128* dst = c->s1_trace ? c->Cq : c->Cm + row0 * oo;
    const int acc = c->s1_trace ? 0 : 1;
    if (c->strassen && c->sVvovv.S)
        CCSD_TRY(strassen_gemm(env, gp(rows, oo, vv, c->Vvovv_p + row0 * vv, vv, c->taup, vv, dst, oo, 1, -1.0, acc), &c->sVvovv,
                               c->strassen_levels_C == 2 ? &c->sTauC : &c->sTau, c->str_C, c->strassen_levels_C));
    else
        CCSD_TRY(run_gemm(env, with_planes(gp(rows, oo, vv, c->Vvovv_p + row0 * vv, vv, c->taup, vv, dst, oo, 1, -1.0, acc),
                                           c->Vvovv_ps ? c->Vvovv_ps + row0 * vv : nullptr, c->taups)));
    if (c->s1_trace) {
        const c128* Cq = c->Cq;
        launch_fill(st, c->Cm, rows, oo, oo, 1, [=] __device__(int64_t r, int64_t IJ) { return Cq[r * oo + IJ]; });
    }
    return CCSD_OK;
}

// S1[i,a] += sum_{k, c<d} <ak||cd> tau[i,k,c,d]  (eq 33) read off the product of C: tau[i,k] = +-tau[(min,max)], so the sum over
// (c<d) is -Cq[(a,k)][(i,k)] for i < k and +Cq[(a,k)][(k,i)] for k < i
static int s1_c_trace(ccsd_ctx* c)
{
    if (!c->s1_trace) return CCSD_OK;
    const c128* Cq = c->Cq;
    const int o = c->o, v = c->v;
    const int64_t oo = c->oo;
    launch_fill(c->st, c->S1, o, v, v, 1, [=] __device__(int64_t i, int64_t a) {
        c128 s = mk(0.0, 0.0);
        for (int k = 0; k < o; k++) {
            if (k == (int)i) continue;
            const c128 x = (int)i < k ? cneg(Cq[(a * o + k) * oo + pair_idx((int)i, k, o)]) : Cq[(a * o + k) * oo + pair_idx(k, (int)i, o)];
            s = cadd(s, x);
        }
        return s;
    });
    return CCSD_OK;
}

static int build_A(ccsd_ctx* c)
{
    cudaStream_t st = c->st;
    const Env& env = c->env;
    const int o = c->o, v = c->v;
    const int64_t oo = c->oo, vv = c->vv;
    const int2* po = c->po;
    // eq 31, stored as Am[(k<l)][(i<j)]
    dcopy(st, c->Am, c->Voooo_p, oo * oo);
    CCSD_TRY(run_gemm(env, gp(oo * o, o, v, c->Vooov_p, v, c->t1, v, c->Z, o, 1, 1.0, 0)));
    const c128* Z = c->Z;
    launch_fill(st, c->Am, oo, oo, oo, 1, [=] __device__(int64_t KL, int64_t IJ) {
        int2 ij = po[IJ];
        return csub(Z[(KL * o + ij.x) * o + ij.y], Z[(KL * o + ij.y) * o + ij.x]);
    });
    if (c->hoo_trace) {   // the quartic term is there already (build_Aq)
        const c128* Aq = c->Aq;
        launch_fill(st, c->Am, oo, oo, oo, 1, [=] __device__(int64_t KL, int64_t IJ) { return Aq[KL * oo + IJ]; });
        return CCSD_OK;
    }
    CCSD_TRY(run_gemm(env, with_planes(gp(oo, oo, vv, c->Voovv_p, vv, c->taup, vv, c->Am, oo, 1, 1.0, 1), c->Voovv_ps, c->taups)));
    return CCSD_OK;
}

// ---- the eight terms of eq 32; each ADDS this rank's slab of the term into S[(i<j)][(a<b)] (struct Shard) --------------
static int s2_driver(ccsd_ctx* c, c128* S)
{
    const c128* V = c->Voovv_p;
    const int64_t vv = c->vv, r0 = c->sh.ij_lo;
    launch_fill(c->st, S + r0 * vv, c->sh.ij_hi - r0, vv, vv, 1,
                [=] __device__(int64_t r, int64_t AB) { return cconj(V[(r0 + r) * vv + AB]); });
    return CCSD_OK;
}
static int s2_pp_ladder(ccsd_ctx* c, c128* S)
{   // sum_{c<d} <ab||cd> tau[i,j,c,d]      M = (a<b), N = (i<j), K = (c<d)
    if (c->opt.cc2) {   // tau = P-(t1 t1): sum_L ( Xv_ai Xv_bj - Xv_aj Xv_bi ), R2[(a,i)][(b,j)] = sum_L Xv_ai Xv_bj
        const int o = c->o;
        const int64_t ov = c->ov, vv = c->vv;
        c128* R2 = c->Xr;
        CCSD_TRY(run_gemm(c->env, with_planes(gp(ov, ov, c->Lp, c->Xv, c->Lp, c->Xv, c->Lp, R2, ov, 1, 1.0, 0), c->Xvs, c->Xvs)));
        const int2 *po = c->po, *pv = c->pv;
        launch_fill(c->st, S, c->oo, vv, vv, 1, [=] __device__(int64_t IJ, int64_t AB) {
            int2 ij = po[IJ], ab = pv[AB];
            const int64_t a = ab.x, b = ab.y;
            return csub(R2[(a * o + ij.x) * ov + b * o + ij.y], R2[(a * o + ij.y) * ov + b * o + ij.x]);
        });
        return CCSD_OK;
    }
    if (c->opt.direct_ladder && c->WslabT) {
        // integral-direct on one GPU, using <ab||cd> = conj <cd||ab>: for the slab of packed rows [r0, r1) only the columns
        // CD >= r0 are rebuilt from B (half the slab-GEMM flops over all slabs), and the block serves twice:
        //   (1) S[:, r0:r1) += W[r0:r1, r0:vv) tau[:, r0:vv)^T                      M = slab rows,  K = vv - r0
        //   (2) S[:, r1:vv) += conj(W[r0:r1, r1:vv))^T tau[:, r0:r1)^T               M = vv - r1,    K = slab rows
        // (2) is what the later slabs would have computed from their columns CD < their r0.  Its left operand is the
        // conj-transposed copy of the block (one bandwidth-bound pass), so that both products stay K-contiguous.
        const int64_t vv = c->vv, oo = c->oo;
        for (int a0 = 0; a0 < c->v - 1; a0 += c->na_slab) {
            int64_t r0 = 0, nrows = 0;
            CCSD_TRY(build_W_slab(c, a0, c->v - 1, c->Wslab, false, &r0, &nrows, true, c->planes ? c->Wslabs : nullptr));
            const int64_t r1 = r0 + nrows, ldt = round_up(nrows, 2);
            CCSD_TRY(run_gemm(c->env, with_planes(gp(nrows, oo, vv - r0, c->Wslab + r0, vv, c->taup + r0, vv, S + r0, 1, vv, 1.0, 1),
                                                  c->planes ? c->Wslabs + r0 : nullptr, c->taups ? c->taups + r0 : nullptr)));
            if (r1 < vv) {
                if (ldt > nrows) CCSD_CUDA_TRY(cudaMemsetAsync(c->WslabT, 0, (size_t)((vv - r1) * ldt) * sizeof(c128), c->st));
                CCSD_TRY(launch_transpose2d_ld(c->st, c->Wslab + r1, vv, c->WslabT, ldt, nrows, vv - r1, 1));
                if (c->planes) launch_sum_plane(c->st, c->WslabT, c->WslabTs, (vv - r1) * ldt);
                CCSD_TRY(run_gemm(c->env, with_planes(gp(vv - r1, oo, nrows, c->WslabT, ldt, c->taup + r0, vv, S + r1, 1, vv, 1.0, 1),
                                                      c->planes ? c->WslabTs : nullptr, c->taups ? c->taups + r0 : nullptr)));
            }
        }
        return CCSD_OK;
    }
    if (c->opt.direct_ladder) {   // integral-direct, sharded: rebuild this rank's rows of <ab||cd> slab by slab and contract them
        for (int a0 = c->sh.wa_lo; a0 < c->sh.wa_hi; a0 += c->na_slab) {
            int64_t r0 = 0, nrows = 0;
            CCSD_TRY(build_W_slab(c, a0, c->sh.wa_hi, c->Wslab, false, &r0, &nrows));
            if (c->planes) launch_sum_plane(c->st, c->Wslab, c->Wslabs, nrows * c->vv);
            CCSD_TRY(run_gemm(c->env, with_planes(gp(nrows, c->oo, c->vv, c->Wslab, c->vv, c->taup, c->vv, S + r0, 1, c->vv, 1.0, 1),
                                                  c->planes ? c->Wslabs : nullptr, c->taups)));
        }
        return CCSD_OK;
    }
    const int64_t rows = c->sh.w_hi - c->sh.w_lo;      // this rank's rows of <ab||cd> (all of them for world = 1)
    if (c->strassen && c->sW.S)      // both operand stacks are ready (ccsd_init, prep_operands): one batched launch + the result sums
        return strassen_gemm(c->env, gp(rows, c->oo, c->vv, c->W, c->vv, c->taup, c->vv, S + c->sh.w_lo, 1, c->vv, 1.0, 1), &c->sW,
                             c->strassen_levels_L == 2 ? &c->sTauC : &c->sTau, c->str_L, c->strassen_levels_L);
    return run_gemm(c->env, with_planes(gp(rows, c->oo, c->vv, c->W, c->vv, c->taup, c->vv, S + c->sh.w_lo, 1, c->vv, 1.0, 1), c->Ws, c->taups));
}
static void fill_AG_hh(ccsd_ctx* c)
{   // AG[(i<j)][(k<l)] = A[k,l,i,j]
    const c128* Am = c->Am;
    const int64_t oo = c->oo;
    launch_fill(c->st, c->AG, oo, oo, 2 * c->oop, 0, [=] __device__(int64_t IJ, int64_t KL) { return Am[KL * oo + IJ]; });
}
static void fill_AG_goo(ccsd_ctx* c)
{   // Ghat[(i<j)][(k<l)] = d_ik Goo[l,j] - d_il Goo[k,j] - d_jk Goo[l,i] + d_jl Goo[k,i]
    //   == P-_ji sum_m Goo[m,j] t2[i,m,a,b] written on packed pairs (reading G7 of eq 32)
    const c128* Goo = c->Goo;
    const int o = c->o;
    const int2* po = c->po;
    launch_fill(c->st, c->AG + c->oop, c->oo, c->oo, 2 * c->oop, 0, [=] __device__(int64_t IJ, int64_t KL) {
        int2 ij = po[IJ], kl = po[KL];
        c128 s = mk(0.0, 0.0);
        if (ij.x == kl.x) s = cadd(s, Goo[kl.y * o + ij.y]);
        if (ij.x == kl.y) s = csub(s, Goo[kl.x * o + ij.y]);
        if (ij.y == kl.x) s = csub(s, Goo[kl.y * o + ij.x]);
        if (ij.y == kl.y) s = cadd(s, Goo[kl.x * o + ij.x]);
        return s;
    });
}
static int fill_TT_t2(ccsd_ctx* c)
{   // TT[(a<b)][oop:oop+oo) = t2^T
    return launch_transpose2d_ld(c->st, c->t2p, c->vv, c->TT + c->oop, 2 * c->oop, c->oo, c->vv, 0);
}
// the three products with M = (a<b) rows of TT run on this rank's rows [w_lo, w_hi)
static int s2_hh_ladder(ccsd_ctx* c, c128* S)
{   // sum_{k<l} A[k,l,i,j] tau[k,l,a,b]
    fill_AG_hh(c);
    const int64_t r0 = c->sh.w_lo, rows = c->sh.w_hi - r0, ld = 2 * c->oop;
    return run_gemm(c->env, gp(rows, c->oo, c->oop, c->TT + r0 * ld, ld, c->AG, ld, S + r0, 1, c->vv, 1.0, 1));
}
static int s2_goo(ccsd_ctx* c, c128* S)
{
    CCSD_TRY(fill_TT_t2(c));
    fill_AG_goo(c);
    const int64_t r0 = c->sh.w_lo, rows = c->sh.w_hi - r0, ld = 2 * c->oop;
    return run_gemm(c->env, gp(rows, c->oo, c->oop, c->TT + r0 * ld + c->oop, ld, c->AG + c->oop, ld, S + r0, 1, c->vv, 1.0, 1));
}
static int s2_hh_and_goo(ccsd_ctx* c, c128* S)
{   // Both terms in ONE product over the pairs (k<l) of tau:  A tau + Ghat t2 = (A + Ghat) tau - Ghat (tau - t2), and the last
    // piece is elementwise because tau - t2 = P-(t1 t1) (eq 23):  with X[j,b] = sum_m Goo[m,j] t1[m,b]
    //   (Ghat (tau - t2))[(ij)][(ab)] = P-_ji ( t1[i,a] X[j,b] - X[j,a] t1[i,b] ).
    // (K = oo instead of the 2 oo of the operand pair [tau | t2] x [A | Ghat]: half the tensor-pipe work of this step.)
    if (c->opt.cc2) {   // CC2 runs this with tau0 = P-(t1 t1) beside the full t2: tau - t2 is not P-(t1 t1); keep the operand pair
        CCSD_TRY(fill_TT_t2(c));
        fill_AG_hh(c);
        fill_AG_goo(c);
        const int64_t r0 = c->sh.w_lo, rows = c->sh.w_hi - r0, ld = 2 * c->oop;
        return run_gemm(c->env, gp(rows, c->oo, 2 * c->oop, c->TT + r0 * ld, ld, c->AG, ld, S + r0, 1, c->vv, 1.0, 1));
    }
    const c128 *Am = c->Am, *Goo = c->Goo, *t1 = c->t1;
    const int o = c->o, v = c->v;
    const int64_t oo = c->oo;
    const int2 *po = c->po, *pv = c->pv;
    launch_fill(c->st, c->AG, oo, oo, 2 * c->oop, 0, [=] __device__(int64_t IJ, int64_t KL) {
        int2 ij = po[IJ], kl = po[KL];
        c128 s = Am[KL * oo + IJ];
        if (ij.x == kl.x) s = cadd(s, Goo[kl.y * o + ij.y]);
        if (ij.x == kl.y) s = csub(s, Goo[kl.x * o + ij.y]);
        if (ij.y == kl.x) s = csub(s, Goo[kl.y * o + ij.x]);
        if (ij.y == kl.y) s = cadd(s, Goo[kl.x * o + ij.x]);
        return s;
    });
    c128* X = c->tmp_ov;     // X[j][b]
    launch_fill(c->st, X, o, v, v, 0, [=] __device__(int64_t j, int64_t b) {
        c128 s = mk(0.0, 0.0);
        for (int m = 0; m < o; m++) cfma(s, Goo[m * o + j], t1[m * v + b]);
        return s;
    });
    const int64_t r0 = c->sh.w_lo, rows = c->sh.w_hi - r0, ld = 2 * c->oop;
    CCSD_TRY(run_gemm(c->env, gp(rows, oo, c->oop, c->TT + r0 * ld, ld, c->AG, ld, S + r0, 1, c->vv, 1.0, 1)));
    launch_fill(c->st, S + r0, oo, rows, c->vv, 1, [=] __device__(int64_t IJ, int64_t rel) {
        const int2 ij = po[IJ], ab = pv[r0 + rel];
        const c128 *ti = t1 + (int64_t)ij.x * v, *tj = t1 + (int64_t)ij.y * v, *Xi = X + (int64_t)ij.x * v, *Xj = X + (int64_t)ij.y * v;
        c128 d = mk(0.0, 0.0);                       // - [ (t_ia X_jb - X_ja t_ib) - (t_ja X_ib - X_ia t_jb) ]
        cfma(d, Xj[ab.x], ti[ab.y]);
        cfma(d, tj[ab.x], Xi[ab.y]);
        d = csub(d, cmul(ti[ab.x], Xj[ab.y]));
        d = csub(d, cmul(Xi[ab.x], tj[ab.y]));
        return d;
    });
    return CCSD_OK;
}
static int ring_gemm(ccsd_ctx* c)
{   // X[i,j,a,b] = sum_{kc} Hvovo[a,k,c,i] t2[j,k,c,b] = Xr[(a,i)][(j,b)]; this rank holds the rows a in [a_lo, a_hi) of H and X
    const int o = c->o;
    const int64_t ov = c->ov;
    const int64_t off = (int64_t)c->sh.a_lo * o * ov, rows = (int64_t)(c->sh.a_hi - c->sh.a_lo) * o;
    if (rows <= 0) return CCSD_OK;
    if (c->strassen)
        return strassen_gemm(c->env, gp(rows, ov, ov, c->Hm + off, ov, c->T2r, ov, c->Xr + off, ov, 1, 1.0, 0), nullptr, nullptr, c->str_ring,
                             c->strassen_levels);
    return run_gemm(c->env, with_planes(gp(rows, ov, ov, c->Hm + off, ov, c->T2r, ov, c->Xr + off, ov, 1, 1.0, 0),
                                        c->Hms ? c->Hms + off : nullptr, c->T2rs));
}
static int ring_add(ccsd_ctx* c, c128* S)
{   // S += P-_ij P-_ab X: this rank adds the terms whose first index is one of its rows a
    const int o = c->o, v = c->v;
    const int64_t vv = c->vv;
    const int alo = c->sh.a_lo, ahi = c->sh.a_hi;
    if (ahi <= alo) return CCSD_OK;
    const c128* Xr = c->Xr;
    const int2 *po = c->po, *pv = c->pv;
    launch_fill(c->st, S, c->oo, vv, vv, 1, [=] __device__(int64_t IJ, int64_t AB) {
        int2 ij = po[IJ], ab = pv[AB];
        int64_t i = ij.x, j = ij.y, a = ab.x, b = ab.y;
        c128 s = mk(0.0, 0.0);
        if (a >= alo && a < ahi) s = csub(Xr[((a * o + i) * o + j) * v + b], Xr[((a * o + j) * o + i) * v + b]);
        if (b >= alo && b < ahi) {
            s = csub(s, Xr[((b * o + i) * o + j) * v + a]);
            s = cadd(s, Xr[((b * o + j) * o + i) * v + a]);
        }
        return s;
    });
    return CCSD_OK;
}
static int s2_ring(ccsd_ctx* c, c128* S)
{
    CCSD_TRY(ring_gemm(c));
    tick(c, 9);
    return ring_add(c, S);
}
// The three remaining small terms, each as its product (into a buffer of its own) and its antisymmetrising add into S:
// in the captured graph the products run inside the parallel branches, the adds after the join (residual_forked).
static int vdag_gemm(ccsd_ctx* c)
{   // P[i][(j,a<b)] = sum_c conj(<cj||ab>) t1[i,c]
    const int o = c->o, v = c->v;
    const int64_t vv = c->vv, r0 = c->sh.w_lo, rows = c->sh.w_hi - c->sh.w_lo;
    if (c->sh.world == 1) return run_gemm(c->env, gp(o * vv, o, v, c->VvovvT, v, c->t1, v, c->P, 1, o * vv, 1.0, 0));
    if (rows <= 0) return CCSD_OK;   // this rank's (a<b) columns only: one product per j
    GemmParams p = gp(rows, o, v, c->VvovvT + r0 * v, v, c->t1, v, c->P + r0, 1, o * vv, 1.0, 0);
    p.batch = o; p.bsA = vv * v; p.bsB = 0; p.bsC = vv;
    return run_gemm(c->env, p);
}
static int vdag_add(ccsd_ctx* c, c128* S)
{   // S += P[(i,j)] - P[(j,i)]
    const int o = c->o;
    const int64_t vv = c->vv, r0 = c->sh.w_lo, rows = c->sh.w_hi - c->sh.w_lo;
    if (rows <= 0) return CCSD_OK;
    const c128* P = c->P;
    const int2* po = c->po;
    launch_fill(c->st, S + r0, c->oo, rows, vv, 1, [=] __device__(int64_t IJ, int64_t col) {
        int2 ij = po[IJ];
        const int64_t AB = r0 + col;
        return csub(P[((int64_t)ij.x * o + ij.y) * vv + AB], P[((int64_t)ij.y * o + ij.x) * vv + AB]);
    });
    return CCSD_OK;
}
static int s2_vdag_t1(ccsd_ctx* c, c128* S)
{   // sum_c conj(<cj||ab>) t1[i,c] - (i<->j)
    CCSD_TRY(vdag_gemm(c));
    return vdag_add(c, S);
}
static void gvv_trace_add(ccsd_ctx* c)
{   // Gvv += gvtr (see ccsd_ctx::gvtr): after fock_like and the linear term of build_Hvovo, before gvv_gemm
    if (!c->gv_trace) return;
    const c128* g = c->gvtr;
    const int v = c->v;
    launch_fill(c->st, c->Gvv, v, v, v, 1, [=] __device__(int64_t a, int64_t cc) { return g[a * v + cc]; });
}
static int gvv_gemm(ccsd_ctx* c)
{   // Qm[(i<j,b)][a] = sum_c t2[i,j,b,c] Gvv[a,c]; rows (i<j) of this rank
    const int v = c->v;
    const int64_t r0 = c->sh.ij_lo, rows = c->sh.ij_hi - c->sh.ij_lo;
    if (rows <= 0) return CCSD_OK;
    return run_gemm(c->env, gp(rows * v, v, v, c->t2hu + r0 * v * v, v, c->Gvv, v, c->Qm + r0 * v * v, v, 1, 1.0, 0));
}
static int gvv_add(ccsd_ctx* c, c128* S)
{   // S += sum_c Gvv[a,c] t2[i,j,c,b] - Gvv[b,c] t2[i,j,c,a] = Qm[(ij,a)][b] - Qm[(ij,b)][a]
    const int v = c->v;
    const int64_t vv = c->vv, r0 = c->sh.ij_lo, rows = c->sh.ij_hi - c->sh.ij_lo;
    if (rows <= 0) return CCSD_OK;
    const c128* Qm = c->Qm;
    const int2* pv = c->pv;
    launch_fill(c->st, S + r0 * vv, rows, vv, vv, 1, [=] __device__(int64_t r, int64_t AB) {
        const int64_t IJ = r0 + r;
        int2 ab = pv[AB];
        return csub(Qm[(IJ * v + ab.x) * v + ab.y], Qm[(IJ * v + ab.y) * v + ab.x]);
    });
    return CCSD_OK;
}
static int s2_gvv(ccsd_ctx* c, c128* S)
{
    CCSD_TRY(gvv_gemm(c));
    return gvv_add(c, S);
}
static int c_t1_gemm(ccsd_ctx* c)
{   // Rr[(a,i<j)][b] = sum_k C[k,a,i,j] t1[k,b]; rows a of this rank
    const int o = c->o, v = c->v;
    const int64_t oo = c->oo;
    const int64_t row0 = (int64_t)c->sh.a_lo * oo, rows = (int64_t)(c->sh.a_hi - c->sh.a_lo) * oo;
    if (rows <= 0) return CCSD_OK;
    const c128* Cm = c->Cm;
    launch_fill(c->st, c->Cm2 + row0 * o, rows, o, o, 0, [=] __device__(int64_t r, int64_t k) {
        const int64_t row = row0 + r, a = row / oo, IJ = row % oo;
        return Cm[(a * o + k) * oo + IJ];
    });
    return run_gemm(c->env, gp(rows, v, o, c->Cm2 + row0 * o, o, c->t1T, o, c->Rr + row0 * v, v, 1, 1.0, 0));
}
static int c_t1_add(ccsd_ctx* c, c128* S)
{   // S += sum_k C[k,a,i,j] t1[k,b] - C[k,b,i,j] t1[k,a], the terms whose C row is one of this rank's
    const int v = c->v;
    const int64_t vv = c->vv, oo = c->oo;
    const int alo = c->sh.a_lo, ahi = c->sh.a_hi;
    if (ahi <= alo) return CCSD_OK;
    const c128* Rr = c->Rr;
    const int2* pv = c->pv;
    launch_fill(c->st, S, oo, vv, vv, 1, [=] __device__(int64_t IJ, int64_t AB) {
        int2 ab = pv[AB];
        c128 s = mk(0.0, 0.0);
        if (ab.x >= alo && ab.x < ahi) s = Rr[((int64_t)ab.x * oo + IJ) * v + ab.y];
        if (ab.y >= alo && ab.y < ahi) s = csub(s, Rr[((int64_t)ab.y * oo + IJ) * v + ab.x]);
        return s;
    });
    return CCSD_OK;
}
static int s2_c_t1(ccsd_ctx* c, c128* S)
{
    CCSD_TRY(c_t1_gemm(c));
    return c_t1_add(c, S);
}

static int build_S1(ccsd_ctx* c)
{
    cudaStream_t st = c->st;
    const Env& env = c->env;
    const int o = c->o, v = c->v, n = c->n;
    const int64_t oo = c->oo, vv = c->vv, ov = c->ov;
    const c128* f = c->f;
    // eq 33
    launch_fill(st, c->S1, o, v, v, 0, [=] __device__(int64_t i, int64_t a) { return cconj(f[i * n + o + a]); });
    CCSD_TRY(run_gemm(env, gp(o, v, v, c->t1, v, c->Hvv, v, c->S1, v, 1, 1.0, 1)));                  // Hvv[a,c] t1[i,c]
    {
        GemmParams p = gp(o, v, o, c->Hoo, 1, c->t1, 1, c->S1, v, 1, 1.0, 1);                         // Hoo[k,i] t1[k,a]
        p.sam = 1; p.sak = o; p.sbn = 1; p.sbk = v;
        CCSD_TRY(run_gemm(env, p));
    }
    CCSD_TRY(run_gemv(env, ov, ov, c->T2r, ov, c->HovT, c->S1, 1, -1.0, 1));                          // Hov[k,c] t2[i,k,a,c]
    const c128* Hov = c->Hov;
    launch_fill(st, c->HF, o, v, v, 0, [=] __device__(int64_t k, int64_t cc) {
        c128 x = f[k * n + o + cc];
        return mk(Hov[k * v + cc].x - 2.0 * x.x, Hov[k * v + cc].y - 2.0 * x.y);
    });
    CCSD_TRY(run_gemm(env, gp(o, o, v, c->HF, v, c->t1, v, c->inner, o, 1, 1.0, 0)));                 // inner[k][i]
    {
        GemmParams p = gp(o, v, o, c->inner, 1, c->t1, 1, c->S1, v, 1, 1.0, 1);
        p.sam = 1; p.sak = o; p.sbn = 1; p.sbk = v;
        CCSD_TRY(run_gemm(env, p));
    }
    if (!c->s1_trace)      // else: s1_c_trace, once C's product is there
        CCSD_TRY(run_gemm(env, gp(v, o, o * vv, c->Vvovv_p, o * vv, c->tauou, o * vv, c->S1, 1, v, 1.0, 1)));  // <ak||cd> tau[i,k,c,d]
    CCSD_TRY(run_gemm(env, gp(o, v, oo * v, c->Vooov_e, oo * v, c->tauc, oo * v, c->S1, v, 1, 1.0, 1)));   // <kl||ic> tau[k,l,c,a]
    CCSD_TRY(run_gemv(env, ov, ov, c->Vvovo_m, ov, c->t1T, c->tmp_ov, 1, 1.0, 0));                         // <ak||ci> t1[k,c]
    const c128* tmp = c->tmp_ov;
    launch_fill(st, c->S1, o, v, v, 1, [=] __device__(int64_t i, int64_t a) { return cneg(tmp[a * o + i]); });
    return CCSD_OK;
}

static int residual(ccsd_ctx* c)
{
    tick(c, 0);
    CCSD_TRY(prep_operands(c));
    tick(c, 1);
    CCSD_TRY(build_Aq(c));      // the quartic term of A: timed with the Fock-like terms, which read H^k_i's quartic term off it
    CCSD_TRY(fock_like(c));
    tick(c, 2);
    CCSD_TRY(build_Hvovo(c));   // ticks 3 inside
    gvv_trace_add(c);
    tick(c, 4);
    CCSD_TRY(build_C(c));
    tick(c, 5);
    CCSD_TRY(build_A(c));
    cudaMemsetAsync(c->S2p, 0, (size_t)(c->oo * c->vv) * sizeof(c128), c->st);
    CCSD_TRY(s2_driver(c, c->S2p));
    tick(c, 6);
    CCSD_TRY(s2_pp_ladder(c, c->S2p));
    tick(c, 7);
    CCSD_TRY(s2_hh_and_goo(c, c->S2p));
    tick(c, 8);
    CCSD_TRY(s2_ring(c, c->S2p));  // ticks 9 inside
    tick(c, 10);
    CCSD_TRY(s2_vdag_t1(c, c->S2p));
    tick(c, 11);
    CCSD_TRY(s2_gvv(c, c->S2p));
    tick(c, 12);
    CCSD_TRY(s2_c_t1(c, c->S2p));
    tick(c, 13);
    CCSD_TRY(build_S1(c));
    CCSD_TRY(s1_c_trace(c));
    tick(c, 14);
    c->have_residual = true;
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

// Fork / join inside ONE stream capture, without further streams: the dependency set of the capturing stream is read
// (cudaStreamGetCaptureInfo) and rewritten (cudaStreamUpdateCaptureDependencies), so that the launches that follow hang off the
// fork point instead of off the previous branch.  The replayed graph then runs independent parts of the residual side by side.
struct CaptureFork {
    cudaStream_t st;
    std::vector<cudaGraphNode_t> base, tails;
    bool snapshot(std::vector<cudaGraphNode_t>& out) const
    {
        cudaStreamCaptureStatus status = cudaStreamCaptureStatusNone;
        const cudaGraphNode_t* deps = nullptr;
        size_t n = 0;
        if (cudaStreamGetCaptureInfo(st, &status, nullptr, nullptr, &deps, &n) != cudaSuccess || status != cudaStreamCaptureStatusActive)
            return false;
        out.assign(deps, deps + n);
        return true;
    }
    bool begin(cudaStream_t s) { st = s; tails.clear(); return snapshot(base); }
    bool end_branch()
    {   // what this branch ended on joins the tails; the next branch starts from the fork point again
        std::vector<cudaGraphNode_t> t;
        if (!snapshot(t)) return false;
        tails.insert(tails.end(), t.begin(), t.end());
        return cudaStreamUpdateCaptureDependencies(st, base.data(), base.size(), cudaStreamSetCaptureDependencies) == cudaSuccess;
    }
    bool join()
    {
        std::vector<cudaGraphNode_t> u;
        for (cudaGraphNode_t n : tails) {
            bool seen = false;
            for (cudaGraphNode_t m : u) seen = seen || m == n;
            if (!seen) u.push_back(n);
        }
        return cudaStreamUpdateCaptureDependencies(st, u.data(), u.size(), cudaStreamSetCaptureDependencies) == cudaSuccess;
    }
};

// The residual with its independent parts as parallel branches of the captured graph (only ever called during capture):
//   after the operand re-layout:   [ H^{ak}_{ci} -> ring product ]   [ Fock-like intermediates -> G_vv t2 product -> S1 ]
//                                  [ C -> C t1 product ]   [ A -> V^dagger t1 product ]   [ S2 = driver + pp-ladder ]
//   joined:                        hh-ladder / G_oo, then the antisymmetrising adds of ring, V^dagger t1, G_vv t2, C t1 into S2
// The small configurations do not fill 148 SMs with one product at a time (cfg1: 108-384 tiles per large GEMM, a chain of
// 25 few-microsecond kernels for the Fock-like terms and S1): side by side they fill each other's partial waves.  Every
// branch writes buffers of its own; split-K scratch comes in one slot per branch.  Same kernels on the same inputs as the
// serial order, so the results are bit-identical to it.
static int residual_forked(ccsd_ctx* c)
{
    CaptureFork fk;
    c128* const partial0 = c->env.partial;
    const int64_t pe0 = c->env.partial_elems;
    auto slot = [&](int k) {   // split-K scratch of branch k
        c->env.partial = k == 0 ? partial0 : c->partial_extra + (int64_t)(k - 1) * c->partial_extra_elems;
        c->env.partial_elems = k == 0 ? pe0 : c->partial_extra_elems;
    };
    int s = prep_operands(c);
    bool ok = s == CCSD_OK && fk.begin(c->st);
    if (ok) {
        slot(0);
        s = build_Hvovo(c);
        if (s == CCSD_OK) s = ring_gemm(c);
        ok = s == CCSD_OK && fk.end_branch();
    }
    if (ok) {
        slot(1);
        s = build_Aq(c);
        if (s == CCSD_OK && c->hoo_trace) s = build_A(c);      // A needs Aq: same branch
        if (s == CCSD_OK) s = fock_like(c);
        if (s == CCSD_OK && !c->gv_trace) s = gvv_gemm(c);     // with gv_trace Gvv is complete only after the join
        if (s == CCSD_OK) s = build_S1(c);
        ok = s == CCSD_OK && fk.end_branch();
    }
    if (ok) {
        slot(2);
        s = build_C(c);
        if (s == CCSD_OK) s = c_t1_gemm(c);
        ok = s == CCSD_OK && fk.end_branch();
    }
    if (ok) {
        slot(3);
        s = c->hoo_trace ? CCSD_OK : build_A(c);
        if (s == CCSD_OK) s = vdag_gemm(c);
        ok = s == CCSD_OK && fk.end_branch();
    }
    if (ok) {
        slot(4);
        cudaMemsetAsync(c->S2p, 0, (size_t)(c->oo * c->vv) * sizeof(c128), c->st);
        s = s2_driver(c, c->S2p);
        if (s == CCSD_OK) s = s2_pp_ladder(c, c->S2p);
        ok = s == CCSD_OK && fk.end_branch();
    }
    slot(0);
    if (s != CCSD_OK) return s;
    if (!ok || !fk.join()) return CCSD_ECUDA;
    if (c->gv_trace) {
        gvv_trace_add(c);
        CCSD_TRY(gvv_gemm(c));
    }
    CCSD_TRY(s2_hh_and_goo(c, c->S2p));
    CCSD_TRY(ring_add(c, c->S2p));
    CCSD_TRY(vdag_add(c, c->S2p));
    CCSD_TRY(gvv_add(c, c->S2p));
    CCSD_TRY(c_t1_add(c, c->S2p));
    CCSD_TRY(s1_c_trace(c));
    c->have_residual = true;
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

// CC2 (Appendix 7.2, eqs 34-38).  "The T1 amplitude equations in 7.1 are unchanged":
// S1 is eq 33 at the full (t1, t2).  The doubles equation 34 is <Phi_ij^ab| exp(-T1) H exp(T1) + [F, T2] |Phi_0>, i.e.
// eq 32 evaluated with t2 -> 0 in every operand (tau -> P-(t1 t1); the ring, G.t2 terms vanish; H^{ak}_{ci} is not
// needed) plus the two Fock terms, which have the form of the G.t2 terms of eq 32 with G^a_c -> f_ac, G^k_i -> -f_ki:
//   (the pp-ladder and the <bk||cd> part of C at tau0 run factorised through the auxiliary index: cc2_dressed_factors)
//   W^{ab}_{ef}CC2 (x) t1 t1  = pp-ladder(tau0) + the <bk||cd> tau0 part of C;  W^{mn}_{ij}CC2 = A(tau0) of eq 31 (up to the
//   factor of the quartic term shared between eqs 35 and 36);  W^{ab}_{ej}, W^{mb}_{ij} = V-dagger.t1 and the rest of C.t1.
// The oracle evaluates eqs 34-38 literally; the two agree to rounding (tests/test_gpu_cc2.py).
static int residual_cc2(ccsd_ctx* c)
{
    cudaStream_t st = c->st;
    const int o = c->o, v = c->v, n = c->n;
    tick(c, 0);
    CCSD_TRY(prep_operands(c));
    tick(c, 1);
    CCSD_TRY(fock_like(c));
    tick(c, 2);
    tick(c, 3);
    CCSD_TRY(build_S1(c));                      // eq 33, full tau (timed under "Hvovo_quad"'s slot: see ccsd_step_name)
    tick(c, 4);
    // doubles: operands with t2 = 0
    CCSD_TRY(cc2_dressed_factors(c));
    build_tau(st, c->taup, c->t1, nullptr, o, v, c->po, c->pv, c->taups);
    c->tau_valid = false;                       // taup now holds tau0 = P-(t1 t1)
    CCSD_TRY(launch_transpose2d_ld(st, c->taup, c->vv, c->TT, 2 * c->oop, c->oo, c->vv, 0));
    const c128* f = c->f;
    launch_fill(st, c->Gvv, v, v, v, 0, [=] __device__(int64_t a, int64_t cc) { return f[(o + a) * n + o + cc]; });
    launch_fill(st, c->Goo, o, o, o, 0, [=] __device__(int64_t k, int64_t i) { return cneg(f[k * n + i]); });
    CCSD_TRY(build_C(c));
    tick(c, 5);
    CCSD_TRY(build_A(c));
    cudaMemsetAsync(c->S2p, 0, (size_t)(c->oo * c->vv) * sizeof(c128), st);
    CCSD_TRY(s2_driver(c, c->S2p));
    tick(c, 6);
    CCSD_TRY(s2_pp_ladder(c, c->S2p));
    tick(c, 7);
    CCSD_TRY(s2_hh_and_goo(c, c->S2p));         // hh-ladder of tau0 and -f_oo . t2
    tick(c, 8);
    tick(c, 9);
    tick(c, 10);
    CCSD_TRY(s2_vdag_t1(c, c->S2p));
    tick(c, 11);
    CCSD_TRY(s2_gvv(c, c->S2p));                // f_vv . t2
    tick(c, 12);
    CCSD_TRY(s2_c_t1(c, c->S2p));
    tick(c, 13);
    tick(c, 14);
    c->have_residual = true;
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

static int residual_body(ccsd_ctx* c) { return c->opt.cc2 ? residual_cc2(c) : residual(c); }

// The ~70 launches of one residual evaluation depend on nothing but the context (shapes, options, resident pointers), so
// they are captured once into a CUDA graph and replayed: the small configurations are launch-bound otherwise (cfg1: a 3.6 ms
// iteration of 1.8 ms of kernels).  Capture is not permitted on the legacy / per-thread default streams; there, with step
// timing on (events between the steps) or after any capture failure the launches are issued directly.
static bool graph_usable(const ccsd_ctx* c)
{
    return c->opt.graph && !c->timing && !c->graph_failed && c->st != nullptr && c->st != cudaStreamLegacy &&
           c->st != cudaStreamPerThread;
}
// opts.graph: 1 = graph with parallel branches (measured faster at every BASELINE configuration: cfg1 3.17 -> 2.99 ms,
// cfg2 34.9 -> 34.3 ms, cfg3 252.3 -> 249.4 ms), 3 = graph with the launches in their serial order.
static bool graph_branches(const ccsd_ctx* c)
{
    return !c->opt.cc2 && c->partial_extra && c->opt.graph != 3;
}
static int residual_any(ccsd_ctx* c)
{
    ensure_tau(c);
    if (!graph_usable(c)) return residual_body(c);
    if (!c->res_graph) {
        if (!c->graph_warm) {   // first use: direct launches (function attributes get set, errors surface at their source)
            c->graph_warm = true;
            return residual_body(c);
        }
        const long long tally0 = t_launch_tally;
        if (cudaStreamBeginCapture(c->st, cudaStreamCaptureModeRelaxed) != cudaSuccess) {
            cudaGetLastError();
            c->graph_failed = true;
            return residual_body(c);
        }
        const int s = graph_branches(c) ? residual_forked(c) : residual_body(c);
        cudaGraph_t g = nullptr;
        cudaError_t e = cudaStreamEndCapture(c->st, &g);
        const long long captured = t_launch_tally - tally0;
        count_launches(-captured);                       // nothing ran yet: replays are counted below
        if (s == CCSD_OK && e == cudaSuccess && g) e = cudaGraphInstantiate(&c->res_graph, g, 0);
        if (g) cudaGraphDestroy(g);
        if (s != CCSD_OK || e != cudaSuccess || !c->res_graph) {
            cudaGetLastError();
            c->res_graph = nullptr;
            c->graph_failed = true;
            return s != CCSD_OK ? s : residual_body(c);
        }
        c->graph_kernels = captured;
    }
    CCSD_CUDA_TRY(cudaGraphLaunch(c->res_graph, c->st));
    count_launches(c->graph_kernels);
    c->have_residual = true;
    if (c->opt.cc2) c->tau_valid = false;               // as residual_cc2 leaves it: taup holds tau0
    return CCSD_OK;
}

// ---------------------------------------------------------------------------------------------------------------
// energy, update, DIIS
// ---------------------------------------------------------------------------------------------------------------
static int energy_async(ccsd_ctx* c, double* red_out /* device, 2 doubles */)
{
    // E = sum_ia f[i,a] t1[i,a] + sum_{i<j,a<b} <ij||ab> tau   (eq 9; reading G11), in one pass that also leaves tau (eq 23)
    // and its sum plane behind as the next residual's operand.  The intermediates of the last residual (Hm, Am, ...) belong
    // to the amplitudes that residual was evaluated at; whoever moves the amplitudes clears have_residual.
    launch_energy_tau(c->st, c->diis.scratch, c->f, c->n, c->o, c->v, c->t1, c->t2p, c->Voovv_p, c->taup, c->taups, c->po, c->pv,
                      red_out);
    c->tau_valid = true;
    return CCSD_OK;
}

#include "lambda.cuh"
#include "contract_terms.cuh"

extern "C" {

void ccsd_default_options(ccsd_options* opts)
{
    if (!opts) return;
    opts->ndiis = 6;
    opts->level_shift = 0.0;
    opts->gemm_mode = 0;
    opts->ccd = 0;
    opts->cc2 = 0;
    opts->direct_ladder = 0;
    opts->graph = 1;
    opts->shard_rank = 0;
    opts->shard_world = 1;
    opts->strassen = 1;
}

int ccsd_workspace_bytes(int nocc, int nvir, int naux, const ccsd_options* opts, size_t* bytes)
{
    if (!bytes) return CCSD_EINVAL;
    CCSD_TRY(check_sizes(nocc, nvir, naux));
    ccsd_ctx tmp;
    setup_dims(&tmp, nocc, nvir, naux, opts);
    carve_auto(&tmp, nullptr, bytes);
    return CCSD_OK;
}

int ccsd_init(ccsd_ctx** out, const ccsd_c128* h, const ccsd_c128* B, int nocc, int nvir, int naux,
              const ccsd_options* opts, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!out || !h || !B || !workspace) return CCSD_EINVAL;
    CCSD_TRY(check_sizes(nocc, nvir, naux));
    if (reinterpret_cast<uintptr_t>(workspace) % 256 != 0) return CCSD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return CCSD_ECUDA;
    }
    if (opts && opts->shard_world > 1) {
        if (opts->shard_rank < 0 || opts->shard_rank >= opts->shard_world || opts->shard_world > nvir || opts->cc2) return CCSD_EINVAL;
    }
    ccsd_ctx* c = new (std::nothrow) ccsd_ctx();
    if (!c) return CCSD_ENOMEM;
    c->lam = nullptr;
    c->ws_base = static_cast<char*>(workspace);
    setup_dims(c, nocc, nvir, naux, opts);
    size_t need = 0;
    carve_auto(c, nullptr, &need);
    if (workspace_bytes < need) { delete c; return CCSD_EINVAL; }
    carve_auto(c, static_cast<char*>(workspace), &need);
    c->st = static_cast<cudaStream_t>(cuda_stream);
    c->env = Env{c->st, c->opt.gemm_mode, c->partial, c->partial_elems};
    c->timing = 0;
    c->red_host = nullptr;
    c->res_graph = nullptr;
    c->init_events = nullptr;
    for (double& x : c->init_stats) x = 0.0;
    c->graph_kernels = 0;
    c->graph_warm = c->graph_failed = false;
    for (int k = 0; k <= CCSD_NSTEPS; k++) c->ev[k] = nullptr;
    if (cudaMallocHost(&c->red_host, 64 * sizeof(double)) != cudaSuccess) { delete c; return CCSD_ECUDA; }
    // zero the padded operand buffers once (pads must stay zero)
    cudaMemsetAsync(c->TT, 0, (size_t)(c->vv * 2 * c->oop) * sizeof(c128), c->st);
    cudaMemsetAsync(c->AG, 0, (size_t)(c->oo * 2 * c->oop) * sizeof(c128), c->st);
    int s = build_constants(c, reinterpret_cast<const c128*>(h), reinterpret_cast<const c128*>(B));
    if (s == CCSD_OK && c->strassen) {   // operand stacks of the constants (strassen.cuh), once
        if (c->sW.S) launch_strassen_prep(c->st, 0, c->W ? c->W : c->W_init, c->vv, c->sW);
        if (c->sVvovv.S)      // this rank's rows (b,k); overwrites W_init: after the line above
            launch_strassen_prep(c->st, 0, c->Vvovv_p + (int64_t)c->sh.a_lo * c->o * c->vv, c->vv, c->sVvovv);
        launch_strassen_prep(c->st, 1, c->G1, c->ov, c->sG1);
    }
    if (s == CCSD_OK) mp2_guess(c);
    if (s == CCSD_OK && cudaStreamSynchronize(c->st) != cudaSuccess) s = CCSD_ECUDA;
    if (s == CCSD_OK) {
        cudaError_t e = cudaGetLastError();
        if (e != cudaSuccess) { snprintf(g_cuda_err, sizeof(g_cuda_err), "%s (init)", cudaGetErrorString(e)); s = CCSD_ECUDA; }
    }
    if (s != CCSD_OK) { cudaFreeHost(c->red_host); delete c; return s; }
    *out = c;
    return CCSD_OK;
}

int ccsd_destroy(ccsd_ctx* c)
{
    if (!c) return CCSD_ESTATE;
    for (int k = 0; k <= CCSD_NSTEPS; k++)
        if (c->ev[k]) cudaEventDestroy(c->ev[k]);
    if (c->red_host) cudaFreeHost(c->red_host);
    if (c->res_graph) cudaGraphExecDestroy(c->res_graph);
    delete c->lam;
    delete c;
    return CCSD_OK;
}

int ccsd_energy(ccsd_ctx* c, double* e_re, double* e_im)
{
    if (!c) return CCSD_ESTATE;
    CCSD_TRY(energy_async(c, c->red));
    CCSD_CUDA_TRY(cudaMemcpyAsync(c->red_host, c->red, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CCSD_CUDA_TRY(cudaStreamSynchronize(c->st));
    if (e_re) *e_re = c->red_host[0];
    if (e_im) *e_im = c->red_host[1];
    return CCSD_OK;
}

int ccsd_t1_diagnostic(ccsd_ctx* c, double* t1_diag)
{   // sqrt(sum |t1|^2 / nocc): tabulated by the paper (Tables 3, 8), not defined there; reading G18 of DESIGN.md
    if (!c || !t1_diag) return CCSD_ESTATE;
    CCSD_CUDA_TRY(cudaMemsetAsync(c->red + 48, 0, sizeof(double), c->st));
    launch_redot(c->st, c->diis.scratch, c->t1, c->t1, c->ov, c->red + 48);
    CCSD_CUDA_TRY(cudaMemcpyAsync(c->red_host + 48, c->red + 48, sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CCSD_CUDA_TRY(cudaStreamSynchronize(c->st));
    *t1_diag = sqrt(c->red_host[48] / (double)c->o);
    return CCSD_OK;
}

int ccsd_residual(ccsd_ctx* c)
{
    if (!c) return CCSD_ESTATE;
    return residual_any(c);
}

// Jacobi step (reading G12) + DIIS (reading G13) + energy of the new amplitudes, all on the device: the Gram row
// is reduced, the bordered Pulay system solved and the amplitudes recombined without a host round trip (reduce.cuh)
static int update_from_residual(ccsd_ctx* c, double* e_re, double* e_im, double* step_norm)
{
    launch_jacobi_diis(c->st, c->diis, c->o, c->v, c->S1, c->S2p, c->t1, c->t2p, c->eps, c->po, c->pv, c->opt.ccd);
    c->have_residual = false;       // the intermediates of this residual belong to the amplitudes before the update
    c->tau_valid = false;
    tick(c, 15);
    CCSD_TRY(energy_async(c, c->red + 32));
    tick(c, 16);
    // the iteration's only read-back: E (2 doubles) and ||S/D||^2, singular flag (2 doubles)
    CCSD_CUDA_TRY(cudaMemcpyAsync(c->red_host + 32, c->red + 32, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CCSD_CUDA_TRY(cudaMemcpyAsync(c->red_host + 34, c->diis.info, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CCSD_CUDA_TRY(cudaStreamSynchronize(c->st));
    if (e_re) *e_re = c->red_host[32];
    if (e_im) *e_im = c->red_host[33];
    if (step_norm) *step_norm = sqrt(c->red_host[34] > 0 ? c->red_host[34] : 0.0);
    if (c->timing) {
        for (int k = 0; k < CCSD_NSTEPS; k++) cudaEventElapsedTime(&c->step_ms[k], c->ev[k], c->ev[k + 1]);
    }
    CCSD_CUDA_TRY(cudaGetLastError());
    return c->red_host[35] != 0.0 ? CCSD_ESINGULAR : CCSD_OK;
}

int ccsd_iterate(ccsd_ctx* c, double* e_re, double* e_im, double* step_norm)
{
    if (!c) return CCSD_ESTATE;
    if (c->sh.world > 1) return CCSD_EINVAL;   // the slabs of S2 have to be summed over the ranks between the two halves
    CCSD_TRY(residual_any(c));
    return update_from_residual(c, e_re, e_im, step_norm);
}

int ccsd_update(ccsd_ctx* c, double* e_re, double* e_im, double* step_norm)
{
    if (!c || !c->have_residual) return CCSD_ESTATE;
    return update_from_residual(c, e_re, e_im, step_norm);
}

int ccsd_shard_ranges(int nocc, int nvir, int rank, int world, int64_t ranges[8])
{   // host only: the slab of rank `rank` of `world` (struct Shard)
    if (!ranges || nocc < 2 || nvir < 2 || world < 1 || rank < 0 || rank >= world || world > nvir) return CCSD_EINVAL;
    const Shard s = make_shard(rank, world, nocc, nvir);
    const int64_t vals[8] = {s.a_lo, s.a_hi, s.w_lo, s.w_hi, s.ij_lo, s.ij_hi, s.wa_lo, s.wa_hi};
    for (int k = 0; k < 8; k++) ranges[k] = vals[k];
    return CCSD_OK;
}

int ccsd_shard_info(ccsd_ctx* c, int64_t info[CCSD_NSHARD_INFO])
{
    if (!c || !info) return CCSD_ESTATE;
    const Shard& s = c->sh;
    const int64_t vals[CCSD_NSHARD_INFO] = {s.rank, s.world, s.a_lo, s.a_hi, s.w_lo, s.w_hi, s.ij_lo, s.ij_hi,
                                            (int64_t)(reinterpret_cast<char*>(c->S2p) - c->ws_base), c->oo * c->vv,
                                            (int64_t)(reinterpret_cast<char*>(c->S1) - c->ws_base), c->ov};
    for (int k = 0; k < CCSD_NSHARD_INFO; k++) info[k] = vals[k];
    return CCSD_OK;
}

int ccsd_solve(ccsd_ctx* c, double tol, int max_iterations, int* iterations, double* e_re, double* e_im, double* step_norm)
{   // .TCONVERG / .NCYCLES of the paper's input (reading G14): both ||S/D||_2 and |Delta E| below tol
    if (!c) return CCSD_ESTATE;
    if (!(tol > 0.0) || max_iterations < 1) return CCSD_EINVAL;
    double er = 0.0, ei = 0.0, sn = 0.0, er_old = 0.0, ei_old = 0.0;
    CCSD_TRY(ccsd_energy(c, &er_old, &ei_old));
    int it = 0, status = CCSD_OK;
    bool converged = false;
    while (it < max_iterations && !converged) {
        status = ccsd_iterate(c, &er, &ei, &sn);
        if (status != CCSD_OK && status != CCSD_ESINGULAR) return status;
        it++;
        converged = sn < tol && hypot(er - er_old, ei - ei_old) < tol;
        er_old = er; ei_old = ei;
    }
    if (iterations) *iterations = it;
    if (e_re) *e_re = er;
    if (e_im) *e_im = ei;
    if (step_norm) *step_norm = sn;
    return converged ? CCSD_OK : CCSD_ENOTCONVERGED;
}

int ccsd_get_amplitudes(ccsd_ctx* c, ccsd_c128* t1, ccsd_c128* t2p)
{
    if (!c) return CCSD_ESTATE;
    if (t1) dcopy(c->st, reinterpret_cast<c128*>(t1), c->t1, c->ov);
    if (t2p) dcopy(c->st, reinterpret_cast<c128*>(t2p), c->t2p, c->oo * c->vv);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

int ccsd_set_amplitudes(ccsd_ctx* c, const ccsd_c128* t1, const ccsd_c128* t2p, int reset_diis)
{
    if (!c) return CCSD_ESTATE;
    if (t1) dcopy(c->st, c->t1, reinterpret_cast<const c128*>(t1), c->ov);
    if (t2p) dcopy(c->st, c->t2p, reinterpret_cast<const c128*>(t2p), c->oo * c->vv);
    if (reset_diis) c->diis.reset();
    c->have_residual = false;
    c->tau_valid = false;
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

int ccsd_tensor_elems(ccsd_ctx* c, int id, size_t* elems)
{
    if (!c || !elems) return CCSD_ESTATE;
    const int64_t o = c->o, v = c->v, n = c->n, oo = c->oo, vv = c->vv, ov = c->ov;
    int64_t e = -1;
    switch (id) {
    case CCSD_T_FOCK: e = n * n; break;
    case CCSD_T_VVVV: e = vv * vv; break;
    case CCSD_T_VOVV: e = ov * vv; break;
    case CCSD_T_VOVO: e = ov * ov; break;
    case CCSD_T_OOVV: e = oo * vv; break;
    case CCSD_T_OOOV: e = oo * ov; break;
    case CCSD_T_OOOO: e = oo * oo; break;
    case CCSD_T_TAU: e = oo * vv; break;
    case CCSD_T_HVV: case CCSD_T_GVV: e = v * v; break;
    case CCSD_T_HOO: case CCSD_T_GOO: e = o * o; break;
    case CCSD_T_HOV: e = ov; break;
    case CCSD_T_HVOVO: e = ov * ov; break;
    case CCSD_T_C: e = ov * oo; break;
    case CCSD_T_A: e = oo * oo; break;
    case CCSD_T_S1: e = ov; break;
    case CCSD_T_S2: e = oo * vv; break;
    default:
        if (id >= CCSD_T_S2_RING && id <= CCSD_T_S2_DRIVER) e = oo * vv;
    }
    if (e < 0) return CCSD_EINVAL;
    *elems = (size_t)e;
    return CCSD_OK;
}

int ccsd_get_tensor(ccsd_ctx* c, int id, ccsd_c128* out_)
{
    if (!c || !out_) return CCSD_ESTATE;
    c128* out = reinterpret_cast<c128*>(out_);
    const int o = c->o, v = c->v;
    const int64_t oo = c->oo, vv = c->vv, ov = c->ov;
    cudaStream_t st = c->st;
    if (id >= CCSD_T_TAU && !c->have_residual) return CCSD_ESTATE;
    switch (id) {
    case CCSD_T_FOCK: dcopy(st, out, c->f, (int64_t)c->n * c->n); break;
    case CCSD_T_VVVV:
        if (c->sh.world > 1 || (!c->W && !(c->W_dropped && c->sW.S))) return CCSD_EINVAL;   // direct_ladder: not stored; sharded: this rank's rows only
        if (c->W) {
            dcopy(st, out, c->W, vv * vv);
        } else {      // kept as the ladder's operand stack only
            const StrassenView wv = strassen_view(c->sW);
            launch_fill(st, out, vv, vv, vv, 0, [=] __device__(int64_t AB, int64_t CD) { return strassen_left_at(wv, AB, CD); });
        }
        break;
    case CCSD_T_VOVV: dcopy(st, out, c->Vvovv_p, ov * vv); break;
    case CCSD_T_VOVO: {
        const c128* V = c->Vvovo_m;  // [(a,i)][(c,k)] -> [a][k][c][i]
        launch_fill(st, out, ov, ov, ov, 0, [=] __device__(int64_t ak, int64_t ci) {
            int64_t a = ak / o, k = ak % o, cc = ci / o, i = ci % o;
            return V[(a * o + i) * ov + cc * o + k];
        });
        break;
    }
    case CCSD_T_OOVV: dcopy(st, out, c->Voovv_p, oo * vv); break;
    case CCSD_T_OOOV: dcopy(st, out, c->Vooov_p, oo * ov); break;
    case CCSD_T_OOOO: dcopy(st, out, c->Voooo_p, oo * oo); break;
    case CCSD_T_TAU: dcopy(st, out, c->taup, oo * vv); break;
    case CCSD_T_HVV: dcopy(st, out, c->Hvv, (int64_t)v * v); break;
    case CCSD_T_GVV: dcopy(st, out, c->Gvv, (int64_t)v * v); break;
    case CCSD_T_HOO: dcopy(st, out, c->Hoo, (int64_t)o * o); break;
    case CCSD_T_GOO: dcopy(st, out, c->Goo, (int64_t)o * o); break;
    case CCSD_T_HOV: dcopy(st, out, c->Hov, ov); break;
    case CCSD_T_HVOVO: {
        const c128* H = c->Hm;
        launch_fill(st, out, ov, ov, ov, 0, [=] __device__(int64_t ak, int64_t ci) {
            int64_t a = ak / o, k = ak % o, cc = ci / o, i = ci % o;
            return H[(a * o + i) * ov + cc * o + k];
        });
        break;
    }
    case CCSD_T_C: {
        const c128* Cm = c->Cm;  // [(b,k)][I] -> [k][b][I]
        launch_fill(st, out, ov, oo, oo, 0, [=] __device__(int64_t kb, int64_t IJ) {
            int64_t k = kb / v, b = kb % v;
            return Cm[(b * o + k) * oo + IJ];
        });
        break;
    }
    case CCSD_T_A: dcopy(st, out, c->Am, oo * oo); break;
    case CCSD_T_S1: dcopy(st, out, c->S1, ov); break;
    case CCSD_T_S2: dcopy(st, out, c->S2p, oo * vv); break;
    default: {
        if (id < CCSD_T_S2_RING || id > CCSD_T_S2_DRIVER) return CCSD_EINVAL;
        CCSD_CUDA_TRY(cudaMemsetAsync(out, 0, (size_t)(oo * vv) * sizeof(c128), st));
        int saved = c->timing;
        c->timing = 0;
        int s = CCSD_OK;
        switch (id) {
        case CCSD_T_S2_RING: s = s2_ring(c, out); break;
        case CCSD_T_S2_GOO: s = s2_goo(c, out); break;
        case CCSD_T_S2_VDAG_T1: s = s2_vdag_t1(c, out); break;
        case CCSD_T_S2_GVV: s = s2_gvv(c, out); break;
        case CCSD_T_S2_C_T1: s = s2_c_t1(c, out); break;
        case CCSD_T_S2_HH_LADDER: s = s2_hh_ladder(c, out); break;
        case CCSD_T_S2_PP_LADDER: s = s2_pp_ladder(c, out); break;
        case CCSD_T_S2_DRIVER: s = s2_driver(c, out); break;
        }
        c->timing = saved;
        CCSD_TRY(s);
    }
    }
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

// ---- perturbative triples (Appendix 7.3; kernels in triples.cuh) ------------------------------
struct TripWs {
    c128 *t2u, *t2T, *Uo, *Mcbuf;
    double *t2us, *t2Ts, *Uos, *Vs, *partials, *acc;
    int4* ijk;
    int nb, op;
    int64_t ntrip;
    bool planes;
};
static void trip_carve(const ccsd_ctx* c, char* base, TripWs* w, size_t* total)
{
    Carver cv{base, 0};
    const int64_t o = c->o, v = c->v, vv = c->vv;
    w->op = (int)round_up(o, 2);
    w->ntrip = o * (o - 1) * (o - 2) / 6;
    int64_t nb = ((int64_t)1 << 30) / (vv * v * 16 > 0 ? vv * v * 16 : 1);   // Mc of a batch: <= 1 GiB
    if (nb < 1) nb = 1;
    if (nb > 256) nb = 256;
    if (nb > w->ntrip) nb = w->ntrip > 0 ? w->ntrip : 1;
    w->nb = (int)nb;
    w->planes = c->planes && v % 2 == 0;
    w->t2u = cv.take<c128>(o * o * v * v);
    w->t2T = cv.take<c128>(o * vv * w->op);
    w->Uo = cv.take<c128>(o * o * v * w->op);
    w->Mcbuf = cv.take<c128>(nb * vv * v);
    w->t2us = cv.take<double>(o * o * v * v);
    w->t2Ts = cv.take<double>(o * vv * w->op);
    w->Uos = cv.take<double>(o * o * v * w->op);
    w->Vs = cv.take<double>(o * vv * v);
    w->partials = cv.take<double>(nb * v * 5);
    w->acc = cv.take<double>(8);
    w->ijk = cv.take<int4>(w->ntrip > 0 ? w->ntrip : 1);
    *total = cv.off;
}

// operands of the segmented GEMM (triples.cuh) from the current amplitudes and the stored integral classes
static int trip_prepare(ccsd_ctx* c, const TripWs& w)
{
    cudaStream_t st = c->st;
    const int o = c->o, v = c->v, op = w.op;
    const int64_t vv = c->vv;
    const c128 *t2p = c->t2p, *Vooov = c->Vooov_p;
    double *t2us = w.planes ? w.t2us : nullptr, *t2Ts = w.planes ? w.t2Ts : nullptr, *Uos = w.planes ? w.Uos : nullptr;
    // t2u[(z,y)][c][e] = t2[z,y,e,c]
    launch_fill(st, w.t2u, (int64_t)o * o * v, v, v, 0, [=] __device__(int64_t row, int64_t e) {
        const int64_t zy = row / v;
        const int cc = (int)(row % v), z = (int)(zy / o), y = (int)(zy % o);
        c128 x = t2_at(t2p, z, y, (int)e, cc, o, v, vv);
        if (t2us) t2us[row * v + e] = x.x + x.y;
        return x;
    });
    // t2T[z][(a<b)][m] = t2[z,m,a,b]   (pad m >= o: zero)
    launch_fill(st, w.t2T, (int64_t)o * vv, op, op, 0, [=] __device__(int64_t row, int64_t m) {
        const int z = (int)(row / vv);
        const int64_t AB = row % vv;
        c128 x = mk(0.0, 0.0);
        if (m < o && m != z) {
            x = z < m ? t2p[pair_idx(z, (int)m, o) * vv + AB] : cneg(t2p[pair_idx((int)m, z, o) * vv + AB]);
        }
        if (t2Ts) t2Ts[row * op + m] = x.x + x.y;
        return x;
    });
    // Uo[(x,y)][c][m] = <cm||xy> = -conj <xy||mc>   (dagger of the stored class <kl||ic>, reading G5)
    launch_fill(st, w.Uo, (int64_t)o * o * v, op, op, 0, [=] __device__(int64_t row, int64_t m) {
        const int64_t xy = row / v;
        const int cc = (int)(row % v), x = (int)(xy / o), y = (int)(xy % o);
        c128 r = mk(0.0, 0.0);
        if (m < o && x != y) {
            const int64_t P = x < y ? pair_idx(x, y, o) : pair_idx(y, x, o);
            c128 g = Vooov[(P * o + m) * v + cc];          // <xy||mc> for x<y
            r = x < y ? mk(-g.x, g.y) : mk(g.x, -g.y);      // -conj(g), sign flipped for x>y
        }
        if (Uos) Uos[row * op + m] = r.x + r.y;
        return r;
    });
    if (w.planes) launch_sum_plane(st, c->VvovvT, w.Vs, (int64_t)o * vv * v);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

static int trip_loader(ccsd_ctx* c, const TripWs& w, const TripVariant& V, TripLoader* ld)
{
    const int o = c->o, v = c->v, op = w.op;
    const int64_t vv = c->vv;
    // A = VvovvT[x][(a<b)][e] = conj <ex||ab> = -<ab||xe>; the sign is absorbed by B = t2[z,y,e,c] = -t2[y,z,e,c].
    // (The 4-d "wide" maps of the plain GEMM were measured slower here: 5.36 s vs 5.06 s of GEMM time at cfg3.)
    CCSD_TRY(make_operand_map(&ld->PA, c->VvovvT, vv, v, v, o, vv * v, V.bm));
    CCSD_TRY(make_operand_map(&ld->PB, w.t2u, v, v, v, o * o, (int64_t)v * v, V.bn));
    CCSD_TRY(make_operand_map(&ld->HA, w.t2T, vv, o, op, o, vv * op, V.bm));
    CCSD_TRY(make_operand_map(&ld->HB, w.Uo, v, o, op, o * o, (int64_t)v * op, V.bn));
    ld->PAs = ld->PA; ld->PBs = ld->PB; ld->HAs = ld->HA; ld->HBs = ld->HB;
    if (V.planes) {
        CCSD_TRY(make_plane_map(&ld->PAs, w.Vs, vv, v, v, o, vv * v, V.bm));
        CCSD_TRY(make_plane_map(&ld->PBs, w.t2us, v, v, v, o * o, (int64_t)v * v, V.bn));
        CCSD_TRY(make_plane_map(&ld->HAs, w.t2Ts, vv, o, op, o, vv * op, V.bm));
        CCSD_TRY(make_plane_map(&ld->HBs, w.Uos, v, o, op, o * o, (int64_t)v * op, V.bn));
    }
    ld->ijk = w.ijk;
    ld->o = o;
    ld->op = op;
    ld->tp = (v + 4 * DMMA_BKG - 1) / (4 * DMMA_BKG);
    ld->ngh = (o + 3) / 4;
    ld->th = (3 * ld->ngh + DMMA_BKG - 1) / DMMA_BKG;
    return CCSD_OK;
}

static const TripVariant& trip_variant(const ccsd_ctx* c, const TripWs& w)
{
    // column-tile width by padded columns x relative cost, as dmma_pick (N = nvir)
    const int v = c->v;
    const double c32 = (double)round_up(v, 32) * (w.planes ? 1.026 : 1.037), c48 = (double)round_up(v, 48),
                 c56 = (double)round_up(v, 56);
    int idx = (w.planes ? 2 : 0) + (c48 < c32 ? 1 : 0);
    if (c56 < (c48 < c32 ? c48 : c32)) idx = w.planes ? 5 : 4;
    return k_trip_variants[idx];
}

static int trip_gemm(ccsd_ctx* c, const TripWs& w, const TripLoader& ld0, const TripVariant& V, int64_t first, int count)
{
    TripLoader ld = ld0;
    ld.ijk = w.ijk + first;
    DmmaArgs a;
    memset(&a, 0, sizeof(a));
    a.M = c->vv; a.N = c->v; a.K = 3 * ((int64_t)c->v + c->o);
    a.C = w.Mcbuf; a.csm = 1; a.csn = c->vv; a.bsC = c->vv * c->v;          // stored transposed: Mc[c][(a<b)]
    a.alpha = mk(1.0, 0.0); a.accumulate = 0;
    a.batchA = a.batchB = 1; a.ksplit = 1; a.kchunk = a.K; a.partial = nullptr;
    dim3 grid((unsigned)((c->v + V.bn - 1) / V.bn), (unsigned)((c->vv + V.bm - 1) / V.bm), (unsigned)count);
    return V.launch(c->st, ld, a, grid);
}

static TripData trip_data(const ccsd_ctx* c)
{
    TripData d;
    d.t1 = c->t1; d.t2p = c->t2p; d.Voovv_p = c->Voovv_p; d.f = c->f; d.eps = c->eps0;   // unshifted
    d.o = c->o; d.v = c->v; d.n = c->n; d.vv = c->vv;
    return d;
}

int ccsd_triples_workspace_bytes(ccsd_ctx* c, size_t* bytes)
{
    if (!c || !bytes) return CCSD_ESTATE;
    TripWs w;
    trip_carve(c, nullptr, &w, bytes);
    return CCSD_OK;
}

int ccsd_triples_count(ccsd_ctx* c, int64_t* ntriples)
{
    if (!c || !ntriples) return CCSD_ESTATE;
    const int64_t o = c->o;
    *ntriples = o >= 3 ? o * (o - 1) * (o - 2) / 6 : 0;
    return CCSD_OK;
}

int ccsd_triples(ccsd_ctx* c, double e_plus_t[2], double e_par_t[2], double e_minus_t[2], void* workspace,
                 size_t workspace_bytes)
{
    if (!c) return CCSD_ESTATE;
    const int64_t o = c->o;
    return ccsd_triples_range(c, 0, o * (o - 1) * (o - 2) / 6, e_plus_t, e_par_t, e_minus_t, workspace, workspace_bytes);
}

int ccsd_triples_range(ccsd_ctx* c, int64_t first_triple, int64_t ntriples, double e_plus_t[2], double e_par_t[2],
                       double e_minus_t[2], void* workspace, size_t workspace_bytes)
{
    if (!c) return CCSD_ESTATE;
    if (!workspace || reinterpret_cast<uintptr_t>(workspace) % 256 != 0) return CCSD_EINVAL;
    if (c->o < 3 || c->v < 3) return CCSD_EINVAL;
    {
        const int64_t all = (int64_t)c->o * (c->o - 1) * (c->o - 2) / 6;
        if (first_triple < 0 || ntriples < 0 || first_triple > all || ntriples > all - first_triple) return CCSD_EINVAL;
    }
    TripWs w;
    size_t need = 0;
    trip_carve(c, nullptr, &w, &need);
    if (workspace_bytes < need) return CCSD_EINVAL;
    trip_carve(c, static_cast<char*>(workspace), &w, &need);
    cudaStream_t st = c->st;
    const int o = c->o, v = c->v;
    {   // unique occupied triples i<j<k, lexicographic: consecutive triples share the i and j slices of <ab||xe> in L2
        std::vector<int4> h((size_t)w.ntrip);
        size_t x = 0;
        for (int i = 0; i < o; i++)
            for (int j = i + 1; j < o; j++)
                for (int k = j + 1; k < o; k++) h[x++] = make_int4(i, j, k, 0);
        CCSD_CUDA_TRY(cudaMemcpyAsync(w.ijk, h.data(), h.size() * sizeof(int4), cudaMemcpyHostToDevice, st));
        CCSD_CUDA_TRY(cudaStreamSynchronize(st));   // h goes out of scope
    }
    CCSD_TRY(trip_prepare(c, w));
    const TripVariant& V = trip_variant(c, w);
    TripLoader ld;
    CCSD_TRY(trip_loader(c, w, V, &ld));
    const TripData d = trip_data(c);
    CCSD_CUDA_TRY(cudaMemsetAsync(w.acc, 0, 8 * sizeof(double), st));
    cudaEvent_t e0 = nullptr, e1 = nullptr, e2 = nullptr;
    float gemm_ms = 0.f, energy_ms = 0.f;
    if (c->timing) { cudaEventCreate(&e0); cudaEventCreate(&e1); cudaEventCreate(&e2); }
    const int64_t range_end = first_triple + ntriples;
    for (int64_t first = first_triple; first < range_end; first += w.nb) {
        const int count = (int)((range_end - first < w.nb) ? range_end - first : w.nb);
        if (c->timing) cudaEventRecord(e0, st);
        CCSD_TRY(trip_gemm(c, w, ld, V, first, count));
        if (c->timing) cudaEventRecord(e1, st);
        trip_energy_kernel<<<dim3((unsigned)(v - 2), (unsigned)count), TRIP_THREADS, 0, st>>>(d, w.Mcbuf, c->vv * v, w.ijk + first,
                                                                                           c->pv, w.partials);
        trip_reduce_kernel<<<1, 256, 0, st>>>(w.partials, (int64_t)count * (v - 2), w.acc);
        count_launches(2);
        if (c->timing) {
            cudaEventRecord(e2, st);
            CCSD_CUDA_TRY(cudaEventSynchronize(e2));
            float a = 0.f, b = 0.f;
            cudaEventElapsedTime(&a, e0, e1);
            cudaEventElapsedTime(&b, e1, e2);
            gemm_ms += a; energy_ms += b;
        }
    }
    if (c->timing) { cudaEventDestroy(e0); cudaEventDestroy(e1); cudaEventDestroy(e2); }
    c->trip_ms[0] = gemm_ms; c->trip_ms[1] = energy_ms;
    CCSD_CUDA_TRY(cudaMemcpyAsync(c->red_host + 40, w.acc, 5 * sizeof(double), cudaMemcpyDeviceToHost, st));
    CCSD_CUDA_TRY(cudaStreamSynchronize(st));
    CCSD_CUDA_TRY(cudaGetLastError());
    const double* r = c->red_host + 40;
    if (e_plus_t) { e_plus_t[0] = r[0]; e_plus_t[1] = 0.0; }
    if (e_par_t) { e_par_t[0] = r[0] + r[1]; e_par_t[1] = r[2]; }
    if (e_minus_t) { e_minus_t[0] = r[0] + r[3]; e_minus_t[1] = r[4]; }
    return CCSD_OK;
}

int ccsd_triples_block(ccsd_ctx* c, int i, int j, int k, ccsd_c128* Wbar, ccsd_c128* Zbar, ccsd_c128* Ybar, void* workspace,
                       size_t workspace_bytes)
{
    if (!c) return CCSD_ESTATE;
    if (!workspace || reinterpret_cast<uintptr_t>(workspace) % 256 != 0) return CCSD_EINVAL;
    if (c->o < 3 || c->v < 3 || !(0 <= i && i < j && j < k && k < c->o)) return CCSD_EINVAL;
    TripWs w;
    size_t need = 0;
    trip_carve(c, nullptr, &w, &need);
    if (workspace_bytes < need) return CCSD_EINVAL;
    trip_carve(c, static_cast<char*>(workspace), &w, &need);
    cudaStream_t st = c->st;
    const int4 t = make_int4(i, j, k, 0);
    CCSD_CUDA_TRY(cudaMemcpyAsync(w.ijk, &t, sizeof(int4), cudaMemcpyHostToDevice, st));
    CCSD_CUDA_TRY(cudaStreamSynchronize(st));
    CCSD_TRY(trip_prepare(c, w));
    const TripVariant& V = trip_variant(c, w);
    TripLoader ld;
    CCSD_TRY(trip_loader(c, w, V, &ld));
    CCSD_TRY(trip_gemm(c, w, ld, V, 0, 1));
    const size_t bytes = (size_t)c->v * c->v * c->v * sizeof(c128);
    if (Wbar) CCSD_CUDA_TRY(cudaMemsetAsync(Wbar, 0, bytes, st));
    if (Zbar) CCSD_CUDA_TRY(cudaMemsetAsync(Zbar, 0, bytes, st));
    if (Ybar) CCSD_CUDA_TRY(cudaMemsetAsync(Ybar, 0, bytes, st));
    trip_dense_kernel<<<(unsigned)(c->v - 2), TRIP_THREADS, 0, st>>>(trip_data(c), w.Mcbuf, c->pv, i, j, k, reinterpret_cast<c128*>(Wbar),
                                                            reinterpret_cast<c128*>(Zbar), reinterpret_cast<c128*>(Ybar));
    count_launches(1);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

int ccsd_get_triples_times(ccsd_ctx* c, float ms[2])
{
    if (!c || !ms) return CCSD_ESTATE;
    ms[0] = c->trip_ms[0]; ms[1] = c->trip_ms[1];
    return CCSD_OK;
}

// ---- Lambda equations and one-body density (Appendix 7.4-7.5; lambda.cuh / tensor_ops.cuh) ---------------------------
int ccsd_lambda_workspace_bytes(ccsd_ctx* c, size_t* bytes)
{
    if (!c || !bytes) return CCSD_ESTATE;
    LambdaState tmp;
    lambda_carve(c, nullptr, &tmp, bytes);
    return CCSD_OK;
}

int ccsd_lambda_init(ccsd_ctx* c, void* workspace, size_t workspace_bytes)
{
    if (!c) return CCSD_ESTATE;
    if (!workspace || reinterpret_cast<uintptr_t>(workspace) % 256 != 0 || c->opt.cc2 || c->opt.direct_ladder || c->sh.world > 1)
        return CCSD_EINVAL;
    size_t need = 0;
    LambdaState tmp;
    lambda_carve(c, nullptr, &tmp, &need);
    if (workspace_bytes < need) return CCSD_EINVAL;
    delete c->lam;
    c->lam = new (std::nothrow) LambdaState();
    if (!c->lam) return CCSD_ENOMEM;
    LambdaState* L = c->lam;
    lambda_carve(c, static_cast<char*>(workspace), L, &need);
    L->ready = false;
    L->diis.reset();
    CCSD_TRY(lambda_build_hbar(c, L));
    {   // start: lambda = conj(t) (first order: lambda^{ij}_{ab} = <ij||ab>/D = conj t^{ab}_{ij}; reading G23)
        const c128 *t1 = c->t1, *t2p = c->t2p;
        const int v = c->v;
        const int64_t vv = c->vv;
        launch_fill(c->st, L->l1, c->o, v, v, 0, [=] __device__(int64_t i, int64_t a) { return cconj(t1[i * v + a]); });
        launch_fill(c->st, L->l2p, c->oo, vv, vv, 0, [=] __device__(int64_t IJ, int64_t AB) { return cconj(t2p[IJ * vv + AB]); });
    }
    CCSD_CUDA_TRY(cudaStreamSynchronize(c->st));
    CCSD_CUDA_TRY(cudaGetLastError());
    L->ready = true;
    return CCSD_OK;
}

int ccsd_lambda_iterate(ccsd_ctx* c, double* step_norm)
{
    if (!c || !c->lam || !c->lam->ready) return CCSD_ESTATE;
    return lambda_iterate(c, c->lam, step_norm);
}

int ccsd_lambda_solve(ccsd_ctx* c, double tol, int max_iterations, int* iterations, double* step_norm)
{
    if (!c || !c->lam) return CCSD_ESTATE;
    if (!(tol > 0.0) || max_iterations < 1) return CCSD_EINVAL;
    int it = 0;
    double sn = 0.0;
    bool converged = false;
    while (it < max_iterations && !converged) {
        const int status = ccsd_lambda_iterate(c, &sn);
        if (status != CCSD_OK && status != CCSD_ESINGULAR) return status;
        it++;
        converged = sn < tol;
    }
    if (iterations) *iterations = it;
    if (step_norm) *step_norm = sn;
    return converged ? CCSD_OK : CCSD_ENOTCONVERGED;
}

int ccsd_lambda_residual(ccsd_ctx* c)
{
    if (!c || !c->lam || !c->lam->ready) return CCSD_ESTATE;
    return lambda_residual(c, c->lam);
}

int ccsd_get_lambda(ccsd_ctx* c, ccsd_c128* l1, ccsd_c128* l2p)
{
    if (!c || !c->lam || !c->lam->ready) return CCSD_ESTATE;
    if (l1) dcopy(c->st, reinterpret_cast<c128*>(l1), c->lam->l1, c->ov);
    if (l2p) dcopy(c->st, reinterpret_cast<c128*>(l2p), c->lam->l2p, c->oo * c->vv);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

int ccsd_set_lambda(ccsd_ctx* c, const ccsd_c128* l1, const ccsd_c128* l2p, int reset_diis)
{
    if (!c || !c->lam || !c->lam->ready) return CCSD_ESTATE;
    if (l1) dcopy(c->st, c->lam->l1, reinterpret_cast<const c128*>(l1), c->ov);
    if (l2p) dcopy(c->st, c->lam->l2p, reinterpret_cast<const c128*>(l2p), c->oo * c->vv);
    if (reset_diis) c->lam->diis.reset();
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

int ccsd_get_lambda_residual(ccsd_ctx* c, ccsd_c128* r1, ccsd_c128* r2p)
{
    if (!c || !c->lam || !c->lam->ready) return CCSD_ESTATE;
    if (r1) dcopy(c->st, reinterpret_cast<c128*>(r1), c->lam->R1, c->ov);
    if (r2p) dcopy(c->st, reinterpret_cast<c128*>(r2p), c->lam->R2p, c->oo * c->vv);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

int ccsd_expectation(ccsd_ctx* c, const ccsd_c128* D_, const ccsd_c128* O_, double* re, double* im)
{   // eq 16: <O> = sum_pq o_pq D[p][q], D[p][q] = <a+_p a_q> as ccsd_density returns it
    if (!c || !D_ || !O_) return CCSD_ESTATE;
    const c128 *D = reinterpret_cast<const c128*>(D_), *O = reinterpret_cast<const c128*>(O_);
    CCSD_CUDA_TRY(cudaMemsetAsync(c->red + 50, 0, 2 * sizeof(double), c->st));
    launch_reduce(c->st, c->diis.scratch, (int64_t)c->n * c->n, c->red + 50, 1, [=] __device__(int64_t x) { return cmul(O[x], D[x]); });
    CCSD_CUDA_TRY(cudaMemcpyAsync(c->red_host + 50, c->red + 50, 2 * sizeof(double), cudaMemcpyDeviceToHost, c->st));
    CCSD_CUDA_TRY(cudaStreamSynchronize(c->st));
    if (re) *re = c->red_host[50];
    if (im) *im = c->red_host[51];
    return CCSD_OK;
}

int ccsd_density(ccsd_ctx* c, ccsd_c128* D)
{
    if (!c || !c->lam || !c->lam->ready || !D) return CCSD_ESTATE;
    return lambda_density(c, c->lam, reinterpret_cast<c128*>(D));
}

// ---- standalone contractions ----------------------------------------------------------------------------------
static int64_t contract_partial_elems(int term, int64_t oo, int64_t vv, int64_t ov)
{
    if (term == CCSD_TERM_TAU) return 0;
    return 8 * (term == CCSD_TERM_RING ? ov * ov : oo * vv);
}

int ccsd_contract_workspace_bytes(int term, int nocc, int nvir, size_t* bytes)
{
    if (!bytes || nocc < 1 || nvir < 1) return CCSD_EINVAL;
    const int64_t o = nocc, v = nvir, oo = o * (o - 1) / 2, vv = v * (v - 1) / 2, ov = o * v, oop = round_up(oo > 0 ? oo : 1, 4);
    if (term >= CCSD_TERM_F_OV && term <= CCSD_TERM_C_OVOO) {
        TermWs tw;
        term_carve(nocc, nvir, nullptr, &tw, bytes);
        return CCSD_OK;
    }
    if (term == CCSD_TERM_S1_RESIDUAL || term == CCSD_TERM_S2_SMALL_TERMS) {
        TermWs tw;
        term_carve(nocc, nvir, nullptr, &tw, bytes);
        return CCSD_OK;
    }
    if (term == CCSD_TERM_ENERGY || term == CCSD_TERM_JACOBI_UPDATE) {
        StreamWs sw;
        stream_carve(nocc, nvir, nullptr, &sw, bytes);
        return CCSD_OK;
    }
    Carver w{nullptr, 0};
    w.take<int2>(oo); w.take<int2>(vv);
    switch (term) {
    case CCSD_TERM_PP_LADDER: break;
    case CCSD_TERM_PP_LADDER_PLANES: break;
    case CCSD_TERM_TAU: break;
    case CCSD_TERM_HH_LADDER: w.take<c128>(vv * oop); w.take<c128>(oo * oop); break;
    case CCSD_TERM_RING: w.take<c128>(ov * ov); w.take<c128>(ov * ov); w.take<c128>(ov * ov); break;
    default: return CCSD_EINVAL;
    }
    w.take<c128>(contract_partial_elems(term, oo, vv, ov));
    *bytes = w.off;
    return CCSD_OK;
}

int ccsd_contract(int term, int nocc, int nvir, const ccsd_c128* const* in_, ccsd_c128* out_, int accumulate,
                  const ccsd_options* opts, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!in_ || !out_ || nocc < 1 || nvir < 1) return CCSD_EINVAL;
    size_t need = 0;
    CCSD_TRY(ccsd_contract_workspace_bytes(term, nocc, nvir, &need));
    if (need > 0 && (!workspace || workspace_bytes < need || reinterpret_cast<uintptr_t>(workspace) % 256)) return CCSD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return CCSD_ECUDA;
    }
    cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
    const int o = nocc, v = nvir;
    const int64_t oo = (int64_t)o * (o - 1) / 2, vv = (int64_t)v * (v - 1) / 2, ov = (int64_t)o * v, oop = round_up(oo > 0 ? oo : 1, 4);
    if (term >= CCSD_TERM_F_OV && term <= CCSD_TERM_C_OVOO) {   // intermediates of eqs 24-31 (contract_terms.cuh)
        if (accumulate || nocc < 2 || nvir < 2) return CCSD_EINVAL;
        static const int k_nin[] = {3, 5, 5, 5, 6, 5};
        Env env2{st, opts ? opts->gemm_mode : 0, nullptr, 0};
        return contract_intermediate(term, nocc, nvir, reinterpret_cast<const c128* const*>(in_), k_nin[term - CCSD_TERM_F_OV],
                                     reinterpret_cast<c128*>(out_), env2, static_cast<char*>(workspace));
    }
    if (term >= CCSD_TERM_S1_RESIDUAL && term <= CCSD_TERM_JACOBI_UPDATE) {   // the remaining rows of one iteration
        if (accumulate || nocc < 2 || nvir < 2) return CCSD_EINVAL;
        static const int k_nin2[] = {9, 7, 4, 5};
        const int nin = k_nin2[term - CCSD_TERM_S1_RESIDUAL];
        if (term == CCSD_TERM_ENERGY || term == CCSD_TERM_JACOBI_UPDATE)
            return contract_stream_term(term, nocc, nvir, reinterpret_cast<const c128* const*>(in_), nin, reinterpret_cast<c128*>(out_),
                                        st, static_cast<char*>(workspace), opts ? opts->level_shift : 0.0, opts ? opts->ccd : 0);
        Env env2{st, opts ? opts->gemm_mode : 0, nullptr, 0};
        return contract_residual_term(term, nocc, nvir, reinterpret_cast<const c128* const*>(in_), nin, reinterpret_cast<c128*>(out_),
                                      env2, static_cast<char*>(workspace));
    }
    Env env{st, opts ? opts->gemm_mode : 0, nullptr, 0};
    {   // split-K partials live at the end of the workspace (same carving order as ccsd_contract_workspace_bytes)
        size_t all = 0;
        ccsd_contract_workspace_bytes(term, nocc, nvir, &all);
        int64_t pe = contract_partial_elems(term, oo, vv, ov);
        size_t pbytes = ((size_t)(pe > 0 ? pe : 1) * sizeof(c128) + 255) & ~(size_t)255;
        if (pe > 0) { env.partial = reinterpret_cast<c128*>(static_cast<char*>(workspace) + (all - pbytes)); env.partial_elems = pe; }
    }
    c128* out = reinterpret_cast<c128*>(out_);
    const c128* in0 = reinterpret_cast<const c128*>(in_[0]);
    const c128* in1 = reinterpret_cast<const c128*>(in_[1]);
    if (!in0 || !in1) return CCSD_EINVAL;
    Carver w{static_cast<char*>(workspace), 0};
    int2* po = w.take<int2>(oo);
    int2* pv = w.take<int2>(vv);
    if (oo == 0 || vv == 0) return CCSD_OK;
    switch (term) {
    case CCSD_TERM_PP_LADDER:
        // out[(i<j)][(a<b)] (+)= sum_{c<d} W[(a<b)][(c<d)] tau[(i<j)][(c<d)]
        return run_gemm(env, gp(vv, oo, vv, in1, vv, in0, vv, out, 1, vv, 1.0, accumulate));
    case CCSD_TERM_PP_LADDER_PLANES: {
        const double* taus = reinterpret_cast<const double*>(in_[2]);
        const double* Ws = reinterpret_cast<const double*>(in_[3]);
        if (!taus || !Ws) return CCSD_EINVAL;
        return run_gemm(env, with_planes(gp(vv, oo, vv, in1, vv, in0, vv, out, 1, vv, 1.0, accumulate), Ws, taus));
    }
    case CCSD_TERM_TAU: {
        pair_table_kernel<<<(unsigned)((oo + 255) / 256), 256, 0, st>>>(po, o);
        pair_table_kernel<<<(unsigned)((vv + 255) / 256), 256, 0, st>>>(pv, v);
        count_launches(2);
        if (accumulate) return CCSD_EINVAL;
        build_tau(st, out, in0, in1, o, v, po, pv, nullptr);
        CCSD_CUDA_TRY(cudaGetLastError());
        return CCSD_OK;
    }
    case CCSD_TERM_HH_LADDER: {
        c128* TT = w.take<c128>(vv * oop);
        c128* AT = w.take<c128>(oo * oop);
        CCSD_CUDA_TRY(cudaMemsetAsync(TT, 0, (size_t)(vv * oop) * sizeof(c128), st));
        CCSD_CUDA_TRY(cudaMemsetAsync(AT, 0, (size_t)(oo * oop) * sizeof(c128), st));
        CCSD_TRY(launch_transpose2d_ld(st, in1, vv, TT, oop, oo, vv, 0));
        CCSD_TRY(launch_transpose2d_ld(st, in0, oo, AT, oop, oo, oo, 0));
        return run_gemm(env, gp(vv, oo, oop, TT, oop, AT, oop, out, 1, vv, 1.0, accumulate));
    }
    case CCSD_TERM_RING: {
        pair_table_kernel<<<(unsigned)((oo + 255) / 256), 256, 0, st>>>(po, o);
        pair_table_kernel<<<(unsigned)((vv + 255) / 256), 256, 0, st>>>(pv, v);
        count_launches(2);
        c128* Hm = w.take<c128>(ov * ov);
        c128* T2r = w.take<c128>(ov * ov);
        c128* Xr = w.take<c128>(ov * ov);
        launch_fill(st, Hm, ov, ov, ov, 0, [=] __device__(int64_t ai, int64_t ck) {   // Hvovo[a][k][c][i] -> [(a,i)][(c,k)]
            int64_t a = ai / o, i = ai % o, cc = ck / o, k = ck % o;
            return in0[((a * o + k) * v + cc) * o + i];
        });
        launch_fill(st, T2r, ov, ov, ov, 0, [=] __device__(int64_t jb, int64_t ck) {
            int j = jb / v, b = jb % v, cc = ck / o, k = ck % o;
            return t2_at(in1, j, k, cc, b, o, v, vv);
        });
        CCSD_TRY(run_gemm(env, gp(ov, ov, ov, Hm, ov, T2r, ov, Xr, ov, 1, 1.0, 0)));
        launch_fill(st, out, oo, vv, vv, accumulate ? 1 : 0, [=] __device__(int64_t IJ, int64_t AB) {
            int2 ij = po[IJ], ab = pv[AB];
            int64_t i = ij.x, j = ij.y, a = ab.x, b = ab.y;
            c128 s = Xr[((a * o + i) * o + j) * v + b];
            s = csub(s, Xr[((a * o + j) * o + i) * v + b]);
            s = csub(s, Xr[((b * o + i) * o + j) * v + a]);
            s = cadd(s, Xr[((b * o + j) * o + i) * v + a]);
            return s;
        });
        CCSD_CUDA_TRY(cudaGetLastError());
        return CCSD_OK;
    }
    default: return CCSD_EINVAL;
    }
}

int ccsd_zgemm_nt(int64_t M, int64_t N, int64_t K, const ccsd_c128* A, int64_t lda, const ccsd_c128* B, int64_t ldb,
                  ccsd_c128* C, int64_t csm, int64_t csn, double alpha_re, double alpha_im, int accumulate, int mode,
                  void* cuda_stream)
{
    if (!A || !B || !C || M < 0 || N < 0 || K < 0 || mode < 0 || (mode > 3 && mode < 100)) return CCSD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return CCSD_ECUDA;
    }
    Env env{static_cast<cudaStream_t>(cuda_stream), mode, nullptr, 0};
    GemmParams p = gp(M, N, K, reinterpret_cast<const c128*>(A), lda, reinterpret_cast<const c128*>(B), ldb,
                      reinterpret_cast<c128*>(C), csm, csn, 1.0, accumulate);
    p.alpha = mk(alpha_re, alpha_im);
    return run_gemm(env, p);
}

int ccsd_zgemm_nt_planes(int64_t M, int64_t N, int64_t K, const ccsd_c128* A, int64_t lda, const double* As,
                         const ccsd_c128* B, int64_t ldb, const double* Bs, ccsd_c128* C, int64_t csm, int64_t csn,
                         double alpha_re, double alpha_im, int accumulate, int mode, void* cuda_stream)
{
    if (!A || !B || !C || !As || !Bs || M < 0 || N < 0 || K < 0) return CCSD_EINVAL;
    if (!(mode == 0 || mode == 3 || mode >= 100)) return CCSD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return CCSD_ECUDA;
    }
    Env env{static_cast<cudaStream_t>(cuda_stream), mode, nullptr, 0};
    GemmParams p = gp(M, N, K, reinterpret_cast<const c128*>(A), lda, reinterpret_cast<const c128*>(B), ldb,
                      reinterpret_cast<c128*>(C), csm, csn, 1.0, accumulate);
    p.alpha = mk(alpha_re, alpha_im);
    return run_gemm(env, with_planes(p, As, Bs));
}

// ccsd_zgemm_nt by one Strassen level (strassen.cuh): both operand stacks, their planes and the seven products live in the
// caller's workspace.  Any extents >= 1 (odd ones are zero-padded inside the stacks).
static void strassen_standalone_carve(int64_t M, int64_t N, int64_t K, int levels, char* base, StrassenScratch* w, size_t* total)
{
    Carver cv{base, 0};
    w->a_elems = strassen_stack_elems(M, K, levels);
    w->b_elems = strassen_stack_elems(N, K, levels);
    w->p_elems = (levels == 2 ? 49 : 7) * strassen_rows(M, levels) * strassen_rows(N, levels);
    w->SA = cv.take<c128>(w->a_elems); w->SAp = cv.take<double>(w->a_elems);
    w->SB = cv.take<c128>(w->b_elems); w->SBp = cv.take<double>(w->b_elems);
    w->P = cv.take<c128>(w->p_elems);
    *total = cv.off;
}

int ccsd_zgemm_nt_strassen_workspace_bytes(int64_t M, int64_t N, int64_t K, int levels, size_t* bytes)
{
    if (!bytes || M < 1 || N < 1 || K < 1 || levels < 1 || levels > 2) return CCSD_EINVAL;
    StrassenScratch w;
    strassen_standalone_carve(M, N, K, levels, nullptr, &w, bytes);
    return CCSD_OK;
}

int ccsd_zgemm_nt_strassen(int64_t M, int64_t N, int64_t K, const ccsd_c128* A, int64_t lda, const ccsd_c128* B, int64_t ldb,
                           ccsd_c128* C, int64_t csm, int64_t csn, double alpha_re, double alpha_im, int accumulate, int mode,
                           int levels, void* workspace, size_t workspace_bytes, void* cuda_stream)
{
    if (!A || !B || !C || M < 1 || N < 1 || K < 1 || lda < K || ldb < K || levels < 1 || levels > 2) return CCSD_EINVAL;
    if (!(mode == 0 || mode == 3 || mode >= 100)) return CCSD_EINVAL;
    size_t need = 0;
    StrassenScratch w;
    strassen_standalone_carve(M, N, K, levels, nullptr, &w, &need);
    if (!workspace || workspace_bytes < need || reinterpret_cast<uintptr_t>(workspace) % 256) return CCSD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return CCSD_ECUDA;
    }
    strassen_standalone_carve(M, N, K, levels, static_cast<char*>(workspace), &w, &need);
    Env env{static_cast<cudaStream_t>(cuda_stream), mode, nullptr, 0};
    GemmParams p = gp(M, N, K, reinterpret_cast<const c128*>(A), lda, reinterpret_cast<const c128*>(B), ldb,
                      reinterpret_cast<c128*>(C), csm, csn, 1.0, accumulate);
    p.alpha = mk(alpha_re, alpha_im);
    return strassen_gemm(env, p, nullptr, nullptr, w, levels);
}

int ccsd_strassen_info(ccsd_ctx* c, int info[4])
{
    if (!c || !info) return CCSD_ESTATE;
    info[0] = c->strassen ? 1 : 0;
    info[1] = c->strassen ? c->strassen_levels : 0;      // the two (ov)^3 products: levels
    info[2] = (c->strassen && c->sW.S) ? c->strassen_levels_L : 0;      // pp-ladder
    info[3] = (c->strassen && c->sVvovv.S) ? c->strassen_levels_C : 0;      // <bk||cd> tau part of C
    return CCSD_OK;
}

int ccsd_sum_plane(const ccsd_c128* in, double* out, int64_t n, void* cuda_stream)
{
    if (!in || !out || n < 0) return CCSD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return CCSD_ECUDA;
    }
    launch_sum_plane(static_cast<cudaStream_t>(cuda_stream), reinterpret_cast<const c128*>(in), out, n);
    CCSD_CUDA_TRY(cudaGetLastError());
    return CCSD_OK;
}

int ccsd_transpose(const ccsd_c128* in, ccsd_c128* out, const int64_t dims[4], const int perm[4], int conj, void* cuda_stream)
{
    if (!in || !out || !dims || !perm) return CCSD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return CCSD_ECUDA;
    }
    return launch_transpose4d(static_cast<cudaStream_t>(cuda_stream), reinterpret_cast<const c128*>(in),
                              reinterpret_cast<c128*>(out), dims, perm, conj);
}

int ccsd_enable_step_timing(ccsd_ctx* c, int enable)
{
    if (!c) return CCSD_ESTATE;
    if (enable && !c->ev[0])
        for (int k = 0; k <= CCSD_NSTEPS; k++) CCSD_CUDA_TRY(cudaEventCreate(&c->ev[k]));
    c->timing = enable ? 1 : 0;
    return CCSD_OK;
}

int ccsd_get_init_stats(ccsd_ctx* c, double stats[CCSD_NINIT_STATS])
{
    if (!c || !stats) return CCSD_ESTATE;
    for (int k = 0; k < CCSD_NINIT_STATS; k++) stats[k] = c->init_stats[k];
    return CCSD_OK;
}

int ccsd_get_step_times(ccsd_ctx* c, float ms[CCSD_NSTEPS])
{
    if (!c || !ms) return CCSD_ESTATE;
    for (int k = 0; k < CCSD_NSTEPS; k++) ms[k] = c->step_ms[k];
    return CCSD_OK;
}

int ccsd_measure_fp64_peak(double* tflops, double* device_scratch, int launches, void* cuda_stream)
{
    if (!tflops || !device_scratch || launches < 1) return CCSD_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        snprintf(g_cuda_err, sizeof(g_cuda_err), "no CUDA device");
        return CCSD_ECUDA;
    }
    return measure_fp64_peak(static_cast<cudaStream_t>(cuda_stream), device_scratch, launches, tflops);
}

int ccsd_gemm_plan(int64_t M, int64_t N, int64_t K, int64_t batch, int mode, int with_planes, int64_t partial_elems, int plan[4])
{   // host only: what ccsd_zgemm_nt / the contractions would launch for this shape (dmma_plan)
    if (!plan || M < 1 || N < 1 || K < 1 || batch < 1) return CCSD_EINVAL;
    const bool m3 = mode == 3 || (mode == 0 && CCSD_DEFAULT_3M != 0);
    if (!(mode == 0 || mode == 2 || mode == 3)) return CCSD_EINVAL;
    const DmmaPlan pl = dmma_plan(M, N, K, batch, m3, m3 && with_planes, partial_elems > 0, partial_elems);
    plan[0] = pl.variant; plan[1] = k_dmma_variants[pl.variant].bm; plan[2] = k_dmma_variants[pl.variant].bn; plan[3] = pl.ksplit;
    return CCSD_OK;
}

int ccsd_real_flops_per_cmac(const ccsd_options* opts)
{
    const int mode = opts ? opts->gemm_mode : 0;
    if (mode >= 100 && mode - 100 < DMMA_NVARIANTS) return k_dmma_variants[mode - 100].m3 ? 6 : 8;
    if (mode == 3 || (mode == 0 && CCSD_DEFAULT_3M != 0)) return 6;
    return 8;
}

const char* ccsd_step_name(int step) { return (step >= 0 && step < CCSD_NSTEPS) ? k_step_names[step] : ""; }

long long ccsd_launch_count(int reset)
{
    long long r = g_launches;
    if (reset) g_launches = 0;
    return r;
}

const char* ccsd_strerror(int s)
{
    switch (s) {
    case CCSD_OK: return "ok";
    case CCSD_EINVAL: return "invalid argument";
    case CCSD_ENOMEM: return "out of host memory";
    case CCSD_ECUDA: return "CUDA error";
    case CCSD_ESTATE: return "invalid state or handle";
    case CCSD_ESINGULAR: return "singular DIIS system";
    case CCSD_ENOTCONVERGED: return "not converged within the iteration limit";
    default: return "unknown status";
    }
}

const char* ccsd_last_cuda_error(void) { return g_cuda_err; }

}  // extern "C"
