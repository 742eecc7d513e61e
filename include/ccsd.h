/*
 * ccsd.h -- C ABI of the B200-native complex spinor-basis CCSD hot path (arXiv 2103.08473, "ExaCorr").
 *
 * What the library computes: one iteration of the CCSD amplitude equations in complex (spinor) algebra,
 * Appendix 7.1 of the paper (eqs 22-33): tau (eq 23), the Fock-like intermediates
 * H^a_c/G^a_c, H^k_i/G^k_i, H^k_c (eqs 24-28), the particle-hole intermediate H^{ak}_{ci} (eq 29), C^{kb}_{ij}
 * (eq 30), the hole-hole intermediate A^{kl}_{ij} (eq 31), the doubles residual S^{ab}_{ij} (eq 32: ring,
 * hole-hole ladder, particle-particle ladder and the small terms) and the singles residual S^a_i (eq 33);
 * followed by the denominator ("Jacobi") update with DIIS and the correlation
 * energy (eq 9; contraction string PAPER.md:178-182).  Inputs are those of eq 5: the
 * one-electron matrix h_pq and the two-electron integrals in factorised (Cholesky-type) form.
 * Reading of the paper's notation: DESIGN.md "Readings of the paper".
 *
 * Conventions for EVERY entry point
 *  - ccsd_c128 is an interleaved (re, im) pair of doubles, 16-byte aligned: binary compatible with
 *    torch.complex128 / numpy.complex128 / CUDA double2.
 *  - All tensor pointers are DEVICE pointers unless the comment says HOST.  Row-major, last index fastest.
 *  - Spinors are ordered occupied first: o = nocc, v = nvir, n = o + v.  oo = o(o-1)/2, vv = v(v-1)/2.
 *    A packed pair (x<y) of a dimension of size m has index  x*m - x(x+1)/2 + (y-x-1)  (row-major strict upper
 *    triangle, the order of numpy.triu_indices(m, 1)).
 *  - Canonical layouts at the boundary:  t1, S1 [i][a];  t2, tau, S2 [(i<j)][(a<b)];  <ab||cd> [(a<b)][(c<d)];
 *    Hvv, Gvv [a][c];  Hoo, Goo [k][i];  Hov [k][c];  Hvovo [a][k][c][i];  C [k][b][(i<j)];  A [(k<l)][(i<j)].
 *  - Ownership: the caller owns every buffer including `workspace`; the library never allocates or frees device
 *    memory and never creates streams.  All work is enqueued on the caller's `cuda_stream` (a cudaStream_t).
 *  - Errors: every call returns a CCSD_* status; nothing is thrown or printed.  There is no CPU fallback: without
 *    a CUDA device every compute entry point returns CCSD_ECUDA.
 *  - Threads and streams: contexts are independent -- every buffer a context's kernels touch (reduction scratch, DIIS Gram
 *    matrix and coefficients, split-K scratch included) lies in ITS workspace, so different contexts may be driven from
 *    different host threads on different streams at the same time.  ONE context must not be entered from two threads at once
 *    (its host-side state -- DIIS ring order, graph handle, pinned read-back buffer -- is not locked), and all its calls are
 *    ordered on the stream given to ccsd_init.  The context-free entry points (ccsd_contract, ccsd_zgemm_nt*, ccsd_transpose,
 *    ccsd_sum_plane) keep no state between calls.  ccsd_launch_count is one process-wide atomic counter; ccsd_last_cuda_error
 *    is per host thread.  The current CUDA device must be the one the workspace lives on.
 */
#ifndef CCSD_B200_H
#define CCSD_B200_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct ccsd_ctx ccsd_ctx; /* opaque, host-side handle */
typedef struct { double re, im; } ccsd_c128;

enum { CCSD_OK = 0, CCSD_EINVAL = 1, CCSD_ENOMEM = 2, CCSD_ECUDA = 3, CCSD_ESTATE = 4, CCSD_ESINGULAR = 5,
       CCSD_ENOTCONVERGED = 6 };

typedef struct {
    int ndiis;          /* DIIS subspace size; 0 = plain Jacobi; default 6 (reading G13) */
    double level_shift; /* added to the virtual orbital energies in the denominators; default 0 */
    int gemm_mode;      /* 0 = auto (FP64 tensor-core DMMA kernels where the shape allows; complex arithmetic by the
                           3M scheme, chosen by measurement), 1 = force the simple FP64-FMA kernels
                           (on-device debugging reference), 2 = DMMA kernels with 4M complex arithmetic,
                           3 = DMMA kernels with 3M; 100+v = one fixed tile variant v (tuning only) */
    int ccd;            /* 1 = CCD: t1 is kept at zero */
    int cc2;            /* 1 = CC2 (Appendix 7.2 eqs 34-38): singles equations of CCSD,
                           doubles equations <Phi_ij^ab| exp(-T1) H exp(T1) + [F, T2] |Phi_0>; ccsd_get_tensor then returns
                           tau, C, A at t2 = 0, GVV = f_vv, GOO = -f_oo, and S2_GVV / S2_GOO the two Fock terms */
    int direct_ladder;  /* 1 = integral-direct pp-ladder: the packed <ab||cd>
                           (vv^2 elements, the largest tensor) is never stored; every iteration rebuilds its rows slab by
                           slab from the factor B and contracts them.  Trades 8 v^4 naux flops per iteration for
                           24 vv^2 bytes of HBM; ccsd_get_tensor(CCSD_T_VVVV) and the Lambda entry points then return
                           CCSD_EINVAL.  Default 0 */
    int graph;          /* 1 (default) = the residual evaluation inside ccsd_iterate / ccsd_residual (~70 kernel launches that
                           depend on nothing but the context) is captured into a CUDA graph on its second use and replayed
                           afterwards; 0 = always launch directly.  Capture needs a stream created by the caller: on the
                           legacy / per-thread default streams (cuda_stream = 0, 1 or 2), and while step timing is enabled,
                           the launches are issued directly whatever this says.  In the graph the independent parts of the
                           residual (H^{ak}_{ci} + ring product; A + Fock-like terms + S1; C; V^dagger t1; driver + pp-ladder) are parallel
                           branches, so that the small products fill the partial waves of the large ones; 3 = a graph with the
                           launches in their serial order.  Results are bit-identical in all cases */
    int shard_rank;     /* slab sharding of the iteration over several GPUs (one process and one context per GPU, */
    int shard_world;    /* every rank gets the same h, B and holds the same amplitudes): with shard_world = P > 1 the context
                           of rank r builds and stores only its 1/P of the rows of the packed <ab||cd>, and ccsd_residual
                           evaluates only its slab of every large contraction of eqs 29-32 (disjoint output rows: the (a<b)
                           rows of the pp-ladder, the (a,i) rows of H^{ak}_{ci} and of the ring product, the (b,k) rows of C),
                           adding them into an S2 that is zero elsewhere.  The caller sums S2 over the ranks (ONE all-reduce of
                           the packed S2 per iteration; ccsd_shard_info locates the buffer) and then calls ccsd_update, which
                           is replicated.  S1 and the small intermediates are replicated too.  The library issues no
                           collective itself.  Defaults 0, 1.  Not with cc2; ccsd_iterate / ccsd_solve, CCSD_T_VVVV and the
                           Lambda entry points return CCSD_EINVAL in a sharded context */
    int strassen;       /* 1 (default) = the four large contractions of an iteration -- the two (ov)^3 products of eq 29 and of
                           the ring term, the pp-ladder and the <bk||cd> tau part of eq 30 -- run by Strassen's algorithm around
                           the DMMA GEMM: seven half-size products in ONE batched launch instead of eight, i.e. 7/8 of the FP64
                           tensor-pipe work, plus three streaming passes; TWO levels (49
                           quarter-size products, 0.766 of the work) for the (ov)^3 products from ov >= 3072 and for the ladder
                           and C where a quarter of the (i<j) extent still fills whole tiles (oo >= 510).  Pure FP64; results
                           differ from strassen = 0 by rounding only (about 1e-14 of the largest element of each product at
                           most).  Costs workspace: the operand stacks of <ab||cd>, <bk||cd> and <kl||cd> are built once and
                           kept (1.75 x - 3 x the bytes of those tensors with their planes); where the ladder and C both use
                           it, the packed <ab||cd> itself is NOT kept beside its stack (ccsd_get_tensor(CCSD_T_VVVV) rebuilds
                           it from the stack, exact up to one rounding per element).  Used on one GPU with the 3M kernels
                           (gemm_mode 0 or 3) where the products are large enough (ov >= 1024); ignored in cc2 mode; in a sharded
                           context the left operands are the rank's row slabs (stacks of this rank's rows only); with
                           direct_ladder the ladder keeps its slab form.  A workspace that would exceed
                           128 GiB (of a 180 GB part) gives levels up step by step -- the ladder's first, then C's, then the
                           (ov)^3 products' -- down to plain products: ccsd_strassen_info reports what is used.  0 = plain products;
                           2 = one level only; 3 = two levels on all four products whatever their size (tests) */
} ccsd_options;

/* Fill *opts with the defaults above. */
void ccsd_default_options(ccsd_options* opts);

/* Bytes of device workspace ccsd_init needs for (nocc, nvir, naux).  HOST out-pointer. */
int ccsd_workspace_bytes(int nocc, int nvir, int naux, const ccsd_options* opts, size_t* bytes);

/*
 * Set up a calculation: builds the Fock matrix f = h + sum_i <pi||qi>, the six
 * antisymmetrised integral classes <pq||rs> = (pr|qs) - (ps|qr) with (pq|rs) = sum_L B[L][p][q] B[L][r][s], the
 * orbital-energy denominators and the MP2 starting amplitudes ("iteration 0").
 *   h  [n][n]         bare one-electron matrix of eq 5, Hermitian
 *   B  [naux][n][n]   factor of the two-electron integrals, every B[L] Hermitian
 *   workspace         at least ccsd_workspace_bytes() bytes, 256-byte aligned; must stay alive until ccsd_destroy
 * h and B may be released after the call returns (the call synchronises the stream).
 * Errors: CCSD_EINVAL (bad sizes / null pointers / workspace too small), CCSD_ECUDA.
 */
int ccsd_init(ccsd_ctx** ctx, const ccsd_c128* h, const ccsd_c128* B, int nocc, int nvir, int naux,
              const ccsd_options* opts, void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * One CCSD iteration at the current amplitudes: eqs 23-33, t <- t + S/D, DIIS extrapolation.
 * HOST outputs: correlation energy (Re, Im) of the NEW amplitudes and ||S/D||_2 over the unique amplitudes of the
 * residual just evaluated.  Synchronises the stream (one small device->host copy).
 * Errors: CCSD_ESTATE (no context), CCSD_ESINGULAR (DIIS system singular even with one vector), CCSD_ECUDA.
 */
int ccsd_iterate(ccsd_ctx* ctx, double* e_re, double* e_im, double* step_norm);

/*
 * The second half of ccsd_iterate on its own: Jacobi step + DIIS + energy from the residuals (S1, S2) held by the context
 * (those of the last ccsd_residual, after the caller's all-reduce of S2 in a sharded run: ccsd_residual; all-reduce;
 * ccsd_update is one iteration).  HOST outputs as ccsd_iterate.  CCSD_ESTATE without a residual of the current amplitudes.
 */
int ccsd_update(ccsd_ctx* ctx, double* e_re, double* e_im, double* step_norm);
/*
 * Where this context's slab lies and where the caller's collective has to act.  HOST out-pointer, info[] =
 * { shard_rank, shard_world, a_lo, a_hi (virtual-index slab of the (ov)^3 / C rows), w_lo, w_hi (packed (a<b) rows of
 *   <ab||cd> this rank stores and contracts), ij_lo, ij_hi (packed (i<j) rows of the row-wise small terms),
 *   byte offset of S2 [(i<j)][(a<b)] in the workspace handed to ccsd_init, its ccsd_c128 element count,
 *   byte offset of S1 [i][a], its element count }.
 */
enum { CCSD_NSHARD_INFO = 12 };
int ccsd_shard_info(ccsd_ctx* ctx, int64_t info[CCSD_NSHARD_INFO]);
/* The same ranges without a context (host arithmetic only, no CUDA device needed): ranges[] = { a_lo, a_hi, w_lo, w_hi,
 * ij_lo, ij_hi, wa_lo, wa_hi } of rank `rank` of `world`; [wa_lo, wa_hi) is the range of the first virtual index whose
 * pairs (a, b > a) are the packed rows [w_lo, w_hi).  Over rank = 0..world-1 each family of ranges tiles its index range
 * exactly once.  CCSD_EINVAL for world > nvir. */
int ccsd_shard_ranges(int nocc, int nvir, int rank, int world, int64_t ranges[8]);

/*
 * ccsd_iterate until ||S/D||_2 < tol and |E - E_previous| < tol, or max_iterations (the paper's .TCONVERG 1e-9 and
 * .NCYCLES 30 keywords; which quantity .TCONVERG tests is not stated: reading G14).  HOST outputs:
 * iterations done, energy of the last amplitudes, last ||S/D||_2.  Returns CCSD_ENOTCONVERGED if the limit was hit.
 */
int ccsd_solve(ccsd_ctx* ctx, double tol, int max_iterations, int* iterations, double* e_re, double* e_im,
               double* step_norm);

/* E_corr = sum f_ia t^a_i + sum_{i<j,a<b} <ij||ab> tau^{ab}_{ij} of the current amplitudes (eq 9).  HOST outputs. */
int ccsd_energy(ccsd_ctx* ctx, double* e_re, double* e_im);

/* T1 diagnostic of the current amplitudes, sqrt(sum_ia |t^a_i|^2 / nocc) (the paper tabulates it, PAPER.md:346-379 and
 * 506-522, without defining it; this is the usual definition with nocc correlated spinors).  HOST output. */
int ccsd_t1_diagnostic(ccsd_ctx* ctx, double* t1_diag);

/* Evaluate eqs 23-33 at the current amplitudes WITHOUT updating them (fills the tensors ccsd_get_tensor returns). */
int ccsd_residual(ccsd_ctx* ctx);

/* Copy the current amplitudes out / in (device pointers): t1 [o][v], t2p [(i<j)][(a<b)].  Asynchronous. */
int ccsd_get_amplitudes(ccsd_ctx* ctx, ccsd_c128* t1, ccsd_c128* t2p);
int ccsd_set_amplitudes(ccsd_ctx* ctx, const ccsd_c128* t1, const ccsd_c128* t2p, int reset_diis);

/* Tensor ids for ccsd_get_tensor; canonical layouts as listed at the top.  S2_* are the eight terms of eq 32. */
enum {
    CCSD_T_FOCK = 0,   /* [n][n] */
    CCSD_T_VVVV = 1,   /* [(a<b)][(c<d)]; CCSD_EINVAL in cc2 and direct_ladder mode, where it is not stored; where the ladder runs
                          through its Strassen operand stack (ccsd_options.strassen) it is rebuilt from that stack */
    CCSD_T_VOVV = 2,   /* [a][k][(c<d)] */
    CCSD_T_VOVO = 3,   /* [a][k][c][i] */
    CCSD_T_OOVV = 4,   /* [(k<l)][(c<d)] */
    CCSD_T_OOOV = 5,   /* [(k<l)][i][c] */
    CCSD_T_OOOO = 6,   /* [(k<l)][(i<j)] */
    CCSD_T_TAU = 10, CCSD_T_HVV = 11, CCSD_T_GVV = 12, CCSD_T_HOO = 13, CCSD_T_GOO = 14, CCSD_T_HOV = 15,
    CCSD_T_HVOVO = 16, CCSD_T_C = 17, CCSD_T_A = 18, CCSD_T_S1 = 19, CCSD_T_S2 = 20,
    CCSD_T_S2_RING = 30, CCSD_T_S2_GOO = 31, CCSD_T_S2_VDAG_T1 = 32, CCSD_T_S2_GVV = 33, CCSD_T_S2_C_T1 = 34,
    CCSD_T_S2_HH_LADDER = 35, CCSD_T_S2_PP_LADDER = 36, CCSD_T_S2_DRIVER = 37
};
/* Number of ccsd_c128 elements of tensor `tensor_id` (HOST out-pointer). */
int ccsd_tensor_elems(ccsd_ctx* ctx, int tensor_id, size_t* elems);
/* Copy tensor `tensor_id` into out (device).  Intermediates, S1, S2 are those of the last ccsd_residual/iterate;
 * the S2_* ids re-evaluate that single term of eq 32 from the stored intermediates.  Asynchronous. */
int ccsd_get_tensor(ccsd_ctx* ctx, int tensor_id, ccsd_c128* out);

int ccsd_destroy(ccsd_ctx* ctx);

/*
 * Perturbative triples corrections at the CURRENT amplitudes (Appendix 7.3, eqs 39-44):
 *   E(+T)  = sum conj(Wbar) Wbar / (36 D)            (eq 39)      Wbar = W^abc + W^bca + W^cab, W of eq 40
 *   E((T)) = E(+T) + sum conj(Zbar) Wbar / (36 D)    (eq 41)      Z of eq 42
 *   E(-T)  = E(+T) + sum conj(Ybar) Wbar / 36        (eq 43)      Y of eq 44
 * with D = eps_i + eps_j + eps_k - eps_a - eps_b - eps_c and the sums over all i,j,k,a,b,c (evaluated over the unique
 * i<j<k, a<b<c).  Reading of the printed equations for complex amplitudes: DESIGN.md G22.
 * HOST outputs, (Re, Im) each.  workspace: device, 256-byte aligned, ccsd_triples_workspace_bytes() bytes, used only
 * during the call.  Needs nocc >= 3 and nvir >= 3 (CCSD_EINVAL otherwise).  Synchronises the stream.
 * With step timing enabled ccsd_get_triples_times returns the summed device times (ms) of {0: the W GEMM launches,
 * 1: the energy kernels} of the last call.
 */
int ccsd_triples_workspace_bytes(ccsd_ctx* ctx, size_t* bytes);
int ccsd_triples(ccsd_ctx* ctx, double e_plus_t[2], double e_par_t[2], double e_minus_t[2], void* workspace,
                 size_t workspace_bytes);
int ccsd_get_triples_times(ccsd_ctx* ctx, float ms[2]);
/*
 * The same energies restricted to the occupied triples number first_triple .. first_triple + ntriples - 1 of the
 * lexicographic list of i<j<k (ccsd_triples_count() entries; "only the unique blocks" of the three nested
 * occupied loops).  The outputs are the partial sums of eq 39/42/44 over those triples: summed over a partition of the
 * list they give the values of ccsd_triples, which is how the correction is shared among GPUs (one context per GPU on
 * the same amplitudes, one range each, one sum of six doubles at the end; binding: CCSD.triples_sharded).
 * ntriples == 0 returns zeros.  CCSD_EINVAL when the range leaves the list.
 */
int ccsd_triples_count(ccsd_ctx* ctx, int64_t* ntriples);
int ccsd_triples_range(ccsd_ctx* ctx, int64_t first_triple, int64_t ntriples, double e_plus_t[2], double e_par_t[2],
                       double e_minus_t[2], void* workspace, size_t workspace_bytes);
/*
 * CCSD Lambda equations and Lagrange one-body density matrix (Appendix 7.4-7.5, eqs 45-61; PAPER.md:109-126,
 * 238), at the CURRENT amplitudes, which should be converged (ccsd_solve): the equations are
 * <0|(1+Lambda)(Hbar - E)|mu> = 0 up to terms proportional to the amplitude residual.  Reading of the incomplete
 * printed equations: DESIGN.md G23, G24.  Not available in CC2 mode (CCSD_EINVAL).
 *   ccsd_lambda_init      builds the elements of Hbar = exp(-T) H exp(T) once (it runs one residual evaluation: the
 *                         tensors of ccsd_get_tensor are refreshed) and sets lambda = conj(t).  workspace: device,
 *                         256-byte aligned, ccsd_lambda_workspace_bytes() bytes; it must stay alive while the Lambda
 *                         entry points are used (until the next ccsd_lambda_init or ccsd_destroy).  Synchronises.
 *   ccsd_lambda_iterate   one iteration: right-hand sides of eqs 52-56, lambda <- lambda + R/D with the CCSD
 *                         denominators, DIIS as for the amplitudes.  HOST output ||R/D||_2 over the unique multipliers.
 *   ccsd_lambda_solve     ccsd_lambda_iterate until ||R/D||_2 < tol or max_iterations (as ccsd_solve; the multipliers have
 *                         no energy of their own to test).  HOST outputs: iterations done, last ||R/D||_2.  Returns
 *                         CCSD_ENOTCONVERGED if the limit was hit.
 *   ccsd_lambda_residual  evaluates the right-hand sides only (ccsd_get_lambda_residual returns them).
 *   ccsd_get/set_lambda   multipliers lambda^i_a [i][a], lambda^{ij}_{ab} [(i<j)][(a<b)] (device, asynchronous).
 *   ccsd_density          D[p][q] = <0|(1+Lambda) exp(-T) a+_p a_q exp(T)|0> - delta_pq (p occupied), [n][n] (device),
 *                         occupied spinors first, assembled from eqs 58-61, unsymmetrised (the paper symmetrises it
 *                         before use).  Uses the residual buffers: call it between iterations.
 * In CCD mode (opts.ccd) the Lagrangian has no singles constraint: lambda^i_a stays zero.
 * Errors: CCSD_ESTATE without ccsd_lambda_init, CCSD_EINVAL (workspace), CCSD_ESINGULAR (DIIS), CCSD_ECUDA.
 */
int ccsd_lambda_workspace_bytes(ccsd_ctx* ctx, size_t* bytes);
int ccsd_lambda_init(ccsd_ctx* ctx, void* workspace, size_t workspace_bytes);
int ccsd_lambda_iterate(ccsd_ctx* ctx, double* step_norm);
int ccsd_lambda_solve(ccsd_ctx* ctx, double tol, int max_iterations, int* iterations, double* step_norm);
int ccsd_lambda_residual(ccsd_ctx* ctx);
int ccsd_get_lambda(ccsd_ctx* ctx, ccsd_c128* l1, ccsd_c128* l2p);
int ccsd_set_lambda(ccsd_ctx* ctx, const ccsd_c128* l1, const ccsd_c128* l2p, int reset_diis);
int ccsd_get_lambda_residual(ccsd_ctx* ctx, ccsd_c128* r1, ccsd_c128* r2p);
int ccsd_density(ccsd_ctx* ctx, ccsd_c128* D);
/* eq 16: expectation value of a one-body operator, sum_pq O[p][q] D[p][q] with D as ccsd_density returns it
 * (correlation part; the reference determinant contributes sum_i O[i][i]).  D, O: device [n][n].  HOST outputs. */
int ccsd_expectation(ccsd_ctx* ctx, const ccsd_c128* D, const ccsd_c128* O, double* re, double* im);

/* Per-term parity hook: the dense, fully antisymmetric blocks Wbar, Zbar, Ybar [a][b][c] (nvir^3 elements each, device;
 * NULL = skip) of one occupied triple i<j<k.  Asynchronous on the stream after an initial synchronisation. */
int ccsd_triples_block(ccsd_ctx* ctx, int i, int j, int k, ccsd_c128* Wbar, ccsd_c128* Zbar, ccsd_c128* Ybar,
                       void* workspace, size_t workspace_bytes);

/*
 * Standalone contractions on caller-supplied tensors (per-term parity and timing; BASELINE config 4).
 *   CCSD_TERM_PP_LADDER (eq 32; string form PAPER.md:176):
 *        in[0] = tau [(i<j)][(c<d)], in[1] = W [(a<b)][(c<d)];  out [(i<j)][(a<b)] = sum_{c<d} W tau
 *   CCSD_TERM_HH_LADDER (eq 32): in[0] = A [(k<l)][(i<j)], in[1] = tau [(k<l)][(a<b)];
 *        out [(i<j)][(a<b)] = sum_{k<l} A tau
 *   CCSD_TERM_RING (eq 32 first line): in[0] = Hvovo [a][k][c][i], in[1] = t2 [(i<j)][(a<b)];
 *        out [(i<j)][(a<b)] = P-_ij P-_ab sum_{kc} Hvovo[a,k,c,i] t2[j,k,c,b]
 *   CCSD_TERM_TAU (eq 23): in[0] = t1 [i][a], in[1] = t2 [(i<j)][(a<b)]; out = tau packed
 *   CCSD_TERM_PP_LADDER_PLANES: CCSD_TERM_PP_LADDER with the operands' 3M "sum planes" supplied by the caller, the way
 *        ccsd_iterate runs it (the plane of the constant W is built once, by ccsd_init / ccsd_sum_plane):
 *        in[2] = (double*) plane of tau [(i<j)][(c<d)], in[3] = (double*) plane of W [(a<b)][(c<d)], plane = Re + Im.
 *        Same result as CCSD_TERM_PP_LADDER up to rounding.
 * accumulate != 0 adds into out.  workspace: ccsd_contract_workspace_bytes() bytes.  Asynchronous on the stream.
 */
enum { CCSD_TERM_PP_LADDER = 0, CCSD_TERM_HH_LADDER = 1, CCSD_TERM_RING = 2, CCSD_TERM_TAU = 3,
       CCSD_TERM_PP_LADDER_PLANES = 4,
       /* The intermediates of eqs 24-31 (BASELINE north_star names: F_me, F_ae, F_mi, W_mnij, W_mbej; DESIGN.md relates them to
        * the paper's H^k_c, G^a_c, G^k_i, A^{kl}_{ij}, H^{ak}_{ci}, C^{kb}_{ij}).  Inputs in the canonical layouts listed at the
        * top of this file, f = the Fock matrix [n][n]; accumulate must be 0:
        *   F_OV   (eq 28)      in = { f, <kl||cd>, t1 }                                  out H^k_c [k][c]
        *   F_VV   (eqs 24-25)  in = { f, <kl||cd>, <ak||cd>, t1, t2 }                    out G^a_c [a][c]
        *   F_OO   (eqs 26-27)  in = { f, <kl||cd>, <kl||ic>, t1, t2 }                    out G^k_i [k][i]
        *   W_OOOO (eq 31)      in = { <kl||ij>, <kl||ic>, <kl||cd>, t1, t2 }             out A [(k<l)][(i<j)]
        *   W_OVVO (eq 29)      in = { <ak||ci>, <ak||cd>, <kl||ic>, <kl||cd>, t1, t2 }   out H^{ak}_{ci} [a][k][c][i]
        *   C_OVOO (eq 30)      in = { <kl||ic>, <ak||ci>, <ak||cd>, t1, t2 }             out C [k][b][(i<j)]                    */
       CCSD_TERM_F_OV = 5, CCSD_TERM_F_VV = 6, CCSD_TERM_F_OO = 7, CCSD_TERM_W_OOOO = 8, CCSD_TERM_W_OVVO = 9,
       CCSD_TERM_C_OVOO = 10,
       /* The remaining rows of one iteration; nocc, nvir >= 2, accumulate must be 0:
        *   S1_RESIDUAL    (eq 33)  in = { f, H^a_c [a][c], H^k_i [k][i], H^k_c [k][c], <ak||cd>, <kl||ic>,
        *                   <ak||ci>, t1, t2 }                                              out S1 [i][a]
        *   S2_SMALL_TERMS (eq 32: the G_oo, V^dagger t1, G_vv, C t1 lines and the driver conj <ij||ab>)
        *                   in = { G^a_c [a][c], G^k_i [k][i], C [k][b][(i<j)], <ak||cd>, <kl||cd>, t1, t2 }
        *                                                                                   out [(i<j)][(a<b)]
        *   ENERGY         (eq 9)        in = { f, <kl||cd>, t1, t2 }          out one ccsd_c128 (device)
        *   JACOBI_UPDATE  (DESIGN reading G12)  in = { f, t1, t2, S1 [i][a], S2 [(i<j)][(a<b)] }
        *                   out [nocc*nvir + oo*vv]: u1 = t1 + S1/D^a_i followed by u2 = t2 + S2/D^{ab}_{ij} (the layout of the
        *                   DIIS vectors), D from eps_p = Re f_pp, opts->level_shift added to the virtual eps; opts->ccd
        *                   keeps u1 = 0 */
       CCSD_TERM_S1_RESIDUAL = 11, CCSD_TERM_S2_SMALL_TERMS = 12, CCSD_TERM_ENERGY = 13, CCSD_TERM_JACOBI_UPDATE = 14 };
int ccsd_contract_workspace_bytes(int term, int nocc, int nvir, size_t* bytes);
int ccsd_contract(int term, int nocc, int nvir, const ccsd_c128* const* in, ccsd_c128* out, int accumulate,
                  const ccsd_options* opts, void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The correlation energy (eq 9, with tau of eq 23; reading G11) WITHOUT a workspace, for callers
 * that cannot allocate one (code under stream capture, tight serving loops, harnesses that forbid cudaMalloc):
 *   e_out = sum_ia f[i][o+a] t1[i][a] + sum_{i<j,a<b} <ij||ab> (t2 + P-(t1 t1))^{ab}_{ij}
 * Same arguments as ccsd_contract(CCSD_TERM_ENERGY): f = Fock matrix [n][n], oovv = <kl||cd> [(k<l)][(c<d)], t1 [i][a],
 * t2p [(i<j)][(a<b)] (device, read only); e_out = one ccsd_c128 on the device, overwritten.  Same kernels in their
 * energy-only form, same summation order: the result equals that of the workspace path bit for bit.
 * The scratch that path carves from the caller's workspace (two pair tables and the per-block partial sums) lives in one
 * file-scope device array of CCSD_ENERGY_STATIC_SCRATCH_BYTES (1.07 MiB) inside the library, which every GPU that loads the
 * library holds until the process exits.  Limits: 2 <= nocc <= CCSD_ENERGY_STATIC_MAX_NOCC, 2 <= nvir <=
 * CCSD_ENERGY_STATIC_MAX_NVIR; anything larger returns CCSD_EINVAL (the reason in ccsd_last_cuda_error()) and enqueues
 * nothing -- use ccsd_contract with a workspace there.  The call makes no cudaMalloc / cudaFree and no allocating
 * library call; it enqueues four kernels on `cuda_stream` and returns (asynchronous).  The first call on a device resolves
 * the array's address (cudaGetSymbolAddress, once per device, with the caller's current device).
 * ALL calls on a device share the one array and it keeps the last call's contents.  Every word a call reads it has
 * written itself first (tables and partials are rewritten each call; nothing needs to start at zero), so calls
 * ordered on one stream are independent, but two calls that OVERLAP on the GPU -- different streams or host threads without
 * an ordering between them -- race on it and give undefined results.  Serialise them, or use the workspace path.
 */
#define CCSD_ENERGY_STATIC_MAX_NOCC 128
#define CCSD_ENERGY_STATIC_MAX_NVIR 512
#define CCSD_ENERGY_STATIC_SCRATCH_BYTES 1121024
int ccsd_energy_static(int nocc, int nvir, const ccsd_c128* f, const ccsd_c128* oovv, const ccsd_c128* t1,
                       const ccsd_c128* t2p, ccsd_c128* e_out, void* cuda_stream);

/*
 * Generic complex GEMM used by every contraction above ("NT" form, both operands K-contiguous):
 *   C[m*csm + n*csn] (+)= alpha * sum_k A[m*lda + k] * B[n*ldb + k]
 * mode: as ccsd_options.gemm_mode (0 auto, 1 simple FMA kernel, 2 DMMA 4M, 3 DMMA 3M, 100+v tile variant v).
 */
int ccsd_zgemm_nt(int64_t M, int64_t N, int64_t K, const ccsd_c128* A, int64_t lda, const ccsd_c128* B, int64_t ldb,
                  ccsd_c128* C, int64_t csm, int64_t csn, double alpha_re, double alpha_im, int accumulate, int mode,
                  void* cuda_stream);

/* Host arithmetic only (no CUDA device needed): the launch plan of the DMMA GEMM for a shape -- tile variant and split-K depth
 * chosen together against wave quantisation on the SMs.  mode 0 / 2 / 3 as above; with_planes: the
 * operands carry 3M sum planes; partial_elems: ccsd_c128 elements of split-K scratch available (0 = no split-K).
 * plan[] = { variant id, tile rows, tile columns, split-K depth }. */
int ccsd_gemm_plan(int64_t M, int64_t N, int64_t K, int64_t batch, int mode, int with_planes, int64_t partial_elems, int plan[4]);

/*
 * 3M operand "sum plane": out[i] = Re in[i] + Im in[i], i < n.  The 3M complex GEMM (three real products per complex
 * MAC: Ar Br, Ai Bi, (Ar + Ai)(Br + Bi)) reads these sums through TMA instead of forming them on the FP64 pipe.
 */
int ccsd_sum_plane(const ccsd_c128* in, double* out, int64_t n, void* cuda_stream);
/* ccsd_zgemm_nt on the 3M kernels with the operands' sum planes As[m*lda + k], Bs[n*ldb + k] supplied (mode 0, 3 or
 * 100+v).  The planes are used when lda and ldb are even and the planes 16-byte aligned (TMA rows); otherwise the
 * kernel forms the sums itself.  Same result as ccsd_zgemm_nt up to rounding. */
int ccsd_zgemm_nt_planes(int64_t M, int64_t N, int64_t K, const ccsd_c128* A, int64_t lda, const double* As,
                         const ccsd_c128* B, int64_t ldb, const double* Bs, ccsd_c128* C, int64_t csm, int64_t csn,
                         double alpha_re, double alpha_im, int accumulate, int mode, void* cuda_stream);

/*
 * ccsd_zgemm_nt by ONE level of Strassen's algorithm around the 3M DMMA kernels (the form ccsd_iterate uses for its four large
 * contractions when ccsd_options.strassen = 1): the operands are split in halves along M, N and K, the seven left and the seven
 * right operand combinations are written as two stacks with their sum planes (one streaming pass each), the seven half-size
 * products are ONE batched launch, and a third pass sums them into C (+)= alpha A B^T.  7/8 of the tensor-pipe work of
 * ccsd_zgemm_nt; same result up to rounding (pure FP64; max error a few 1e-15 of the largest element of C).  Any extents
 * >= 1 (odd halves are zero-padded inside the stacks); it pays from roughly M, K >= 1024, N >= 96.  mode 0, 3 or 100+v.
 * levels = 2 applies the scheme twice: 49 quarter-size products in one batched launch (0.766 of the plain work), the 49
 * operand combinations written straight from the 4 x 4 blocks of the operand and the 16 blocks of C summed straight from the
 * 49 products (one pass each, as for one level); it pays from roughly M, K >= 4096.
 * workspace: ccsd_zgemm_nt_strassen_workspace_bytes() bytes, 256-byte aligned, device.  Asynchronous on the stream.
 */
int ccsd_zgemm_nt_strassen_workspace_bytes(int64_t M, int64_t N, int64_t K, int levels, size_t* bytes);
int ccsd_zgemm_nt_strassen(int64_t M, int64_t N, int64_t K, const ccsd_c128* A, int64_t lda, const ccsd_c128* B, int64_t ldb,
                           ccsd_c128* C, int64_t csm, int64_t csn, double alpha_re, double alpha_im, int accumulate, int mode,
                           int levels, void* workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Tensor transposition ("A(a,c,b,d)+=B(a,b,c,d)"):  out[permuted index] = in[index]
 * (conj != 0: complex conjugate).  dims = extents of `in`; out dimension d is in dimension perm[d].
 */
int ccsd_transpose(const ccsd_c128* in, ccsd_c128* out, const int64_t dims[4], const int perm[4], int conj,
                   void* cuda_stream);

/* Real flops the DMMA GEMM kernels EXECUTE per complex multiply-add under `opts` (NULL = defaults): 8 for the 4M
 * scheme, 6 for 3M.  Algorithmic rates are always quoted on the 8-flop (ZGEMM) convention; the fraction of the FP64
 * peak must be computed from the executed flops so that it cannot exceed 1. */
int ccsd_real_flops_per_cmac(const ccsd_options* opts);

/* Per-step device times (ms, CUDA events) of the last ccsd_iterate/ccsd_residual when timing was enabled. */
enum { CCSD_NSTEPS = 16 };
int ccsd_enable_step_timing(ccsd_ctx* ctx, int enable);
int ccsd_get_step_times(ccsd_ctx* ctx, float ms[CCSD_NSTEPS]);
const char* ccsd_step_name(int step);
/* How ccsd_init built the packed <ab||cd> (the "transposes" metric; zeros in cc2 / direct_ladder mode):
 * stats[0..2] = summed device ms of {the slab GEMMs (ac|bd) over the auxiliary index, the slab transpositions, the
 * antisymmetrise-and-pack fills}, stats[3] = complex elements the transpositions moved (16 B read + 16 B written each),
 * stats[4] = packed elements written (two 16 B reads + one 16 B write each).  HOST out-pointer. */
enum { CCSD_NINIT_STATS = 5 };
int ccsd_get_init_stats(ccsd_ctx* ctx, double stats[CCSD_NINIT_STATS]);
/* Where this context uses the Strassen level (ccsd_options.strassen; it needs one GPU, the 3M kernels and ov >= 1024):
 * info[] = { any, the two (ov)^3 products (H^{ak}_{ci} quadratic term, ring), the pp-ladder, the <bk||cd> tau part of C }: the
 * number of levels L (0 = plain product).  Such a product executes (7/8)^L of the real flops of the plain one.  HOST out-pointer. */
int ccsd_strassen_info(ccsd_ctx* ctx, int info[4]);
/* Kernel launches issued by the library since the last reset (all contexts, this process). */
long long ccsd_launch_count(int reset);

/*
 * FP64 tensor-pipe yardstick: times a register-resident DMMA.8x8x4 (mma.sync.m8n8k4.f64) issue loop with no memory
 * traffic and returns the best of `launches` (~1 ms each) in TFLOP/s (HOST out-pointer).  device_scratch: >= 8 bytes.
 * This is the denominator of the "fraction of FP64 peak" numbers (148 SMs x 64 FMA/clk x 2 x SM clock).
 */
int ccsd_measure_fp64_peak(double* tflops, double* device_scratch, int launches, void* cuda_stream);

const char* ccsd_strerror(int status);
/* Last CUDA error string seen by the library on this thread ("" if none). */
const char* ccsd_last_cuda_error(void);

#ifdef __cplusplus
}
#endif
#endif /* CCSD_B200_H */
