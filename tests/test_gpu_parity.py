"""GPU parity: the CUDA library (through its C ABI) against the CPU oracle, element by element.

Tolerances (BASELINE.json north_star): per contraction output max|delta| / max|oracle| <= 1e-12; energies <= 1e-10 Eh
(observed ~1e-14).  All inputs are seeded synthetic (ccsd_inputs.py); nothing reads /root/reference.
"""
import numpy as np
import pytest

import ccsd_inputs as ci

pytestmark = pytest.mark.gpu

REL_TOL = 1e-12
E_TOL = 1e-10


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2103_08473_b200 as lib
    lib.load_library()
    return lib


def _rel(a, b):
    a = np.asarray(a)
    b = np.asarray(b)
    scale = np.abs(b).max()
    return np.abs(a - b).max() / (scale if scale > 0 else 1.0)


def _triu(m):
    return np.triu_indices(m, 1)


def oracle_canonical(oc):
    """Oracle tensors re-laid-out in the canonical ABI layouts of include/ccsd.h."""
    from oracle.ccsd_oracle import pack_t2
    o, v = oc.o, oc.v
    io, jo = _triu(o)
    av, bv = _triu(v)
    d = {
        "fock": oc.f,
        "vvvv": oc.vvvv[av[:, None], bv[:, None], av[None, :], bv[None, :]],
        "vovv": oc.vovv[:, :, av, bv],
        "vovo": oc.vovo,
        "oovv": oc.oovv[io[:, None], jo[:, None], av[None, :], bv[None, :]],
        "ooov": oc.ooov[io, jo],
        "oooo": oc.oooo[io[:, None], jo[:, None], io[None, :], jo[None, :]],
        "tau": pack_t2(oc.tau),
        "Hvv": oc.Hvv, "Gvv": oc.Gvv, "Hoo": oc.Hoo, "Goo": oc.Goo, "Hov": oc.Hov, "Hvovo": oc.Hvovo,
        "C": oc.C[:, :, io, jo],
        "A": oc.A[io[:, None], jo[:, None], io[None, :], jo[None, :]],
        "S1": oc.S1, "S2": pack_t2(oc.S2),
    }
    for name in oc.TERMS:
        d["S2_" + name] = pack_t2(oc.s2_term(name))
    return {k: np.ascontiguousarray(x).ravel() for k, x in d.items()}


def compare_all(oc, gc, names=None, tol=REL_TOL):
    ref = oracle_canonical(oc)
    worst = {}
    for name, r in ref.items():
        if names is not None and name not in names:
            continue
        got = gc.get_tensor(name).cpu().numpy()
        assert got.shape == r.shape, name
        worst[name] = _rel(got, r)
    bad = {k: x for k, x in worst.items() if not x <= tol}
    assert not bad, f"parity failures (rel max-abs): {bad}\nall: {worst}"
    return worst


# the last two shapes have more occupied spinors than one 48-column GEMM tile and more occupied than virtual spinors
@pytest.mark.parametrize("o,v,L,gemm_mode", [(5, 11, 20, 1), (5, 11, 20, 0), (6, 16, 30, 0), (3, 9, 10, 0), (6, 16, 30, 2),
                                            (6, 16, 30, 3), (50, 20, 30, 0), (52, 7, 12, 0)])
def test_every_tensor_matches_oracle(gpu, o, v, L, gemm_mode):
    """All integral classes, all intermediates of eqs 24-31, all eight terms of eq 32, S1, S2: ragged sizes."""
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    inp = ci.make_inputs(o, v, L, seed=100 + o + v, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    gc = gpu.CCSD(inp.h, inp.B, o, v, gemm_mode=gemm_mode)
    # iteration 0: MP2 amplitudes (computed independently on each side)
    t1g, t2g = gc.get_amplitudes()
    assert _rel(t1g.cpu().numpy(), oc.t1) < REL_TOL
    assert _rel(t2g.cpu().numpy(), pack_t2(oc.t2)) < REL_TOL
    oc.residual()
    gc.residual()
    compare_all(oc, gc)
    assert abs(gc.energy() - oc.energy()) < 1e-13 * max(1.0, abs(oc.energy()))
    # seeded random antisymmetric amplitudes, CN(0, 0.01^2) and larger
    for seed, scale in ((1, 0.01), (2, 0.2)):
        t1, t2p = ci.random_amplitudes(o, v, seed, scale)
        oc.set_amplitudes(t1, unpack_t2(t2p, o, v))
        gc.set_amplitudes(t1, t2p)
        oc.residual()
        gc.residual()
        compare_all(oc, gc)
        assert abs(gc.energy() - oc.energy()) < 1e-12 * max(1.0, abs(oc.energy()))
    gc.close()


@pytest.mark.parametrize("o,v,L,gemm_mode", [(6, 16, 30, 0), (5, 11, 20, 0), (7, 13, 18, 0), (9, 8, 12, 0), (6, 16, 30, 3)])
def test_every_tensor_matches_oracle_with_strassen_levels_forced(gpu, o, v, L, gemm_mode):
    """ccsd_options.strassen = 3: all four large contractions as 49 quarter-size products at sizes the oracle finishes in seconds
    (odd halves and quarters: every zero-padding path), the packed <ab||cd> kept as the ladder's operand stack only (the "vvvv"
    entry below is rebuilt from it), S1 / G_vv / H_oo quartic terms read off the products of C, H^{ak}_{ci} and A.  Every tensor
    against the oracle, then six iterations in lock step."""
    from oracle.ccsd_oracle import OracleCCSD, unpack_t2
    inp = ci.make_inputs(o, v, L, seed=300 + o + v, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    gc = gpu.CCSD(inp.h, inp.B, o, v, strassen=3, gemm_mode=gemm_mode)
    assert gc.strassen_steps() == {"Hvovo_quad": 2, "ring_gemm": 2, "pp_ladder": 2, "C_ovoo": 2}
    for mode in (1, 2):      # the levels need the 3M kernels with sum planes: forced simple / 4M kernels run plain products
        other = gpu.CCSD(inp.h, inp.B, o, v, strassen=3, gemm_mode=mode)
        assert other.strassen_steps() == {}
        other.close()
    oc.residual()
    gc.residual()
    compare_all(oc, gc)
    t1, t2p = ci.random_amplitudes(o, v, 5, 0.2)
    oc.set_amplitudes(t1, unpack_t2(t2p, o, v))
    gc.set_amplitudes(t1, t2p)
    oc.residual()
    gc.residual()
    compare_all(oc, gc)
    assert abs(gc.energy() - oc.energy()) < 1e-12 * max(1.0, abs(oc.energy()))
    for it in range(6):
        eo, so = oc.iterate()
        eg, sg = gc.iterate()
        assert abs(eg - eo) < 1e-12 * max(1.0, abs(eo)), (it, eg, eo)
        assert abs(sg - so) < 1e-11 * max(1.0, so), (it, sg, so)
    gc.close()


@pytest.mark.parametrize("cfg,niter", [("cfg0_2e", 8), ("cfg0", 10)])
def test_lockstep_energies_tiny_configs(gpu, cfg, niter):
    from oracle.ccsd_oracle import OracleCCSD
    inp = ci.make_config(cfg)
    oc = OracleCCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    assert abs(gc.energy() - oc.energy()) < 1e-14
    for it in range(niter):
        eo, so = oc.iterate()
        eg, sg = gc.iterate()
        assert abs(eg - eo) < 1e-13, (it, eg, eo)
        assert abs(sg - so) < 1e-12 * max(1.0, so) + 1e-15, (it, sg, so)
    assert so < 1e-10          # converged: this is the converged-energy comparison of north_star
    assert abs(eg - eo) < E_TOL
    gc.close()


def test_lockstep_no_diis_and_level_shift(gpu):
    from oracle.ccsd_oracle import OracleCCSD
    inp = ci.make_inputs(4, 10, 24, seed=77, b_scale=0.06, f_offdiag=0.02)
    oc = OracleCCSD(inp.h, inp.B, 4, 10, ndiis=0, level_shift=0.25)
    gc = gpu.CCSD(inp.h, inp.B, 4, 10, ndiis=0, level_shift=0.25)
    for it in range(6):
        eo, so = oc.iterate()
        eg, sg = gc.iterate()
        assert abs(eg - eo) < 1e-13 and abs(sg - so) < 1e-13
    gc.close()


@pytest.mark.parametrize("strassen", [1, 3])
def test_ccd_mode_keeps_t1_zero(gpu, strassen):
    """CCD (PAPER.md:1044 .CCDOUBLES): t1 = 0 throughout; plain Jacobi on both sides."""
    from oracle.ccsd_oracle import OracleCCSD
    inp = ci.make_inputs(4, 10, 24, seed=78, b_scale=0.08, f_offdiag=0.03)
    gc = gpu.CCSD(inp.h, inp.B, 4, 10, ccd=True, ndiis=0, strassen=strassen)
    oc = OracleCCSD(inp.h, inp.B, 4, 10, ndiis=0)
    oc.set_amplitudes(np.zeros_like(oc.t1), oc.t2)
    for it in range(4):
        _, S2 = oc.residual()
        oc.set_amplitudes(np.zeros_like(oc.t1), oc.t2 + S2 / oc.D2)
        eg, _ = gc.iterate()
        assert abs(eg - oc.energy()) < 1e-13, it
    t1g, _ = gc.get_amplitudes()
    assert np.abs(t1g.cpu().numpy()).max() == 0.0
    gc.close()


def test_cfg1_lockstep_15_iterations(gpu):
    """BASELINE config 1 (nocc=16, nvir=96, L=336, DIIS(6), 15 iterations): energies after every iteration."""
    from oracle.ccsd_oracle import OracleCCSD
    inp = ci.make_config("cfg1")
    oc = OracleCCSD(inp.h, inp.B, inp.nocc, inp.nvir, restricted=True)
    gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    assert abs(gc.energy() - oc.energy()) < 1e-12
    oc.residual()
    gc.residual()
    compare_all(oc, gc, names={"Hvv", "Gvv", "Hoo", "Goo", "Hov", "Hvovo", "C", "A", "S1", "S2", "S2_pp_ladder",
                               "S2_ring", "S2_hh_ladder", "tau", "vvvv", "vovv"})
    for it in range(15):
        eo, so = oc.iterate()
        eg, sg = gc.iterate()
        assert abs(eg - eo) < 1e-11, (it, eg, eo)
    assert abs(eg - eo) < E_TOL
    gc.close()


# ------------------------------------------------------------------------------------------- standalone entries
@pytest.mark.parametrize("o,v", [(5, 12), (7, 20), (4, 9)])
def test_contract_terms(gpu, o, v):
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    inp = ci.make_inputs(o, v, 16, seed=5 + o, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    t1, t2p = ci.random_amplitudes(o, v, 3, 0.1)
    oc.set_amplitudes(t1, unpack_t2(t2p, o, v))
    oc.residual()
    ref = oracle_canonical(oc)
    oo, vv = ci.pair_count(o), ci.pair_count(v)
    tau = ref["tau"].reshape(oo, vv)
    got = gpu.contract("tau", o, v, [t1, t2p]).cpu().numpy()
    assert _rel(got.ravel(), ref["tau"]) < REL_TOL
    got = gpu.contract("pp_ladder", o, v, [tau, ref["vvvv"].reshape(vv, vv)]).cpu().numpy()
    assert _rel(got.ravel(), ref["S2_pp_ladder"]) < REL_TOL
    # the same contraction on the 4M kernels, the 3M kernels, and 3M with caller-supplied sum planes (as ccsd_iterate runs it)
    W = ref["vvvv"].reshape(vv, vv)
    for mode in (2, 3):
        got = gpu.contract("pp_ladder", o, v, [tau, W], gemm_mode=mode).cpu().numpy()
        assert _rel(got.ravel(), ref["S2_pp_ladder"]) < REL_TOL, mode
    taus, Ws = gpu.sum_plane(tau), gpu.sum_plane(W)
    assert np.array_equal(taus.cpu().numpy(), tau.real + tau.imag)
    got = gpu.contract("pp_ladder_planes", o, v, [tau, W, taus, Ws]).cpu().numpy()
    assert _rel(got.ravel(), ref["S2_pp_ladder"]) < REL_TOL
    got = gpu.contract("hh_ladder", o, v, [ref["A"].reshape(oo, oo), tau]).cpu().numpy()
    assert _rel(got.ravel(), ref["S2_hh_ladder"]) < REL_TOL
    got = gpu.contract("ring", o, v, [ref["Hvovo"].reshape(v, o, v, o), t2p]).cpu().numpy()
    assert _rel(got.ravel(), ref["S2_ring"]) < REL_TOL
    # accumulate
    import torch
    base = torch.from_numpy(t2p).cuda()
    out = gpu.contract("pp_ladder", o, v, [tau, ref["vvvv"].reshape(vv, vv)], out=base.clone(), accumulate=True)
    assert _rel(out.cpu().numpy().ravel(), ref["S2_pp_ladder"] + t2p.ravel()) < REL_TOL


@pytest.mark.parametrize("M,N,K", [(1, 1, 1), (37, 53, 29), (130, 70, 260), (64, 64, 64), (300, 9, 1000), (5, 700, 36)])
@pytest.mark.parametrize("mode", [0, 1, 2, 3])
def test_zgemm_nt_matches_oracle_samples(gpu, M, N, K, mode):
    from oracle.ccsd_oracle import nt_samples
    rng = np.random.default_rng(M * 1000 + N + K)
    A = rng.standard_normal((M, K)) + 1j * rng.standard_normal((M, K))
    B = rng.standard_normal((N, K)) + 1j * rng.standard_normal((N, K))
    C = gpu.zgemm_nt(A, B, alpha=0.5 - 0.25j, mode=mode).cpu().numpy()
    ms, ns = np.meshgrid(np.arange(M), np.arange(N), indexing="ij")
    ref = (0.5 - 0.25j) * nt_samples(A, B, ms.ravel(), ns.ravel()).reshape(M, N)
    assert _rel(C, ref) < REL_TOL
    Ct = gpu.zgemm_nt(A, B, alpha=0.5 - 0.25j, mode=mode, transposed_out=True).cpu().numpy()
    assert _rel(Ct.T, ref) < REL_TOL


@pytest.mark.parametrize("M,N,K", [(37, 53, 30), (130, 70, 260), (300, 9, 1002), (5, 700, 36), (129, 49, 18)])
@pytest.mark.parametrize("mode", [0, 111, 112])
def test_zgemm_nt_with_sum_planes(gpu, M, N, K, mode):
    """The 3M kernels reading caller-supplied sum planes (even K = leading dimension, ragged everything else)."""
    from oracle.ccsd_oracle import nt_samples
    rng = np.random.default_rng(M * 1000 + N + K)
    A = rng.standard_normal((M, K)) + 1j * rng.standard_normal((M, K))
    B = rng.standard_normal((N, K)) + 1j * rng.standard_normal((N, K))
    As, Bs = gpu.sum_plane(A), gpu.sum_plane(B)
    C = gpu.zgemm_nt(A, B, alpha=-0.75 + 0.5j, mode=mode, planes=(As, Bs)).cpu().numpy()
    ms, ns = np.meshgrid(np.arange(M), np.arange(N), indexing="ij")
    ref = (-0.75 + 0.5j) * nt_samples(A, B, ms.ravel(), ns.ravel()).reshape(M, N)
    assert _rel(C, ref) < REL_TOL


# the later shapes walk the tile variants of transpose.cuh: one 40-, 48- or 64-row tile for 32 < ny <= 64, merged y groups
# (two and three sub-dims) longer than one tile, ragged x, unit dims
@pytest.mark.parametrize("dims", [(3, 5, 7, 9), (34, 33, 2, 65), (1, 1, 40, 40), (8, 8, 8, 8), (5, 7, 33, 37),
                                  (34, 3, 70, 65), (66, 2, 2, 31), (3, 129, 5, 2), (64, 33, 9, 1), (47, 2, 41, 3)])
def test_transpose_all_permutations(gpu, dims):
    import itertools
    import torch
    rng = np.random.default_rng(7)
    x = rng.standard_normal(dims) + 1j * rng.standard_normal(dims)
    xd = torch.from_numpy(x).cuda()
    for perm in itertools.permutations(range(4)):
        for conj in (False, True):
            got = gpu.transpose(xd, list(perm), conj=conj).cpu().numpy()
            ref = np.transpose(x, perm)            # bit-exact data movement
            if conj:
                ref = ref.conj()
            assert np.array_equal(got, ref), (perm, conj)


def test_error_paths(gpu):
    import ctypes
    from paper_2103_08473_b200.binding import CCSDError
    inp = ci.make_config("cfg0_2e")
    with pytest.raises(CCSDError):
        gpu.CCSD(inp.h, inp.B, 1, inp.nvir + 1)          # nocc < 2 is rejected
    lib = gpu.load_library()
    assert lib.ccsd_iterate(None, None, None, None) == 4  # CCSD_ESTATE
    n = ctypes.c_size_t(0)
    assert lib.ccsd_contract_workspace_bytes(99, 4, 4, ctypes.byref(n)) == 1


def test_t1_diagnostic(gpu):
    """sqrt(sum |t1|^2 / nocc) of the amplitudes held by the library (reading G18)."""
    inp = ci.make_config("cfg0")
    gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    for _ in range(3):
        gc.iterate()
    t1 = gc.get_amplitudes()[0].cpu().numpy()
    ref = np.sqrt((np.abs(t1) ** 2).sum() / inp.nocc)
    assert abs(gc.t1_diagnostic() - ref) <= 1e-15 + 1e-13 * ref
    gc.close()


def test_solve_to_convergence(gpu):
    """ccsd_solve (.TCONVERG / .NCYCLES): stops when ||S/D|| and |dE| < tol; the converged energy
    equals the oracle's converged energy (independent of the DIIS details); the iteration limit is reported."""
    from oracle.ccsd_oracle import OracleCCSD
    inp = ci.make_config("cfg0")
    oc = OracleCCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    e_ref = oc.run(60, tol=1e-13)[-1][0]
    gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    ok, nit, e, sn = gc.solve(1e-11, 40)
    assert ok and nit < 40 and sn < 1e-11 and abs(e - e_ref) < E_TOL
    gc.close()
    gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    ok, nit, e, sn = gc.solve(1e-13, 2)
    assert not ok and nit == 2
    gc.close()


@pytest.mark.parametrize("o,v,L", [(5, 11, 20), (7, 29, 37)])
def test_direct_ladder_matches_oracle(gpu, o, v, L):
    """Integral-direct pp-ladder (opts.direct_ladder): <ab||cd> is rebuilt from B slab by slab in every iteration and never
    stored.  Same residuals and energies as the oracle; the pp-ladder term alone too; VVVV and Lambda are refused."""
    from oracle.ccsd_oracle import OracleCCSD, pack_t2
    from paper_2103_08473_b200.binding import CCSDError
    inp = ci.make_inputs(o, v, L, seed=990 + o)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    gc = gpu.CCSD(inp.h, inp.B, o, v, direct_ladder=True)
    t1, t2p = ci.random_amplitudes(o, v, 3, 0.05)
    from oracle.ccsd_oracle import unpack_t2
    oc.set_amplitudes(t1, unpack_t2(t2p, o, v))
    gc.set_amplitudes(t1, t2p)
    S1, S2 = oc.residual()
    gc.residual()
    assert _rel(gc.get_tensor("S2").cpu().numpy(), pack_t2(S2).ravel()) <= REL_TOL
    assert _rel(gc.get_tensor("S2_pp_ladder").cpu().numpy(), pack_t2(oc.s2_term("pp_ladder")).ravel()) <= REL_TOL
    assert _rel(gc.get_tensor("S1").cpu().numpy(), S1.ravel()) <= REL_TOL
    with pytest.raises(CCSDError):
        gc.get_tensor("vvvv")
    with pytest.raises(CCSDError):
        gc.lambda_init()
    oc.mp2_guess()
    gc.close()
    gc = gpu.CCSD(inp.h, inp.B, o, v, direct_ladder=True)
    for _ in range(5):
        eo, so = oc.iterate()
        eg, sg = gc.iterate()
        assert abs(eg - eo) < E_TOL and abs(sg - so) < 1e-9 * max(1.0, so)
    gc.close()


@pytest.mark.parametrize("strassen", [1, 3])
def test_two_contexts_on_two_streams_concurrently(gpu, strassen):
    """The C ABI takes a stream per context: two contexts iterating at the same time on two streams (from two host threads)
    share no scratch -- reduction partials, Gram matrix and DIIS coefficients (strassen = 3: the Strassen operand stacks and
    products too) are carved from each context's workspace -- and both reproduce the oracle's lock-step energies."""
    import threading
    import torch
    from oracle.ccsd_oracle import OracleCCSD
    cases = [ci.make_inputs(6, 20, 40, seed=4101, b_scale=0.06), ci.make_inputs(5, 24, 40, seed=4102, b_scale=0.06)]
    refs = []
    for inp in cases:
        oc = OracleCCSD(inp.h, inp.B, inp.nocc, inp.nvir)
        refs.append([oc.iterate() for _ in range(12)])
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    solvers = [gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir, stream=st, strassen=strassen) for inp, st in zip(cases, streams)]
    assert solvers[0].stream.cuda_stream != solvers[1].stream.cuda_stream
    out = [[], []]

    def work(k):
        torch.cuda.set_device(0)
        for _ in range(12):
            out[k].append(solvers[k].iterate())

    for rep in range(3):                       # several rounds: a race would not show every time
        out[0].clear(); out[1].clear()
        for k, inp in enumerate(cases):
            solvers[k].close()
            solvers[k] = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir, stream=streams[k], strassen=strassen)
        threads = [threading.Thread(target=work, args=(k,)) for k in range(2)]
        for t in threads:
            t.start()
        for t in threads:
            t.join()
        for k in range(2):
            for (eg, sg), (eo, so) in zip(out[k], refs[k]):
                assert abs(eg - eo) < E_TOL and abs(sg - so) < 1e-9 * max(1.0, so), (rep, k, eg, eo)
    for s_ in solvers:
        s_.close()


@pytest.mark.parametrize("strassen", [1, 3])
def test_graph_replay_equals_direct_launches_and_stale_tensors_are_refused(gpu, strassen):
    """opts.graph: the residual replayed as a CUDA graph gives bit-identical iterates to direct launches (same kernels, same
    data flow; strassen = 3: with two Strassen levels forced on the four large products); after ccsd_iterate the intermediates
    of the residual no longer belong to the current amplitudes, so ccsd_get_tensor refuses them (CCSD_ESTATE) until the next
    ccsd_residual."""
    from paper_2103_08473_b200.binding import CCSDError
    inp = ci.make_inputs(7, 30, 50, seed=4103, b_scale=0.05)
    a = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir, graph=True, strassen=strassen)
    b = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir, graph=False, strassen=strassen)
    n0 = gpu.launch_count()
    for it in range(8):
        ea, eb = a.iterate(), b.iterate()
        assert ea == eb, (it, ea, eb)
    assert gpu.launch_count() - n0 > 8 * 2 * 60           # replays are counted kernel by kernel
    with pytest.raises(CCSDError):
        a.get_tensor("Hvv")
    a.get_tensor("oovv")                                   # constants are always there
    a.residual()
    b.residual()
    for name in ("tau", "Hvv", "Hvovo", "S2", "S1"):
        assert torch_equal(a.get_tensor(name), b.get_tensor(name)), name
    a.close(); b.close()


def torch_equal(x, y):
    import torch
    return bool(torch.equal(x, y))
