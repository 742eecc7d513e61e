"""GPU parity of the Lambda equations and the one-body density (Appendix 7.4-7.5) against the
Lambda oracle (oracle/lambda_oracle.py, pinned by tests/test_lambda_pins.py).

Compared element by element (1e-12 relative max-abs): the right-hand sides of eqs 52-56 at seeded RANDOM multipliers
(every element of Hbar and every term enters) and at lambda = conj(t); the density matrix of eqs 58-61; lock-step
||R/D||_2 and multipliers over the iterations with DIIS(6).  Both sides start from their own converged amplitudes.
"""
import numpy as np
import pytest

import ccsd_inputs as ci

pytestmark = pytest.mark.gpu

REL_TOL = 1e-12


@pytest.fixture(scope="module")
def gpu():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import paper_2103_08473_b200 as lib
    lib.load_library()
    return lib


def _rel(a, b):
    scale = np.abs(b).max()
    return np.abs(np.asarray(a) - np.asarray(b)).max() / (scale if scale > 0 else 1.0)


def _pair(gpu, name):
    from oracle.ccsd_oracle import OracleCCSD
    from oracle.lambda_oracle import OracleLambda
    if name == "ragged":
        inp = ci.make_inputs(5, 13, 21, seed=4713, b_scale=0.06, f_offdiag=0.03)
    elif name == "ragged2":
        inp = ci.make_inputs(7, 18, 30, seed=4714)
    else:
        inp = ci.make_config(name)
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v)
    oc.run(80, tol=1e-13)
    gc = gpu.CCSD(inp.h, inp.B, o, v)
    ok, _, _, _ = gc.solve(1e-13, 80)
    assert ok
    return inp, oc, OracleLambda(oc), gc


@pytest.mark.parametrize("name", ["cfg0_2e", "cfg0", "ragged", "ragged2"])
def test_lambda_residual_and_density_match_oracle(gpu, name):
    from oracle.ccsd_oracle import pack_t2, unpack_t2
    inp, oc, ol, gc = _pair(gpu, name)
    o, v = inp.nocc, inp.nvir
    gc.lambda_init()
    # (a) at the start multipliers conj(t)
    R1, R2 = ol.residual()
    r1, r2p = gc.lambda_residual()
    assert _rel(r1.cpu().numpy(), R1) <= 1e-10 and _rel(r2p.cpu().numpy(), pack_t2(R2)) <= 1e-10   # t differs by ~1e-13
    # (b) at seeded random multipliers, same on both sides
    l1, l2p = ci.random_amplitudes(o, v, 44, 0.2)
    gc.set_lambda(l1, l2p)
    R1, R2 = ol.residual(l1, unpack_t2(l2p, o, v))
    r1, r2p = gc.lambda_residual()
    assert _rel(r1.cpu().numpy(), R1) <= 1e-10
    assert _rel(r2p.cpu().numpy(), pack_t2(R2)) <= 1e-10
    D = gc.density().cpu().numpy()
    assert _rel(D, ol.density(l1, unpack_t2(l2p, o, v))) <= 1e-10
    gc.close()


@pytest.mark.parametrize("strassen", [1, 3])
def test_lambda_exact_parity_at_identical_amplitudes(gpu, strassen):
    """Same amplitudes on both sides (the oracle's converged ones are handed to the library): 1e-12.  strassen = 3: the Lambda
    iteration's ladder and (ov)^3 product as 49 quarter-size products, <ab||cd> read back from the ladder's operand stack."""
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    from oracle.lambda_oracle import OracleLambda
    inp = ci.make_inputs(6, 15, 24, seed=4715)
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v)
    oc.run(80, tol=1e-13)
    ol = OracleLambda(oc)
    gc = gpu.CCSD(inp.h, inp.B, o, v, strassen=strassen)
    gc.set_amplitudes(oc.t1, pack_t2(oc.t2))
    gc.lambda_init()
    l1, l2p = ci.random_amplitudes(o, v, 45, 0.2)
    gc.set_lambda(l1, l2p)
    R1, R2 = ol.residual(l1, unpack_t2(l2p, o, v))
    r1, r2p = gc.lambda_residual()
    assert _rel(r1.cpu().numpy(), R1) <= REL_TOL
    assert _rel(r2p.cpu().numpy(), pack_t2(R2)) <= REL_TOL
    assert _rel(gc.density().cpu().numpy(), ol.density(l1, unpack_t2(l2p, o, v))) <= REL_TOL
    gc.close()


@pytest.mark.parametrize("name,nit", [("cfg0", 14), ("ragged", 10)])
def test_lambda_lockstep_iterations(gpu, name, nit):
    from oracle.ccsd_oracle import pack_t2
    inp, oc, ol, gc = _pair(gpu, name)
    gc.lambda_init()
    for _ in range(nit):
        so = ol.iterate()
        sg = gc.lambda_iterate()
        assert abs(sg - so) <= 1e-9 * max(1.0, so) + 1e-12
    l1, l2p = gc.get_lambda()
    assert _rel(l1.cpu().numpy(), ol.l1) <= 1e-9 and _rel(l2p.cpu().numpy(), pack_t2(ol.l2)) <= 1e-9
    assert _rel(gc.density().cpu().numpy(), ol.density()) <= 1e-9
    gc.close()


def test_lambda_cfg1_identical_amplitudes(gpu):
    """cfg1 (16/96): several DMMA tiles in every GEMM of the Lambda path.  The oracle's amplitudes after two CCSD
    iterations are handed to the library (the working equations are compared term for term; convergence of T is not
    needed for that); residuals at random multipliers, density, two lock-step iterations."""
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    from oracle.lambda_oracle import OracleLambda
    inp = ci.make_config("cfg1")
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v, restricted=True)
    for _ in range(2):
        oc.iterate()
    ol = OracleLambda(oc)
    gc = gpu.CCSD(inp.h, inp.B, o, v)
    gc.set_amplitudes(oc.t1, pack_t2(oc.t2))
    gc.lambda_init()
    l1, l2p = ci.random_amplitudes(o, v, 46, 0.05)
    gc.set_lambda(l1, l2p)
    R1, R2 = ol.residual(l1, unpack_t2(l2p, o, v))
    r1, r2p = gc.lambda_residual()
    assert _rel(r1.cpu().numpy(), R1) <= REL_TOL
    assert _rel(r2p.cpu().numpy(), pack_t2(R2)) <= REL_TOL
    assert _rel(gc.density().cpu().numpy(), ol.density(l1, unpack_t2(l2p, o, v))) <= REL_TOL
    gc.set_lambda(np.conj(oc.t1), np.conj(pack_t2(oc.t2)))
    for _ in range(2):
        so, sg = ol.iterate(), gc.lambda_iterate()
        assert abs(sg - so) <= 1e-10 * max(1.0, so)
    gc.close()


@pytest.mark.parametrize("cfg", ["cfg1", "cfg2", "cfg3"])
def test_fullsize_density_is_the_energy_derivative(gpu, cfg):
    """A property that holds at any size (eqs 15-16): with the converged Lambda, Tr(P D) equals
    dE_CCSD/d(eps) for h -> h + eps P.  The derivative is taken by central differences (Richardson) of CCSD energies
    the library converges itself (their parity with the oracle is tested elsewhere); the oracle-side version of this
    pin is tests/test_lambda_pins.py::test_l4."""
    inp = ci.make_config(cfg)
    o, v = inp.nocc, inp.nvir
    n = o + v
    rng = np.random.default_rng(7)
    X = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    P = 0.5 * (X + X.conj().T)

    def e_corr(eps):
        g = gpu.CCSD(inp.h + eps * P, inp.B, o, v)
        ok, _, e, _ = g.solve(1e-12, 200)
        g.close()
        assert ok
        return e

    gc = gpu.CCSD(inp.h, inp.B, o, v)
    ok, _, _, _ = gc.solve(1e-12, 200)
    assert ok
    gc.lambda_init()
    for it in range(300):
        if gc.lambda_iterate() < 1e-12:
            break
    else:
        raise AssertionError("Lambda iteration did not converge")
    D_dev = gc.density()
    D = D_dev.cpu().numpy()
    assert abs(gc.expectation(D_dev, P) - np.sum(P * D)) < 1e-13 * max(1.0, abs(np.sum(P * D)))     # eq 16 on the device
    gc.close()
    assert abs(np.trace(D)) < 1e-12
    h1, h2 = 2.5e-4, 5e-4             # eps |P| stays small against the orbital-energy gaps: truncation ~1e-10, round-off ~3e-9
    d1 = (e_corr(h1) - e_corr(-h1)) / (2 * h1)
    d2 = (e_corr(h2) - e_corr(-h2)) / (2 * h2)
    deriv = (4 * d1 - d2) / 3
    got = np.sum(P * D)
    assert abs(deriv - got) < 2e-8 * max(1.0, abs(deriv)), (deriv, got)


def test_lambda_edge_cases(gpu):
    """Minimal system (two occupied, two virtual spinors: one pair each), plain Jacobi (ndiis = 0) with shifted
    denominators, CC2 mode rejected, calls before ccsd_lambda_init rejected."""
    from paper_2103_08473_b200.binding import CCSDError
    from oracle.ccsd_oracle import OracleCCSD, pack_t2
    from oracle.lambda_oracle import OracleLambda
    for (o, v, nd, shift) in ((2, 2, 6, 0.0), (3, 5, 0, 0.3), (2, 7, 3, 0.0)):
        inp = ci.make_inputs(o, v, 6, seed=60 + o + v, b_scale=0.1, f_offdiag=0.05)
        oc = OracleCCSD(inp.h, inp.B, o, v, ndiis=nd, level_shift=shift)
        for _ in range(4):
            oc.iterate()
        ol = OracleLambda(oc, ndiis=nd)
        gc = gpu.CCSD(inp.h, inp.B, o, v, ndiis=nd, level_shift=shift)
        with pytest.raises(CCSDError):
            gc.lambda_iterate()
        gc.set_amplitudes(oc.t1, pack_t2(oc.t2))
        gc.lambda_init()
        for _ in range(5):
            so, sg = ol.iterate(), gc.lambda_iterate()
            assert abs(sg - so) <= 1e-11 * max(1.0, so) + 1e-14
        assert _rel(gc.density().cpu().numpy(), ol.density()) <= 1e-11
        gc.close()
    inp = ci.make_config("cfg0")
    gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir, cc2=True)
    with pytest.raises(CCSDError):
        gc.lambda_init()
    gc.close()


@pytest.mark.parametrize("gemm_mode", [1, 2, 3])
def test_lambda_under_every_gemm_mode(gpu, gemm_mode):
    """The Lambda path on the simple FMA kernels (1), the 4M DMMA kernels (2, no sum planes) and forced 3M (3)."""
    from oracle.ccsd_oracle import OracleCCSD, pack_t2
    from oracle.lambda_oracle import OracleLambda
    inp = ci.make_inputs(6, 14, 20, seed=4716)
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v)
    for _ in range(5):
        oc.iterate()
    ol = OracleLambda(oc)
    gc = gpu.CCSD(inp.h, inp.B, o, v, gemm_mode=gemm_mode)
    gc.set_amplitudes(oc.t1, pack_t2(oc.t2))
    gc.lambda_init()
    for _ in range(3):
        so, sg = ol.iterate(), gc.lambda_iterate()
        assert abs(sg - so) <= 1e-11 * max(1.0, so)
    assert _rel(gc.density().cpu().numpy(), ol.density()) <= 1e-11
    gc.close()


def test_lambda_in_ccd_mode_keeps_singles_multipliers_zero(gpu):
    """CCD: t1 = 0 and no singles constraint in the Lagrangian, so lambda^i_a = 0 throughout; the
    doubles multipliers follow eqs 52-54 with t1 = lambda1 = 0 (oracle: the same equations with both zeroed)."""
    from oracle.ccsd_oracle import OracleCCSD, pack_t2
    from oracle.lambda_oracle import OracleLambda
    inp = ci.make_inputs(4, 10, 24, seed=79, b_scale=0.08, f_offdiag=0.03)
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v, ndiis=0)
    oc.set_amplitudes(np.zeros_like(oc.t1), oc.t2)
    for _ in range(6):                                   # plain Jacobi CCD on the oracle side (as in the CCD parity test)
        _, S2 = oc.residual()
        oc.set_amplitudes(np.zeros_like(oc.t1), oc.t2 + S2 / oc.D2)
    gc = gpu.CCSD(inp.h, inp.B, o, v, ccd=True, ndiis=0)
    gc.set_amplitudes(oc.t1, pack_t2(oc.t2))
    ol = OracleLambda(oc, ndiis=0)
    ol.l1[:] = 0.0
    gc.lambda_init()
    for _ in range(4):
        so = ol.iterate()
        ol.l1[:] = 0.0
        gc.lambda_iterate()
    l1, l2p = gc.get_lambda()
    assert float(l1.abs().max()) == 0.0
    assert _rel(l2p.cpu().numpy(), pack_t2(ol.l2)) <= 1e-11
    gc.close()


def test_lambda_solve_converges_like_the_oracle_loop(gpu):
    """ccsd_lambda_solve: the same number of iterations to ||R/D||_2 < tol as the oracle's loop with the same test, the
    same converged multipliers and density; the iteration limit reports CCSD_ENOTCONVERGED (binding: converged False)."""
    from oracle.ccsd_oracle import pack_t2
    from paper_2103_08473_b200.binding import CCSDError
    inp, oc, ol, gc = _pair(gpu, "ragged")
    with pytest.raises(CCSDError):
        gc.lambda_solve(1e-10, 50)                       # before ccsd_lambda_init
    gc.lambda_init()
    tol, it_o = 1e-10, 0
    while it_o < 60:
        it_o += 1
        if ol.iterate() < tol:
            break
    ok, it_g, sn = gc.lambda_solve(tol, 60)
    assert ok and it_g == it_o and sn < tol
    l1, l2p = gc.get_lambda()
    assert _rel(l1.cpu().numpy(), ol.l1) <= 1e-9 and _rel(l2p.cpu().numpy(), pack_t2(ol.l2)) <= 1e-9
    assert _rel(gc.density().cpu().numpy(), ol.density()) <= 1e-9
    gc.lambda_init()
    ok, it_g, sn = gc.lambda_solve(1e-14, 2)
    assert not ok and it_g == 2 and sn > 1e-14
    with pytest.raises(CCSDError):
        gc.lambda_solve(0.0, 5)
    gc.close()
