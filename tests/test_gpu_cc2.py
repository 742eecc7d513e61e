"""GPU parity of the CC2 mode (Appendix 7.2) against the CC2 oracle (eqs 34-38 written out).

The library evaluates eq 34 as eq 32 with t2 -> 0 in the operands plus the two Fock terms; the oracle
evaluates eqs 34-38 literally.  Compared: S1, S2 (element by element), the terms that correspond one to one (driver,
f_vv.t2, f_oo.t2) and the sum of the other four; lock-step energies with DIIS(6) from the MP2 start.
Tolerances: 1e-12 relative max-abs per output tensor, 1e-10 Eh on energies (BASELINE.json north_star).
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
    scale = np.abs(b).max()
    return np.abs(np.asarray(a) - np.asarray(b)).max() / (scale if scale > 0 else 1.0)


def _g(gc, name):
    return gc.get_tensor(name).cpu().numpy().ravel()


CASES = [("cfg0", 0.2), ("cfg0_2e", 0.2), ("ragged", 0.05), ("cfg1", 0.01)]


@pytest.mark.parametrize("cfg,scale", CASES)
def test_cc2_residual_matches_oracle(gpu, cfg, scale):
    from oracle.cc2_oracle import OracleCC2
    from oracle.ccsd_oracle import pack_t2, unpack_t2
    if cfg == "ragged":
        o, v = 7, 29                      # several DMMA tiles with ragged tails in every dimension
        inp = ci.make_inputs(o, v, 37, seed=4711)
    else:
        inp = ci.make_config(cfg)
        o, v = inp.nocc, inp.nvir
    t1, t2p = ci.random_amplitudes(o, v, 21, scale)
    oc = OracleCC2(inp.h, inp.B, o, v)
    oc.set_amplitudes(t1, unpack_t2(t2p, o, v))
    S1, S2 = oc.residual()
    gc = gpu.CCSD(inp.h, inp.B, o, v, cc2=True)
    gc.set_amplitudes(t1, t2p)
    gc.residual()
    assert _rel(_g(gc, "S1"), S1.ravel()) <= REL_TOL
    assert _rel(_g(gc, "S2"), pack_t2(S2).ravel()) <= REL_TOL
    terms = {name: pack_t2(oc.cc2_s2(k)).ravel() for k, name in enumerate(oc.CC2_TERMS)}
    assert _rel(_g(gc, "S2_driver"), terms["driver"]) <= REL_TOL
    assert _rel(_g(gc, "S2_gvv"), terms["fvv_t2"]) <= REL_TOL
    assert _rel(_g(gc, "S2_goo"), terms["foo_t2"]) <= REL_TOL
    rest_gpu = _g(gc, "S2_vdag_t1") + _g(gc, "S2_c_t1") + _g(gc, "S2_hh_ladder") + _g(gc, "S2_pp_ladder")
    rest_orc = terms["t1_Wvvvo"] + terms["t1_Wovoo"] + terms["t1t1_Woooo"] + terms["t1t1_Wvvvv"]
    assert _rel(rest_gpu, rest_orc) <= REL_TOL
    gc.close()


@pytest.mark.parametrize("cfg,nit", [("cfg0", 12), ("cfg0_2e", 10), ("cfg1", 4)])
def test_cc2_lockstep_energies(gpu, cfg, nit):
    from oracle.cc2_oracle import OracleCC2
    inp = ci.make_config(cfg)
    oc = OracleCC2(inp.h, inp.B, inp.nocc, inp.nvir, ndiis=6)
    gc = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir, ndiis=6, cc2=True)
    assert abs(gc.energy() - oc.energy()) < E_TOL
    for _ in range(nit):
        eo, so = oc.iterate()
        eg, sg = gc.iterate()
        assert abs(eg - eo) < E_TOL, (eg, eo)
        assert abs(sg - so) < 1e-9 * max(1.0, so)
    gc.close()


def test_cc2_and_ccsd_modes_differ(gpu):
    """Guards against the flag being ignored: one CC2 and one CCSD iteration from the same start give different E."""
    inp = ci.make_config("cfg0")
    a = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir, cc2=True)
    b = gpu.CCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    ea, _ = a.iterate()
    eb, _ = b.iterate()
    assert abs(ea - eb) > 1e-8
    a.close(); b.close()


def test_cc2_minimal_size_and_level_shift(gpu):
    """nocc = nvir = 2 (one occupied pair, one virtual pair) and shifted denominators, lock-step against the oracle."""
    from oracle.cc2_oracle import OracleCC2
    for (o, v, shift) in ((2, 2, 0.0), (3, 5, 0.25)):
        inp = ci.make_inputs(o, v, 6, seed=50 + o, b_scale=0.1, f_offdiag=0.05)
        oc = OracleCC2(inp.h, inp.B, o, v, ndiis=3, level_shift=shift)
        gc = gpu.CCSD(inp.h, inp.B, o, v, ndiis=3, level_shift=shift, cc2=True)
        for _ in range(6):
            eo, so = oc.iterate()
            eg, sg = gc.iterate()
            assert abs(eg - eo) < E_TOL and abs(sg - so) < 1e-9 * max(1.0, so)
        gc.close()
