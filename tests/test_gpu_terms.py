"""GPU parity of the standalone intermediates: ccsd_contract terms F_OV, F_VV, F_OO, W_OOOO, W_OVVO, C_OVOO
(eqs 24-31) against the CPU oracle's intermediates at random amplitudes, element by element,
every input handed over in the canonical layouts of include/ccsd.h (made from the oracle's integral classes).
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
    return np.abs(np.asarray(a).ravel() - np.asarray(b).ravel()).max() / (scale if scale > 0 else 1.0)


def _setup(o, v, naux, seed):
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    inp = ci.make_inputs(o, v, naux, seed, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    t1, t2p = ci.random_amplitudes(o, v, seed + 1, scale=0.05)
    oc.set_amplitudes(t1, unpack_t2(t2p, o, v))
    oc.build_intermediates()
    io, jo = np.triu_indices(o, 1)
    av, bv = np.triu_indices(v, 1)
    can = {
        "f": oc.f,
        "oovv": oc.oovv[io[:, None], jo[:, None], av[None, :], bv[None, :]],
        "ooov": oc.ooov[io, jo],
        "oooo": oc.oooo[io[:, None], jo[:, None], io[None, :], jo[None, :]],
        "vovv": oc.vovv[:, :, av, bv],
        "vovo": oc.vovo,
        "t1": oc.t1, "t2": pack_t2(oc.t2),
    }
    can = {k: np.ascontiguousarray(x) for k, x in can.items()}
    want = {
        "f_ov": oc.Hov, "f_vv": oc.Gvv, "f_oo": oc.Goo,
        "w_oooo": oc.A[io[:, None], jo[:, None], io[None, :], jo[None, :]],
        "w_ovvo": oc.Hvovo, "c_ovoo": oc.C[:, :, io, jo],
    }
    return can, want


INPUTS = {
    "f_ov": ("f", "oovv", "t1"),
    "f_vv": ("f", "oovv", "vovv", "t1", "t2"),
    "f_oo": ("f", "oovv", "ooov", "t1", "t2"),
    "w_oooo": ("oooo", "ooov", "oovv", "t1", "t2"),
    "w_ovvo": ("vovo", "vovv", "ooov", "oovv", "t1", "t2"),
    "c_ovoo": ("ooov", "vovo", "vovv", "t1", "t2"),
}


@pytest.mark.parametrize("o,v,naux,seed", [(4, 6, 10, 31), (5, 11, 17, 32), (2, 2, 3, 33), (7, 13, 20, 34), (3, 30, 25, 35)])
def test_intermediate_terms(gpu, o, v, naux, seed):
    can, want = _setup(o, v, naux, seed)
    for term, names in INPUTS.items():
        got = gpu.contract(term, o, v, [can[k] for k in names]).cpu().numpy()
        assert got.shape == want[term].shape, term
        assert _rel(got, want[term]) < REL_TOL, (term, _rel(got, want[term]))


def test_intermediate_terms_gemm_modes(gpu):
    o, v = 6, 14
    can, want = _setup(o, v, 18, 41)
    for mode in (1, 2, 3):
        for term, names in INPUTS.items():
            got = gpu.contract(term, o, v, [can[k] for k in names], gemm_mode=mode).cpu().numpy()
            assert _rel(got, want[term]) < REL_TOL, (mode, term)


def test_intermediate_terms_feed_the_s2_terms(gpu):
    """The standalone intermediates chained into the standalone S2 contractions reproduce the oracle's S2 terms."""
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    o, v = 5, 9
    can, want = _setup(o, v, 14, 51)
    inp = ci.make_inputs(o, v, 14, 51, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    oc.set_amplitudes(can["t1"], unpack_t2(can["t2"], o, v))
    oc.build_intermediates()
    tau = gpu.contract("tau", o, v, [can["t1"], can["t2"]])
    A = gpu.contract("w_oooo", o, v, [can[k] for k in INPUTS["w_oooo"]])
    H = gpu.contract("w_ovvo", o, v, [can[k] for k in INPUTS["w_ovvo"]])
    hh = gpu.contract("hh_ladder", o, v, [A, tau]).cpu().numpy()
    ring = gpu.contract("ring", o, v, [H, can["t2"]]).cpu().numpy()
    assert _rel(hh, pack_t2(oc.s2_term("hh_ladder"))) < REL_TOL
    assert _rel(ring, pack_t2(oc.s2_term("ring"))) < REL_TOL


def test_intermediate_terms_errors(gpu):
    can, _ = _setup(4, 6, 10, 31)
    with pytest.raises(RuntimeError):
        gpu.contract("f_ov", 4, 6, [can[k] for k in INPUTS["f_ov"]], accumulate=True)
    with pytest.raises(RuntimeError):
        gpu.contract("f_ov", 1, 6, [can["f"], can["oovv"], can["t1"]])


# ---- the remaining rows of one iteration as standalone terms: S1 (eq 33), the small S2 terms (eq 32), energy, update ----
def _setup_residual(o, v, naux, seed, level_shift=0.0):
    from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
    can, _ = _setup(o, v, naux, seed)
    inp = ci.make_inputs(o, v, naux, seed, b_scale=0.1, f_offdiag=0.05)
    oc = OracleCCSD(inp.h, inp.B, o, v, ndiis=0, level_shift=level_shift)
    oc.set_amplitudes(can["t1"], unpack_t2(can["t2"], o, v))
    S1, S2 = oc.residual()
    io, jo = np.triu_indices(o, 1)
    can.update({"hvv": oc.Hvv, "hoo": oc.Hoo, "hov": oc.Hov, "gvv": oc.Gvv, "goo": oc.Goo,
                "c": oc.C[:, :, io, jo], "s1": S1, "s2": pack_t2(S2)})
    can = {k: np.ascontiguousarray(x) for k, x in can.items()}
    return can, oc


RESIDUAL_INPUTS = {
    "s1_residual": ("f", "hvv", "hoo", "hov", "vovv", "ooov", "vovo", "t1", "t2"),
    "s2_small_terms": ("gvv", "goo", "c", "vovv", "oovv", "t1", "t2"),
    "energy": ("f", "oovv", "t1", "t2"),
    "jacobi_update": ("f", "t1", "t2", "s1", "s2"),
}


@pytest.mark.parametrize("o,v,naux,seed", [(4, 6, 10, 61), (5, 11, 17, 62), (2, 2, 3, 63), (7, 13, 20, 64), (3, 30, 25, 65),
                                           (9, 4, 12, 66)])
def test_residual_terms(gpu, o, v, naux, seed):
    from oracle.ccsd_oracle import pack_t2
    can, oc = _setup_residual(o, v, naux, seed)
    got = gpu.contract("s1_residual", o, v, [can[k] for k in RESIDUAL_INPUTS["s1_residual"]]).cpu().numpy()
    assert _rel(got, oc.S1) < REL_TOL, ("s1", _rel(got, oc.S1))
    small = sum(oc.s2_term(name) for name in ("goo", "vdag_t1", "gvv", "c_t1", "driver"))
    got = gpu.contract("s2_small_terms", o, v, [can[k] for k in RESIDUAL_INPUTS["s2_small_terms"]]).cpu().numpy()
    assert _rel(got, pack_t2(small)) < REL_TOL, ("s2_small", _rel(got, pack_t2(small)))
    e = gpu.contract("energy", o, v, [can[k] for k in RESIDUAL_INPUTS["energy"]]).cpu().numpy()[0]
    want = oc.energy()
    assert abs(e - want) < 1e-12 * max(1.0, abs(want)), (e, want)


def test_small_terms_complete_the_residual(gpu):
    """Standalone intermediates -> ring + hh-ladder + pp-ladder + small terms = the oracle's full S2 (eq 32)."""
    from oracle.ccsd_oracle import pack_t2
    o, v = 5, 9
    can, oc = _setup_residual(o, v, 14, 71)
    av, bv = np.triu_indices(v, 1)
    Wp = np.ascontiguousarray(oc.vvvv[av[:, None], bv[:, None], av[None, :], bv[None, :]])
    tau = gpu.contract("tau", o, v, [can["t1"], can["t2"]])
    A = gpu.contract("w_oooo", o, v, [can[k] for k in INPUTS["w_oooo"]])
    H = gpu.contract("w_ovvo", o, v, [can[k] for k in INPUTS["w_ovvo"]])
    S2 = gpu.contract("s2_small_terms", o, v, [can[k] for k in RESIDUAL_INPUTS["s2_small_terms"]])
    gpu.contract("ring", o, v, [H, can["t2"]], out=S2, accumulate=True)
    gpu.contract("hh_ladder", o, v, [A, tau], out=S2, accumulate=True)
    gpu.contract("pp_ladder", o, v, [tau, Wp], out=S2, accumulate=True)
    assert _rel(S2.cpu().numpy(), can["s2"]) < REL_TOL


@pytest.mark.parametrize("shift,ccd", [(0.0, False), (0.35, False), (0.0, True)])
def test_jacobi_update_term(gpu, shift, ccd):
    """u = t + S/D (reading G12) against the oracle's plain-Jacobi step (ndiis = 0), with the level shift
    of PAPER.md:1062 and the CCD switch."""
    from oracle.ccsd_oracle import pack_t2
    o, v = 6, 11
    can, oc = _setup_residual(o, v, 16, 81, level_shift=shift)
    got = gpu.contract("jacobi_update", o, v, [can[k] for k in RESIDUAL_INPUTS["jacobi_update"]], level_shift=shift,
                       ccd=ccd).cpu().numpy()
    oc.iterate()   # ndiis = 0: t <- t + S/D
    want1 = np.zeros_like(oc.t1) if ccd else oc.t1
    assert _rel(got[: o * v].reshape(o, v), want1) < REL_TOL
    assert _rel(got[o * v:], pack_t2(oc.t2).ravel()) < REL_TOL


def test_residual_terms_gemm_modes_and_errors(gpu):
    from oracle.ccsd_oracle import pack_t2
    o, v = 6, 14
    can, oc = _setup_residual(o, v, 18, 91)
    small = pack_t2(sum(oc.s2_term(name) for name in ("goo", "vdag_t1", "gvv", "c_t1", "driver")))
    for mode in (1, 2, 3):
        got = gpu.contract("s1_residual", o, v, [can[k] for k in RESIDUAL_INPUTS["s1_residual"]], gemm_mode=mode).cpu().numpy()
        assert _rel(got, oc.S1) < REL_TOL, mode
        got = gpu.contract("s2_small_terms", o, v, [can[k] for k in RESIDUAL_INPUTS["s2_small_terms"]], gemm_mode=mode).cpu().numpy()
        assert _rel(got, small) < REL_TOL, mode
    for term, names in RESIDUAL_INPUTS.items():
        with pytest.raises(RuntimeError):
            gpu.contract(term, o, v, [can[k] for k in names], accumulate=True)
        with pytest.raises(RuntimeError):
            gpu.contract(term, 1, v, [can[k] for k in names])
