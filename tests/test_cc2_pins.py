"""Pins of the CC2 oracle (Appendix 7.2, eqs 34-38) against things other than itself (CPU only).

C1  determinant-space definition of the CC2 doubles residual, brute force over all Slater determinants:
        S2 = <Phi_ij^ab| exp(-T1) H exp(T1) |Phi_0> + <Phi_ij^ab| [F, T2] |Phi_0>,   F = sum_pq f_pq a+_p a_q
    (CC2 = CCSD with the doubles equations kept to first order in the fluctuation potential, T1 treated as zeroth
    order; ref. 102 of the paper).  Pins every term, sign, factor 1/2, 1/4 and conjugation of eqs 34-38.
C2  the same doubles residual written through Appendix 7.1: CCSD eq 32 evaluated at t2 = 0 (pinned by P1) plus the
    two Fock terms -- a second, independently pinned route to every t1-only term.
C3  antisymmetry of each of the seven terms of eq 34.
C4  for two electrons with t1 = 0 and t2 = 0 the CC2 and CCSD doubles residuals coincide with <ab||ij>.
"""
import numpy as np
import pytest

import ccsd_inputs as ci
from oracle.cc2_oracle import OracleCC2
from oracle.ccsd_oracle import OracleCCSD, unpack_t2
from tests.detspace import DetSpace, antisymmetrised_integrals


def _amps(o, v, seed, scale):
    t1, t2p = ci.random_amplitudes(o, v, seed, scale)
    return t1, unpack_t2(t2p, o, v)


def _cc2_doubles_bruteforce(inp, o, v, f, t1, t2):
    ds = DetSpace(o + v, o)
    H = ds.hamiltonian(inp.h, antisymmetrised_integrals(inp.B))
    T1 = ds.cluster_operator(t1, np.zeros_like(t2))
    T2 = ds.cluster_operator(np.zeros_like(t1), t2)
    F = ds.one_body(f)
    w = ds.similarity_transformed_column(H, T1)
    phi0 = np.zeros(ds.dim, dtype=np.complex128)
    phi0[ds.iref] = 1.0
    w = w + F @ (T2 @ phi0) - T2 @ (F @ phi0)
    return ds.project_doubles(w)


@pytest.mark.parametrize("o,v", [(2, 3), (3, 3), (3, 4), (4, 4), (2, 5)])
def test_c1_cc2_doubles_equal_determinant_space_definition(o, v):
    inp = ci.make_inputs(o, v, 7, seed=700 + 10 * o + v, b_scale=0.3, f_offdiag=0.2)
    t1, t2 = _amps(o, v, 31 + o + v, 0.3)
    oc = OracleCC2(inp.h, inp.B, o, v)
    oc.set_amplitudes(t1, t2)
    S1, S2 = oc.residual()
    S2_bf = _cc2_doubles_bruteforce(inp, o, v, oc.f, t1, t2)
    assert np.abs(S2_bf).max() > 0.5
    assert np.abs(S2 - S2_bf).max() < 2e-13
    # singles are those of CCSD
    cc = OracleCCSD(inp.h, inp.B, o, v)
    cc.set_amplitudes(t1, t2)
    assert np.abs(S1 - cc.residual()[0]).max() == 0.0


def test_c1_sectors_t1_only_and_t2_only():
    o, v = 3, 4
    inp = ci.make_inputs(o, v, 5, seed=4343, b_scale=0.3, f_offdiag=0.2)
    t1, t2 = _amps(o, v, 6, 0.3)
    oc = OracleCC2(inp.h, inp.B, o, v)
    for a1, a2 in ((np.zeros_like(t1), t2), (t1, np.zeros_like(t2))):
        oc.set_amplitudes(a1, a2)
        S2 = oc.residual()[1]
        assert np.abs(S2 - _cc2_doubles_bruteforce(inp, o, v, oc.f, a1, a2)).max() < 2e-13


def test_c2_cc2_doubles_equal_ccsd_at_zero_t2_plus_fock_terms():
    o, v = 4, 6
    inp = ci.make_inputs(o, v, 9, seed=99, b_scale=0.3, f_offdiag=0.2)
    t1, t2 = _amps(o, v, 3, 0.3)
    oc = OracleCC2(inp.h, inp.B, o, v)
    oc.set_amplitudes(t1, t2)
    S2 = oc.residual()[1]
    cc = OracleCCSD(inp.h, inp.B, o, v)
    cc.set_amplitudes(t1, np.zeros_like(t2))
    ref = cc.residual()[1].copy()
    fvv, foo = oc.f[o:, o:], oc.f[:o, :o]
    x = np.einsum("be,ijae->ijab", fvv, t2)
    ref += x - x.transpose(0, 1, 3, 2)
    y = np.einsum("mj,imab->ijab", foo, t2)
    ref -= y - y.transpose(1, 0, 2, 3)
    assert np.abs(S2 - ref).max() < 2e-13


def test_c3_antisymmetry_of_every_term():
    o, v = 4, 5
    inp = ci.make_inputs(o, v, 6, seed=5, b_scale=0.3, f_offdiag=0.2)
    t1, t2 = _amps(o, v, 8, 0.3)
    oc = OracleCC2(inp.h, inp.B, o, v)
    oc.set_amplitudes(t1, t2)
    oc.cc2_intermediates()
    total = np.zeros_like(t2)
    for k, name in enumerate(oc.CC2_TERMS):
        x = oc.cc2_s2(k)
        assert np.abs(x).max() > 1e-3, name
        assert np.abs(x + x.transpose(1, 0, 2, 3)).max() < 1e-14, name
        assert np.abs(x + x.transpose(0, 1, 3, 2)).max() < 1e-14, name
        total += x
    assert np.abs(total - oc.cc2_s2(-1)).max() < 1e-13


def test_c4_zero_amplitudes_give_the_driver():
    o, v = 2, 4
    inp = ci.make_inputs(o, v, 5, seed=17)
    oc = OracleCC2(inp.h, inp.B, o, v)
    oc.set_amplitudes(np.zeros((o, v), complex), np.zeros((o, o, v, v), complex))
    S2 = oc.residual()[1]
    g = antisymmetrised_integrals(inp.B)
    assert np.abs(S2 - g[o:, o:, :o, :o].transpose(2, 3, 0, 1)).max() < 1e-15


def test_cc2_iteration_converges_near_ccsd_and_energy_real_under_kramers_symmetry():
    """CC2 run end to end from the MP2 start with DIIS: converges to an energy close to (not equal to) CCSD; under
    Kramers (time-reversal) symmetry the CC2 energy is real at every iteration, as for CCSD (pin P5)."""
    o, v, L, seed = ci.CONFIGS["cfg0"]
    inp = ci.make_inputs(o, v, L, seed)
    oc = OracleCC2(inp.h, inp.B, o, v)
    hist = oc.run(40, tol=1e-13)
    assert hist[-1][1] < 1e-13
    cc = OracleCCSD(inp.h, inp.B, o, v)
    e_ccsd = cc.run(40, tol=1e-13)[-1][0]
    assert 1e-9 < abs(hist[-1][0] - e_ccsd) < 1e-4
    kin = ci.make_kramers_inputs(2, 5, 12, seed=5)
    ok = OracleCC2(kin.h, kin.B, kin.nocc, kin.nvir)
    for e, _ in ok.run(12, tol=1e-14):
        assert abs(e.imag) < 1e-16 * max(1.0, abs(e.real)) + 1e-17
