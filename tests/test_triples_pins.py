"""Pins of the triples oracle (Appendix 7.3, eqs 39-44) against things other than itself (CPU).

All pins are determinant-space brute force (tests/detspace.py knows no working equation).  With V_N = H - F - const
(F = sum_pq f_pq a+_p a_q the Fock operator), P3 the projector on triply excited determinants and
R3 = sum_triples |Phi><Phi| / D:
  Q1  Wbar = <Phi_ijk^abc| V_N T2 |Phi_0>                      (eq 40 + the cyclic sum; every term, sign, bracket)
  Q2  Zbar = <Phi_ijk^abc| V_N T1 + F T2 |Phi_0>               (eq 42)
  Q3  Ybar = <Phi_ijk^abc| T1 T2 + T1^3/6 |Phi_0>              (eq 44)
  Q4  E(+T) = <0|T2+ V_N R3 V_N T2|0>;  E((T)) - E(+T) = <0|(T1+ V_N + T2+ F) R3 V_N T2|0>;
      E(-T) - E(+T) = <0|(T1 T2 + T1^3/6)+ P3 V_N T2|0>        (eqs 39, 41, 43: factors 1/36, denominators, conjugation)
  Q5  restricted (i<j<k) == full sum; the input re-indexing <ab||ie>, <am||ij>, <ab||ij> against the definition;
      E(+T) real and negative; all three real under Kramers symmetry.
"""
import itertools

import numpy as np
import pytest

import ccsd_inputs as ci
from oracle.ccsd_oracle import OracleCCSD, unpack_t2
from oracle.triples_oracle import OracleTriples
from tests.detspace import DetSpace, antisymmetrised_integrals, apply_string


def _setup(o, v, seed):
    inp = ci.make_inputs(o, v, 7, seed=seed, b_scale=0.3, f_offdiag=0.2)
    t1, t2p = ci.random_amplitudes(o, v, seed + 1, 0.3)
    t2 = unpack_t2(t2p, o, v)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    oc.set_amplitudes(t1, t2)
    return inp, oc, t1, t2


def _detspace(inp, oc, t1, t2):
    o, v = oc.o, oc.v
    ds = DetSpace(o + v, o)
    g = antisymmetrised_integrals(inp.B)
    H = ds.hamiltonian(inp.h, g)
    F = ds.one_body(oc.f)
    T1 = ds.cluster_operator(t1, np.zeros_like(t2))
    T2 = ds.cluster_operator(np.zeros_like(t1), t2)
    phi0 = np.zeros(ds.dim, dtype=np.complex128)
    phi0[ds.iref] = 1.0
    VN = H - F                                   # + a multiple of 1, which P3 removes below
    x = VN @ (T2 @ phi0)
    z = VN @ (T1 @ phi0) + F @ (T2 @ phi0)
    y = T1 @ (T2 @ phi0) + T1 @ (T1 @ (T1 @ phi0)) / 6.0
    return ds, x, z, y


def _triples_index(ds, o, v):
    """[(i,j,k,a,b,c, determinant index, sign)] for i<j<k, a<b<c: |Phi_ijk^abc> = a+_a a+_b a+_c a_k a_j a_i |Phi_0>."""
    out = []
    for i, j, k in itertools.combinations(range(o), 3):
        for a, b, c in itertools.combinations(range(v), 3):
            d2, s = apply_string(ds.ref, [o + a, o + b, o + c], [k, j, i])
            out.append((i, j, k, a, b, c, ds.index[d2], s))
    return out


@pytest.mark.parametrize("o,v", [(3, 3), (3, 4), (4, 4)])
def test_q1_q2_q3_drivers_equal_determinant_space(o, v):
    inp, oc, t1, t2 = _setup(o, v, 300 + 10 * o + v)
    ds, x, z, y = _detspace(inp, oc, t1, t2)
    ot = OracleTriples(oc)
    worst = {"W": 0.0, "Z": 0.0, "Y": 0.0}
    big = {"W": 0.0, "Z": 0.0, "Y": 0.0}
    cache = {}
    for i, j, k, a, b, c, idx, s in _triples_index(ds, o, v):
        if (i, j, k) not in cache:
            cache[(i, j, k)] = (ot.W(i, j, k)[1], ot.Z(i, j, k)[1], ot.Y(i, j, k)[1])
        Wb, Zb, Yb = cache[(i, j, k)]
        for name, blk, vec in (("W", Wb, x), ("Z", Zb, z), ("Y", Yb, y)):
            worst[name] = max(worst[name], abs(blk[a, b, c] - s * vec[idx]))
            big[name] = max(big[name], abs(vec[idx]))
    assert min(big.values()) > 0.05, big
    assert max(worst.values()) < 2e-13, worst
    # full antisymmetry of the cyclic sums (all index orders are then fixed by the i<j<k, a<b<c values)
    Wb = ot.W(0, 1, 2)[1]
    assert np.abs(Wb + Wb.transpose(1, 0, 2)).max() < 1e-13 and np.abs(Wb + Wb.transpose(0, 2, 1)).max() < 1e-13
    assert np.abs(Wb + ot.W(1, 0, 2)[1]).max() < 1e-13 and np.abs(Wb - ot.W(1, 2, 0)[1]).max() < 1e-13


@pytest.mark.parametrize("o,v", [(3, 3), (3, 4), (4, 4)])
def test_q4_energies_equal_perturbation_theory_in_determinant_space(o, v):
    inp, oc, t1, t2 = _setup(o, v, 500 + 10 * o + v)
    ds, x, z, y = _detspace(inp, oc, t1, t2)
    eps = oc.eps
    e4 = e5 = ey = 0.0
    for i, j, k, a, b, c, idx, s in _triples_index(ds, o, v):
        D = eps[i] + eps[j] + eps[k] - eps[o + a] - eps[o + b] - eps[o + c]
        e4 += np.conj(x[idx]) * x[idx] / D
        e5 += np.conj(z[idx]) * x[idx] / D
        ey += np.conj(y[idx]) * x[idx]
    ot = OracleTriples(oc)
    for restricted in (False, True):
        e = ot.energies(restricted=restricted)
        assert abs(e["+T"] - e4) < 1e-13 * max(1.0, abs(e4))
        assert abs(e["(T)"] - (e4 + e5)) < 1e-13 * max(1.0, abs(e4))
        assert abs(e["-T"] - (e4 + ey)) < 1e-13 * max(1.0, abs(e4))
    assert abs(e4) > 1e-3 and abs(e5) > 1e-4 and abs(ey) > 1e-4
    assert e4.real < 0 and abs(e4.imag) < 1e-15


def test_q5_reindexed_integrals_equal_definition():
    o, v = 3, 5
    inp, oc, t1, t2 = _setup(o, v, 42)
    g = antisymmetrised_integrals(inp.B)
    ot = OracleTriples(oc)
    assert np.abs(ot.vvov - g[o:, o:, :o, o:]).max() < 1e-14
    assert np.abs(ot.vooo - g[o:, :o, :o, :o]).max() < 1e-14
    assert np.abs(ot.vvoo - g[o:, o:, :o, :o]).max() < 1e-14


def test_q5_real_under_kramers_symmetry_complex_otherwise():
    kin = ci.make_kramers_inputs(2, 4, 12, seed=9)
    oc = OracleCCSD(kin.h, kin.B, kin.nocc, kin.nvir)
    oc.run(6)
    e = OracleTriples(oc).energies()
    for key in ("+T", "(T)", "-T"):
        assert abs(e[key].imag) < 1e-17 + 1e-14 * abs(e[key].real), (key, e[key])
        assert e[key].real < 0
    inp = ci.make_inputs(4, 8, 12, seed=9, b_scale=0.08)
    oc = OracleCCSD(inp.h, inp.B, 4, 8)
    oc.run(6)
    e = OracleTriples(oc).energies()
    assert abs(e["+T"].imag) < 1e-17 and abs(e["(T)"].imag) > 1e-12


def test_q6_single_element_evaluator_equals_plain_loop_oracle():
    """The from-B evaluator used for the full-size GPU spot checks equals the plain-loop oracle on a ragged system."""
    from oracle.ccsd_oracle import pack_t2
    from oracle.triples_oracle import wbar_samples_from_B
    o, v = 5, 7
    inp, oc, t1, t2 = _setup(o, v, 77)
    ot = OracleTriples(oc)
    rng = np.random.default_rng(3)
    ijk = [(0, 1, 2), (1, 3, 4), (0, 2, 4)]
    abc = [tuple(rng.permutation(v)[:3]) for _ in ijk]
    got = wbar_samples_from_B(inp.B, o, pack_t2(t2), ijk, abc)
    ref = np.array([ot.W(*t)[1][x] for t, x in zip(ijk, abc)])
    assert np.abs(got - ref).max() < 1e-13 * np.abs(ref).max() + 1e-15


def test_q7_partial_sums_over_occupied_triples_equal_determinant_space():
    """energies_of(list of i<j<k) = the determinant-space sums restricted to the triply excited determinants with those
    three holes (the unit of the multi-GPU split); the pieces of a partition add up to energies()."""
    o, v = 4, 4
    inp, oc, t1, t2 = _setup(o, v, 577)
    ds, x, z, y = _detspace(inp, oc, t1, t2)
    eps = oc.eps
    ot = OracleTriples(oc)
    all_triples = list(itertools.combinations(range(o), 3))
    parts = [all_triples[:1], all_triples[1:3], all_triples[3:], []]
    tot = {"+T": 0.0, "(T)": 0.0, "-T": 0.0}
    for part in parts:
        e4 = e5 = ey = 0.0
        for i, j, k, a, b, c, idx, s in _triples_index(ds, o, v):
            if tuple(sorted((i, j, k))) not in part:
                continue
            D = eps[i] + eps[j] + eps[k] - eps[o + a] - eps[o + b] - eps[o + c]
            e4 += np.conj(x[idx]) * x[idx] / D
            e5 += np.conj(z[idx]) * x[idx] / D
            ey += np.conj(y[idx]) * x[idx]
        e = ot.energies_of(part)
        assert abs(e["+T"] - e4) < 1e-13 and abs(e["(T)"] - (e4 + e5)) < 1e-13 and abs(e["-T"] - (e4 + ey)) < 1e-13
        if part:
            assert abs(e4) > 1e-5
        for key in tot:
            tot[key] += e[key]
    full = ot.energies(restricted=True)
    for key in tot:
        assert abs(tot[key] - full[key]) < 1e-13


def test_q8_triples_corrections_do_not_depend_on_the_level_shift():
    """The level shift (.LSHIFT) only preconditions the amplitude iterations: the converged amplitudes, and
    with them +T / (T) / -T (whose denominators are the spinor energies Re f_pp, eqs 39/41), must not depend on it."""
    o, v = 4, 7
    inp = ci.make_inputs(o, v, 12, seed=881, b_scale=0.12, f_offdiag=0.08)
    ref = None
    for shift in (0.0, 0.3):
        oc = OracleCCSD(inp.h, inp.B, o, v, level_shift=shift)
        hist = oc.run(400, tol=1e-13)
        assert hist[-1][1] < 1e-12
        e = OracleTriples(oc).energies(restricted=True)
        assert abs(e["+T"]) > 1e-6
        if ref is None:
            ref = e
        else:
            for key in ref:
                assert abs(e[key] - ref[key]) < 1e-10, (key, e[key], ref[key])
