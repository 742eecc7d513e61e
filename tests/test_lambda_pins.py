"""Pins of the Lambda / density oracle (Appendix 7.4-7.5, eqs 45-61) against things other than itself.

All CPU, determinant-space brute force (tests/detspace.py knows no working equation) or finite differences of the
pinned CCSD oracle:
  L1  R_mu = <0|(1+Lambda)(Hbar - E_CC)|mu> for singles and doubles, at converged T and RANDOM multipliers: pins every
      element of Hbar the equations use (eqs 45-49, 57 and the ones the paper leaves to its ref. 39; reading G23) and
      every term, sign, factor and permutation operator of eqs 50-56.
  L2  two electrons: the converged (1 + Lambda) is the left eigenvector of Hbar over the WHOLE determinant space
      (singles and doubles are all there is), with eigenvalue E_CC = E_FCI: pins the Jacobi/DIIS iteration end to end.
  L3  density blocks of eqs 58-61 = <0|(1+Lambda) exp(-T) a+_p a_q exp(T)|0> for random multipliers (reading G24);
      its trace vanishes.
  L4  the defining property of the Lagrange density (eqs 15-16): dE_CCSD/d(eps) for h -> h + eps P
      (central differences of the pinned CCSD oracle, re-converged at every eps) equals Tr(P D) with the CONVERGED
      Lambda: pins the Lambda solve and the density together against the amplitude equations.
  L5  re-indexed integral blocks against the definition; antisymmetry of R2.
"""
import itertools

import numpy as np
import pytest

import ccsd_inputs as ci
from oracle.ccsd_oracle import OracleCCSD, unpack_t2
from oracle.lambda_oracle import OracleLambda
from tests.detspace import DetSpace, antisymmetrised_integrals, apply_string


def _converged(o, v, seed, b_scale=0.12, f_off=0.08):
    inp = ci.make_inputs(o, v, 7, seed=seed, b_scale=b_scale, f_offdiag=f_off)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    hist = oc.run(300, tol=1e-14)
    assert hist[-1][1] < 1e-13
    return inp, oc


def _expm_nilpotent(ds, A, sign):
    out = np.eye(ds.dim, dtype=np.complex128)
    term = out.copy()
    for k in range(1, ds.nelec + 3):
        term = sign * (A @ term) / k
        out = out + term
    return out


def _left_vector(ds, o, v, l1, l2):
    """<0|(1 + Lambda) as a row vector; returns it with the (index, sign) maps of the singles and doubles."""
    L = np.zeros(ds.dim, dtype=np.complex128)
    L[ds.iref] = 1.0
    sing, doub = {}, {}
    for i in range(o):
        for a in range(v):
            d2, s = apply_string(ds.ref, [o + a], [i])
            sing[(i, a)] = (ds.index[d2], s)
            L[ds.index[d2]] += s * l1[i, a]
    for i, j in itertools.combinations(range(o), 2):
        for a, b in itertools.combinations(range(v), 2):
            d2, s = apply_string(ds.ref, [o + a, o + b], [j, i])
            doub[(i, j, a, b)] = (ds.index[d2], s)
            L[ds.index[d2]] += s * l2[i, j, a, b]
    return L, sing, doub


def _random_multipliers(o, v, seed, scale=0.3):
    l1, l2p = ci.random_amplitudes(o, v, seed, scale)
    return l1, unpack_t2(l2p, o, v)


@pytest.mark.parametrize("o,v", [(2, 3), (3, 3), (3, 4), (2, 5), (4, 4)])
def test_l1_residuals_equal_determinant_space_definition(o, v):
    inp, oc = _converged(o, v, 11 + o + v)
    ol = OracleLambda(oc)
    l1, l2 = _random_multipliers(o, v, 9)
    R1, R2 = ol.residual(l1, l2)
    ds = DetSpace(o + v, o)
    H = ds.hamiltonian(inp.h, antisymmetrised_integrals(inp.B))
    T = ds.cluster_operator(oc.t1, oc.t2)
    Hbar = _expm_nilpotent(ds, T, -1.0) @ H @ _expm_nilpotent(ds, T, 1.0)
    e_cc = Hbar[ds.iref, ds.iref]
    L, sing, doub = _left_vector(ds, o, v, l1, l2)
    row = L @ Hbar - e_cc * L
    e1 = max(abs(s * row[idx] - R1[i, a]) for (i, a), (idx, s) in sing.items())
    e2 = max(abs(s * row[idx] - R2[i, j, a, b]) for (i, j, a, b), (idx, s) in doub.items()) if doub else 0.0
    assert np.abs(R1).max() > 0.3 and np.abs(R2).max() > 0.3
    assert e1 < 5e-13 and e2 < 5e-13, (e1, e2)
    assert np.abs(R2 + R2.transpose(1, 0, 2, 3)).max() < 1e-13 and np.abs(R2 + R2.transpose(0, 1, 3, 2)).max() < 1e-13


def test_l2_two_electron_lambda_is_the_left_eigenvector():
    o, v = 2, 5
    inp, oc = _converged(o, v, 21, b_scale=0.15, f_off=0.1)
    ol = OracleLambda(oc)
    hist = ol.run(200, tol=1e-13)
    assert hist[-1] < 1e-13
    ds = DetSpace(o + v, o)
    H = ds.hamiltonian(inp.h, antisymmetrised_integrals(inp.B))
    T = ds.cluster_operator(oc.t1, oc.t2)
    Hbar = _expm_nilpotent(ds, T, -1.0) @ H @ _expm_nilpotent(ds, T, 1.0)
    L, _, _ = _left_vector(ds, o, v, ol.l1, ol.l2)
    e_cc = Hbar[ds.iref, ds.iref]
    assert np.abs(L @ Hbar - e_cc * L).max() < 1e-11
    assert abs(e_cc - np.linalg.eigvalsh(H)[0]) < 1e-11                      # = FCI for two electrons (pin P2)


@pytest.mark.parametrize("o,v", [(2, 3), (3, 4)])
def test_l3_density_blocks_equal_determinant_space(o, v):
    inp, oc = _converged(o, v, 31 + o)
    ol = OracleLambda(oc)
    l1, l2 = _random_multipliers(o, v, 5)
    D = ol.density(l1, l2)
    n = o + v
    ds = DetSpace(n, o)
    T = ds.cluster_operator(oc.t1, oc.t2)
    em, ep = _expm_nilpotent(ds, T, -1.0), _expm_nilpotent(ds, T, 1.0)
    L, _, _ = _left_vector(ds, o, v, l1, l2)
    left = L @ em
    ref = np.zeros((n, n), dtype=np.complex128)
    for p in range(n):
        for q in range(n):
            e = np.zeros((n, n)); e[p, q] = 1.0
            ref[p, q] = (left @ ds.one_body(e) @ ep)[ds.iref]
    ref -= np.diag([1.0] * o + [0.0] * v)
    assert np.abs(ref).max() > 0.01
    assert np.abs(D - ref).max() < 1e-14
    assert abs(np.trace(D)) < 1e-14


def test_l4_density_is_the_energy_derivative():
    o, v = 3, 5
    inp, oc = _converged(o, v, 41)
    ol = OracleLambda(oc)
    assert ol.run(200, tol=1e-13)[-1] < 1e-13
    D = ol.density()
    n = o + v
    rng = np.random.default_rng(3)
    X = rng.standard_normal((n, n)) + 1j * rng.standard_normal((n, n))
    P = 0.5 * (X + X.conj().T)                                              # Hermitian one-body perturbation

    def e_corr(eps):
        c = OracleCCSD(inp.h + eps * P, inp.B, o, v)
        return c.run(300, tol=1e-14)[-1][0]

    h1, h2 = 1e-3, 2e-3
    d1 = (e_corr(h1) - e_corr(-h1)) / (2 * h1)
    d2 = (e_corr(h2) - e_corr(-h2)) / (2 * h2)
    deriv = (4 * d1 - d2) / 3                                               # Richardson: error O(h^4)
    assert abs(deriv - np.sum(P * D)) < 1e-9 * max(1.0, abs(deriv)), (deriv, np.sum(P * D))
    assert abs(deriv) > 1e-3


def test_l5_reindexed_blocks_equal_definition():
    o, v = 3, 4
    inp, oc = _converged(o, v, 51)
    ol = OracleLambda(oc)
    g = antisymmetrised_integrals(inp.B)
    O, V = slice(0, o), slice(o, o + v)
    for got, ref in ((ol.ovvo, g[O, V, V, O]), (ol.ovoo, g[O, V, O, O]), (ol.vvvo, g[V, V, V, O]),
                     (ol.ovvv, g[O, V, V, V]), (ol.oovo, g[O, O, V, O])):
        assert np.abs(got - ref).max() < 1e-14
