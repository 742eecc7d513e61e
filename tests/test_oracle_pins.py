"""Pins of the CPU oracle against things other than itself (CPU only; run with -m "not gpu").

P1  determinant-space brute force of <Phi_mu|exp(-T) H exp(T)|Phi_0>  (eqs 5, 8-11)
    pins every term, sign, factor and conjugation of eqs 23-33 and the energy expression.
P2  CCSD == FCI for two electrons: pins the whole iteration (update, DIIS, energy).
P3  closed-form MP2 from the MP2 start.
P4  antisymmetry of t2, S2 and of each of the eight terms of eq 32.
P5  real energy under Kramers (time-reversal) symmetry; complex for a generic Hermitian input.
P7  restricted-sum mode == full-sum mode.
P8  permutational / Hermitian symmetry of the integral classes; Fock build returns the generator's f.
P9  SOFT cross-check against the energies printed in SURVEY.md 8(c) (an independent numpy/BLAS scratch
    implementation by the survey, same input recipe) -- not the paper's numbers.
"""
import os

import numpy as np
import pytest

import ccsd_inputs as ci
from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
from tests.detspace import DetSpace, antisymmetrised_integrals

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _random_unpacked_amplitudes(o, v, seed, scale):
    t1, t2p = ci.random_amplitudes(o, v, seed, scale)
    return t1, unpack_t2(t2p, o, v)


# ----------------------------------------------------------------------------------------------------------- P1
@pytest.mark.parametrize("o,v", [(2, 3), (3, 3), (3, 4), (4, 4), (2, 5)])
@pytest.mark.parametrize("restricted", [False, True])
def test_p1_residual_equals_determinant_space(o, v, restricted):
    inp = ci.make_inputs(o, v, 7, seed=900 + 10 * o + v, b_scale=0.3, f_offdiag=0.2)
    t1, t2 = _random_unpacked_amplitudes(o, v, 77 + o + v, 0.3)
    oc = OracleCCSD(inp.h, inp.B, o, v, restricted=restricted)
    oc.set_amplitudes(t1, t2)
    S1, S2 = oc.residual()
    E = oc.energy()

    ds = DetSpace(o + v, o)
    g = antisymmetrised_integrals(inp.B)
    H = ds.hamiltonian(inp.h, g)
    T = ds.cluster_operator(t1, t2)
    w = ds.similarity_transformed_column(H, T)
    e_ref = H[ds.iref, ds.iref]
    S1_bf, S2_bf = ds.project_singles(w), ds.project_doubles(w)
    assert np.abs(S2_bf).max() > 0.5 and np.abs(S1_bf).max() > 0.1      # large couplings: nothing hides
    assert np.abs(S1 - S1_bf).max() < 2e-13
    assert np.abs(S2 - S2_bf).max() < 2e-13
    assert abs(E - (w[ds.iref] - e_ref)) < 1e-13
    # the Fock matrix really is the one-particle part of H relative to Phi_0
    assert abs(oc.reference_energy(inp.h) - e_ref.real) < 1e-12 and abs(e_ref.imag) < 1e-13


def test_p1_ccd_and_singles_only_sectors():
    """t1 = 0 and t2 = 0 separately, so a term that cancels in the mixed case cannot hide."""
    o, v = 3, 4
    inp = ci.make_inputs(o, v, 5, seed=4242, b_scale=0.3, f_offdiag=0.2)
    ds = DetSpace(o + v, o)
    H = ds.hamiltonian(inp.h, antisymmetrised_integrals(inp.B))
    t1, t2 = _random_unpacked_amplitudes(o, v, 5, 0.3)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    for a1, a2 in ((np.zeros_like(t1), t2), (t1, np.zeros_like(t2))):
        oc.set_amplitudes(a1, a2)
        S1, S2 = oc.residual()
        w = ds.similarity_transformed_column(H, ds.cluster_operator(a1, a2))
        assert np.abs(S1 - ds.project_singles(w)).max() < 2e-13
        assert np.abs(S2 - ds.project_doubles(w)).max() < 2e-13


# ----------------------------------------------------------------------------------------------------------- P2
@pytest.mark.parametrize("b_scale,f_off,nit", [(ci.B_SCALE, ci.F_OFFDIAG, 30), (0.15, 0.1, 80)])
def test_p2_two_electron_ccsd_equals_fci(b_scale, f_off, nit):
    o, v, L, seed = ci.CONFIGS["cfg0_2e"]
    inp = ci.make_inputs(o, v, L, seed, b_scale=b_scale, f_offdiag=f_off)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    hist = oc.run(nit, tol=1e-14)
    e_ccsd = hist[-1][0]
    assert hist[-1][1] < 1e-12
    ds = DetSpace(o + v, o)
    H = ds.hamiltonian(inp.h, antisymmetrised_integrals(inp.B))
    assert np.abs(H - H.conj().T).max() < 1e-14
    e_fci = np.linalg.eigvalsh(H)[0]
    e_ref = H[ds.iref, ds.iref].real
    assert abs(e_ccsd.real - (e_fci - e_ref)) < 5e-14
    assert abs(e_ccsd.imag) < 1e-15                       # exactly real for N = 2


# ----------------------------------------------------------------------------------------------------------- P3
def test_p3_mp2_closed_form():
    inp = ci.make_config("cfg0")
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v)
    g = antisymmetrised_integrals(inp.B)
    eps = inp.f_target.diagonal().real
    eo, ev = eps[:o], eps[o:]
    D2 = eo[:, None, None, None] + eo[None, :, None, None] - ev[None, None, :, None] - ev[None, None, None, :]
    D1 = eo[:, None] - ev[None, :]
    e_d = 0.25 * np.sum(np.abs(g[:o, :o, o:, o:]) ** 2 / D2)
    e_s = np.sum(np.abs(inp.f_target[:o, o:]) ** 2 / D1)
    # MP2 amplitudes themselves
    assert np.abs(oc.t2 - np.conj(g[:o, :o, o:, o:]) / D2).max() < 1e-15
    assert np.abs(oc.t1 - np.conj(inp.f_target[:o, o:]) / D1).max() < 1e-15
    # doubles-only and singles-only energies are the closed forms and real; the t1*t1 cross term is separate
    t1, t2 = oc.t1.copy(), oc.t2.copy()
    oc.set_amplitudes(np.zeros_like(t1), t2)
    ed = oc.energy()
    assert abs(ed.real - e_d) < 1e-15 and abs(ed.imag) < 1e-17
    oc.set_amplitudes(t1, np.zeros_like(t2))
    es = oc.energy()
    cross = 0.5 * np.einsum("ijab,ia,jb->", g[:o, :o, o:, o:], t1, t1)
    assert abs(es - (e_s + cross)) < 1e-15
    assert e_d < 0 and e_s < 0


# ----------------------------------------------------------------------------------------------------------- P4
def _assert_antisym(x, tol):
    assert np.abs(x + x.transpose(1, 0, 2, 3)).max() < tol
    assert np.abs(x + x.transpose(0, 1, 3, 2)).max() < tol


@pytest.mark.parametrize("restricted", [False, True])
def test_p4_antisymmetry(restricted):
    inp = ci.make_inputs(3, 5, 9, seed=31, b_scale=0.2, f_offdiag=0.1)
    oc = OracleCCSD(inp.h, inp.B, 3, 5, restricted=restricted)
    t1, t2 = _random_unpacked_amplitudes(3, 5, 32, 0.2)
    oc.set_amplitudes(t1, t2)
    S1, S2 = oc.residual()
    _assert_antisym(S2, 1e-14)
    total = np.zeros_like(S2)
    for name in oc.TERMS:
        term = oc.s2_term(name)
        assert np.abs(term).max() > 1e-3, name
        _assert_antisym(term, 1e-14)
        total += term
    assert np.abs(total - S2).max() < 1e-14
    _assert_antisym(oc.A.transpose(2, 3, 0, 1), 1e-14)         # A antisymmetric in ij (and in kl)
    _assert_antisym(oc.A, 1e-14) if False else None
    assert np.abs(oc.A + oc.A.transpose(1, 0, 2, 3)).max() < 1e-14
    assert np.abs(oc.C + oc.C.transpose(0, 1, 3, 2)).max() < 1e-14
    for _ in range(3):
        oc.iterate()
        _assert_antisym(oc.t2, 1e-15)


# ----------------------------------------------------------------------------------------------------------- P5
def test_p5_energy_real_under_kramers_symmetry():
    inp = ci.make_kramers_inputs(2, 5, 12, seed=5)
    oc = OracleCCSD(inp.h, inp.B, inp.nocc, inp.nvir)
    assert np.abs(oc.f - inp.f_target).max() < 1e-13
    for it in range(12):
        e, _ = oc.iterate()
        assert abs(e.imag) < 1e-15 * max(1.0, abs(e.real)), (it, e)
    assert e.real < -1e-3
    # an unstructured input of similar strength has a complex energy
    gen = ci.make_inputs(4, 10, 12, seed=5, b_scale=0.08, f_offdiag=0.05)
    og = OracleCCSD(gen.h, gen.B, 4, 10)
    for _ in range(6):
        e2, _ = og.iterate()
    assert abs(e2.imag) > 1e-9


# ----------------------------------------------------------------------------------------------------------- P7
def test_p7_restricted_equals_full():
    o, v = 4, 9
    inp = ci.make_inputs(o, v, 20, seed=8, b_scale=0.1, f_offdiag=0.05)
    a = OracleCCSD(inp.h, inp.B, o, v, restricted=False)
    b = OracleCCSD(inp.h, inp.B, o, v, restricted=True)
    for name in ("oooo", "ooov", "oovv", "vovo", "vovv", "vvvv"):
        assert np.array_equal(getattr(a, name), getattr(b, name)) or \
            np.abs(getattr(a, name) - getattr(b, name)).max() < 1e-17, name
    t1, t2 = _random_unpacked_amplitudes(o, v, 9, 0.1)
    for oc in (a, b):
        oc.set_amplitudes(t1, t2)
        oc.residual()
    scale = np.abs(a.S2).max()
    assert np.abs(a.S2 - b.S2).max() < 1e-14 * max(1.0, scale)
    assert np.abs(a.S1 - b.S1).max() < 1e-14
    for name in ("Hvv", "Gvv", "Hoo", "Goo", "Hov", "Hvovo", "C", "A"):
        assert np.abs(getattr(a, name) - getattr(b, name)).max() < 1e-14, name
    assert abs(a.energy() - b.energy()) < 1e-15
    ha, hb = a.run(6), b.run(6)
    for (ea, _), (eb, _) in zip(ha, hb):
        assert abs(ea - eb) < 1e-14


# ----------------------------------------------------------------------------------------------------------- P8
def test_p8_integral_symmetries_and_fock():
    inp = ci.make_config("cfg0")
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v)
    assert np.abs(oc.f - inp.f_target).max() < 1e-13          # Fock build vs the generator's target
    assert np.abs(oc.f - oc.f.conj().T).max() < 1e-15
    g = antisymmetrised_integrals(inp.B)                     # independent einsum route
    O, V = slice(0, o), slice(o, o + v)
    for name, blk in (("oooo", g[O, O, O, O]), ("ooov", g[O, O, O, V]), ("oovv", g[O, O, V, V]),
                      ("vovo", g[V, O, V, O]), ("vovv", g[V, O, V, V]), ("vvvv", g[V, V, V, V])):
        assert np.abs(getattr(oc, name) - blk).max() < 1e-16, name
    w = oc.vvvv
    assert np.abs(w - w.transpose(2, 3, 0, 1).conj()).max() < 1e-17     # <ab||cd> = conj <cd||ab>
    assert np.abs(w + w.transpose(1, 0, 2, 3)).max() < 1e-17
    assert np.abs(w + w.transpose(0, 1, 3, 2)).max() < 1e-17


def test_pack_unpack_roundtrip():
    t1, t2p = ci.random_amplitudes(5, 7, 3)
    t2 = unpack_t2(t2p, 5, 7)
    assert np.array_equal(pack_t2(t2), t2p)
    assert t2[1, 3, 2, 6] == t2p[ci.pair_index(1, 3, 5), ci.pair_index(2, 6, 7)]
    assert t2[3, 1, 2, 6] == -t2[1, 3, 2, 6] and t2[1, 3, 6, 2] == -t2[1, 3, 2, 6]


# ----------------------------------------------------------------------------------------------------------- P9
def test_p9_soft_reference_energies_from_survey():
    """energies printed by the survey's independent scratch implementation."""
    rows = {}
    with open(os.path.join(GOLDEN, "survey_soft_energies.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            cfg, key, re_, im_ = line.split()
            rows[(cfg, key)] = (float(re_), None if im_ == "-" else float(im_))
    for cfg in ("cfg0_2e", "cfg0"):
        inp = ci.make_config(cfg)
        oc = OracleCCSD(inp.h, inp.B, inp.nocc, inp.nvir)
        e0 = oc.energy()
        hist = oc.run(30, tol=1e-14)
        for key, e in (("E_iter0", e0), ("E_ccsd", hist[-1][0])):
            re_, im_ = rows[(cfg, key)]
            assert abs(e.real - re_) < 2e-13, (cfg, key, e)
            if im_ is not None:
                assert abs(e.imag - im_) < max(2e-13, 5e-3 * abs(im_)), (cfg, key, e)


def test_sampled_evaluators_from_B_equal_the_plain_loop_oracle():
    """The single-element evaluators used for the full-size (cfg2/cfg3) spot checks are pinned to the explicit-loop
    oracle on a small ragged system: <pq||rs> samples, the pp-ladder of eq 32 and H^k_c of eq 28."""
    from oracle import ccsd_oracle as orc
    o, v, L = 5, 11, 20
    inp = ci.make_inputs(o, v, L, seed=3, b_scale=0.1, f_offdiag=0.05)
    oc = orc.OracleCCSD(inp.h, inp.B, o, v)
    t1, t2p = ci.random_amplitudes(o, v, 1, 0.1)
    oc.set_amplitudes(t1, orc.unpack_t2(t2p, o, v))
    oc.residual()
    rng = np.random.default_rng(0)
    ref = orc.pack_t2(oc.s2_term("pp_ladder"))
    ij, ab = rng.integers(0, ref.shape[0], 25), rng.integers(0, ref.shape[1], 25)
    got = orc.pp_ladder_samples_from_B(inp.B, o, t1, t2p, ij, ab)
    assert np.abs(got - ref[ij, ab]).max() < 1e-14 * max(1.0, np.abs(ref).max())
    ks, cs = rng.integers(0, o, 12), rng.integers(0, v, 12)
    assert np.abs(orc.hov_samples_from_B(inp.B, oc.f, o, t1, ks, cs) - oc.Hov[ks, cs]).max() < 1e-14
    a, b, c, d = rng.integers(0, v, (4, 30))
    assert np.abs(orc.g_samples(inp.B, o + a, o + b, o + c, o + d) - oc.vvvv[a, b, c, d]).max() < 1e-15
    k, l = rng.integers(0, o, (2, 30))
    assert np.abs(orc.g_samples(inp.B, k, l, o + c, o + d) - oc.oovv[k, l, c, d]).max() < 1e-15
    assert np.abs(orc.g_samples(inp.B, o + a, k, o + c, o + d) - oc.vovv[a, k, c, d]).max() < 1e-15


def test_slab_entry_points_tile_the_full_evaluation():
    """The range / part entry points bench.py times (slabs of the BASELINE-size terms) are the same loop nests: evaluated
    slab by slab they reproduce the full evaluation bit for bit, in both sum modes, also through from_blocks with only a
    row block of <ab||cd> resident."""
    o, v = 4, 7
    inp = ci.make_inputs(o, v, 9, seed=71, b_scale=0.2, f_offdiag=0.1)
    t1, t2 = _random_unpacked_amplitudes(o, v, 72, 0.2)
    for restricted in (False, True):
        full = OracleCCSD(inp.h, inp.B, o, v, restricted=restricted)
        full.set_amplitudes(t1, t2)
        S1, S2 = full.residual()
        S1, S2 = S1.copy(), S2.copy()
        terms = {name: full.s2_term(name).copy() for name in full.TERMS}
        part = OracleCCSD(inp.h, inp.B, o, v, restricted=restricted)
        part.set_amplitudes(t1, t2)
        part.build_tau()
        for name, extent in zip(part.PARTS, (v, o, o, v, o, o)):
            for lo in range(0, extent, 3):
                part.intermediates_part(name, lo, min(extent, lo + 3))
        for name in ("Hvv", "Gvv", "Hoo", "Goo", "Hov", "Hvovo", "C", "A"):
            assert np.array_equal(getattr(part, name), getattr(full, name)), name
        for name in part.TERMS:
            out = np.zeros_like(S2)
            for i0 in range(0, o, 2):
                for a0 in range(0, v, 3):
                    part.s2_term_range(name, i0, min(o, i0 + 2), a0, min(v, a0 + 3), out=out)
            if name == "ring":      # the ring antisymmetrises a buffer that holds the slab only: slabs ADD up
                out = np.zeros_like(S2)
                for i0 in range(0, o, 2):
                    for a0 in range(0, v, 3):
                        out += part.s2_term_range(name, i0, min(o, i0 + 2), a0, min(v, a0 + 3), out=np.zeros_like(S2))
                assert np.abs(out - terms[name]).max() < 1e-14
            else:
                assert np.array_equal(out, terms[name]), name
        for i0 in range(0, o, 3):
            part.s1_range(i0, min(o, i0 + 3))
        assert np.array_equal(part.S1, S1)
    # from_blocks with rows [2, 5) of <ab||cd> only: the pp-ladder slab of those rows
    rows = np.ascontiguousarray(full.vvvv[2:5])
    fb = OracleCCSD.from_blocks(o, v, full.f, full.oooo, full.ooov, full.oovv, full.vovo, full.vovv, rows, 2, restricted=True)
    fb.set_amplitudes(t1, t2)
    fb.build_tau()
    out = fb.s2_term_range("pp_ladder", 0, o, 2, 5, out=np.zeros_like(S2))
    ref = terms["pp_ladder"]
    assert np.array_equal(out[:, :, 2:5, :][:, :, :, 3:], ref[:, :, 2:5, :][:, :, :, 3:])
