"""Pins of the oracle's DIIS step (reading G13 of DESIGN.md) against things other than itself (CPU only).

The paper says only "DIIS was implemented", so the definition is DESIGN.md's reading G13:
error vector e = S/D, stored pairs (u = t + e, e) over the UNIQUE amplitudes (t1, then t2 packed i<j, a<b), real
coefficients c minimising |sum_l c_l e_l|_2 subject to sum_l c_l = 1 (Pulay), extrapolation as soon as two pairs exist,
FIFO of the last m = 6 pairs, energy evaluated at the extrapolated amplitudes.  Every cfg1/cfg2/cfg3 lock-step parity
claim compares two DIIS trajectories BEFORE convergence, so the trajectory itself needs a pin:

D1  the per-iteration energies SURVEY.md 8(c) pin P9 prints from the survey's INDEPENDENT numpy/BLAS scratch (cfg2
    iterations 0..10, cfg1 iterations 0, 15 and converged) against the committed oracle runs
    tests/golden/oracle_lockstep_cfg{1,2}.txt, at the printed precision (file against file).
D2  a live trajectory where DIIS matters long before convergence: the oracle's residual and energy (pinned by P1) are
    driven by a DIIS written here as the DEFINITION -- a constrained least-squares problem solved by numpy's lstsq
    in the null space of the constraint; no Gram matrix, no bordered system -- and compared with OracleCCSD.iterate()
    at every iteration, past the point where the FIFO drops vectors.  A different metric (unpacked weighting, a
    complex Gram matrix), a different start (extrapolating from 1 or 3 pairs), a different subspace size or an energy
    taken before the extrapolation all change the trajectory at O(1e-3) and fail.
D3  the same for the Lambda oracle's iteration (start lambda = conj(t), Jacobi + DIIS as G12/G13; reading G23).
D4  DIIS off (ndiis = 0) is the plain Jacobi iteration t <- t + S/D.
"""
import os

import numpy as np
import pytest

import ccsd_inputs as ci
from oracle.ccsd_oracle import OracleCCSD, pack_t2, unpack_t2
from oracle.lambda_oracle import OracleLambda

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ------------------------------------------------------------------------------------------------------------ D1
def _survey_rows():
    rows = {}
    with open(os.path.join(GOLDEN, "survey_soft_energies.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            cfg, key, re_, im_ = line.split()
            rows[(cfg, key)] = (re_, im_)
    return rows


def _golden_rows(cfg):
    out = {}
    with open(os.path.join(GOLDEN, f"oracle_lockstep_{cfg}.txt")) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            it, re_, im_, sn = line.split()
            out[int(it)] = (complex(float(re_), float(im_)), float(sn))
    return out


def _printed_tolerance(text):
    """Half a unit of the last printed digit (plus a rounding margin): '-6.081230344181' -> 0.6e-12."""
    mant = text.lower().split("e")
    digits = len(mant[0].split(".")[1]) if "." in mant[0] else 0
    expo = int(mant[1]) if len(mant) > 1 else 0
    return 0.6 * 10.0 ** (expo - digits)


@pytest.mark.parametrize("cfg", ["cfg1", "cfg2"])
def test_d1_oracle_lockstep_files_reproduce_the_surveys_independent_trajectory(cfg):
    survey = _survey_rows()
    golden = _golden_rows(cfg)
    keys = [k for (c, k) in survey if c == cfg and k.startswith("E_iter")]
    assert len(keys) >= (11 if cfg == "cfg2" else 2)
    checked_after_diis = 0
    for key in keys:
        it = int(key[len("E_iter"):])
        re_txt, im_txt = survey[(cfg, key)]
        e, _ = golden[it]
        assert abs(e.real - float(re_txt)) <= _printed_tolerance(re_txt), (cfg, key, e.real, re_txt)
        if im_txt != "-":
            assert abs(e.imag - float(im_txt)) <= _printed_tolerance(im_txt), (cfg, key, e.imag, im_txt)
        checked_after_diis += it >= 2          # from iteration 2 on the energy depends on the extrapolation
    assert checked_after_diis >= (9 if cfg == "cfg2" else 1)
    if (cfg, "E_ccsd") in survey:              # converged value (independent of DIIS; printed to 13 decimals); the
        re_txt, _ = survey[(cfg, "E_ccsd")]    # committed run stops at ||S/D|| = 4e-11, i.e. a few 1e-13 Eh short of it
        last = golden[max(golden)]
        assert last[1] < 1e-10 and abs(last[0].real - float(re_txt)) <= 5e-13


# ------------------------------------------------------------------------------------------------------------ D2
def _pulay_by_least_squares(errs):
    """argmin_c | sum_l c_l e_l |_2  subject to  sum_l c_l = 1, c real -- the definition, solved without a Gram matrix:
    c = c0 + Z y with c0 = 1/m and Z an orthonormal basis of the null space of the constraint; the complex vectors are
    stacked as (Re, Im) so that real coefficients minimise the complex 2-norm."""
    m = len(errs)
    M = np.stack([np.concatenate([e.real, e.imag]) for e in errs], axis=1)          # (2N, m) real
    c0 = np.full(m, 1.0 / m)
    q, _ = np.linalg.qr(np.concatenate([np.ones((m, 1)), np.eye(m)[:, : m - 1]], axis=1))
    Z = q[:, 1:]                                                                    # columns orthogonal to (1,...,1)
    assert np.abs(np.ones(m) @ Z).max() < 1e-14
    y = np.linalg.lstsq(M @ Z, -(M @ c0), rcond=None)[0]
    return c0 + Z @ y


class _DefinitionDIIS:
    """Jacobi + DIIS(m) around a residual callback, written from reading G13 alone."""

    def __init__(self, m):
        self.m, self.us, self.es = m, [], []

    def step(self, t_vec, e_vec):
        u = t_vec + e_vec
        if self.m <= 0:
            return u
        self.us.append(u); self.es.append(e_vec)
        self.us, self.es = self.us[-self.m:], self.es[-self.m:]
        if len(self.us) < 2:
            return u
        c = _pulay_by_least_squares(self.es)
        return sum(cl * ul for cl, ul in zip(c, self.us))


def _vec(a1, a2):
    return np.concatenate([a1.ravel(), pack_t2(a2).ravel()])


def _unvec(x, o, v):
    return x[: o * v].reshape(o, v), unpack_t2(x[o * v:].reshape(o * (o - 1) // 2, v * (v - 1) // 2), o, v)


@pytest.mark.parametrize("o,v,naux,seed,b_scale,f_off,ndiis,nit,min_moved", [
    (4, 16, 60, 2021030801, ci.B_SCALE, ci.F_OFFDIAG, 6, 7, 1e-8),  # BASELINE cfg0 (weak coupling, converges in 8)
    (4, 9, 14, 77, 0.16, 0.10, 6, 14, 1e-4),                        # strong coupling: the FIFO drops vectors
    (3, 8, 12, 78, 0.15, 0.10, 3, 10, 1e-4),                        # a smaller subspace
])
def test_d2_oracle_diis_trajectory_equals_the_definition(o, v, naux, seed, b_scale, f_off, ndiis, nit, min_moved):
    inp = ci.make_inputs(o, v, naux, seed, b_scale=b_scale, f_offdiag=f_off)
    ref = OracleCCSD(inp.h, inp.B, o, v, ndiis=ndiis)          # iterates with its own DIIS
    drv = OracleCCSD(inp.h, inp.B, o, v, ndiis=0)              # only its (pinned) residual and energy are used
    eps = drv.f.diagonal().real
    eo, ev = eps[:o], eps[o:]
    D1 = eo[:, None] - ev[None, :]
    D2 = eo[:, None, None, None] + eo[None, :, None, None] - ev[None, None, :, None] - ev[None, None, None, :]
    diis = _DefinitionDIIS(ndiis)
    moved = 0.0
    for it in range(1, nit + 1):
        e_ref, sn_ref = ref.iterate()
        S1, S2 = drv.residual()
        e_vec = _vec(S1 / D1, S2 / D2)
        t_new = diis.step(_vec(drv.t1, drv.t2), e_vec)
        plain = _vec(drv.t1, drv.t2) + e_vec
        moved = max(moved, np.abs(t_new - plain).max())
        drv.set_amplitudes(*_unvec(t_new, o, v))
        e_def = drv.energy()
        sn_def = float(np.linalg.norm(e_vec))
        assert abs(sn_def - sn_ref) <= 1e-9 * max(sn_ref, 1e-6), (it, sn_def, sn_ref)
        assert abs(e_def - e_ref) <= 1e-11 * max(1.0, abs(e_ref)), (it, e_def, e_ref)
        assert np.abs(drv.t1 - ref.t1).max() < 1e-9 and np.abs(drv.t2 - ref.t2).max() < 1e-9, it
    assert moved > min_moved     # the extrapolation really changed the iterates (nothing hides behind convergence)
    assert sn_ref > 1e-9 or nit <= 8   # the comparison ended before the subspace became numerically degenerate


def test_d2_alternative_conventions_are_distinguishable():
    """The trajectory test has teeth: an unpacked (4x-weighted t2) metric or a 1-pair start moves the energies by far
    more than its tolerance."""
    o, v = 4, 9
    inp = ci.make_inputs(o, v, 14, 77, b_scale=0.16, f_offdiag=0.10)
    ref = OracleCCSD(inp.h, inp.B, o, v, ndiis=6)
    alt = OracleCCSD(inp.h, inp.B, o, v, ndiis=0)
    us, es, ws = [], [], []
    diff = 0.0
    for it in range(6):
        e_ref, _ = ref.iterate()
        S1, S2 = alt.residual()
        e1, e2 = S1 / alt.D1, S2 / alt.D2
        us.append(_vec(alt.t1 + e1, alt.t2 + e2)); es.append(np.concatenate([e1.ravel(), e2.ravel()]))   # unpacked metric
        c = _pulay_by_least_squares(es[-6:]) if len(es) >= 2 else np.ones(1)
        t_new = sum(cl * ul for cl, ul in zip(c, us[-6:]))
        alt.set_amplitudes(*_unvec(t_new, o, v))
        diff = max(diff, abs(alt.energy() - e_ref))
    assert diff > 1e-6


# ------------------------------------------------------------------------------------------------------------ D3
def test_d3_lambda_oracle_iteration_equals_the_definition():
    o, v = 3, 7
    inp = ci.make_inputs(o, v, 10, seed=505, b_scale=0.14, f_offdiag=0.08)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    assert oc.run(300, tol=1e-13)[-1][1] < 1e-12
    ref = OracleLambda(oc, ndiis=6)
    drv = OracleLambda(oc, ndiis=0)
    assert np.array_equal(drv.l1, np.conj(oc.t1)) and np.array_equal(drv.l2, np.conj(oc.t2))     # start (G23)
    diis = _DefinitionDIIS(6)
    l1, l2 = np.conj(oc.t1), np.conj(oc.t2)
    moved = 0.0
    for it in range(1, 11):
        sn_ref = ref.iterate()
        R1, R2 = drv.residual(l1, l2)
        e_vec = _vec(R1 / oc.D1, R2 / oc.D2)
        new = diis.step(_vec(l1, l2), e_vec)
        moved = max(moved, np.abs(new - _vec(l1, l2) - e_vec).max())
        l1, l2 = _unvec(new, o, v)
        assert abs(np.linalg.norm(e_vec) - sn_ref) <= 1e-9 * max(sn_ref, 1e-6), (it, sn_ref)
        assert np.abs(l1 - ref.l1).max() < 1e-9 and np.abs(l2 - ref.l2).max() < 1e-9, it
    assert moved > 1e-5


# ------------------------------------------------------------------------------------------------------------ D4
def test_d4_no_diis_is_plain_jacobi():
    inp = ci.make_config("cfg0")
    o, v = inp.nocc, inp.nvir
    oc = OracleCCSD(inp.h, inp.B, o, v, ndiis=0)
    for _ in range(3):
        t1, t2 = oc.t1.copy(), oc.t2.copy()
        S1, S2 = oc.residual()
        want1, want2 = t1 + S1 / oc.D1, t2 + S2 / oc.D2
        oc.set_amplitudes(t1, t2)
        oc.iterate()
        assert np.array_equal(oc.t1, want1) and np.array_equal(oc.t2, want2)
