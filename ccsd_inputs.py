"""Seeded synthetic inputs for the complex spinor-basis CCSD hot path.

This module serves BOTH the CPU oracle (``oracle/``) and the CUDA library
(``paper_2103_08473_b200/``).  It holds no CCSD arithmetic: it draws random
numbers and shapes them into the Hamiltonian of PAPER.md:65-75 (eq 5): a
complex Hermitian one-electron matrix ``h[n][n]`` and a factorised two-electron
tensor ``B[L][n][n]`` with (pq|rs) = sum_L B[L,p,q]*B[L,r,s] (the Cholesky-type
factor ExaCorr accepts).  Recipe: SURVEY.md 8(d),
restated in DESIGN.md "Input recipe".  They stand in for the paper's
heavy-element workloads (uranyl with 24 / 34 correlated electrons,
PAPER.md:29), whose molecular inputs are not available.

The only formula here besides the distributions is step 5 of the recipe: the
caller-visible ``h`` is chosen so that the Fock matrix the solver rebuilds,
f = h + sum_i <pi||qi>, has the prescribed statistics
(diagonal = orbital energies, off-diagonal CN(0, 0.01^2)).  Both sides rebuild f
from (h, B) with their own code.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

# name -> (nocc, nvir, naux, seed)     BASELINE.json configs[0..3] (+ the 2-electron variant)
CONFIGS = {
    "cfg0_2e": (2, 10, 60, 2021030800),
    "cfg0": (4, 16, 60, 2021030801),
    "cfg1": (16, 96, 336, 2021030802),
    "cfg2": (24, 160, 552, 2021030803),
    "cfg3": (34, 224, 774, 2021030804),
}
# BASELINE.json configs[4]: isolated pp-ladder sweep shapes (nocc, nvir)
LADDER_SWEEP = [(20, 128), (20, 192), (20, 256), (40, 128), (40, 192), (40, 256)]
LADDER_SEED0 = 2021030805

B_SCALE = 0.05 / math.sqrt(20.0)
F_OFFDIAG = 0.01


@dataclasses.dataclass
class CCSDInputs:
    nocc: int
    nvir: int
    naux: int
    seed: int
    h: np.ndarray        # [n][n] complex128, Hermitian, bare one-electron matrix of eq 5
    B: np.ndarray        # [naux][n][n] complex128, B[L] Hermitian
    f_target: np.ndarray  # [n][n] the Fock matrix the recipe aimed at (test pin for the Fock build)

    @property
    def n(self) -> int:
        return self.nocc + self.nvir


def _fock_shift(B: np.ndarray, nocc: int) -> np.ndarray:
    """u_pq = sum_{i<nocc} <pi||qi> = sum_{i,L} (B[L,p,q] B[L,i,i] - B[L,p,i] B[L,i,q]) (recipe step 5)."""
    d = np.einsum("lii->l", B[:, :nocc, :nocc])
    coul = np.einsum("lpq,l->pq", B, d)
    exch = np.einsum("lpi,liq->pq", B[:, :, :nocc], B[:, :nocc, :])
    return coul - exch


def make_inputs(nocc: int, nvir: int, naux: int, seed: int,
                b_scale: float = B_SCALE, f_offdiag: float = F_OFFDIAG) -> CCSDInputs:
    """SURVEY.md 8(d) steps 1-6.  Draw order is part of the recipe."""
    n = nocc + nvir
    rng = np.random.default_rng(seed)
    zre = rng.standard_normal((naux, n, n))
    zim = rng.standard_normal((naux, n, n))
    eo = np.sort(rng.uniform(-2.0, -0.5, nocc))
    ev = np.sort(rng.uniform(0.3, 5.0, nvir))
    xre = rng.standard_normal((n, n))
    xim = rng.standard_normal((n, n))
    z = (zre + 1j * zim) / math.sqrt(2.0)
    del zre, zim
    B = (b_scale / math.sqrt(2.0)) * (z + np.conj(np.transpose(z, (0, 2, 1))))
    del z
    x = f_offdiag * (xre + 1j * xim) / math.sqrt(2.0)
    f = (x + x.conj().T) / math.sqrt(2.0)
    f[np.arange(n), np.arange(n)] = np.concatenate([eo, ev])
    h = f - _fock_shift(B, nocc)
    h = 0.5 * (h + h.conj().T)
    return CCSDInputs(nocc, nvir, naux, seed, np.ascontiguousarray(h), np.ascontiguousarray(B), f)


def make_config(name: str) -> CCSDInputs:
    o, v, L, seed = CONFIGS[name]
    return make_inputs(o, v, L, seed)


def make_kramers_inputs(m_occ: int, m_vir: int, naux: int, seed: int,
                        b_scale: float = 0.08, f_offdiag: float = 0.05) -> CCSDInputs:
    """Time-reversal (Kramers) structured input, SURVEY.md 8(c) pin P5.

    Every matrix is M = [[A, C], [-conj(C), conj(A)]] in the basis (p_1..p_m, pbar_1..pbar_m) with A Hermitian and
    C antisymmetric; complete pairs are occupied; spinors are then permuted to occupied-first order.
    """
    m = m_occ + m_vir
    rng = np.random.default_rng(seed)

    def kramers(herm_diag=None, scale=1.0):
        a = (rng.standard_normal((m, m)) + 1j * rng.standard_normal((m, m))) / math.sqrt(2.0)
        a = scale * (a + a.conj().T) / math.sqrt(2.0)
        c = (rng.standard_normal((m, m)) + 1j * rng.standard_normal((m, m))) / math.sqrt(2.0)
        c = scale * (c - c.T) / math.sqrt(2.0)
        if herm_diag is not None:
            a[np.arange(m), np.arange(m)] = herm_diag
        return np.block([[a, c], [-c.conj(), a.conj()]])

    eps = np.concatenate([np.sort(rng.uniform(-2.0, -0.5, m_occ)), np.sort(rng.uniform(0.3, 5.0, m_vir))])
    f = kramers(eps, f_offdiag)
    B = np.stack([kramers(None, b_scale) for _ in range(naux)])
    occ = list(range(m_occ)) + list(range(m, m + m_occ))
    vir = list(range(m_occ, m)) + list(range(m + m_occ, 2 * m))
    order = np.array(occ + vir)
    f = f[np.ix_(order, order)]
    B = B[:, order][:, :, order]
    nocc, nvir = 2 * m_occ, 2 * m_vir
    h = f - _fock_shift(B, nocc)
    return CCSDInputs(nocc, nvir, naux, seed, np.ascontiguousarray(h), np.ascontiguousarray(B), f)


def pair_count(m: int) -> int:
    return m * (m - 1) // 2


def pair_index(x: int, y: int, m: int) -> int:
    """Packed index of x<y in a dimension of size m (row-major strict upper triangle = numpy.triu_indices(m, 1))."""
    return x * m - x * (x + 1) // 2 + (y - x - 1)


def random_amplitudes(nocc: int, nvir: int, seed: int, scale: float = 0.01):
    """Seeded antisymmetric amplitudes: t1[o][v] and packed t2p[(i<j)][(a<b)], entries CN(0, scale^2)."""
    rng = np.random.default_rng(seed)
    oo, vv = pair_count(nocc), pair_count(nvir)
    t1 = scale * (rng.standard_normal((nocc, nvir)) + 1j * rng.standard_normal((nocc, nvir))) / math.sqrt(2.0)
    t2p = scale * (rng.standard_normal((oo, vv)) + 1j * rng.standard_normal((oo, vv))) / math.sqrt(2.0)
    return np.ascontiguousarray(t1), np.ascontiguousarray(t2p)


def ladder_inputs(nocc: int, nvir: int, seed: int, w_scale: float = 5.0e-3, t_scale: float = 0.01):
    """BASELINE.json configs[4] / SURVEY.md 8(d) step 7: W[(a<b)][(c<d)] Hermitian CN(0, w_scale^2), tau[(i<j)][(c<d)]
    i.i.d. CN(0, t_scale^2).  Returned as (tau, W)."""
    rng = np.random.default_rng(seed)
    oo, vv = pair_count(nocc), pair_count(nvir)
    W = np.empty((vv, vv), dtype=np.complex128)
    W.real = rng.standard_normal((vv, vv))
    W.imag = rng.standard_normal((vv, vv))
    W *= w_scale / 2.0
    W = W + W.conj().T
    tau = np.empty((oo, vv), dtype=np.complex128)
    tau.real = rng.standard_normal((oo, vv))
    tau.imag = rng.standard_normal((oo, vv))
    tau *= t_scale / math.sqrt(2.0)
    return tau, W
