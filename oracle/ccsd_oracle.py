"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Driver of the plain CPU CCSD oracle: the heavy explicit loops are in ``ccsd_oracle.c`` (eqs 22-33 of
arXiv 2103.08473); this file holds the iteration around them, in plain numpy:

* MP2 start: t1 = f_ai / D^a_i, t2 = <ab||ij> / D^ab_ij.
* Jacobi step ("Jacobi preconditioning during amplitude updates"; reading G12):
  u = t + S / D with D^a_i = eps_i - eps_a, D^ab_ij = eps_i + eps_j - eps_a - eps_b, eps_p = Re f_pp.
* DIIS (PAPER.md:107, 234 say only "DIIS was implemented"; reading G13 of DESIGN.md): error vector e = S/D,
  stored pairs (u, e) over the unique amplitudes (t1 followed by t2 packed i<j, a<b), real Gram matrix
  B_kl = Re <e_k|e_l>, bordered Pulay system, extrapolate as soon as two pairs exist, keep the last m pairs.
  "parity unpinned": the paper does not define these details; the converged energy is independent of them and is
  pinned (FCI for two electrons, determinant-space residuals).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
It imports nothing from paper_2103_08473_b200.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from oracle._build import compile_oracle

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "liboracle.so")
_SRC_PATH = os.path.join(_HERE, "ccsd_oracle.c")
_lib = None

C128 = np.complex128


def build(force: bool = False) -> str:
    """Compile ccsd_oracle.c -> liboracle.so (gcc -O2 -fopenmp, no -ffast-math)."""
    return compile_oracle(_SRC_PATH, _LIB_PATH, force)


class _Sys(ctypes.Structure):
    _fields_ = [("o", ctypes.c_int), ("v", ctypes.c_int), ("restricted", ctypes.c_int),
                ("f", ctypes.c_void_p), ("oooo", ctypes.c_void_p), ("ooov", ctypes.c_void_p),
                ("oovv", ctypes.c_void_p), ("vovo", ctypes.c_void_p), ("vovv", ctypes.c_void_p),
                ("vvvv", ctypes.c_void_p)]


class _Inter(ctypes.Structure):
    _fields_ = [(k, ctypes.c_void_p) for k in ("tau", "Hvv", "Gvv", "Hoo", "Goo", "Hov", "Hvovo", "C", "A")]


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.oracle_num_threads.restype = ctypes.c_int
    return _lib


def _p(a: np.ndarray):
    assert a.flags["C_CONTIGUOUS"]
    return ctypes.c_void_p(a.ctypes.data)


def num_threads() -> int:
    return int(lib().oracle_num_threads())


# ---------------------------------------------------------------------------------------------------------------
# packing helpers (row-major strict upper triangle == numpy.triu_indices(m, 1))
# ---------------------------------------------------------------------------------------------------------------
def pack_t2(t2: np.ndarray) -> np.ndarray:
    o, v = t2.shape[0], t2.shape[2]
    io, jo = np.triu_indices(o, 1)
    av, bv = np.triu_indices(v, 1)
    return np.ascontiguousarray(t2[io[:, None], jo[:, None], av[None, :], bv[None, :]])


def unpack_t2(t2p: np.ndarray, o: int, v: int) -> np.ndarray:
    io, jo = np.triu_indices(o, 1)
    av, bv = np.triu_indices(v, 1)
    t2 = np.zeros((o, o, v, v), dtype=C128)
    t2[io[:, None], jo[:, None], av[None, :], bv[None, :]] = t2p
    t2[jo[:, None], io[:, None], av[None, :], bv[None, :]] = -t2p
    t2[io[:, None], jo[:, None], bv[None, :], av[None, :]] = -t2p
    t2[jo[:, None], io[:, None], bv[None, :], av[None, :]] = t2p
    return t2


class OracleCCSD:
    """The oracle's CCSD solver.  ``restricted=False`` is the definition (full sums); ``True`` the c<d form."""

    TERMS = ("ring", "goo", "vdag_t1", "gvv", "c_t1", "hh_ladder", "pp_ladder", "driver")

    def __init__(self, h: np.ndarray, B: np.ndarray, nocc: int, nvir: int, ndiis: int = 6,
                 restricted: bool = False, level_shift: float = 0.0):
        L = lib()
        self.o, self.v, self.n = nocc, nvir, nocc + nvir
        o, v, n = self.o, self.v, self.n
        self.naux = B.shape[0]
        self.restricted = bool(restricted)
        self.ndiis = ndiis
        h = np.ascontiguousarray(h, dtype=C128)
        B = np.ascontiguousarray(B, dtype=C128)
        assert h.shape == (n, n) and B.shape == (self.naux, n, n)
        # Fock matrix
        self.f = np.zeros((n, n), dtype=C128)
        L.oracle_fock(n, o, self.naux, _p(h), _p(B), _p(self.f))
        # eps_fock = Re f_pp, the spinor energies themselves: what the triples denominators of eqs 39/41 are made of
        # (PAPER.md:645-663).  The level shift (.LSHIFT) is a convergence aid of the amplitude iterations
        # only: eps = eps_fock + shift on the virtuals feeds D1 / D2 of the Jacobi step and of the MP2 start.
        self.eps_fock = self.f.diagonal().real.copy()
        self.eps = self.eps_fock.copy()
        self.eps[o:] += level_shift
        # the six integral classes, each by the definition <pq||rs> = (pr|qs) - (ps|qr)
        self.Bt = np.zeros((n, n, self.naux), dtype=C128)
        L.oracle_transpose_B(n, self.naux, _p(B), _p(self.Bt))
        r = int(self.restricted)
        O, V = (0, o), (o, v)
        self.oooo = self._g(O, O, O, O, r, r)
        self.ooov = self._g(O, O, O, V, r, 0)
        self.oovv = self._g(O, O, V, V, r, r)
        self.vovo = self._g(V, O, V, O, 0, 0)
        self.vovv = self._g(V, O, V, V, 0, r)
        self.vvvv = self._g(V, V, V, V, r, r)
        self.sys = _Sys(o, v, r, *[a.ctypes.data for a in
                                  (self.f, self.oooo, self.ooov, self.oovv, self.vovo, self.vovv, self.vvvv)])
        eo, ev = self.eps[:o], self.eps[o:]
        self.D1 = eo[:, None] - ev[None, :]
        self.D2 = eo[:, None, None, None] + eo[None, :, None, None] - ev[None, None, :, None] - ev[None, None, None, :]
        self._alloc_work()      # intermediates, residuals
        self.mp2_guess()

    @classmethod
    def from_blocks(cls, nocc: int, nvir: int, f, oooo, ooov, oovv, vovo, vovv, vvvv_rows=None, vvvv_row0: int = 0,
                    restricted: bool = True, ndiis: int = 6):
        """An oracle object on CALLER-SUPPLIED Fock matrix and integral blocks (no Fock / integral build, amplitudes zero):
        bench.py's cpu_baseline leg times slabs of the BASELINE-size terms with it, on synthetic-valued blocks of the true
        shapes (building the real v^4 block takes the oracle tens of minutes at cfg3).  `vvvv_rows` holds rows
        [vvvv_row0, vvvv_row0 + len) of <ab||cd> [a][b][c][d] only; s2_term_range must then stay inside that a-range."""
        self = cls.__new__(cls)
        o, v = int(nocc), int(nvir)
        self.o, self.v, self.n, self.naux = o, v, o + v, 0
        self.restricted, self.ndiis = bool(restricted), ndiis
        self.f, self.oooo, self.ooov, self.oovv, self.vovo, self.vovv = f, oooo, ooov, oovv, vovo, vovv
        self.vvvv = vvvv_rows
        for a, shp in ((f, (o + v, o + v)), (oooo, (o, o, o, o)), (ooov, (o, o, o, v)), (oovv, (o, o, v, v)),
                       (vovo, (v, o, v, o)), (vovv, (v, o, v, v))):
            assert a.dtype == C128 and a.shape == shp and a.flags["C_CONTIGUOUS"]
        vvvv_ptr = 0
        if vvvv_rows is not None:
            assert vvvv_rows.dtype == C128 and vvvv_rows.shape[1:] == (v, v, v) and vvvv_rows.flags["C_CONTIGUOUS"]
            vvvv_ptr = vvvv_rows.ctypes.data - int(vvvv_row0) * v ** 3 * 16
        self.vvvv_range = (int(vvvv_row0), int(vvvv_row0) + (0 if vvvv_rows is None else vvvv_rows.shape[0]))
        self.sys = _Sys(o, v, int(self.restricted), f.ctypes.data, oooo.ctypes.data, ooov.ctypes.data, oovv.ctypes.data,
                        vovo.ctypes.data, vovv.ctypes.data, vvvv_ptr)
        self.eps_fock = f.diagonal().real.copy()
        self.eps = self.eps_fock.copy()
        eo, ev = self.eps[:o], self.eps[o:]
        self.D1 = eo[:, None] - ev[None, :]
        self.D2 = None
        self._alloc_work()
        self.t1 = np.zeros((o, v), dtype=C128)
        self.t2 = np.zeros((o, o, v, v), dtype=C128)
        self._diis_u, self._diis_e = [], []
        return self

    def _alloc_work(self):
        o, v = self.o, self.v
        self.tau = np.zeros((o, o, v, v), dtype=C128)
        self.Hvv = np.zeros((v, v), dtype=C128); self.Gvv = np.zeros((v, v), dtype=C128)
        self.Hoo = np.zeros((o, o), dtype=C128); self.Goo = np.zeros((o, o), dtype=C128)
        self.Hov = np.zeros((o, v), dtype=C128)
        self.Hvovo = np.zeros((v, o, v, o), dtype=C128)
        self.C = np.zeros((o, v, o, o), dtype=C128)
        self.A = np.zeros((o, o, o, o), dtype=C128)
        self.inter = _Inter(*[a.ctypes.data for a in (self.tau, self.Hvv, self.Gvv, self.Hoo, self.Goo, self.Hov,
                                                      self.Hvovo, self.C, self.A)])
        self.S1 = np.zeros((o, v), dtype=C128)
        self.S2 = np.zeros((o, o, v, v), dtype=C128)
        self._scratch = np.zeros((o, o, v, v), dtype=C128)

    def _g(self, P, Q, Rr, S, apq, ars):
        out = np.zeros((P[1], Q[1], Rr[1], S[1]), dtype=C128)
        lib().oracle_g_block(self.n, self.naux, _p(self.Bt), P[0], P[1], Q[0], Q[1], Rr[0], Rr[1], S[0], S[1],
                             apq, ars, _p(out))
        return out

    # --- amplitudes -------------------------------------------------------------------------------------------
    def mp2_guess(self):
        """MP2 amplitudes as the initial guess.  t1 = f_ai/D = conj(f_ia)/D; t2 = <ab||ij>/D = conj(<ij||ab>)/D."""
        o = self.o
        self.t1 = np.conj(self.f[:o, o:]) / self.D1
        self.t2 = np.conj(self.oovv) / self.D2
        self._diis_u, self._diis_e = [], []
        return self

    def set_amplitudes(self, t1, t2, reset_diis=True):
        self.t1 = np.ascontiguousarray(t1, dtype=C128).copy()
        self.t2 = np.ascontiguousarray(t2, dtype=C128).copy()
        if reset_diis:
            self._diis_u, self._diis_e = [], []

    # --- one residual evaluation --------------------------------------------------------------------------------
    def build_intermediates(self):
        L = lib()
        L.oracle_tau(self.o, self.v, _p(self.t1), _p(self.t2), _p(self.tau))
        L.oracle_intermediates(ctypes.byref(self.sys), _p(self.t1), _p(self.t2), ctypes.byref(self.inter))

    def s2_term(self, name: str) -> np.ndarray:
        out = np.zeros_like(self.S2)
        lib().oracle_s2_term(ctypes.byref(self.sys), _p(self.t1), _p(self.t2), ctypes.byref(self.inter),
                             self.TERMS.index(name), _p(out))
        return out

    # --- slabs of the same loop nests (timing of BASELINE-size terms in bench.py; results land in the usual arrays) ------
    PARTS = ("Hvv_Gvv", "Hoo_Goo", "Hov", "Hvovo", "C", "A")          # eqs 24-25, 26-27, 28, 29, 30, 31

    def build_tau(self):
        lib().oracle_tau(self.o, self.v, _p(self.t1), _p(self.t2), _p(self.tau))

    def intermediates_part(self, name: str, lo: int, hi: int):
        """One group of eqs 24-31 for its outermost output index in [lo, hi) (tau must be current)."""
        lib().oracle_intermediates_part(ctypes.byref(self.sys), _p(self.t1), _p(self.t2), ctypes.byref(self.inter),
                                        self.PARTS.index(name), int(lo), int(hi))

    def s2_term_range(self, name: str, i_lo: int, i_hi: int, a_lo: int, a_hi: int, out=None) -> np.ndarray:
        """One term of eq 32 for i in [i_lo, i_hi) and a in [a_lo, a_hi) (other elements of `out` untouched)."""
        out = self._scratch if out is None else out
        lib().oracle_s2_term_range(ctypes.byref(self.sys), _p(self.t1), _p(self.t2), ctypes.byref(self.inter),
                                   self.TERMS.index(name), int(i_lo), int(i_hi), int(a_lo), int(a_hi), _p(out))
        return out

    def s1_range(self, i_lo: int, i_hi: int) -> np.ndarray:
        lib().oracle_s1_range(ctypes.byref(self.sys), _p(self.t1), _p(self.t2), ctypes.byref(self.inter), int(i_lo),
                              int(i_hi), _p(self.S1))
        return self.S1

    def residual(self):
        """eqs 23-33 at the current amplitudes -> (S1[i][a], S2[i][j][a][b])."""
        L = lib()
        self.build_intermediates()
        L.oracle_s2(ctypes.byref(self.sys), _p(self.t1), _p(self.t2), ctypes.byref(self.inter), _p(self.S2),
                    _p(self._scratch))
        L.oracle_s1(ctypes.byref(self.sys), _p(self.t1), _p(self.t2), ctypes.byref(self.inter), _p(self.S1))
        return self.S1, self.S2

    def energy(self) -> complex:
        """E_corr of the current amplitudes (eq 9; reading G11)."""
        L = lib()
        L.oracle_tau(self.o, self.v, _p(self.t1), _p(self.t2), _p(self.tau))
        e = np.zeros(1, dtype=C128)
        L.oracle_energy(ctypes.byref(self.sys), _p(self.t1), _p(self.tau), _p(e))
        return complex(e[0])

    # --- update -------------------------------------------------------------------------------------------------
    def _vec(self, a1, a2):
        return np.concatenate([a1.ravel(), pack_t2(a2).ravel()])

    def iterate(self):
        """One CCSD iteration: residual, Jacobi step, DIIS.  Returns (E, ||S/D||_2 over unique amplitudes)."""
        S1, S2 = self.residual()
        e1, e2 = S1 / self.D1, S2 / self.D2
        u1, u2 = self.t1 + e1, self.t2 + e2
        evec = self._vec(e1, e2)
        step_norm = float(np.sqrt(np.vdot(evec, evec).real))
        if self.ndiis > 0:
            self._diis_u.append(self._vec(u1, u2))
            self._diis_e.append(evec)
            if len(self._diis_u) > self.ndiis:
                self._diis_u.pop(0)
                self._diis_e.pop(0)
            m = len(self._diis_u)
            if m >= 2:
                c = self._diis_coefficients()
                unew = np.zeros_like(self._diis_u[0])
                for cl, ul in zip(c, self._diis_u):
                    unew += cl * ul
                o, v = self.o, self.v
                u1 = unew[: o * v].reshape(o, v)
                oo, vv = o * (o - 1) // 2, v * (v - 1) // 2
                u2 = unpack_t2(unew[o * v:].reshape(oo, vv), o, v)
        self.t1, self.t2 = np.ascontiguousarray(u1), np.ascontiguousarray(u2)
        return self.energy(), step_norm

    def _diis_coefficients(self):
        """Pulay: minimise |sum_l c_l e_l|^2 with sum_l c_l = 1, real coefficients, Gram matrix Re<e_k|e_l>."""
        m = len(self._diis_e)
        while True:
            G = np.zeros((m + 1, m + 1))
            for k in range(m):
                for l in range(m):
                    G[k, l] = np.vdot(self._diis_e[-m + k], self._diis_e[-m + l]).real
            G[:m, m] = -1.0
            G[m, :m] = -1.0
            rhs = np.zeros(m + 1)
            rhs[m] = -1.0
            try:
                sol = np.linalg.solve(G, rhs)
                c = np.zeros(len(self._diis_e))
                c[len(c) - m:] = sol[:m]
                return c
            except np.linalg.LinAlgError:
                m -= 1
                if m < 1:
                    raise

    def run(self, niter: int = 50, tol: float = 1e-11, verbose: bool = False):
        """Iterate from the current amplitudes; returns the list of (E, step_norm) per iteration."""
        hist = []
        e_old = self.energy()
        for it in range(niter):
            e, sn = self.iterate()
            hist.append((e, sn))
            if verbose:
                print(f"  oracle iter {it + 1:3d}  E = {e.real:+.13f} {e.imag:+.3e}i  |S/D| = {sn:.3e}")
            if sn < tol and abs(e - e_old) < tol:
                break
            e_old = e
        return hist

    # --- reference energy for the FCI pin (reading G11): E_ref = sum_i h_ii + 1/2 sum_ij <ij||ij> -----------------
    def reference_energy(self, h) -> float:
        o = self.o
        e = sum(h[i, i] for i in range(o))
        e += 0.5 * sum(self.oooo[i, j, i, j] for i in range(o) for j in range(o))
        return float(np.real(e))


# ---------------------------------------------------------------------------------------------------------------
# sampled single-element evaluators (full-size spot checks)
# ---------------------------------------------------------------------------------------------------------------
def pp_ladder_samples(taup: np.ndarray, W: np.ndarray, ij: np.ndarray, ab: np.ndarray) -> np.ndarray:
    """R[(i<j)][(a<b)] = sum_{c<d} W[(a<b)][(c<d)] tau[(i<j)][(c<d)] at the sampled (ij, ab) pairs (eq 32)."""
    ij = np.ascontiguousarray(ij, dtype=np.int64)
    ab = np.ascontiguousarray(ab, dtype=np.int64)
    out = np.zeros(len(ij), dtype=C128)
    assert taup.shape[1] == W.shape[1]
    lib().oracle_pp_ladder_samples(ctypes.c_long(taup.shape[0]), ctypes.c_long(W.shape[1]), _p(taup), _p(W),
                                   len(ij), _p(ij), _p(ab), _p(out))
    return out


def nt_samples(A: np.ndarray, B: np.ndarray, ms, ns, conjB: bool = False) -> np.ndarray:
    """C[m][n] = sum_k A[m][k] * B[n][k] at sampled (m, n)."""
    ms = np.ascontiguousarray(ms, dtype=np.int64)
    ns = np.ascontiguousarray(ns, dtype=np.int64)
    assert A.ndim == 2 and B.ndim == 2 and A.shape[1] == B.shape[1]
    out = np.zeros(len(ms), dtype=C128)
    lib().oracle_nt_samples(ctypes.c_long(A.shape[1]), _p(A), ctypes.c_long(A.shape[1]), _p(B),
                            ctypes.c_long(B.shape[1]), int(conjB), len(ms), _p(ms), _p(ns), _p(out))
    return out


# ---------------------------------------------------------------------------------------------------------------
# single-element evaluators straight from the factorised integrals (full-size spot checks at cfg2/cfg3, where the
# unpacked <ab||cd> of OracleCCSD would need v^4 * 16 bytes).  Each is the definition written out for one element.
# ---------------------------------------------------------------------------------------------------------------
def g_samples(B: np.ndarray, p, q, r, s) -> np.ndarray:
    """<pq||rs> = (pr|qs) - (ps|qr) with (pq|rs) = sum_L B[L,p,q] B[L,r,s]  (eq 6 PAPER.md:71 in
    reading G1) at sampled index quadruples (absolute spinor indices)."""
    p, q, r, s = (np.asarray(x, dtype=np.int64) for x in (p, q, r, s))
    out = np.zeros(len(p), dtype=C128)
    for n in range(len(p)):
        out[n] = np.sum(B[:, p[n], r[n]] * B[:, q[n], s[n]]) - np.sum(B[:, p[n], s[n]] * B[:, q[n], r[n]])
    return out


def vvvv_row_packed(B: np.ndarray, nocc: int, a: int, b: int) -> np.ndarray:
    """Row (a<b) of <ab||cd>, all c<d in packed order: (ac|bd) - (ad|bc), the sum over L as one matrix product."""
    o = nocc
    Ba, Bb = B[:, o + a, o:], B[:, o + b, o:]            # [L][c], [L][d]
    J = Ba.T @ Bb                                          # J[c][d] = (ac|bd)
    K = J.T                                                # K[c][d] = (ad|bc)
    c, d = np.triu_indices(B.shape[1] - o, 1)
    return (J - K)[c, d]


def tau_row_packed(t1: np.ndarray, t2p_row: np.ndarray, i: int, j: int) -> np.ndarray:
    """Row (i<j) of tau = t2 + t1[i,a] t1[j,b] - t1[j,a] t1[i,b] (eq 23), all a<b packed."""
    a, b = np.triu_indices(t1.shape[1], 1)
    return t2p_row + t1[i, a] * t1[j, b] - t1[j, a] * t1[i, b]


def pp_ladder_samples_from_B(B: np.ndarray, nocc: int, t1: np.ndarray, t2p: np.ndarray, ij, ab) -> np.ndarray:
    """1/2 sum_cd <ab||cd> tau^cd_ij = sum_{c<d} (eq 32 last line) at sampled packed (ij, ab) pairs,
    from the factorised integrals and the amplitudes (t2p packed [(i<j)][(a<b)])."""
    o, v = nocc, B.shape[1] - nocc
    io, jo = np.triu_indices(o, 1)
    av, bv = np.triu_indices(v, 1)
    out = np.zeros(len(ij), dtype=C128)
    for n, (IJ, AB) in enumerate(zip(ij, ab)):
        w = vvvv_row_packed(B, o, int(av[AB]), int(bv[AB]))
        tau = tau_row_packed(t1, t2p[IJ], int(io[IJ]), int(jo[IJ]))
        out[n] = np.sum(w * tau)
    return out


def hov_samples_from_B(B: np.ndarray, f: np.ndarray, nocc: int, t1: np.ndarray, ks, cs) -> np.ndarray:
    """H^k_c = f_kc + sum_ld <kl||cd> t^d_l (eq 28) at sampled (k, c)."""
    o = nocc
    out = np.zeros(len(ks), dtype=C128)
    Bov = B[:, :o, o:]                                      # [L][l][d]
    for n, (k, c) in enumerate(zip(ks, cs)):
        # (kc|ld) - (kd|lc)
        coul = np.einsum("L,Lld->ld", B[:, k, o + c], Bov)
        exch = np.einsum("Ld,Ll->ld", B[:, k, o:], B[:, :o, o + c])
        out[n] = f[k, o + c] + np.sum((coul - exch) * t1)
    return out
