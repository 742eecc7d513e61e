"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Perturbative triples +T, (T), -T (arXiv 2103.08473 Appendix 7.3, eqs 39-44) on top of the CCSD
oracle's amplitudes and integral classes.  The explicit loops are in ``triples_oracle.c`` (reading G22 there and in
DESIGN.md); this file only re-indexes the stored integral classes ("dagger" = swap bra/ket and conjugate, G5):
    <ab||ie> = -conj <ei||ab>,   <am||ij> = -conj <ij||ma>,   <ab||ij> = conj <ij||ab>.

Pins: tests/test_triples_pins.py (determinant-space definitions of the drivers and of the three energies).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from oracle._build import compile_oracle

from oracle.ccsd_oracle import C128, _p

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtriples_oracle.so")
_SRC_PATH = os.path.join(_HERE, "triples_oracle.c")
_lib = None


def build(force: bool = False) -> str:
    return compile_oracle(_SRC_PATH, _LIB_PATH, force)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    return _lib


class OracleTriples:
    """+T / (T) / -T at the amplitudes (t1[i][a], t2[i][j][a][b]) of an OracleCCSD-like object `oc`
    (uses oc.f, oc.eps_fock, oc.vovv, oc.ooov, oc.oovv).  The denominators D^{abc}_{ijk} of eqs 39/41
    are built from the spinor energies Re f_pp WITHOUT the level shift of the amplitude iterations: the
    converged amplitudes do not depend on the shift, so neither may the triples corrections."""

    def __init__(self, oc, t1=None, t2=None):
        self.o, self.v = oc.o, oc.v
        o = self.o
        self.eps = np.ascontiguousarray(oc.eps_fock, dtype=np.float64)
        self.fov = np.ascontiguousarray(oc.f[:o, o:], dtype=C128)
        self.t1 = np.ascontiguousarray(oc.t1 if t1 is None else t1, dtype=C128)
        self.t2 = np.ascontiguousarray(oc.t2 if t2 is None else t2, dtype=C128)
        self.vvov = np.ascontiguousarray(-np.conj(oc.vovv).transpose(2, 3, 1, 0))     # [a][b][i][e] = <ab||ie>
        self.vooo = np.ascontiguousarray(-np.conj(oc.ooov).transpose(3, 2, 0, 1))     # [a][m][i][j] = <am||ij>
        self.vvoo = np.ascontiguousarray(np.conj(oc.oovv).transpose(2, 3, 0, 1))      # [a][b][i][j] = <ab||ij>

    def _block(self, fn, *args):
        v = self.v
        q = np.zeros((v, v, v), dtype=C128)
        qb = np.zeros((v, v, v), dtype=C128)
        fn(*args, _p(q))
        lib().oracle_triples_cyclic(v, _p(q), _p(qb))
        return q, qb

    def W(self, i, j, k):
        """(W, Wbar) of eq 40 for one occupied triple: [a][b][c]."""
        return self._block(lib().oracle_triples_W, self.o, self.v, _p(self.t2), _p(self.vvov), _p(self.vooo), i, j, k)

    def Z(self, i, j, k):
        return self._block(lib().oracle_triples_Z, self.o, self.v, _p(self.fov), _p(self.t1), _p(self.t2),
                           _p(self.vvoo), i, j, k)

    def Y(self, i, j, k):
        return self._block(lib().oracle_triples_Y, self.o, self.v, _p(self.t1), _p(self.t2), i, j, k)

    def energies(self, restricted: bool = False) -> dict:
        """{"+T": E(+T), "(T)": E((T)), "-T": E(-T)} (complex), eqs 39, 41, 43."""
        v = self.v
        work = np.zeros(6 * v ** 3, dtype=C128)
        out = np.zeros(3, dtype=C128)
        lib().oracle_triples_energies(self.o, v, int(bool(restricted)), _p(self.eps), _p(self.fov), _p(self.t1),
                                      _p(self.t2), _p(self.vvov), _p(self.vooo), _p(self.vvoo), _p(work), _p(out))
        return {"+T": complex(out[0]), "(T)": complex(out[0] + out[1]), "-T": complex(out[0] + out[2])}

    def energies_of(self, triples) -> dict:
        """Partial sums of the same three energies over a list of unique occupied triples (i<j<k): what one rank of a
        multi-GPU split evaluates ("only the unique blocks").  Over all C(o,3) triples = energies()."""
        v = self.v
        ijk = np.ascontiguousarray(np.asarray(list(triples), dtype=np.int32).reshape(-1, 3))
        assert all(0 <= a < b < c < self.o for a, b, c in ijk)
        work = np.zeros(6 * v ** 3, dtype=C128)
        out = np.zeros(3, dtype=C128)
        lib().oracle_triples_energies_list(self.o, v, int(ijk.shape[0]), ijk.ctypes.data_as(ctypes.c_void_p), _p(self.eps),
                                           _p(self.fov), _p(self.t1), _p(self.t2), _p(self.vvov), _p(self.vooo),
                                           _p(self.vvoo), _p(work), _p(out))
        return {"+T": complex(out[0]), "(T)": complex(out[0] + out[1]), "-T": complex(out[0] + out[2])}


# ---------------------------------------------------------------------------------------------------------------
# single-element evaluator straight from the factorised integrals (full-size spot checks at cfg2 / cfg3, where the
# plain-loop oracle would need hours): eq 40 + the cyclic sum written out for one (i,j,k,a,b,c).
# ---------------------------------------------------------------------------------------------------------------
def _g(B, p, q, r, s):
    """<pq||rs> = (pr|qs) - (ps|qr), (pq|rs) = sum_L B[L,p,q] B[L,r,s]; any of p,q,r,s may be an index array."""
    return np.einsum("l...,l...->...", B[:, p, r], B[:, q, s]) - np.einsum("l...,l...->...", B[:, p, s], B[:, q, r])


def _t2(t2p, o, v, i, j, a, b):
    """signed lookup t2[i,j,a,b] in the packed array [(i<j)][(a<b)]; a or b may be arrays (the other scalar)."""
    if i == j:
        return np.zeros(np.broadcast(a, b).shape, dtype=C128)
    sg = 1.0
    if i > j:
        i, j, sg = j, i, -sg
    row = t2p[i * o - i * (i + 1) // 2 + (j - i - 1)]
    a, b = np.broadcast_arrays(np.asarray(a), np.asarray(b))
    lo, hi = np.minimum(a, b), np.maximum(a, b)
    idx = lo * v - lo * (lo + 1) // 2 + (hi - lo - 1)
    val = np.where(a == b, 0.0, row[np.where(a == b, 0, idx)])
    return sg * np.where(a < b, 1.0, -1.0) * val


def w_element_from_B(B, nocc, t2p, i, j, k, a, b, c):
    """W[i,j,k,a,b,c] of eq 40 (reading G22) for one index sextuple."""
    o, v = nocc, B.shape[1] - nocc
    e = np.arange(v)
    m = np.arange(o)
    s = 0.0
    for (x, y, z) in ((i, j, k), (j, k, i), (k, i, j)):
        s += np.sum(_g(B, o + a, o + b, x, o + e) * _t2(t2p, o, v, y, z, e, c))          # <ab||xe> t2[y,z,e,c]
        gm = _g(B, o + a, m, x, y)                                                       # <am||xy>
        tm = np.array([_t2(t2p, o, v, z, mm, b, c) for mm in range(o)]).reshape(o)       # t2[z,m,b,c]
        s += np.sum(gm * tm)
    return s


def wbar_samples_from_B(B, nocc, t2p, ijk, abc):
    """Wbar = W^abc + W^bca + W^cab at sampled (i,j,k), (a,b,c)."""
    out = np.zeros(len(ijk), dtype=C128)
    for n, ((i, j, k), (a, b, c)) in enumerate(zip(ijk, abc)):
        out[n] = (w_element_from_B(B, nocc, t2p, i, j, k, a, b, c) + w_element_from_B(B, nocc, t2p, i, j, k, b, c, a) +
                  w_element_from_B(B, nocc, t2p, i, j, k, c, a, b))
    return out
