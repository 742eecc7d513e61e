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
import subprocess

import numpy as np

from oracle.ccsd_oracle import C128, _p

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libtriples_oracle.so")
_SRC_PATH = os.path.join(_HERE, "triples_oracle.c")
_lib = None


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB_PATH) or os.path.getmtime(_LIB_PATH) < os.path.getmtime(_SRC_PATH):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-fcx-limited-range", "-shared", "-fPIC", "-o", _LIB_PATH,
                               _SRC_PATH])
    return _LIB_PATH


def lib():
    global _lib
    if _lib is None:
        build()
        _lib = ctypes.CDLL(_LIB_PATH)
    return _lib


class OracleTriples:
    """+T / (T) / -T at the amplitudes (t1[i][a], t2[i][j][a][b]) of an OracleCCSD-like object `oc`
    (uses oc.f, oc.eps, oc.vovv, oc.ooov, oc.oovv)."""

    def __init__(self, oc, t1=None, t2=None):
        self.o, self.v = oc.o, oc.v
        o = self.o
        self.eps = np.ascontiguousarray(oc.eps, dtype=np.float64)
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
