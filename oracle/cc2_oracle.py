"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

CC2 on top of the plain CPU CCSD oracle (arXiv 2103.08473 Appendix 7.2, eqs 34-38).

"In the CC2 method the T1 amplitude equations in 7.1 are unchanged whereas the T2 amplitude equations are given by"
eq 34 with the intermediates of eqs 35-38.  The explicit loops for eqs 34-38 are in ``cc2_oracle.c``;
the singles residual (eq 33), the integral classes, the MP2 start, the Jacobi step, DIIS (reading G13) and the energy
expression (reading G11) are those of ``ccsd_oracle``.

Pins: tests/test_cc2_pins.py (determinant-space definition of the CC2 doubles residual; CCSD(t2=0) identity).
Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may import this module.
"""
from __future__ import annotations

import ctypes
import os

import numpy as np

from oracle._build import compile_oracle

from oracle.ccsd_oracle import C128, OracleCCSD, _p

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libcc2_oracle.so")
_SRC_PATH = os.path.join(_HERE, "cc2_oracle.c")
_lib = None


def build(force: bool = False) -> str:
    return compile_oracle(_SRC_PATH, _LIB_PATH, force)


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
    return _lib


class OracleCC2(OracleCCSD):
    """CC2: singles residual = eq 33 (unchanged), doubles residual = eq 34.  Needs the unpacked <ab||ef> (v^4)."""

    CC2_TERMS = ("driver", "t1_Wvvvo", "t1_Wovoo", "t1t1_Woooo", "t1t1_Wvvvv", "fvv_t2", "foo_t2")

    def __init__(self, h, B, nocc, nvir, ndiis: int = 6, level_shift: float = 0.0):
        super().__init__(h, B, nocc, nvir, ndiis=ndiis, restricted=False, level_shift=level_shift)
        o, v = self.o, self.v
        self.Woooo = np.zeros((o, o, o, o), dtype=C128)
        self.Wvvvv = np.zeros((v, v, v, v), dtype=C128)
        self.Wvvvo = np.zeros((v, v, v, o), dtype=C128)
        self.Wovoo = np.zeros((o, v, o, o), dtype=C128)

    def cc2_intermediates(self):
        L = lib()
        o, v = self.o, self.v
        L.oracle_cc2_Woooo(o, v, _p(self.t1), _p(self.oooo), _p(self.ooov), _p(self.oovv), _p(self.Woooo))
        L.oracle_cc2_Wvvvv(o, v, _p(self.t1), _p(self.vvvv), _p(self.vovv), _p(self.oovv), _p(self.Wvvvv))
        L.oracle_cc2_Wvvvo(o, v, _p(self.t1), _p(self.vovv), _p(self.vovo), _p(self.Wvvvo))
        L.oracle_cc2_Wovoo(o, v, _p(self.t1), _p(self.ooov), _p(self.vovo), _p(self.Wovoo))

    def cc2_s2(self, term: int = -1) -> np.ndarray:
        """eq 34 from the current W intermediates; term = index into CC2_TERMS or -1 for the sum."""
        out = np.zeros_like(self.S2)
        lib().oracle_cc2_s2(self.o, self.v, _p(self.f), _p(self.t1), _p(self.t2), _p(self.oovv), _p(self.Woooo),
                            _p(self.Wvvvv), _p(self.Wvvvo), _p(self.Wovoo), int(term), _p(out))
        return out

    def residual(self):
        """S1 by eq 33 with the full (t1, t2) ("unchanged"), S2 by eqs 34-38."""
        from oracle.ccsd_oracle import lib as ccsd_lib
        self.build_intermediates()
        ccsd_lib().oracle_s1(ctypes.byref(self.sys), _p(self.t1), _p(self.t2), ctypes.byref(self.inter), _p(self.S1))
        self.cc2_intermediates()
        self.S2 = self.cc2_s2(-1)
        return self.S1, self.S2
