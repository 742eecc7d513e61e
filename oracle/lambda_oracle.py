"""ORACLE -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

CCSD Lambda equations and the Lagrange one-body density matrix (arXiv 2103.08473 Appendix 7.4-7.5, PAPER.md:674-730,
eqs 45-61; eqs 12-16) in plain numpy, one ``einsum`` per printed term, on top of the
amplitudes and integral classes of the plain CPU CCSD oracle.  It is the reference the CUDA Lambda solver
(ccsd_lambda_* / ccsd_density) is compared with and shares no code with it.

The paper prints the two Lambda equations (eqs 52-56), G (eqs 50-51), three of the similarity-transformed-Hamiltonian
elements (eqs 45-49: W^{ij}_{mn}, W^{mb}_{ej}, W^{ef}_{am}) and Fbar^e_a (eq 57), and refers to its ref. 39 for "the
full list including intermediates".  Reading G23: the missing elements (Fbar^j_m, Fbar^j_b,
W^{ef}_{ab}, W^{ej}_{ab}, W^{ij}_{mb}, W^{nf}_{am}) are the one- and two-body elements of Hbar = exp(-T) H exp(T) in
the form of Gauss and Stanton, J. Chem. Phys. 103, 3561 (1995); eqs 48-49 are garbled in extraction and are taken in
that form too.  EVERY element is pinned, through the residuals, by the determinant-space definition
    R_mu = <0| (1 + Lambda) (Hbar - E_CC) |mu>          (tests/test_lambda_pins.py, brute force at converged T)
so a wrong sign, factor or index in any of them fails the pin.  Index conventions as in 7.1 (G1): V^{pq}_{rs} = <pq||rs>;
lambda^i_a = l1[i,a], lambda^{ij}_{ab} = l2[i,j,a,b] (antisymmetric in ij and in ab).

Pins: tests/test_lambda_pins.py.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this module.  It imports nothing from paper_2103_08473_b200.
"""
from __future__ import annotations

import numpy as np

from oracle.ccsd_oracle import C128, pack_t2, unpack_t2



def E(subscripts, *operands):
    """One printed term = one einsum; optimize=True lets numpy hand the two-operand products to its matmul."""
    return np.einsum(subscripts, *operands, optimize=True)



def _p_ij(x):
    return x - x.transpose(1, 0, 2, 3)


def _p_ab(x):
    return x - x.transpose(0, 1, 3, 2)


class OracleLambda:
    """Lambda equations at the amplitudes of an OracleCCSD object `oc` (which should be converged: the working
    equations are <0|(1+Lambda)(Hbar - E)|mu> = 0 only up to terms proportional to the CC residual)."""

    def __init__(self, oc, ndiis: int = 6):
        o, v = oc.o, oc.v
        self.o, self.v, self.ndiis = o, v, ndiis
        self.t1, self.t2 = oc.t1.copy(), oc.t2.copy()
        f = oc.f
        self.foo, self.fov, self.fvv = f[:o, :o], f[:o, o:], f[o:, o:]
        self.D1, self.D2 = oc.D1, oc.D2
        # the six stored classes and their daggers / antisymmetry images (reading G5)
        self.oooo, self.ooov, self.oovv, self.vovv, self.vvvv = oc.oooo, oc.ooov, oc.oovv, oc.vovv, oc.vvvv
        self.ovvo = -oc.vovo.transpose(1, 0, 2, 3)                 # <mb||ej> = -<bm||ej>
        self.ovoo = np.conj(oc.ooov).transpose(2, 3, 0, 1)         # <mb||ij> = conj <ij||mb>
        self.vvvo = np.conj(oc.vovv).transpose(2, 3, 0, 1)         # <ab||ei> = conj <ei||ab>
        self.ovvv = -oc.vovv.transpose(1, 0, 2, 3)                 # <mb||ef> = -<bm||ef>
        self.oovo = -oc.ooov.transpose(0, 1, 3, 2)                 # <mn||ej> = -<mn||je>
        self.build_hbar()
        # start: lambda = conj(t) (first order: lambda^{ij}_{ab} = <ij||ab>/D = conj t^{ab}_{ij}); the paper is silent
        self.l1, self.l2 = np.conj(self.t1), np.conj(self.t2)
        self._diis_u, self._diis_e = [], []

    # --- elements of Hbar (eqs 45-49, 57 and the rest of the list of ref. 39; reading G23) -----------------------
    def build_hbar(self):
        t1, t2 = self.t1, self.t2
        oovv, ooov, vovv, oooo, vvvv = self.oovv, self.ooov, self.vovv, self.oooo, self.vvvv
        ovvo, ovoo, vvvo, ovvv, oovo = self.ovvo, self.ovoo, self.vvvo, self.ovvv, self.oovo
        tau = t2 + E("ia,jb->ijab", t1, t1) - E("ib,ja->ijab", t1, t1)                      # eq 23
        # Fbar^m_e, Fbar^m_i, Fbar^a_e (eq 57: f - f t + V t - sum_{m>n} V tau)
        self.Fov = self.fov + E("nf,mnef->me", t1, oovv)
        self.Foo = (self.foo + E("ie,me->mi", t1, self.fov) + E("ne,mnie->mi", t1, ooov)
                    + 0.5 * E("inef,mnef->mi", tau, oovv))
        self.Fvv = (self.fvv - E("ma,me->ae", t1, self.fov) + E("mf,amef->ae", t1, vovv)
                    - 0.5 * E("mnaf,mnef->ae", tau, oovv))
        # eq 45: W^{mn}_{ij} = V + P(ij) V t + sum_{e<f} V tau
        x = E("je,mnie->mnij", t1, ooov)
        self.Woooo = oooo + x - x.transpose(0, 1, 3, 2) + 0.5 * E("ijef,mnef->mnij", tau, oovv)
        # W^{ab}_{ef} = V - P(ab) t V + sum_{m<n} tau V
        self.Wvvvv = vvvv - E("mb,amef->abef", t1, vovv) + E("ma,bmef->abef", t1, vovv) \
            + 0.5 * E("mnab,mnef->abef", tau, oovv)
        self.Wvovv = vovv - E("na,nmef->amef", t1, oovv)                                   # W^{am}_{ef}
        self.Wooov = ooov + E("if,mnfe->mnie", t1, oovv)                                   # W^{mn}_{ie}
        # eqs 46-47: W^{mb}_{ej} = V + V t - V t - sum V (t2 + t1 t1)
        self.Wovvo = (ovvo + E("jf,mbef->mbej", t1, ovvv) - E("nb,mnej->mbej", t1, oovo)
                      - E("jnfb,mnef->mbej", t2, oovv) - E("jf,nb,mnef->mbej", t1, t1, oovv))
        # W^{mb}_{ij}
        inner = ovvo - E("njbf,mnef->mbej", t2, oovv)
        x = E("jnbe,mnie->mbij", t2, ooov) + E("ie,mbej->mbij", t1, inner)
        self.Wovoo = (ovoo - E("me,ijbe->mbij", self.Fov, t2) - E("nb,mnij->mbij", t1, self.Woooo)
                      + 0.5 * E("ijef,mbef->mbij", tau, ovvv) + x - x.transpose(0, 1, 3, 2))
        # eqs 48-49: W^{ab}_{ei}
        x = E("miaf,mbef->abei", t2, ovvv) + E("ma,mbei->abei", t1, inner)
        self.Wvvvo = (vvvo - E("me,miab->abei", self.Fov, t2) + E("if,abef->abei", t1, self.Wvvvv)
                      + 0.5 * E("mnab,mnei->abei", tau, oovo) - (x - x.transpose(1, 0, 2, 3)))

    # --- eqs 50-56 -----------------------------------------------------------------------------------------------
    def residual(self, l1=None, l2=None):
        """Right-hand sides of eqs 55-56 (R1[i,a]) and 52-54 (R2[i,j,a,b]) at (l1, l2) (default: the current ones)."""
        l1 = self.l1 if l1 is None else l1
        l2 = self.l2 if l2 is None else l2
        t2, oovv = self.t2, self.oovv
        Gvv = -0.5 * E("mnef,mnaf->ae", t2, l2)                                            # eq 50
        Goo = 0.5 * E("mnef,inef->mi", t2, l2)                                             # eq 51
        R1 = (self.Fov + E("ie,ea->ia", l1, self.Fvv) - E("ma,im->ia", l1, self.Foo)
              - E("mn,mina->ia", Goo, self.Wooov) - E("ef,eifa->ia", Gvv, self.Wvovv)
              + E("me,ieam->ia", l1, self.Wovvo) - 0.5 * E("mnae,iemn->ia", l2, self.Wovoo)
              + 0.5 * E("imef,efam->ia", l2, self.Wvvvo))
        R2 = (oovv + _p_ab(E("ijae,eb->ijab", l2, self.Fvv)) - _p_ij(E("imab,jm->ijab", l2, self.Foo))
              + 0.5 * E("mnab,ijmn->ijab", l2, self.Woooo)
              + _p_ij(_p_ab(E("imae,jebm->ijab", l2, self.Wovvo)))
              + _p_ab(E("ijae,be->ijab", oovv, Gvv)) - _p_ab(E("ma,ijmb->ijab", l1, self.Wooov))
              - _p_ij(E("imab,mj->ijab", oovv, Goo)) + _p_ij(E("ie,ejab->ijab", l1, self.Wvovv))
              + _p_ij(_p_ab(E("ia,jb->ijab", l1, self.Fov)))
              + 0.5 * E("ijef,efab->ijab", l2, self.Wvvvv))
        return R1, R2

    # --- iteration: Jacobi step lambda <- lambda + R / D and DIIS exactly as for the amplitudes (G12, G13) ----------
    def _vec(self, a1, a2):
        return np.concatenate([a1.ravel(), pack_t2(a2).ravel()])

    def iterate(self):
        """One Lambda iteration.  Returns ||R/D||_2 over the unique multipliers."""
        R1, R2 = self.residual()
        e1, e2 = R1 / self.D1, R2 / self.D2
        u1, u2 = self.l1 + e1, self.l2 + e2
        evec = self._vec(e1, e2)
        step = float(np.sqrt(np.vdot(evec, evec).real))
        if self.ndiis > 0:
            self._diis_u.append(self._vec(u1, u2)); self._diis_e.append(evec)
            if len(self._diis_u) > self.ndiis:
                self._diis_u.pop(0); self._diis_e.pop(0)
            m = len(self._diis_u)
            if m >= 2:
                G = np.zeros((m + 1, m + 1))
                for k in range(m):
                    for l in range(m):
                        G[k, l] = np.vdot(self._diis_e[k], self._diis_e[l]).real
                G[:m, m] = -1.0; G[m, :m] = -1.0
                rhs = np.zeros(m + 1); rhs[m] = -1.0
                c = np.linalg.solve(G, rhs)[:m]
                unew = sum(cl * ul for cl, ul in zip(c, self._diis_u))
                o, v = self.o, self.v
                u1 = unew[: o * v].reshape(o, v)
                u2 = unpack_t2(unew[o * v:].reshape(o * (o - 1) // 2, v * (v - 1) // 2), o, v)
        self.l1, self.l2 = np.ascontiguousarray(u1, dtype=C128), np.ascontiguousarray(u2, dtype=C128)
        return step

    def run(self, niter: int = 60, tol: float = 1e-12):
        hist = []
        for _ in range(niter):
            hist.append(self.iterate())
            if hist[-1] < tol:
                break
        return hist

    # --- eqs 58-61: one-body density matrix ---------------------------------------------------------------------------
    def density(self, l1=None, l2=None):
        """D[p][q] = <0|(1+Lambda) exp(-T) a+_p a_q exp(T)|0> - delta_pq (p occupied): the correlation part of the Lagrange
        one-body density (eqs 15-16), [n][n] with occupied spinors first, assembled from eqs 58-61.
        Reading G24: the printed blocks are gamma_ij = <a+_i a_j> (eq 58), gamma_ab = <a+_b a_a> (eq 61),
        gamma_ia = <a+_a a_i> (eq 59), gamma_ai = <a+_i a_a> (eq 60) -- fixed by the determinant-space pin; the paper
        symmetrises the matrix before use, this returns it unsymmetrised."""
        l1 = self.l1 if l1 is None else l1
        l2 = self.l2 if l2 is None else l2
        t1, t2, o, v = self.t1, self.t2, self.o, self.v
        g_ij = -0.5 * E("imef,jmef->ij", t2, l2) - E("ie,je->ij", t1, l1)                   # eq 58 (lambda^{mj} = -lambda^{jm})
        g_ia = l1                                                                          # eq 59
        g_ai = (t1 + E("me,imae->ia", l1, t2) - E("me,ie,ma->ia", l1, t1, t1)
                - 0.5 * E("mnef,inef,ma->ia", l2, t2, t1) - 0.5 * E("mnef,ie,mnaf->ia", l2, t1, t2))   # eq 60, as [i][a]
        g_ab = 0.5 * E("mnae,mnbe->ab", t2, l2) + E("ma,mb->ab", t1, l1)                    # eq 61
        D = np.zeros((o + v, o + v), dtype=C128)
        D[:o, :o] = g_ij
        D[o:, o:] = g_ab.T
        D[:o, o:] = g_ai
        D[o:, :o] = g_ia.T
        return D
