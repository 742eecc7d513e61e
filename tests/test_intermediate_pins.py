"""Pin P6: the oracle's INDIVIDUAL intermediates of eqs 24-31 against the textbook
spin-orbital CCSD intermediates BASELINE.json's north_star names (F_ae, F_mi, F_me, W_mnij, W_mbej, in the form of
Stanton, Gauss, Watts and Bartlett, J. Chem. Phys. 94, 4334 (1991)), written out here independently with numpy.einsum
on the full antisymmetrised integral tensor <pq||rs> of tests/detspace.py.  CPU only.

The GPU tests compare Hvv, Gvv, Hoo, Goo, Hov, Hvovo, C and A one by one with the oracle; pin P1 fixes them only through
the sums S1 and S2.  The identities below give each a second, independently derived formula:

    H^k_c        =  F_me[k,c]
    G^a_c        =  F_ae[a,c] - 1/2 sum_m t^a_m F_me[m,c]
    G^k_i        = -( F_mi[k,i] + 1/2 sum_e t^e_i F_me[k,e] )
    A^{kl}_{ij}  =  W_mnij[k,l,i,j] + 1/4 sum_ef tau^{ef}_{ij} <kl||ef>
    H^{ak}_{ci}  = -W_mbej[k,a,c,i]
with the textbook definitions (f WITH its diagonal, reading G4; tau~ = t2 + 1/2 P-(t1 t1), tau = t2 + P-(t1 t1)):
    F_ae   = f_ae - 1/2 sum_m f_me t^a_m + sum_mf t^f_m <ma||fe> - 1/2 sum_mnf tau~^{af}_{mn} <mn||ef>
    F_mi   = f_mi + 1/2 sum_e t^e_i f_me + sum_en t^e_n <mn||ie> + 1/2 sum_nef tau~^{ef}_{in} <mn||ef>
    F_me   = f_me + sum_nf t^f_n <mn||ef>
    W_mnij = <mn||ij> + P-_ij sum_e t^e_j <mn||ie> + 1/4 sum_ef tau^{ef}_{ij} <mn||ef>
    W_mbej = <mb||ej> + sum_f t^f_j <mb||ef> - sum_n t^b_n <mn||ej> - sum_nf (1/2 t^{fb}_{jn} + t^f_j t^b_n) <mn||ef>
H^a_c and H^k_i (eqs 24, 26) are the same textbook pieces with tau instead of tau~ and without the t1 terms; they are
checked in that form.  C^{kb}_{ij} (eq 30) has no textbook counterpart of its own (the paper folds <mb||ij>, part of the
t1-dressing of W_mbej and that of W_abef into it): it stays pinned through S2, here additionally against the complete
textbook doubles equation built from F_ae, F_mi, W_mnij, W_abef, W_mbej.
"""
import numpy as np
import pytest

import ccsd_inputs as ci
from oracle.ccsd_oracle import OracleCCSD, unpack_t2
from tests.detspace import antisymmetrised_integrals


def _textbook(f, g, t1, t2, o):
    """Stanton-Gauss-Watts-Bartlett intermediates; f[n][n], g[p,q,r,s] = <pq||rs>, t1[i,a], t2[i,j,a,b]."""
    O, V = slice(0, o), slice(o, None)
    fov, foo, fvv = f[O, V], f[O, O], f[V, V]
    t1t1 = np.einsum("ia,jb->ijab", t1, t1) - np.einsum("ib,ja->ijab", t1, t1)
    tau_t = t2 + 0.5 * t1t1
    tau = t2 + t1t1
    F_me = fov + np.einsum("nf,mnef->me", t1, g[O, O, V, V])
    F_ae = (fvv - 0.5 * np.einsum("me,ma->ae", fov, t1) + np.einsum("mf,mafe->ae", t1, g[O, V, V, V])
            - 0.5 * np.einsum("mnaf,mnef->ae", tau_t, g[O, O, V, V]))
    F_mi = (foo + 0.5 * np.einsum("ie,me->mi", t1, fov) + np.einsum("ne,mnie->mi", t1, g[O, O, O, V])
            + 0.5 * np.einsum("inef,mnef->mi", tau_t, g[O, O, V, V]))
    x = np.einsum("je,mnie->mnij", t1, g[O, O, O, V])
    W_mnij = g[O, O, O, O] + x - x.transpose(0, 1, 3, 2) + 0.25 * np.einsum("ijef,mnef->mnij", tau, g[O, O, V, V])
    W_mbej = (g[O, V, V, O] + np.einsum("jf,mbef->mbej", t1, g[O, V, V, V]) - np.einsum("nb,mnej->mbej", t1, g[O, O, V, O])
              - np.einsum("jnfb,mnef->mbej", 0.5 * t2, g[O, O, V, V])
              - np.einsum("jf,nb,mnef->mbej", t1, t1, g[O, O, V, V]))
    return dict(F_me=F_me, F_ae=F_ae, F_mi=F_mi, W_mnij=W_mnij, W_mbej=W_mbej, tau=tau)


@pytest.mark.parametrize("o,v,restricted", [(3, 5, False), (4, 7, True), (2, 6, False), (5, 4, True)])
def test_p6_oracle_intermediates_equal_textbook_intermediates(o, v, restricted):
    inp = ci.make_inputs(o, v, 9, seed=600 + 10 * o + v, b_scale=0.25, f_offdiag=0.15)
    t1, t2p = ci.random_amplitudes(o, v, 61 + o, 0.3)
    t2 = unpack_t2(t2p, o, v)
    oc = OracleCCSD(inp.h, inp.B, o, v, restricted=restricted)
    oc.set_amplitudes(t1, t2)
    oc.build_intermediates()
    g = antisymmetrised_integrals(inp.B)
    O, V = slice(0, o), slice(o, None)
    tb = _textbook(inp.f_target, g, t1, t2, o)
    tol = 2e-14
    for name in ("F_me", "F_ae", "F_mi", "W_mnij", "W_mbej"):
        assert np.abs(tb[name]).max() > 0.05, name                  # large couplings: nothing hides
    assert np.abs(oc.tau - tb["tau"]).max() < tol                   # eq 23
    assert np.abs(oc.Hov - tb["F_me"]).max() < tol                  # eq 28
    assert np.abs(oc.Gvv - (tb["F_ae"] - 0.5 * np.einsum("ma,mc->ac", t1, tb["F_me"]))).max() < tol      # eq 25
    assert np.abs(oc.Goo + (tb["F_mi"] + 0.5 * np.einsum("ie,ke->ki", t1, tb["F_me"]))).max() < tol      # eq 27
    A_ref = tb["W_mnij"] + 0.25 * np.einsum("ijef,klef->klij", tb["tau"], g[O, O, V, V])
    assert np.abs(oc.A - A_ref).max() < tol                         # eq 31
    assert np.abs(oc.Hvovo + tb["W_mbej"].transpose(1, 0, 2, 3)).max() < tol       # eq 29: H[a,k,c,i] = -W_mbej[k,a,c,i]
    # eqs 24, 26: H differs from G by the two printed t1 terms; expressed through textbook pieces only
    Hvv_ref = oc.Gvv - np.einsum("kd,akcd->ac", t1, g[V, O, V, V]) + np.einsum("kc,ka->ac", inp.f_target[O, V], t1)
    Hoo_ref = oc.Goo + np.einsum("lc,klic->ki", t1, g[O, O, O, V]) + np.einsum("kc,ic->ki", inp.f_target[O, V], t1)
    assert np.abs(oc.Hvv - Hvv_ref).max() < tol and np.abs(oc.Hoo - Hoo_ref).max() < tol
    # ... and on their own: H^a_c = f_ac + 1/2 V tau (eq 24), H^k_i = -f_ki + 1/2 V tau (eq 26) as tau~-forms:
    #   F_ae + 1/2 f_me t - V t1 + 1/4 P-(t1t1)V  (the difference tau - tau~ = 1/2 P-(t1 t1))
    t1t1 = np.einsum("ia,jb->ijab", t1, t1) - np.einsum("ib,ja->ijab", t1, t1)
    Hvv_tb = (tb["F_ae"] + 0.5 * np.einsum("me,ma->ae", inp.f_target[O, V], t1) - np.einsum("mf,mafe->ae", t1, g[O, V, V, V])
              - 0.25 * np.einsum("mnaf,mnef->ae", t1t1, g[O, O, V, V]))
    Hoo_tb = -(tb["F_mi"] - 0.5 * np.einsum("ie,me->mi", t1, inp.f_target[O, V]) - np.einsum("ne,mnie->mi", t1, g[O, O, O, V])
               + 0.25 * np.einsum("inef,mnef->mi", t1t1, g[O, O, V, V]))
    assert np.abs(oc.Hvv - Hvv_tb).max() < tol and np.abs(oc.Hoo - Hoo_tb).max() < tol


def test_p6_c_intermediate_through_the_textbook_doubles_equation():
    """C^{kb}_{ij} (eq 30) has no textbook name: in the Stanton form its content is split between <mb||ij>, the t1-dressing
    of W_mbej and that of W_abef.  It enters S2 only through P-_ab sum_k C^{ka}_{ij} t^b_k, so it is pinned by requiring the
    oracle's eight terms of eq 32 with ITS C to equal the textbook doubles equation term by term where they match one to
    one, and in the sum elsewhere -- here: the whole textbook D2 equation (with W_abef) against the oracle's S2."""
    o, v = 3, 5
    inp = ci.make_inputs(o, v, 9, seed=6035, b_scale=0.25, f_offdiag=0.15)
    t1, t2p = ci.random_amplitudes(o, v, 64, 0.3)
    t2 = unpack_t2(t2p, o, v)
    oc = OracleCCSD(inp.h, inp.B, o, v)
    oc.set_amplitudes(t1, t2)
    _, S2 = oc.residual()
    g = antisymmetrised_integrals(inp.B)
    f = inp.f_target
    O, V = slice(0, o), slice(o, None)
    tb = _textbook(f, g, t1, t2, o)
    tau, F_me = tb["tau"], tb["F_me"]
    x = np.einsum("mb,amef->abef", t1, g[V, O, V, V])
    W_abef = g[V, V, V, V] - (x - x.transpose(1, 0, 2, 3)) + 0.25 * np.einsum("mnab,mnef->abef", tau, g[O, O, V, V])
    Fae = tb["F_ae"] - 0.5 * np.einsum("mb,me->be", t1, F_me)
    Fmi = tb["F_mi"] + 0.5 * np.einsum("je,me->mj", t1, F_me)

    def pab(y):
        return y - y.transpose(0, 1, 3, 2)

    def pij(y):
        return y - y.transpose(1, 0, 2, 3)

    D2 = (g[O, O, V, V].conj()                                                    # <ab||ij> as [i,j,a,b]
          + pab(np.einsum("ijae,be->ijab", t2, Fae)) - pij(np.einsum("imab,mj->ijab", t2, Fmi))
          + 0.5 * np.einsum("mnab,mnij->ijab", tau, tb["W_mnij"]) + 0.5 * np.einsum("ijef,abef->ijab", tau, W_abef)
          + pij(pab(np.einsum("imae,mbej->ijab", t2, tb["W_mbej"]) - np.einsum("ie,ma,mbej->ijab", t1, t1, g[O, V, V, O])))
          + pij(np.einsum("ie,abej->ijab", t1, g[V, V, V, O])) - pab(np.einsum("ma,mbij->ijab", t1, g[O, V, O, O])))
    assert np.abs(D2).max() > 0.5
    assert np.abs(S2 - D2).max() < 5e-13
