"""Brute-force determinant-space machinery used to PIN the oracle (tests only; tiny systems).

Nothing here knows the CCSD working equations.  It builds the Hamiltonian of eq 5 and the cluster
operator of eq 8 (normalised as T2 = 1/4 sum t_ij^ab a+_a a+_b a_j a_i, reading G2) as dense
matrices over all N-electron Slater determinants and evaluates the DEFINITIONS of eqs 9-11:
    E      = <Phi_0| exp(-T) H exp(T) |Phi_0>
    S_mu   = <Phi_mu| exp(-T) H exp(T) |Phi_0>
and the full-CI ground state (lowest eigenvalue of H).

Determinant |D> = a+_{p1} a+_{p2} ... |0> with p1 < p2 < ...; bit p of the integer D set <=> spinor p occupied.
a_p |D> = (-1)^{#occupied q<p} |D - p>,  a+_p |D> = (-1)^{#occupied q<p} |D + p>.
"""
from __future__ import annotations

import itertools

import numpy as np


def antisymmetrised_integrals(B: np.ndarray) -> np.ndarray:
    """<pq||rs> = (pr|qs) - (ps|qr),  (pq|rs) = sum_L B[L,p,q] B[L,r,s]   (eq 6)."""
    eri = np.einsum("lpq,lrs->pqrs", B, B)           # chemists' (pq|rs)
    return eri.transpose(0, 2, 1, 3) - eri.transpose(0, 2, 3, 1)


def _ann(det: int, p: int):
    if not (det >> p) & 1:
        return 0, 0
    sign = -1 if bin(det & ((1 << p) - 1)).count("1") & 1 else 1
    return det ^ (1 << p), sign


def _cre(det: int, p: int):
    if (det >> p) & 1:
        return 0, 0
    sign = -1 if bin(det & ((1 << p) - 1)).count("1") & 1 else 1
    return det | (1 << p), sign


def apply_string(det: int, creators, annihilators):
    """(a+_{c0} a+_{c1} ... a_{x0} a_{x1} ...) |det>: the right-most operator acts first."""
    sign = 1
    for p in reversed(annihilators):
        det, s = _ann(det, p)
        if s == 0:
            return 0, 0
        sign *= s
    for p in reversed(creators):
        det, s = _cre(det, p)
        if s == 0:
            return 0, 0
        sign *= s
    return det, sign


class DetSpace:
    def __init__(self, n: int, nelec: int):
        self.n, self.nelec = n, nelec
        self.dets = [sum(1 << p for p in occ) for occ in itertools.combinations(range(n), nelec)]
        self.index = {d: k for k, d in enumerate(self.dets)}
        self.dim = len(self.dets)
        self.ref = (1 << nelec) - 1          # spinors 0..nelec-1 occupied
        self.iref = self.index[self.ref]

    def one_body(self, h: np.ndarray) -> np.ndarray:
        """sum_pq h[p,q] a+_p a_q"""
        M = np.zeros((self.dim, self.dim), dtype=np.complex128)
        for col, d in enumerate(self.dets):
            for p in range(self.n):
                for q in range(self.n):
                    if h[p, q] == 0:
                        continue
                    d2, s = apply_string(d, [p], [q])
                    if s:
                        M[self.index[d2], col] += s * h[p, q]
        return M

    def two_body(self, g: np.ndarray) -> np.ndarray:
        """1/4 sum_pqrs g[p,q,r,s] a+_p a+_q a_s a_r   (g[p,q,r,s] = <pq||rs>)"""
        M = np.zeros((self.dim, self.dim), dtype=np.complex128)
        n = self.n
        for col, d in enumerate(self.dets):
            for p, q, r, s in itertools.product(range(n), repeat=4):
                if p == q or r == s or g[p, q, r, s] == 0:
                    continue
                d2, sg = apply_string(d, [p, q], [s, r])
                if sg:
                    M[self.index[d2], col] += 0.25 * sg * g[p, q, r, s]
        return M

    def hamiltonian(self, h: np.ndarray, g: np.ndarray) -> np.ndarray:
        return self.one_body(h) + self.two_body(g)

    def cluster_operator(self, t1: np.ndarray, t2: np.ndarray) -> np.ndarray:
        """T = sum_ia t1[i,a] a+_a a_i + 1/4 sum_ijab t2[i,j,a,b] a+_a a+_b a_j a_i   (virtual a -> spinor o+a)."""
        o = self.nelec
        v = self.n - o
        M = np.zeros((self.dim, self.dim), dtype=np.complex128)
        for col, d in enumerate(self.dets):
            for i in range(o):
                for a in range(v):
                    d2, s = apply_string(d, [o + a], [i])
                    if s:
                        M[self.index[d2], col] += s * t1[i, a]
            for i, j in itertools.product(range(o), repeat=2):
                for a, b in itertools.product(range(v), repeat=2):
                    if i == j or a == b:
                        continue
                    d2, s = apply_string(d, [o + a, o + b], [j, i])
                    if s:
                        M[self.index[d2], col] += 0.25 * s * t2[i, j, a, b]
        return M

    def exp_nilpotent(self, T: np.ndarray, vec: np.ndarray, sign: float = 1.0) -> np.ndarray:
        """exp(sign*T) vec by the (terminating) power series."""
        out = vec.copy()
        term = vec.copy()
        for k in range(1, self.nelec + 2):
            term = sign * (T @ term) / k
            out = out + term
        return out

    def similarity_transformed_column(self, H: np.ndarray, T: np.ndarray) -> np.ndarray:
        """w = exp(-T) H exp(T) |Phi_0>"""
        phi0 = np.zeros(self.dim, dtype=np.complex128)
        phi0[self.iref] = 1.0
        return self.exp_nilpotent(T, H @ self.exp_nilpotent(T, phi0, +1.0), -1.0)

    def project_singles(self, w: np.ndarray) -> np.ndarray:
        """S1[i,a] = <Phi_i^a | w>,  |Phi_i^a> = a+_a a_i |Phi_0>"""
        o, v = self.nelec, self.n - self.nelec
        S1 = np.zeros((o, v), dtype=np.complex128)
        for i in range(o):
            for a in range(v):
                d2, s = apply_string(self.ref, [o + a], [i])
                S1[i, a] = s * w[self.index[d2]]
        return S1

    def project_doubles(self, w: np.ndarray) -> np.ndarray:
        """S2[i,j,a,b] = <Phi_ij^ab | w>,  |Phi_ij^ab> = a+_a a+_b a_j a_i |Phi_0>"""
        o, v = self.nelec, self.n - self.nelec
        S2 = np.zeros((o, o, v, v), dtype=np.complex128)
        for i, j in itertools.product(range(o), repeat=2):
            for a, b in itertools.product(range(v), repeat=2):
                if i == j or a == b:
                    continue
                d2, s = apply_string(self.ref, [o + a, o + b], [j, i])
                S2[i, j, a, b] = s * w[self.index[d2]]
        return S2
