"""Fock-space brute force of PAPER.md Eq. 2, 3-4, 7, 13-15 for micro inputs.

Independent of ``oracle/``: no determinants, no inverses, no Wick's theorem.  Many-body
states are dense vectors over the 2^(2N) occupation bit strings of the 2N spin orbitals
(alpha orbital p -> bit p, beta orbital p -> bit N+p); a_j / a+_j act with the
Jordan-Wigner sign (-1)^(number of occupied spin orbitals below j).

A basis determinant with ascending alpha string then ascending beta string is
a+_{p1} a+_{p2} ... |0> with p1 < p2 < ..., which is +|bit string> in this convention
(reading A6 of DESIGN.md).  A walker is  prod_i (sum_p psi_a[p,i] a+_{p,alpha})
prod_j (sum_q psi_b[q,j] a+_{q,beta}) |0>.
"""
from __future__ import annotations

import numpy as np


class Fock:
    def __init__(self, N: int):
        self.N = N
        self.M = 2 * N
        self.dim = 1 << self.M
        idx = np.arange(self.dim, dtype=np.int64)
        self.idx = idx
        self.occ = [((idx >> j) & 1).astype(bool) for j in range(self.M)]
        self.sign = []
        for j in range(self.M):
            below = idx & ((1 << j) - 1)
            pc = np.zeros(self.dim, dtype=np.int64)
            b = below.copy()
            while b.any():
                pc += b & 1
                b >>= 1
            self.sign.append(1.0 - 2.0 * (pc & 1))

    def so(self, p: int, spin: int) -> int:
        return p + spin * self.N

    def annihilate(self, j: int, v: np.ndarray) -> np.ndarray:
        out = np.zeros_like(v)
        src = self.idx[self.occ[j]]
        out[src ^ (1 << j)] = self.sign[j][src] * v[src]
        return out

    def create(self, j: int, v: np.ndarray) -> np.ndarray:
        out = np.zeros_like(v)
        src = self.idx[~self.occ[j]]
        out[src | (1 << j)] = self.sign[j][src] * v[src]
        return out

    def vacuum(self) -> np.ndarray:
        v = np.zeros(self.dim, dtype=np.complex128)
        v[0] = 1.0
        return v

    def basis_det(self, occ_a, occ_b) -> np.ndarray:
        v = self.vacuum()
        ops = [self.so(int(p), 0) for p in occ_a] + [self.so(int(q), 1) for q in occ_b]
        for j in reversed(ops):          # rightmost operator acts first
            v = self.create(j, v)
        return v

    def walker(self, psi_a: np.ndarray, psi_b: np.ndarray) -> np.ndarray:
        v = self.vacuum()
        cols = [(psi_b[:, j], 1) for j in range(psi_b.shape[1])][::-1] + \
               [(psi_a[:, i], 0) for i in range(psi_a.shape[1])][::-1]
        for col, spin in cols:           # last beta column first, first alpha column last
            acc = np.zeros_like(v)
            for p in range(self.N):
                if col[p] != 0:
                    acc += col[p] * self.create(self.so(p, spin), v)
            v = acc
        return v

    def trial(self, ci, occa, occb) -> np.ndarray:
        v = np.zeros(self.dim, dtype=np.complex128)
        for c, oa, ob in zip(ci, occa, occb):
            v += c * self.basis_det(oa, ob)
        return v


def brute_force(h1, L, e0, occa, occb, ci, psi_a, psi_b, hamiltonian="eq2"):
    """<Psi_T|psi>, G, force bias (Eq. 7 without -sqrt(dt)) and mixed energy for ONE walker.

    hamiltonian="eq2": H = sum h a+a + 1/2 sum (ps|qr) a+_p a+_q a_r a_s        (Eq. 2)
    hamiltonian="eq3": H = sum h' a+a + 1/2 sum_g (sum_pq L^g_pq a+_p a_q)^2,
                       h'_pq = h_pq - 1/2 sum_r (pr|rq)                          (Eq. 3-4)
    """
    N = h1.shape[0]
    F = Fock(N)
    T = F.trial(ci, occa, occb)        # real coefficients: <Psi_T| = T^dagger = T^T conj (T real)
    psi = F.walker(psi_a, psi_b)
    ovlp = np.vdot(T, psi)
    eri = np.einsum("gps,gqr->psqr", L, L)     # (ps|qr)

    # one-body: <T| a+_p a_q |psi> = (a_p T)^dagger (a_q psi)
    aT = [[F.annihilate(F.so(p, s), T) for p in range(N)] for s in range(2)]
    aP = [[F.annihilate(F.so(p, s), psi) for p in range(N)] for s in range(2)]
    G = np.zeros((2, N, N), dtype=np.complex128)
    for s in range(2):
        for p in range(N):
            for q in range(N):
                G[s, p, q] = np.vdot(aT[s][p], aP[s][q]) / ovlp
    fb = np.einsum("gpq,pq->g", L, G[0] + G[1])
    E1 = np.sum(h1 * (G[0] + G[1]))

    if hamiltonian == "eq2":
        # <T| a+_ps a+_qt a_rt a_ss |psi> = (a_qt a_ps T)^dagger (a_rt a_ss psi)
        E2 = 0.0j
        for s in range(2):
            for t in range(2):
                aaT = {(p, q): F.annihilate(F.so(q, t), aT[s][p]) for p in range(N) for q in range(N)}
                aaP = {(r, ss): F.annihilate(F.so(r, t), aP[s][ss]) for r in range(N) for ss in range(N)}
                for p in range(N):
                    for q in range(N):
                        for r in range(N):
                            for ss in range(N):
                                if eri[p, ss, q, r] != 0.0:
                                    E2 += 0.5 * eri[p, ss, q, r] * np.vdot(aaT[(p, q)], aaP[(r, ss)])
        E2 = E2 / ovlp
        return dict(ovlp=ovlp, G=G, fb=fb, E=np.array([e0 + E1 + E2, E1, E2]))

    # Eq. 3-4: apply the one-body operator v_g = sum_pq L^g_pq sum_sigma a+_p a_q twice
    hp = h1 - 0.5 * np.einsum("prrq->pq", eri)

    def apply_one_body(mat, v):
        out = np.zeros_like(v)
        for s in range(2):
            for q in range(N):
                aq = F.annihilate(F.so(q, s), v)
                if not aq.any():
                    continue
                for p in range(N):
                    if mat[p, q] != 0.0:
                        out += mat[p, q] * F.create(F.so(p, s), aq)
        return out

    Hpsi = apply_one_body(hp, psi)
    for g in range(L.shape[0]):
        Hpsi += 0.5 * apply_one_body(L[g], apply_one_body(L[g], psi))
    Etot = np.vdot(T, Hpsi) / ovlp
    return dict(ovlp=ovlp, G=G, fb=fb, E=np.array([e0 + Etot, np.nan, np.nan]))
