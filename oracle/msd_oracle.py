"""Oracle tiers O0 and O1 in plain numpy, complex128 / float64.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Each function cites the passage
of /root/reference/PAPER.md it follows.  No blocking, fusion or reordering
beyond what the definitions state.

Conventions (readings A1, A2, A3, A5, A6):
  * a determinant D_I is the ascending-ordered string of its occupied orbitals,
    alpha string first:  <D_I|psi> = det psi_a[occ_I^a, :] * det psi_b[occ_I^b, :]
    (Eq. 13 with Psi_T = the columns occ_I of the identity).
  * G[p][q] = <a+_p a_q> = [phi (Psi_T^+ phi)^-1 Psi_T^+]_{qp}            (Eq. 14)
  * H = sum h_pq a+_p a_q + 1/2 sum (ps|qr) a+_p a+_q a_r a_s,
    (pq|rs) = sum_g L^g_pq L^g_rs                                          (Eq. 2)
  * <Psi_T| = sum_I c_I <D_I|  with real c_I                                (Eq. 15)
"""
from __future__ import annotations

import numpy as np


# ----------------------------------------------------------------------------
# O1: the definition with dense per-determinant Green's functions
# ----------------------------------------------------------------------------
def sd_overlap_and_greens(psi: np.ndarray, occ: np.ndarray):
    """One spin sector of one determinant.  Eq. 13: d = det(Psi_T^+ psi) with
    Psi_T^+ psi = psi[occ, :];  Eq. 14: G[p][q] = [psi (Psi_T^+ psi)^-1 Psi_T^+]_{qp},
    i.e. G[occ[l], q] = Theta[q, l] with Theta = psi O^-1, all other rows zero."""
    N = psi.shape[0]
    O = psi[occ, :]
    d = np.linalg.det(O) if O.shape[0] > 0 else 1.0 + 0.0j
    G = np.zeros((N, N), dtype=np.complex128)
    if O.shape[0] > 0:
        theta = psi @ np.linalg.inv(O)          # N x n
        G[occ, :] = theta.T
    return d, G


def sd_energy_terms(h1: np.ndarray, L: np.ndarray, Ga: np.ndarray, Gb: np.ndarray):
    """Mixed energy of ONE determinant pair from its Green's functions (PAPER.md:L98:
    2-RDM from the 1-RDM by the generalized Wick's theorem; Eq. 2 for H).
      E1 = sum_pq h_pq (Ga+Gb)_pq
      E2 = 1/2 sum_g [ X_g^2 - sum_sigma sum_pqrs L^g_pq L^g_rs G^s_ps G^s_rq ],
      X_g = sum_pq L^g_pq (Ga+Gb)_pq."""
    Gt = Ga + Gb
    E1 = np.sum(h1 * Gt)
    X = np.einsum("gpq,pq->g", L, Gt)
    exch = 0.0
    for G in (Ga, Gb):
        # sum_pqrs L_pq L_rs G_ps G_rq = sum_pr (L G^T)_pr (L G^T)_rp
        LG = L @ G.T                                    # [g][p][r] = sum_q L^g_pq G_rq
        exch = exch + np.einsum("gpr,grp->g", LG, LG)
    E2 = 0.5 * np.sum(X * X - exch)
    return E1, E2, X


def o1_definition(h1, L, e0, occa, occb, ci, phi_a, phi_b, want_greens=True):
    """SURVEY 8(c) steps 1-6 = PAPER.md:L114 (one SD evaluation per determinant) combined
    by Eq. 15.  Returns dict(ovlp[nw], G[nw,2,N,N], fb[nw,ng], E[nw,3]=(E,E1,E2))."""
    nw = phi_a.shape[0]
    N = h1.shape[0]
    ng = L.shape[0]
    nd = len(ci)
    ovlp = np.zeros(nw, dtype=np.complex128)
    Gout = np.zeros((nw, 2, N, N), dtype=np.complex128)
    fb = np.zeros((nw, ng), dtype=np.complex128)
    E = np.zeros((nw, 3), dtype=np.complex128)
    for w in range(nw):
        num_G = np.zeros((2, N, N), dtype=np.complex128)
        num_E1 = 0.0j
        num_E2 = 0.0j
        den = 0.0j
        for I in range(nd):
            da, Ga = sd_overlap_and_greens(phi_a[w], occa[I])
            db, Gb = sd_overlap_and_greens(phi_b[w], occb[I])
            wI = ci[I] * da * db                     # c_I <D_I|psi>
            e1, e2, _ = sd_energy_terms(h1, L, Ga, Gb)
            den += wI
            num_G[0] += wI * Ga
            num_G[1] += wI * Gb
            num_E1 += wI * e1
            num_E2 += wI * e2
        ovlp[w] = den                                # step 2
        Gout[w] = num_G / den                        # step 3
        fb[w] = np.einsum("gpq,pq->g", L, Gout[w, 0] + Gout[w, 1])   # step 4 = Eq. 7 without -sqrt(dt)
        E[w, 1] = num_E1 / den
        E[w, 2] = num_E2 / den
        E[w, 0] = e0 + E[w, 1] + E[w, 2]             # step 6
    return dict(ovlp=ovlp, G=Gout, fb=fb, E=E)


# ----------------------------------------------------------------------------
# O0: explicit determinants only (no inverse; valid for singular O_I)
# ----------------------------------------------------------------------------
def _det(a: np.ndarray) -> complex:
    return complex(np.linalg.det(a)) if a.shape[0] > 0 else 1.0 + 0.0j


def _one_body_numerators(psi: np.ndarray, occ: np.ndarray) -> np.ndarray:
    """g1[p, q] = <D|a+_p a_q|psi> (one spin sector) = det psi[occ(p->q), :] for p in occ,
    the row of p replaced IN PLACE by row q; zero for p not in occ."""
    N = psi.shape[0]
    g1 = np.zeros((N, N), dtype=np.complex128)
    for l, p in enumerate(occ):
        for q in range(N):
            rows = np.array(occ, dtype=np.int64)
            rows[l] = q
            g1[p, q] = _det(psi[rows, :])
    return g1


def _two_body_numerators(psi: np.ndarray, occ: np.ndarray) -> np.ndarray:
    """g2[p, q, r, s] = <D|a+_p a+_q a_r a_s|psi> (same spin) = det psi[occ(p->s, q->r), :]
    for p != q both in occ; zero otherwise."""
    N = psi.shape[0]
    g2 = np.zeros((N, N, N, N), dtype=np.complex128)
    for lp, p in enumerate(occ):
        for lq, q in enumerate(occ):
            if lp == lq:
                continue
            for r in range(N):
                for s in range(N):
                    rows = np.array(occ, dtype=np.int64)
                    rows[lp] = s
                    rows[lq] = r
                    g2[p, q, r, s] = _det(psi[rows, :])
    return g2


def o0_pure_determinants(h1, L, e0, occa, occb, ci, phi_a, phi_b):
    """Tiny inputs only.  Numerators of Eq. 7 / Eq. 14 / the energy as explicit determinants
    of row-substituted matrices; divides only by the total overlap.  Eq. 2 for H with
    (ps|qr) = sum_g L^g_ps L^g_qr."""
    nw = phi_a.shape[0]
    N = h1.shape[0]
    ng = L.shape[0]
    eri = np.einsum("gps,gqr->psqr", L, L)            # (ps|qr)
    ovlp = np.zeros(nw, dtype=np.complex128)
    Gout = np.zeros((nw, 2, N, N), dtype=np.complex128)
    fb = np.zeros((nw, ng), dtype=np.complex128)
    E = np.zeros((nw, 3), dtype=np.complex128)
    for w in range(nw):
        den = 0.0j
        nG = np.zeros((2, N, N), dtype=np.complex128)
        nE1 = 0.0j
        nE2 = 0.0j
        for I in range(len(ci)):
            da = _det(phi_a[w][occa[I], :])
            db = _det(phi_b[w][occb[I], :])
            g1a = _one_body_numerators(phi_a[w], occa[I])
            g1b = _one_body_numerators(phi_b[w], occb[I])
            g2a = _two_body_numerators(phi_a[w], occa[I])
            g2b = _two_body_numerators(phi_b[w], occb[I])
            den += ci[I] * da * db
            nG[0] += ci[I] * g1a * db
            nG[1] += ci[I] * da * g1b
            nE1 += ci[I] * np.sum(h1 * (g1a * db + da * g1b))
            # 1/2 sum_{sigma tau} sum (ps|qr) <a+_p,s a+_q,t a_r,t a_s,s>
            same = np.einsum("psqr,pqrs->", eri, g2a) * db + da * np.einsum("psqr,pqrs->", eri, g2b)
            # opposite spin: <a+_p a_s>_sigma <a+_q a_r>_tau, both orderings of (sigma,tau)
            opp = 2.0 * np.einsum("psqr,ps,qr->", eri, g1a, g1b)
            nE2 += ci[I] * 0.5 * (same + opp)
        ovlp[w] = den
        Gout[w] = nG / den
        fb[w] = np.einsum("gpq,pq->g", L, Gout[w, 0] + Gout[w, 1])
        E[w, 1] = nE1 / den
        E[w, 2] = nE2 / den
        E[w, 0] = e0 + E[w, 1] + E[w, 2]
    return dict(ovlp=ovlp, G=Gout, fb=fb, E=E)


def run(inp, tier: str = "o1", walkers=None):
    """Convenience: run a tier on an msd_inputs.MSDInputs (optionally a walker subset)."""
    pa, pb = inp.phi_a, inp.phi_b
    if walkers is not None:
        pa, pb = pa[walkers], pb[walkers]
    f = {"o0": o0_pure_determinants, "o1": o1_definition}[tier]
    return f(inp.h1, inp.L, inp.e0, inp.occa, inp.occb, inp.ci, pa, pb)
