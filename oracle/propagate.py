"""Oracle of ONE phaseless-AFQMC propagation step around the hot path.  TEST INFRASTRUCTURE.

PAPER.md Eq. 5 and Eq. 7-12, step by step, in numpy (float64 / complex128), on top of oracle tier O2 for the two
quantities the hot path supplies (overlap Eq. 13+15, force bias Eq. 7).  Nothing here is shared with the CUDA path.

    h'        = h - 1/2 sum_g L^g L^g                                                  Eq. 4,  (pr|rq) = sum_g L^g_pr L^g_rq
    v_g       = <Psi_T| sum_pq L^g_pq a+_p a_q |psi> / <Psi_T|psi>                    Eq. 7 without its prefactor (O2)
    xbar_g    = -i sqrt(dt) v_g                                                        Eq. 7, reading A20 (below)
    B(dt, y)  = exp(-dt h'/2) exp(i sqrt(dt) sum_g y_g L^g) exp(-dt h'/2)              Eq. 5, reading A20
    psi'      = B(dt, x - xbar) psi                                                    (Thouless: B acts on the orbital matrix)
    S         = <Psi_T|psi'> / <Psi_T|psi>                                             Eq. 8
    theta     = arg S                                                                  Eq. 9
    I         = S exp(x.xbar - xbar.xbar/2)                                            Eq. 10 (plain sums, no conjugation)
    I_ph      = |I| max(0, cos theta),  w' = I_ph w                                    Eq. 11-12

Readings (the paper prints neither B nor how its exponential is applied):
  A20  Eq. 3 has +1/2 sum_g (L^g)^2, so the Hubbard-Stratonovich field couples as exp(i sqrt(dt) x_g L^g)
       (exp(-dt v^2/2) = int p(x) exp(i sqrt(dt) x v)); the optimal shift is then xbar = -i sqrt(dt) v: Eq. 7 as printed
       lacks the factor i (it would be right for L -> iL).  The symmetric split of the one-body part is the usual one and
       keeps Eq. 5's O(dt^2) error.  Pinned by the Fock-space test of Eq. 5 in tests/test_oracle_propagate.py.
  A21  exp(-dt h'/2) is the exact matrix exponential (here: eigendecomposition of the real symmetric h');
       exp(A) psi with A = i sqrt(dt) sum_g y_g L^g is the Taylor series truncated after order n_taylor (default 6, the
       value of the ipie code the paper extends): psi + A psi + A(A psi)/2 + ... ; n_taylor is an argument of the step.
"""
from __future__ import annotations

import numpy as np

from . import o2


def h_prime(h1: np.ndarray, L: np.ndarray) -> np.ndarray:
    """Eq. 4 with (pr|rq) = sum_g L^g_pr L^g_rq."""
    return h1 - 0.5 * np.einsum("gpr,grq->pq", L, L)


def exp_one_body(h1: np.ndarray, L: np.ndarray, dt: float) -> np.ndarray:
    """exp(-dt h'/2), h' real symmetric (A21)."""
    w, U = np.linalg.eigh(h_prime(h1, L))
    return (U * np.exp(-0.5 * dt * w)) @ U.T


def apply_taylor(A: np.ndarray, psi: np.ndarray, n_taylor: int) -> np.ndarray:
    """sum_{k <= n} A^k psi / k!  (A21), term by term."""
    out = psi.copy()
    term = psi.copy()
    for k in range(1, n_taylor + 1):
        term = (A @ term) / k
        out = out + term
    return out


def apply_B(h1, L, dt, y, psi, n_taylor=6):
    """B(dt, y) psi for ONE walker's orbital matrix psi [N][n] (Eq. 5, A20-A21); y complex [n_chol]."""
    E = exp_one_body(h1, L, dt)
    A = 1j * np.sqrt(dt) * np.einsum("g,gpq->pq", y, L)
    return E @ apply_taylor(A, E @ psi, n_taylor)


def step(inp, x, dt, weights=None, n_taylor=6, walkers=None):
    """One propagation step of the walkers of `inp` with the auxiliary fields x [n_w][n_chol] (real, drawn by the caller).

    Returns dict(phi_a, phi_b (the propagated walkers), ovlp_old, ovlp_new, fb (v), xbar, S, theta, I, I_ph, w)."""
    ws = np.arange(inp.n_w) if walkers is None else np.asarray(walkers)
    x = np.asarray(x, dtype=np.float64)[ws]
    w0 = np.ones(len(ws)) if weights is None else np.asarray(weights, dtype=np.float64)[ws]
    r = o2.run(inp, walkers=ws, want=("ovlp", "greens"), return_G=False)
    v = r["fb"]
    xbar = -1j * np.sqrt(dt) * v
    E = exp_one_body(inp.h1, inp.L, dt)
    pa = np.empty_like(inp.phi_a[ws])
    pb = np.empty_like(inp.phi_b[ws])
    for k, w in enumerate(ws):
        A = 1j * np.sqrt(dt) * np.einsum("g,gpq->pq", x[k] - xbar[k], inp.L)
        pa[k] = E @ apply_taylor(A, E @ inp.phi_a[w], n_taylor)
        pb[k] = E @ apply_taylor(A, E @ inp.phi_b[w], n_taylor)
    new = o2.o2(inp.h1, inp.L, inp.e0, inp.occa, inp.occb, inp.ci, pa, pb, want=("ovlp",))
    S = new["ovlp"] / r["ovlp"]
    theta = np.angle(S)
    I = S * np.exp(np.sum(x * xbar, axis=1) - 0.5 * np.sum(xbar * xbar, axis=1))
    I_ph = np.abs(I) * np.maximum(0.0, np.cos(theta))
    return dict(phi_a=pa, phi_b=pb, ovlp_old=r["ovlp"], ovlp_new=new["ovlp"], fb=v, xbar=xbar, S=S, theta=theta, I=I,
                I_ph=I_ph, w=I_ph * w0)
