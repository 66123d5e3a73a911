"""Pins of oracle/propagate.py (one phaseless-AFQMC step, Eq. 5, 7-12) -- no GPU.

The paper prints no numbers for a step, so the oracle is pinned by what Eq. 5 and Eq. 10 themselves assert:
  Q1  Eq. 5 in Fock space: int dx p(x) B(x) = exp(-dt H) + O(dt^2), H of Eq. 3-4, on the micro input.  Left side by
      Gauss-Hermite quadrature over all auxiliary fields with B(x)|phi> built from the propagated orbital matrix (Thouless);
      right side by diagonalising H on the full 2^(2N) Fock space (tests/fock_bruteforce.py: no determinants, no Wick).
      Fixes the sign and the factor i of the field coupling, h' of Eq. 4 and the symmetric split (reading A20).
  Q2  the force-bias shift is an identity: int p(x) I(x, xbar) <T|phi> = int p(x) <T|B(x)|phi>  (Eq. 8, Eq. 10)
  Q3  dt -> 0:  (I(x = 0) - 1)/dt -> -(sum h'_pq G_pq + 1/2 sum_g v_g^2), with G and v from oracle tier O2
  Q4  the truncated Taylor series (reading A21) converges to the matrix exponential; order 6 error is bounded
  Q5  Eq. 9, 11, 12: theta = arg S, I_ph = |I| max(0, cos theta) real and non-negative, weights scale
"""
import itertools

import numpy as np
import pytest
import scipy.linalg

import msd_inputs as mi
from fock_bruteforce import Fock
from oracle import o2
from oracle import propagate as op


def _fock_h(F, hp, L):
    """Dense matrix of H = sum h' a+a + 1/2 sum_g (sum L^g a+a)^2 (Eq. 3) on the full Fock space."""
    N = F.N

    def one_body(mat):
        M = np.zeros((F.dim, F.dim))
        eye = np.eye(F.dim)
        for s in range(2):
            for q in range(N):
                for p in range(N):
                    if mat[p, q] != 0.0:
                        for col in range(F.dim):
                            aq = F.annihilate(F.so(q, s), eye[:, col].astype(complex))
                            if aq.any():
                                M[:, col] += mat[p, q] * F.create(F.so(p, s), aq).real
        return M

    H = one_body(hp)
    for g in range(L.shape[0]):
        V = one_body(L[g])
        H += 0.5 * V @ V
    return H


@pytest.fixture(scope="module")
def micro():
    x = mi.generate("micro")
    F = Fock(x.N)
    H = _fock_h(F, op.h_prime(x.h1, x.L), x.L)
    assert np.abs(H - H.T).max() < 1e-12
    return x, F, H, F.trial(x.ci, x.occa, x.occb)


def _quadrature(n_fields, n_nodes):
    t, w = np.polynomial.hermite_e.hermegauss(n_nodes)
    w = w / np.sqrt(2.0 * np.pi)
    for idx in itertools.product(range(n_nodes), repeat=n_fields):
        yield t[list(idx)], float(np.prod(w[list(idx)]))


def _hs_average(x, F, T, w, dt, xbar=None, n_nodes=6):
    acc = 0.0j
    for xs, wt in _quadrature(x.n_chol, n_nodes):
        y = xs if xbar is None else xs - xbar
        pa = op.apply_B(x.h1, x.L, dt, y, x.phi_a[w], n_taylor=24)
        pb = op.apply_B(x.h1, x.L, dt, y, x.phi_b[w], n_taylor=24)
        val = np.vdot(T, F.walker(pa, pb))
        if xbar is not None:
            val *= np.exp(np.sum(xs * xbar) - 0.5 * np.sum(xbar * xbar))
        acc += wt * val
    return acc


def test_q1_eq5_hubbard_stratonovich_in_fock_space(micro):
    x, F, H, T = micro
    ev, U = np.linalg.eigh(H)
    errs = []
    for dt in (0.04, 0.02):
        exact = np.vdot(T, (U * np.exp(-dt * ev)) @ (U.T @ F.walker(x.phi_a[0], x.phi_b[0])))
        hs = _hs_average(x, F, T, 0, dt)
        errs.append(abs(hs - exact) / abs(exact))
    assert errs[0] < 2e-3 and errs[1] < 5e-4, errs          # a Trotter error, not O(dt) or O(1)
    assert errs[0] / errs[1] > 3.0, errs                    # halving dt at least quarters it (Eq. 5: O(dt^2); the symmetric
                                                            # split is in fact third order on this input: ratio ~ 9)
    # the wrong field coupling (no factor i: exp(+dt v^2/2)) is off at first order in dt
    dt = 0.02
    exact = np.vdot(T, (U * np.exp(-dt * ev)) @ (U.T @ F.walker(x.phi_a[0], x.phi_b[0])))
    wrong = 0.0j
    for xs, wt in _quadrature(x.n_chol, 6):
        pa = op.apply_B(x.h1, x.L, dt, -1j * xs, x.phi_a[0], n_taylor=24)
        pb = op.apply_B(x.h1, x.L, dt, -1j * xs, x.phi_b[0], n_taylor=24)
        wrong += wt * np.vdot(T, F.walker(pa, pb))
    assert abs(wrong - exact) / abs(exact) > 20 * errs[1]


def test_q2_force_bias_shift_is_an_identity(micro):
    x, F, H, T = micro
    dt = 0.02
    r = o2.run(x, walkers=[1], want=("ovlp", "greens"), return_G=False)
    xbar = -1j * np.sqrt(dt) * r["fb"][0]
    plain = _hs_average(x, F, T, 1, dt, n_nodes=6)
    shifted = _hs_average(x, F, T, 1, dt, xbar=xbar, n_nodes=6)
    assert abs(shifted - plain) / abs(plain) < 1e-8
    # and the step's own S, I are what the integrand uses (Eq. 8, Eq. 10) for one field vector
    xs = np.random.default_rng(2).standard_normal((x.n_w, x.n_chol))
    s = op.step(x, xs, dt, n_taylor=24)
    pa = op.apply_B(x.h1, x.L, dt, xs[1] - s["xbar"][1], x.phi_a[1], n_taylor=24)
    pb = op.apply_B(x.h1, x.L, dt, xs[1] - s["xbar"][1], x.phi_b[1], n_taylor=24)
    S = np.vdot(T, F.walker(pa, pb)) / np.vdot(T, F.walker(x.phi_a[1], x.phi_b[1]))
    assert abs(S - s["S"][1]) < 1e-12 * abs(S)
    assert abs(s["xbar"][1] - xbar).max() < 1e-14


@pytest.mark.parametrize("name", ["micro", "tiny", "open-shell"])
def test_q3_small_dt_limit_of_the_importance_function(name):
    x = mi.generate(name)
    r = o2.run(x)
    hp = op.h_prime(x.h1, x.L)
    want = -(np.einsum("pq,wpq->w", hp, r["G"][:, 0] + r["G"][:, 1]) + 0.5 * np.sum(r["fb"] ** 2, axis=1))
    errs = []
    for dt in (1e-4, 1e-5):
        s = op.step(x, np.zeros((x.n_w, x.n_chol)), dt, n_taylor=12)
        got = (s["I"] - 1.0) / dt
        errs.append(np.abs(got - want).max() / np.abs(want).max())
    assert errs[1] < 5e-3 and errs[1] < 0.2 * errs[0], errs        # O(dt) remainder: a wrong sign, a missing 1/2 or h instead
                                                                    # of h' leaves an O(1) mismatch


def test_q4_taylor_series_against_expm():
    x = mi.generate("tiny")
    rng = np.random.default_rng(0)
    y = rng.standard_normal(x.n_chol) + 0.1j * rng.standard_normal(x.n_chol)
    A = 1j * np.sqrt(0.01) * np.einsum("g,gpq->pq", y, x.L)
    ref = scipy.linalg.expm(A) @ x.phi_a[0]
    assert np.abs(op.apply_taylor(A, x.phi_a[0], 30) - ref).max() < 1e-14
    nrm = np.linalg.norm(A, 2)
    e6 = np.abs(op.apply_taylor(A, x.phi_a[0], 6) - ref).max()
    assert e6 <= 1.5 * nrm ** 7 / 5040.0 * np.exp(nrm)            # Lagrange remainder of the order-6 series
    E = op.exp_one_body(x.h1, x.L, 0.01)
    assert np.abs(E - scipy.linalg.expm(-0.005 * op.h_prime(x.h1, x.L))).max() < 1e-13
    assert np.abs(op.h_prime(x.h1, x.L) - (x.h1 - 0.5 * np.einsum("gprrq->pq", np.einsum("gps,gqr->gpsqr", x.L, x.L)))).max() < 1e-13


def test_q5_phaseless_weight_update():
    x = mi.generate("small", n_w=6, n_det=200)
    xs = np.random.default_rng(5).standard_normal((x.n_w, x.n_chol))
    w0 = np.linspace(0.5, 2.0, x.n_w)
    s = op.step(x, xs, 0.005, weights=w0)
    assert np.allclose(s["theta"], np.angle(s["ovlp_new"] / s["ovlp_old"]))
    assert (s["I_ph"] >= 0).all() and np.isrealobj(s["I_ph"])
    assert np.allclose(s["I_ph"], np.abs(s["I"]) * np.clip(np.cos(s["theta"]), 0, None))
    assert np.allclose(s["w"], s["I_ph"] * w0)
    sub = op.step(x, xs, 0.005, weights=w0, walkers=[1, 4])
    assert np.allclose(sub["w"], s["w"][[1, 4]]) and np.allclose(sub["phi_a"], s["phi_a"][[1, 4]])
