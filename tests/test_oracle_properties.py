"""Property-based pins of the oracle (hypothesis): the statements below hold for EVERY admissible input, so they are
checked on randomly generated small problems rather than on a few fixed seeds.  CPU only, a few seconds."""
import math

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

from oracle import zfac_oracle as O

SETTINGS = dict(max_examples=30, deadline=None)


def problem(n, seed, kappa, spread):
    """SPD S with condition number kappa and a NON-symmetric start Z0 = S^-1/2 (I + spread G / sqrt(n)), ||R0||_2 < 1."""
    rng = np.random.default_rng(seed)
    Q, _ = np.linalg.qr(rng.standard_normal((n, n)))
    lam = np.geomspace(1.0 / kappa, 1.0, n) if n > 1 else np.array([1.0])
    S = (Q * lam) @ Q.T
    S = 0.5 * (S + S.T)
    Zs = (Q / np.sqrt(lam)) @ Q.T
    Z0 = Zs @ (np.eye(n) + spread * rng.standard_normal((n, n)) / math.sqrt(n))
    return S, Z0


dims = st.integers(min_value=1, max_value=14)
seeds = st.integers(min_value=0, max_value=2 ** 31 - 1)
kappas = st.floats(min_value=1.0, max_value=1e4)
spreads = st.floats(min_value=0.0, max_value=0.25)


@settings(**SETTINGS)
@given(dims, seeds, kappas, spreads)
def test_x_form_and_delta_form_are_the_same_polynomial(n, seed, kappa, spread):
    """Eq. 13 (a_k) and Eq. 16 written in R = I - X give the same update for every Z, S."""
    S, Z0 = problem(n, seed, kappa, spread)
    X = O.triple_product(S, Z0)
    a = O.update_x_form(Z0, X)
    b = O.update_delta_form(Z0, np.eye(n) - X)
    assert np.linalg.norm(a - b) <= 1e-13 * max(1.0, np.linalg.norm(b))


@settings(**SETTINGS)
@given(dims, seeds, kappas, spreads, st.sampled_from([2, 3, 4]))
def test_one_step_obeys_the_error_polynomial_bound(n, seed, kappa, spread, m):
    """||R_1||_2 <= ||R_0||_2^(m+1) whenever ||R_0||_2 < 1 (Eq. 36-38 with nu_max = m + 1: the tail coefficients are
    positive and sum to 1), for symmetric R_0 -- which Z^T S Z always gives."""
    S, Z0 = problem(n, seed, kappa, spread)
    R0 = O.residual(S, Z0)
    r0 = np.linalg.norm(R0, 2)
    if not (1e-6 < r0 < 0.95):
        return
    Z1 = O.update_delta_form(Z0, R0) if m == 2 else O.update_order_m(Z0, R0, m)
    r1 = np.linalg.norm(O.residual(S, Z1), 2)
    assert r1 <= r0 ** (m + 1) * (1 + 1e-9) + 1e-13 * kappa


@settings(**SETTINGS)
@given(dims, seeds, kappas, spreads, st.floats(min_value=1e-3, max_value=1e3))
def test_scaling_covariance(n, seed, kappa, spread, c):
    """(S, Z0) -> (c S, Z0 / sqrt(c)) leaves X, hence the whole Err[] history and the stop index, unchanged, and
    scales Z by 1 / sqrt(c)."""
    S, Z0 = problem(n, seed, kappa, spread)
    a = O.refine(S, Z0, 6, O.STOP_FIXED)
    b = O.refine(c * S, Z0 / math.sqrt(c), 6, O.STOP_FIXED)
    assert a.iters == b.iters
    for ea, eb in zip(a.err, b.err):
        assert eb == pytest.approx(ea, rel=1e-6, abs=1e-12 * kappa)
    assert np.linalg.norm(b.Z * math.sqrt(c) - a.Z) <= 1e-9 * np.linalg.norm(a.Z)


@settings(**SETTINGS)
@given(st.integers(min_value=2, max_value=12), seeds, kappas, spreads)
def test_permutation_covariance(n, seed, kappa, spread):
    """A simultaneous row / column permutation P of S and Z0 permutes every iterate: Z_n -> P Z_n P^T; Err[] unchanged."""
    S, Z0 = problem(n, seed, kappa, spread)
    perm = np.random.default_rng(seed ^ 0x5bd1e995).permutation(n)
    P = np.eye(n)[perm]
    a = O.refine(S, Z0, 5, O.STOP_FIXED)
    b = O.refine(P @ S @ P.T, P @ Z0 @ P.T, 5, O.STOP_FIXED)
    assert np.linalg.norm(b.Z - P @ a.Z @ P.T) <= 1e-9 * np.linalg.norm(a.Z)
    assert np.allclose(a.err, b.err, rtol=1e-6, atol=1e-12 * kappa)


@settings(**SETTINGS)
@given(dims, seeds, st.floats(min_value=1.0, max_value=1e3), spreads)
def test_converged_factor_inverts_s(n, seed, kappa, spread):
    """Whatever the (admissible, non-symmetric) start, the limit satisfies Z Z^T = S^-1 (Eq. 10) and Z^T S Z = I."""
    S, Z0 = problem(n, seed, kappa, spread)
    if np.linalg.norm(O.residual(S, Z0), 2) >= 0.95:
        return
    res = O.refine(S, Z0, 60, O.STOP_PAPER)
    assert res.flags & (O.R_STOPPED | O.R_MAXITER)
    Sinv = np.linalg.inv(S)
    assert np.linalg.norm(res.Z @ res.Z.T - Sinv) <= 1e-10 * kappa * np.linalg.norm(Sinv)
    assert O.final_residual_per_sqrt_n(S, res.Z) <= 1e-12 * kappa
