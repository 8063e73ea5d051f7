"""Pins of the oracle's higher-order update (m = 3, 4) against what the
paper and the mathematics fix -- none of them re-uses the oracle's closed form c_k = C(2k,k)/4^k.

CPU only.  Exact rational arithmetic (fractions.Fraction) wherever a statement is exact.
"""
from fractions import Fraction as F
import math
import os

import numpy as np
import pytest

from oracle import zfac_oracle as O

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ----------------------------------------------------------------------------- exact polynomial helpers (test-local)
def pmul(a, b):
    out = [F(0)] * (len(a) + len(b) - 1)
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            out[i + j] += x * y
    return out


def derive_coefficients(m):
    """Solve the paper's condition directly: with Z' = Z p(R), X' = p(R)(I - R)p(R), choose
    c_1..c_m one at a time so that the coefficient of r^k in (1 - r) p(r)^2 vanishes for k = 1..m (c_0 = 1).
    The coefficient of r^k is linear in c_k with slope 2 c_0 = 2, so each step is one exact division."""
    c = [F(1)]
    for k in range(1, m + 1):
        trial = c + [F(0)]
        e = pmul([F(1), F(-1)], pmul(trial, trial))
        c.append(-e[k] / 2)                      # d/dc_k of coeff_k[(1 - r) p^2] = 2 c_0
    return c


def tail(c):
    """t(r) = 1 - (1 - r) p(r)^2 as an exact coefficient list."""
    e = pmul([F(1), F(-1)], pmul(c, c))
    t = [-x for x in e]
    t[0] += 1
    return t


def paper_constants():
    """tests/golden/paper_constants.txt: the values PAPER.md:451 and :267 print ("name value" per line)."""
    want = {}
    for line in open(os.path.join(GOLDEN, "paper_constants.txt")):
        line = line.split("#")[0].split()
        if len(line) == 2:
            want[line[0]] = F(line[1])
    return want


def random_problem(n, seed, nonsym=True, spread=0.3):
    rng = np.random.default_rng(seed)
    A = rng.standard_normal((n, n))
    S = A @ A.T / n + np.eye(n)
    lam, V = np.linalg.eigh(S)
    Zs = (V / np.sqrt(lam)) @ V.T
    if nonsym:
        Z0 = Zs @ (np.eye(n) + spread * rng.standard_normal((n, n)) / math.sqrt(n))
    else:
        Z0 = np.eye(n) / math.sqrt(lam[-1] * 1.01)
    return S, Z0, Zs


# ----------------------------------------------------------------------------- coefficients
@pytest.mark.parametrize("m", [2, 3, 4])
def test_coefficients_follow_from_the_vanishing_condition(m):
    c = derive_coefficients(m)
    got = O.order_coefficients(m)
    assert len(got) == m + 1
    for k in range(m + 1):
        assert F(got[k]) == c[k], (k, got[k], c[k])          # dyadic rationals: exact in binary FP
    e = pmul([F(1), F(-1)], pmul(c, c))
    assert e[0] == 1 and all(e[k] == 0 for k in range(1, m + 1))


def test_order_2_maps_onto_the_printed_a_k():
    """PAPER.md:451 prints a = (15/8, -5/4, 3/8) for Z(a0 I + a1 X + a2 X^2); substituting R = I - X into
    c_0 + c_1 R + c_2 R^2 must give exactly that."""
    want = paper_constants()
    c = derive_coefficients(2)
    one_minus_x = [F(1), F(-1)]
    poly = [c[0]]
    term = [F(1)]
    for k in (1, 2):
        term = pmul(term, one_minus_x)
        poly = [a + b for a, b in zip(poly + [F(0)] * (len(term) - len(poly)), [c[k] * t for t in term])]
    assert poly == [want["a0"], want["a1"], want["a2"]]


@pytest.mark.parametrize("m", [2, 3, 4])
def test_tail_is_positive_and_sums_to_one(m):
    """The stop test's exponent: R' = sum_{k=m+1}^{2m+1} t_k R^k with t_k > 0, sum t_k = 1,
    so ||R'|| <= ||R||^(m+1) while ||R|| < 1 -- Eq. 36-38 with nu_max = m + 1.  For m = 2 the t_k are the printed
    c, d, e = 5/8, 15/64, 9/64 in magnitude."""
    t = tail(derive_coefficients(m))
    assert all(x == 0 for x in t[: m + 1])
    assert len(t) == 2 * m + 2
    assert all(x > 0 for x in t[m + 1:])
    assert sum(t) == 1
    if m == 2:
        # printed in delta = X - I = -R: delta' = c delta^3 + d delta^4 + e delta^5; with R = -delta the
        # even power changes sign, so the R-form tail is (c, -d, e)
        g = paper_constants()
        assert t[3:] == [g["c"], -g["d"], g["e"]]


# ----------------------------------------------------------------------------- the update itself
@pytest.mark.parametrize("m", [3, 4])
def test_scalar_step_in_exact_rationals(m):
    """N = 1 brute force: one oracle update against the same step in Fractions (inputs are dyadic, so the
    only difference is FP64 rounding of a handful of operations)."""
    s, z = F(3, 2), F(3, 4)
    r = 1 - z * s * z
    c = derive_coefficients(m)
    z1 = z * sum(c[k] * r ** k for k in range(m + 1))
    r1 = 1 - z1 * s * z1
    res = O.refine(np.array([[float(s)]]), np.array([[float(z)]]), 1, O.STOP_FIXED, order=m)
    assert res.Z[0, 0] == pytest.approx(float(z1), rel=4e-16)
    assert res.err[0] == pytest.approx(abs(float(r)), rel=4e-16)
    assert res.err[1] == pytest.approx(abs(float(r1)), rel=1e-12, abs=1e-17)
    t = tail(c)
    assert r1 == sum(t[k] * r ** k for k in range(len(t)))    # exact identity, ties the tail to the update


@pytest.mark.parametrize("m", [3, 4])
def test_matrix_error_identity_nonsymmetric_start(m):
    """R_1 = sum_k t_k R_0^k as a MATRIX identity for a non-symmetric, non-commuting Z0 (a transposed operand or
    a wrong power in the update breaks it)."""
    S, Z0, _ = random_problem(24, seed=11, nonsym=True, spread=0.25)
    assert np.linalg.norm(Z0 - Z0.T) > 1e-2
    R0 = O.residual(S, Z0)
    Z1 = O.update_order_m(Z0, R0, m)
    R1 = O.residual(S, Z1)
    t = [float(x) for x in tail(derive_coefficients(m))]
    want = np.zeros_like(R0)
    Rk = np.eye(24)
    for k in range(len(t)):
        if k:
            Rk = Rk @ R0
        want += t[k] * Rk
    assert np.linalg.norm(R1 - want) <= 1e-13 * max(1.0, np.linalg.norm(R0))


def test_general_update_reduces_to_the_m2_form():
    S, Z0, _ = random_problem(20, seed=3)
    R = O.residual(S, Z0)
    a = O.update_order_m(Z0, R, 2)
    b = O.update_delta_form(Z0, R)
    assert np.linalg.norm(a - b) <= 1e-15 * np.linalg.norm(b)


@pytest.mark.parametrize("m", [3, 4])
@pytest.mark.parametrize("kappa", [20.0, 1e3])
def test_converges_to_inverse_square_root_from_eigendecomposition(m, kappa):
    n = 48
    rng = np.random.default_rng(5)
    Qm, _ = np.linalg.qr(rng.standard_normal((n, n)))
    lam = np.geomspace(1.0 / kappa, 1.0, n)
    S = (Qm * lam) @ Qm.T
    S = 0.5 * (S + S.T)
    Z0 = np.eye(n) / math.sqrt(1.01)
    res = O.refine(S, Z0, 60, O.STOP_PAPER, order=m)
    w, V = np.linalg.eigh(S)
    Zref = (V / np.sqrt(w)) @ V.T
    assert res.flags & O.R_STOPPED
    assert np.linalg.norm(res.Z - Zref) / np.linalg.norm(Zref) <= 5e-14 * kappa ** 0.5
    assert O.final_residual_per_sqrt_n(S, res.Z) <= 1e-13 * kappa ** 0.5


@pytest.mark.parametrize("m", [2, 3, 4])
def test_observed_order_is_m_plus_one(m):
    """nu_max = m + 1.  Err[1] = C Err[0]^(m+1) with a constant C that depends on the direction of
    R_0 only, so scaling ONE perturbation direction by eps and taking the slope d log Err[1] / d log Err[0]
    between two eps isolates the order (a single log/log ratio cannot tell m + 1 from m + 2: C is unknown).
    Both steps stay well above the FP64 floor."""
    n = 32
    rng = np.random.default_rng(7)
    A = rng.standard_normal((n, n))
    S = A @ A.T / n + np.eye(n)
    lam, V = np.linalg.eigh(S)
    Zs = (V / np.sqrt(lam)) @ V.T
    G = rng.standard_normal((n, n)) / math.sqrt(n)              # non-symmetric direction
    pts = []
    for eps in (0.01, 0.02):
        res = O.refine(S, Zs @ (np.eye(n) + eps * G), 1, O.STOP_FIXED, order=m)
        assert 1e-2 < res.err[0] < 0.5 and res.err[1] > 1e-11, res.err
        assert res.err[1] <= res.err[0] ** (m + 1)              # Eq. 38 holds away from the floor
        pts.append((math.log(res.err[0]), math.log(res.err[1])))
    slope = (pts[1][1] - pts[0][1]) / (pts[1][0] - pts[0][0])
    assert abs(slope - (m + 1)) < 0.05, (slope, pts)      # measured: 2.99994, 4.0004, 5.0014


@pytest.mark.parametrize("m", [3, 4])
def test_generalised_stop_rule(m):
    """Away from the floor the test Err[n] > Err[n-1]^(m+1) never fires (tail coefficients sum to 1); it fires at
    the FP64 floor; the history has iters + 1 entries; FIXED runs exactly max_iter updates."""
    S, Z0, _ = random_problem(40, seed=9, nonsym=True, spread=0.3)
    res = O.refine(S, Z0, 50, O.STOP_PAPER, order=m)
    e = res.err
    assert res.flags == O.R_STOPPED and len(e) == res.iters + 1
    for k in range(1, len(e) - 1):
        assert e[k] <= e[k - 1] ** (m + 1)
    assert e[-1] > e[-2] ** (m + 1) and e[-1] < 1e-12
    # a higher order needs no more updates than a lower one
    assert res.iters <= O.refine(S, Z0, 50, O.STOP_PAPER, order=m - 1).iters
    fx = O.refine(S, Z0, 3, O.STOP_FIXED, order=m)
    assert fx.iters == 3 and fx.flags == O.R_MAXITER and len(fx.err) == 4
    with pytest.raises(ValueError):
        O.refine(S, Z0, 3, order=5)
    with pytest.raises(ValueError):
        O.refine(S, Z0, 3, order=3, form="x")
