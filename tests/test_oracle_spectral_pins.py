"""Pins of oracle.spectral_closed_form: the refinement for Z0 = alpha I written as N scalar
recursions.  It is the parity reference at N = 16384, where the matrix iteration is too slow, so it is pinned here
against routes that share none of its code.  CPU only."""
import math
import os

import numpy as np
import pytest

from oracle import zfac_oracle as O
from paper_2404_19163_b200 import workloads as W

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


@pytest.mark.parametrize("m", [2, 3, 4])
@pytest.mark.parametrize("n,kappa", [(64, 1e3), (256, 1e2)])
def test_against_the_matrix_iteration(n, kappa, m):
    """`refine` multiplies N x N matrices, the closed form never forms one: Err[] and Z = Q diag(z) Q^T must agree."""
    w = W.spectral_workload(n, 1.0 / kappa, 1.0, seed=4)
    k = {2: 9, 3: 7, 4: 6}[m]
    ref = O.refine(w.S, w.Z0, k, O.STOP_FIXED, order=m)
    cf = O.spectral_closed_form(w.lam, w.alpha, k, order=m)
    assert len(cf.err) == k + 1 and cf.z.shape == (n,)
    for i in range(k + 1):
        if ref.err[i] > 1e-9:
            assert cf.err[i] == pytest.approx(ref.err[i], rel=1e-9)
    Z = (w.Q * cf.z) @ w.Q.T
    assert np.linalg.norm(Z - ref.Z) / np.linalg.norm(ref.Z) < 1e-13 * math.sqrt(kappa)
    assert ref.err[0] > 1.0 and ref.err[k] < 1e-6                 # the run really spans start to convergence


@pytest.mark.parametrize("m", [2, 3, 4])
def test_limit_is_inverse_square_root(m):
    lam = np.geomspace(1e-4, 1.0, 500)
    cf = O.spectral_closed_form(lam, 1.0, 40, order=m)
    assert np.max(np.abs(cf.z * np.sqrt(lam) - 1.0)) < 1e-14
    assert cf.err[-1] < 1e-13
    assert all(cf.err[i + 1] <= cf.err[i] for i in range(len(cf.err) - 1) if cf.err[i] > 1e-12)   # monotone (Q10)


def test_against_the_surveys_80_bit_tables():
    """SURVEY.md §8(c) prints Err_F[n] for configs 1, 3, 5 from an independent 80-bit computation (golden file,
    with its citation).  alpha = 1/sqrt(lam_max) exactly, as the table states."""
    rows = 0
    for line in open(os.path.join(GOLDEN, "survey_closed_form_err.txt")):
        f = line.split("#")[0].split()
        if not f:
            continue
        n, lo, hi = int(f[1]), float(f[2]), float(f[3])
        want = [float(x) for x in f[4:]]
        lam = lo * (hi / lo) ** (np.arange(n) / (n - 1))
        cf = O.spectral_closed_form(lam, 1.0 / math.sqrt(hi), len(want) - 1)
        for i, v in enumerate(want):
            assert cf.err[i] == pytest.approx(v, rel=2e-6), (f[0], i)    # 7 printed digits
        rows += 1
    assert rows == 3


def _decimal_history(n, lo, hi, updates, digits=50):
    """The same N scalar recursions in `decimal` arithmetic at `digits` significant digits (test-local, no numpy):
    lam_i = lo (hi/lo)^(i/(N-1)), z_0 = 1/sqrt(hi), r = 1 - lam z^2, z <- z (1 + r/2 + 3 r^2/8)."""
    import decimal
    D = decimal.Decimal
    with decimal.localcontext() as ctx:
        ctx.prec = digits
        ratio = D(hi) / D(lo)
        lam = [D(lo) * ratio ** (D(i) / D(n - 1)) for i in range(n)]
        z = [D(1) / D(hi).sqrt()] * n
        out = []
        for k in range(updates + 1):
            r = [D(1) - l * zi * zi for l, zi in zip(lam, z)]
            out.append(float(sum(x * x for x in r).sqrt()))
            z = [zi * (D(1) + x / 2 + D(3) * x * x / 8) for zi, x in zip(z, r)]
        return [float(l) for l in lam], out


def test_against_50_digit_decimal_arithmetic_and_provenance_of_the_stored_table():
    """Brute force in extended precision (pin list): the FP64 closed form agrees with 50-digit
    decimal arithmetic to FP64 rounding, and every value of the stored table (golden/survey_closed_form_err.txt, the
    surveyor's 80-bit numbers) is reproduced by that decimal computation to its 7 printed digits -- so the fixture's
    content is checkable inside the repository, not taken on trust."""
    for line in open(os.path.join(GOLDEN, "survey_closed_form_err.txt")):
        f = line.split("#")[0].split()
        if not f or int(f[1]) > 1000:                  # the N = 256 row in full; the large rows below on a prefix
            continue
        n, lo, hi = int(f[1]), f[2], f[3]
        want = [float(x) for x in f[4:]]
        lam, dec = _decimal_history(n, lo, hi, len(want) + 1)
        for i, v in enumerate(want):
            assert dec[i] == pytest.approx(v, rel=2e-6), (f[0], i)
        cf = O.spectral_closed_form(np.array(lam), 1.0 / math.sqrt(float(hi)), len(want) + 1)
        for i in range(len(want) + 2):
            if dec[i] > 1e-9:
                assert cf.err[i] == pytest.approx(dec[i], rel=1e-11), i
        assert dec[len(want)] < 1e-5 and dec[len(want) + 1] < 1e-15      # 5.7e-7, then below FP64 resolution
    # the two large rows: first four entries (4617 / 8192 recursions x 4 updates in decimal is still a second or two)
    for line in open(os.path.join(GOLDEN, "survey_closed_form_err.txt")):
        f = line.split("#")[0].split()
        if not f or int(f[1]) <= 1000:
            continue
        _, dec = _decimal_history(int(f[1]), f[2], f[3], 3, digits=30)
        for i in range(4):
            assert dec[i] == pytest.approx(float(f[4 + i]), rel=2e-6), (f[0], i)


def test_argument_checks():
    with pytest.raises(ValueError):
        O.spectral_closed_form(np.ones(4), 1.0, 3, order=5)
    cf = O.spectral_closed_form(np.array([2.0]), 0.5, 0)
    assert len(cf.err) == 1 and cf.err[0] == pytest.approx(0.5) and cf.z[0] == 0.5
