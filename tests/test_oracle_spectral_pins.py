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


def test_argument_checks():
    with pytest.raises(ValueError):
        O.spectral_closed_form(np.ones(4), 1.0, 3, order=5)
    cf = O.spectral_closed_form(np.array([2.0]), 0.5, 0)
    assert len(cf.err) == 1 and cf.err[0] == pytest.approx(0.5) and cf.z[0] == 0.5
