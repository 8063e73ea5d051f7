"""Pins of the oracle's Algorithm 3 (`refine_with_refi`, `update_mixed`) -- CPU only.

Alg. 3 (Sec. IV.B) has no closed form, so it is pinned against what the paper
and the mathematics fix:
  * the err[] layout, entry by entry, against Frobenius norms formed directly (numpy.linalg.norm of
    I - Z^T S Z) from the low-precision run's own Z and from the returned Z;
  * a single-precision refinement of an (h)(h)-level run lands at the `single` level;
  * a double-precision refinement reaches the FP64 level, a single-precision one cannot
    on an ill-conditioned S;
  * the algebra of one update: R_1 = c R_0^3 + ... holds for the FP64 step, and a correction
    evaluated in a lower precision u leaves an O(u ||R_0||) term behind -- measured slope 1 in ||R_0||.
None of these re-uses the function under test to produce its own expected value.
"""
import math

import numpy as np
import pytest

from oracle import zfac_oracle as O
from paper_2404_19163_b200 import workloads as W


def _fro_residual(S, Z):
    S = np.asarray(S, np.float64); Z = np.asarray(Z, np.float64)
    return float(np.linalg.norm(np.eye(S.shape[0]) - Z.T @ S @ Z, "fro"))


@pytest.mark.parametrize("steps,final_check", [(1, True), (2, True), (1, False), (3, False)])
def test_err_layout_entry_by_entry(steps, final_check):
    w = W.random_spd_general(40, 3, kappa=200.0, pert=0.1, fp32_stored=True)
    low = O.refine(w.S, w.Z0, 30, O.STOP_PAPER, dtype=np.float32)
    k = low.iters
    res = O.refine_with_refi(w.S, w.Z0, 30, low_dtype=np.float32, refi_steps=steps, final_check=final_check)
    assert res.iters == k + steps and res.flags == low.flags
    assert len(res.err) == (k + 1) + steps + (1 if final_check else 0)
    assert np.array_equal(res.err[: k + 1], low.err)                      # the low-precision history, untouched
    # err[k+1]: the FP64 re-evaluation of the SAME Z the low-precision run returned (step 2 of Sec. IV.B)
    assert res.err[k + 1] == pytest.approx(_fro_residual(w.S, low.Z), rel=1e-9)
    # entries k+1 .. k+steps are taken BEFORE each update: replay the updates with plain numpy expressions
    Z = np.asarray(low.Z, np.float64)
    for j in range(steps):
        assert res.err[k + 1 + j] == pytest.approx(_fro_residual(w.S, Z), rel=1e-6, abs=1e-15)
        R = np.eye(w.n) - Z.T @ w.S @ Z
        Z = Z @ (np.eye(w.n) + 0.5 * R + 0.375 * R @ R)
    if final_check:
        assert res.err[-1] == pytest.approx(_fro_residual(w.S, res.Z), rel=1e-6, abs=1e-15)
    assert np.allclose(res.Z, Z, rtol=1e-12, atol=1e-14)
    with pytest.raises(ValueError):
        O.refine_with_refi(w.S, w.Z0, 30, refi_steps=0)


def test_single_precision_refinement_of_a_half_precision_run_reaches_the_single_level():
    """"(h)(h) + refi ... the 2-norm error drops to the same level as that of the single
    method".  float16 stands in for the (h)(h) arithmetic (11-bit operands)."""
    w = W.random_spd_general(48, 11, kappa=8.0, pert=0.05, fp32_stored=True)
    half = O.refine(w.S, w.Z0, 30, O.STOP_PAPER, dtype=np.float16)
    single = O.refine(w.S, w.Z0, 30, O.STOP_PAPER, dtype=np.float32)
    res = O.refine_with_refi(w.S, w.Z0, 30, low_dtype=np.float16, refi_steps=2, refi_dtype=np.float32)
    assert res.Z.dtype == np.float32
    r_half, r_single, r_refi = (_fro_residual(w.S, z) for z in (half.Z, single.Z, res.Z))
    assert r_half > 30.0 * r_single                     # the (h)(h)-level run is far from the single level ...
    assert r_refi < 3.0 * r_single                      # ... the single-precision refinement brings it there
    assert r_refi > 1e-9                                # ... and no further: it IS single precision


def test_double_refinement_reaches_fp64_level_single_cannot_when_ill_conditioned():
    """"Because of the large condition number, it is important to do the refinement step in
    double precision.  A single precision refinement only lowers the error to around 1e-3"; after the double
    precision step "the error is around 1e-11"."""
    w = W.random_spd_general(64, 5, kappa=1e5, pert=0.02, fp32_stored=True)
    r64 = O.refine_with_refi(w.S, w.Z0, 40, low_dtype=np.float32, refi_steps=2, refi_dtype=np.float64)
    r32 = O.refine_with_refi(w.S, w.Z0, 40, low_dtype=np.float32, refi_steps=2, refi_dtype=np.float32)
    a, b = _fro_residual(w.S, r64.Z) / math.sqrt(w.n), _fro_residual(w.S, r32.Z) / math.sqrt(w.n)
    assert a < 1e-10
    assert b > 1e3 * a and b > 1e-7
    # both are inverse factors of the same S to their precision: Z Z^T = S^-1 (Eq. 10)
    Sinv = np.linalg.inv(w.S)
    assert np.linalg.norm(r64.Z @ r64.Z.T - Sinv) / np.linalg.norm(Sinv) < 1e-9


def test_fp64_refinement_step_obeys_the_printed_error_polynomial():
    """One FP64 refinement update maps R_0 to 5/8 R_0^3 + 15/64 R_0^4 + 9/64 R_0^5 (PAPER.md:267 with R = -delta):
    err[k+2] of a final_check run must be that norm, formed here from the printed coefficients."""
    w = W.random_spd_general(24, 17, kappa=30.0, pert=0.2, fp32_stored=True)
    res = O.refine_with_refi(w.S, w.Z0, 0, low_dtype=np.float32, refi_steps=1)      # no low-precision update: Z = Z0
    R0 = np.eye(w.n) - w.Z0.T @ w.S @ w.Z0
    R3 = R0 @ R0 @ R0
    R1 = 5 / 8 * R3 + 15 / 64 * R3 @ R0 + 9 / 64 * R3 @ R0 @ R0
    assert res.err[1] == pytest.approx(np.linalg.norm(R0, "fro"), rel=1e-12)
    assert res.err[2] == pytest.approx(np.linalg.norm(R1, "fro"), rel=1e-9)


def test_mixed_update_leaves_u_times_r_and_two_steps_reach_the_fp64_floor():
    """`update_mixed`: the correction Z(1/2 R + 3/8 R R) in float32, added to a float64 master.  With the exact
    correction, R_1 is cubic in R_0 (above); rounding the correction to u = 2^-24 adds a term linear in
    ||R_0||: R_1 ~ -(dQ + dQ^T), ||dQ|| ~ u ||Q||.  Pinned by (i) the size of what is left, between 0.01 u and
    100 u times ||R_0|| and far above the cubic term, (ii) its slope 1 in ||R_0|| (two starts whose R_0 differ by
    10x), (iii) two mixed steps at the FP64 floor, where a float32 MASTER is stuck ~1e-7 above it, and
    (iv) update_dtype = float64 being the plain update, bit for bit."""
    u = 2.0 ** -24
    base = W.random_spd_general(48, 23, kappa=50.0, pert=0.0, fp32_stored=False)
    lam, V = np.linalg.eigh(base.S)
    Zex = (V / np.sqrt(lam)) @ V.T
    G = np.random.default_rng(1).standard_normal((48, 48)) / math.sqrt(48)
    left = []
    for eps in (1e-5, 1e-6):
        Z = Zex @ (np.eye(48) + eps * G)
        R0 = O.residual(base.S, Z)
        Z1 = O.update_mixed(Z, R0, np.float32)
        assert Z1.dtype == np.float64
        r0, r1 = O.err_fro(R0), _fro_residual(base.S, Z1)
        cubic = _fro_residual(base.S, O.update_delta_form(Z, R0))
        assert 0.01 * u * r0 < r1 < 100.0 * u * r0
        assert r1 > 20.0 * cubic                                          # it is the rounding term, not the cubic one
        left.append(r1)
        assert np.array_equal(O.update_mixed(Z, R0, np.float64), O.update_delta_form(Z, R0))
    assert left[0] / left[1] == pytest.approx(10.0, rel=0.5)              # linear in ||R_0||
    w = W.random_spd_general(48, 29, kappa=1e4, pert=0.05, fp32_stored=True)
    mixed = O.refine_with_refi(w.S, w.Z0, 40, low_dtype=np.float32, refi_steps=2, update_dtype=np.float32)
    full = O.refine_with_refi(w.S, w.Z0, 40, low_dtype=np.float32, refi_steps=2)
    single_master = O.refine_with_refi(w.S, w.Z0, 40, low_dtype=np.float32, refi_steps=2, refi_dtype=np.float32)
    fm, ff, fs = (_fro_residual(w.S, r.Z) / math.sqrt(w.n) for r in (mixed, full, single_master))
    assert mixed.Z.dtype == np.float64
    assert fm < 1e-11 and ff < 1e-11
    assert fs > 1e3 * fm
    # the mixed history: first FP64 Err equals the full run's (same Z); the second is the u ||R|| term, above the cubic one
    k = mixed.iters - 2
    assert mixed.err[k + 1] == full.err[k + 1]
    assert mixed.err[k + 2] < 1e-4 * mixed.err[k + 1]


def test_alg2_with_mixed_update_converges_to_the_fp64_floor_one_iteration_late_at_most():
    """`refine(..., update_dtype=float32)`: FP64 residual, float32 correction, in every iteration of Alg. 2.  The
    rounding of the correction leaves u ||R_n|| behind (pinned above), which is below the cubic term until
    ||R_n||^2 ~ u: the run tracks the FP64 run entry by entry down to Err ~ 1e-4, reaches the FP64 floor, and needs
    at most one update more.  A float32 MASTER (dtype = float32) stalls ~1e5 higher."""
    w = W.random_spd_general(40, 31, kappa=1e3, pert=0.1, fp32_stored=True)
    full = O.refine(w.S, w.Z0, 40, O.STOP_PAPER)
    mixed = O.refine(w.S, w.Z0, 40, O.STOP_PAPER, update_dtype=np.float32)
    single = O.refine(w.S, w.Z0, 40, O.STOP_PAPER, dtype=np.float32)
    assert full.iters <= mixed.iters <= full.iters + 1
    for k in range(min(full.iters, mixed.iters)):
        if full.err[k] > 1e-4:
            assert mixed.err[k] == pytest.approx(full.err[k], rel=1e-4)
    fm, ff, fs = (_fro_residual(w.S, r.Z) / math.sqrt(w.n) for r in (mixed, full, single))
    assert fm < 1e-12 and ff < 1e-12 and fs > 1e3 * fm
    same = O.refine(w.S, w.Z0, 40, O.STOP_PAPER, update_dtype=np.float64)
    assert same.iters == full.iters and np.array_equal(same.Z, full.Z) and np.array_equal(same.err, full.err)
    # both are the inverse factor reached from the same start: the rotation the float32 correction adds is ~u ||R_0||
    assert np.linalg.norm(mixed.Z - full.Z) / np.linalg.norm(full.Z) < 1e-6
    with pytest.raises(ValueError):
        O.refine(w.S, w.Z0, 5, order=3, update_dtype=np.float32)


def test_mixed_update_makes_the_papers_test_fire_one_update_short_of_the_fp64_floor_on_a_cold_start():
    """What ZFAC_OPT_EXTRA_UPDATE (include/zfac.h) is for, on the oracle's own model of the FP64-master update.  From a
    cold start at kappa = 1e5 the last cubic step goes from Err ~ 3e-4 to the u ||R|| sqrt(kappa)-class term the float32
    correction leaves (pinned above), which is ABOVE Err^3: the test of Alg. 2 fires there, one update before
    the all-FP64 run stops, with an invariant ~1e2-1e3 times the FP64 floor.  One more mixed update -- Alg. 3's single
    refinement step -- lands on the floor."""
    w = W.spectral_workload(300, 1e-5, 1.0, seed=0)
    full = O.refine(w.S, w.Z0, 40, O.STOP_PAPER)
    mixed = O.refine(w.S, w.Z0, 40, O.STOP_PAPER, update_dtype=np.float32)
    assert mixed.iters == full.iters - 1 and (mixed.flags & O.R_STOPPED)
    k = mixed.iters
    assert mixed.err[k] > mixed.err[k - 1] ** 3                          # the test fired ...
    assert mixed.err[k] < 1e-4 * mixed.err[k - 1]                        # ... on a residual that had just dropped 1e4-fold
    f_m, f_f = (_fro_residual(w.S, r.Z) / math.sqrt(w.n) for r in (mixed, full))
    assert f_m > 50.0 * f_f and f_m < 1e-8
    Z1 = O.update_mixed(mixed.Z, O.residual(w.S, mixed.Z), np.float32)
    assert _fro_residual(w.S, Z1) / math.sqrt(w.n) < 3.0 * f_f
