"""CPU FP64 ORACLE for the Z-refinement hot path -- TEST INFRASTRUCTURE ONLY.

This file is test infrastructure.  Only `tests/`, `__graft_entry__.smoke()` and
`bench.py`'s `cpu_baseline` / `--impl reference` legs may import it.  It shares
no code with the CUDA path (paper_2404_19163_b200/csrc, binding.py) and imports
nothing from it; it is plain numpy in FP64, with `numpy.matmul` as the only
library primitive.  No blocking, fusion, symmetry trick or reordering beyond
what the paper's algorithm states.

What it computes (PAPER.md = /root/reference/PAPER.md):

  Algorithm 2, m = 2, Frobenius norm
  (PAPER.md:289):

      Z = initial guess; iter = 0; X = Z^T S Z
      for iter < Nmax:
          Err[iter] = ||X - I||_F
          if iter > 0 and Err[iter] > Err[iter-1]^3: break          (Eq. 38)
          iter += 1
          Z = Z (a0 I + a1 X + a2 X^2),  a = (15/8, -5/4, 3/8)        (Eq. 13)
          X = Z^T S Z

  The triple product is formed as A = S Z, then X = Z^T A (Eq. 22, 26,
  PAPER.md:181-205).  Two algebraically identical forms of the update are
  provided: the printed X-form above, and the delta-form of Eq. 16
   written in the residual R = I - X = -delta:

      Z = Z + Z (1/2 R + 3/8 R R)         <=>   Z (15/8 I - 5/4 X + 3/8 X^2)

  (substitute X = I - R).  The delta-form is the default because it is the one
  BASELINE.json's north_star names; tests pin the two against each other.

  Higher orders m = 3, 4.  The paper does not
  print the coefficients for m > 2 ("Reference 1 gives a table"); it fixes them by
  the condition that "the error terms delta^nu = (X_n - I)^nu should vanish up to
  the highest possible order" after each iteration.  In the
  residual R = I - X with Z_{n+1} = Z_n p(R_n), X_{n+1} = p(R)(I - R)p(R), so the
  condition is p(R)^2 (I - R) = I + O(R^{m+1}): p is the degree-m Taylor polynomial
  of (1 - R)^{-1/2},  c_k = C(2k, k) / 4^k = 1, 1/2, 3/8, 5/16, 35/128  (reading Q18;
  for m = 2 it is the printed a_k under X = I - R).  The error then obeys
  R_{n+1} = sum_{k=m+1}^{2m+1} t_k R_n^k with t_k > 0, sum t_k = 1 (for m = 2 the
  printed 5/8, 15/64, 9/64), so the argument of Sec. IV.A
   carries over with the exponent nu_max = m + 1:
  the test is  Err[n] > Err[n-1]^(m+1).

Readings of silent / ambiguous points (repeated in DESIGN.md):
  Q5  the Z returned at the break is the current one (Alg. 2 never rolls back);
  Q6  `iters` = number of Z updates performed = the stop index; Err has iters+1 entries;
  Q7  Err of the final Z is always recorded (also when Nmax is reached);
  Q9  strict '>' as printed; a non-finite Err stops the loop with a flag;
  Q10 the test is applied unconditionally (as Alg. 2), not only when Err < 1;
  Q11 Frobenius norm, one sqrt of an FP64 sum of squares.

Pins (tests/test_oracle_pins.py): exact-rational brute force at N <= 4; the
printed error polynomial c,d,e = 5/8,-15/64,9/64 as a matrix
identity for non-symmetric Z0; Z -> S^-1/2 from a dense eigendecomposition when
Z0 ∝ I; Z Z^T = S^-1 for non-commuting Z0; cubic order; stop-rule cases;
scaling / permutation covariances; diagonal S reduces to N scalar recursions;
`congruence` against the generalized eigenvalues of (H, S) from scipy.linalg.eigh.
`spectral_closed_form` (N scalar recursions for Z0 = alpha I): against the matrix iteration of `refine` at N = 64
and 256 (the two routes share only the coefficients), against z -> lam^-1/2, against 50-digit `decimal` arithmetic,
and against the Err tables SURVEY.md §8(c) prints from an independent 80-bit computation.
Order m = 3, 4 (tests/test_oracle_order_pins.py): the coefficients re-derived in exact
rationals from the vanishing condition alone; m = 2 mapped onto the printed a_k; the
tail t_k > 0 with sum 1 and, for m = 2, equal to the printed c, d, e; a scalar
exact-rational step; the matrix identity R_1 = sum t_k R_0^k for non-symmetric Z0;
Z -> S^-1/2 from numpy.linalg.eigh; observed order m + 1; the generalised stop test.
`refine_with_refi` / `update_mixed` (Alg. 3; tests/test_oracle_refi_pins.py): the err[] layout entry by entry
against norms formed directly from the returned low-precision Z; a float32 refinement of a float16 run lands at
the level of a pure float32 run; a float64 refinement reaches the FP64 floor;
the mixed update leaves u_update ||R|| in the next residual and two mixed steps reach the FP64 floor, while a
run whose MASTER is float32 cannot; update_dtype = float64 reproduces the plain update bit for bit.
Every function below is pinned; none is "parity unpinned".
"""
from __future__ import annotations

import math
from typing import NamedTuple

import numpy as np

# result flags (same meaning as include/zfac.h, values restated, not imported)
R_STOPPED = 1     # the parameter-free test fired (Eq. 38 violated)
R_MAXITER = 2     # Nmax updates were performed without the test firing
R_NONFINITE = 4   # Err became inf/NaN

STOP_PAPER = 0    # Alg. 2 test
STOP_FIXED = 1    # run exactly max_iter updates (benchmark / parity mode)

# Polynomial coefficients for m = 2, from Ref. 1's Table I as quoted at PAPER.md:451.
A0, A1, A2 = 15.0 / 8.0, -5.0 / 4.0, 3.0 / 8.0


class RefineResult(NamedTuple):
    Z: np.ndarray        # final iterate
    iters: int           # number of Z updates performed
    err: np.ndarray      # Err[0..iters], ||Z_n^T S Z_n - I||_F
    flags: int


def triple_product(S: np.ndarray, Z: np.ndarray) -> np.ndarray:
    """X = Z^T S Z via A = S Z, X = Z^T A   (Eq. 22 and Eq. 26)."""
    A = S @ Z
    return Z.T @ A


def residual(S: np.ndarray, Z: np.ndarray) -> np.ndarray:
    """R = I - Z^T S Z = -(X - I) = -delta   (Eq. 12, Eq. 33)."""
    X = triple_product(S, Z)
    return np.eye(S.shape[0], dtype=X.dtype) - X


def err_fro(R: np.ndarray) -> float:
    """Err = ||X - I||_F = ||R||_F   (Alg. 2; norm choice PAPER.md:289)."""
    return float(math.sqrt(float(np.sum(R.astype(np.float64) * R.astype(np.float64)))))


def update_delta_form(Z: np.ndarray, R: np.ndarray) -> np.ndarray:
    """Z_{n+1} = Z_n + Z_n (1/2 R + 3/8 R R)   (Eq. 16 form of Eq. 13 with m = 2)."""
    Q = 0.5 * R + 0.375 * (R @ R)
    return Z + Z @ Q


def update_x_form(Z: np.ndarray, X: np.ndarray) -> np.ndarray:
    """Z_{n+1} = Z_n (a0 I + a1 X + a2 X^2)   (Eq. 13 as printed; Alg. 2)."""
    n = X.shape[0]
    P = A0 * np.eye(n, dtype=X.dtype) + A1 * X + A2 * (X @ X)
    return Z @ P


def update_mixed(Z: np.ndarray, R: np.ndarray, update_dtype) -> np.ndarray:
    """Z_{n+1} = Z_n + D with the correction D = Z_n (1/2 R + 3/8 R R) (Eq. 16 form of Eq. 13, m = 2) evaluated
    in `update_dtype` from the operands rounded to it, and ADDED to the master Z in Z's own precision.  This is
    step 3 of Sec. IV.B when only the residual of step 2 is recomputed in the enhanced
    precision: D is a correction of relative size ||R||, so its rounding error u_update ||R|| is what is left
    of the update in the next residual (reading Q-R2)."""
    Ru = np.asarray(R, dtype=update_dtype)
    Zu = np.asarray(Z, dtype=update_dtype)
    Q = 0.5 * Ru + 0.375 * (Ru @ Ru)
    D = Zu @ Q
    return Z + np.asarray(D, dtype=Z.dtype)


def order_coefficients(m: int) -> list:
    """c_0..c_m of p(R) = sum c_k R^k, the degree-m Taylor polynomial of (1 - R)^{-1/2}:
    c_k = C(2k, k) / 4^k  (the vanishing-order condition of PAPER.md:121-123; reading Q18)."""
    if m < 1:
        raise ValueError("order m must be >= 1")
    return [math.comb(2 * k, k) / 4.0 ** k for k in range(m + 1)]


def update_order_m(Z: np.ndarray, R: np.ndarray, m: int) -> np.ndarray:
    """Z_{n+1} = Z_n + Z_n (c_1 R + c_2 R^2 + ... + c_m R^m)   (Eq. 13 / Eq. 16 with general m,
    PAPER.md:112-131).  The powers of R are formed one by one, R^k = R^{k-1} R, and summed in
    increasing k: no Horner form, no regrouping."""
    c = order_coefficients(m)
    Rk = R
    Q = c[1] * R
    for k in range(2, m + 1):
        Rk = Rk @ R
        Q = Q + c[k] * Rk
    return Z + Z @ Q


def refine(S: np.ndarray, Z0: np.ndarray, max_iter: int, stop: int = STOP_PAPER,
           form: str = "delta", dtype=np.float64, order: int = 2, update_dtype=None) -> RefineResult:
    """Algorithm 2.  `dtype` exists only so that the paper's
    `single` scheme (Table I) can be emulated in a pin; the oracle
    proper is FP64.  `order` = m of Eq. 13 (2 = the paper's tests; 3, 4 = SURVEY.md §8(f3));
    the stop test uses the exponent nu_max = m + 1 (Eq. 38).
    `update_dtype` (m = 2 only): the correction of every update is evaluated in that precision and added to the
    `dtype` master (`update_mixed`): Alg. 2 with the enhanced-precision residual of Sec. IV.B in EVERY iteration."""
    if max_iter < 0:
        raise ValueError("max_iter must be >= 0")
    if order < 2 or order > 4:
        raise ValueError("order must be 2, 3 or 4")
    if order != 2 and form != "delta":
        raise ValueError("the X-form is printed for m = 2 only (PAPER.md:303, :451)")
    if update_dtype is not None and (order != 2 or form != "delta"):
        raise ValueError("the mixed update is defined for m = 2 in the delta form")
    S = np.asarray(S, dtype=dtype)
    Z = np.array(Z0, dtype=dtype, copy=True)
    n = S.shape[0]
    eye = np.eye(n, dtype=dtype)
    err = []
    flags = 0
    it = 0
    X = triple_product(S, Z)
    while True:
        R = eye - X
        err.append(err_fro(R))
        if not math.isfinite(err[it]):
            flags |= R_NONFINITE
            break
        if stop == STOP_PAPER and it > 0 and err[it] > err[it - 1] ** (order + 1):
            flags |= R_STOPPED
            break
        if it == max_iter:
            flags |= R_MAXITER
            break
        it += 1
        if order != 2:
            Z = update_order_m(Z, R, order)
        elif update_dtype is not None:
            Z = update_mixed(Z, R, update_dtype)
        elif form == "delta":
            Z = update_delta_form(Z, R)
        elif form == "x":
            Z = update_x_form(Z, X)
        else:
            raise ValueError(form)
        X = triple_product(S, Z)
    return RefineResult(Z, it, np.asarray(err, dtype=np.float64), flags)


class SpectralResult(NamedTuple):
    z: np.ndarray        # z_n per eigenvalue: Z_n = Q diag(z_n) Q^T
    err: np.ndarray      # Err[0..iters] = (sum_i r_{n,i}^2)^(1/2)


def spectral_closed_form(lam: np.ndarray, alpha: float, iters: int, order: int = 2) -> SpectralResult:
    """The refinement for the special start Z0 = alpha I, written per eigenvalue.

    With S = Q diag(lam) Q^T and Z0 = alpha I, every Z_n is a polynomial in S: Z_n = Q diag(z_n) Q^T, and
    Eq. 13 / Eq. 16 decouple into N independent scalar recursions

        r_i = 1 - lam_i z_i^2,      z_i <- z_i (1 + c_1 r_i + ... + c_m r_i^m),

    with Err[n] = ||R_n||_F = (sum_i r_{n,i}^2)^(1/2) because Q is orthogonal.  No matrix is
    formed: this is the parity reference at sizes where the matrix iteration is too slow (N = 16384), after ONE
    N^3 reconstruction Q diag(z) Q^T by the caller.  Runs exactly `iters` updates (no stop test).  Exact only when
    `lam` are the eigenvalues of the S actually used: for FP32-stored S they are perturbed by ~6e-8 ||S||."""
    if order < 2 or order > 4:
        raise ValueError("order must be 2, 3 or 4")
    lam = np.asarray(lam, dtype=np.float64)
    c = order_coefficients(order)
    z = np.full(lam.shape, float(alpha), dtype=np.float64)
    err = []
    for n in range(iters + 1):
        r = 1.0 - lam * z * z
        err.append(math.sqrt(float(np.sum(r * r))))
        if n == iters:
            break
        rk = r
        q = c[1] * r
        for k in range(2, order + 1):
            rk = rk * r
            q = q + c[k] * rk
        z = z + z * q
    return SpectralResult(z, np.asarray(err, dtype=np.float64))


def refine_with_refi(S: np.ndarray, Z0: np.ndarray, max_iter: int, low_dtype=np.float32,
                     refi_steps: int = 1, refi_dtype=np.float64, update_dtype=None,
                     final_check: bool = True) -> RefineResult:
    """Algorithm 3 (Sec. IV.B):
      1. Alg. 2 in the lower precision `low_dtype` until the test of Eq. 38 fires (or max_iter updates);
      2. "Z = FP32[Z] or FP64[Z]": Z is converted to the enhanced precision `refi_dtype`
         (float32 = the paper's single-precision refinement; float64)
         and X = Z^T S Z is recomputed in it (S converted to it as well);
      3. Z_{n+1} is computed in the enhanced precision -- or, with `update_dtype` given, its correction
         Z (1/2 R + 3/8 R R) alone is evaluated in `update_dtype` and added to the `refi_dtype` master
         (`update_mixed`).
    Steps 2-3 are repeated `refi_steps` times ("Typically we would only do one extra refinement step,
    although we could continue").

    err[] layout (k = stop index of the low-precision run):
        err[0..k]               the low-precision history, Err[n] = ||R_n||_F in `low_dtype`
        err[k+1 .. k+refi_steps] the enhanced-precision Err evaluated BEFORE each refinement update
        err[k+refi_steps+1]      (final_check only) the enhanced-precision Err of the returned Z;
                                 Alg. 3 as printed ends after the update (final_check = False).
    iters = k + refi_steps; flags are those of the low-precision run."""
    if refi_steps < 1:
        raise ValueError("refi_steps must be >= 1")
    low = refine(S, Z0, max_iter, STOP_PAPER, dtype=low_dtype)
    Sr = np.asarray(S, dtype=refi_dtype)
    Z = np.asarray(low.Z, dtype=refi_dtype)
    err = list(low.err)
    for _ in range(refi_steps):
        R = residual(Sr, Z)
        err.append(err_fro(R))
        Z = update_delta_form(Z, R) if update_dtype is None else update_mixed(Z, R, update_dtype)
    if final_check:
        err.append(err_fro(residual(Sr, Z)))
    return RefineResult(Z, low.iters + refi_steps, np.asarray(err), low.flags)


def congruence(H: np.ndarray, Z: np.ndarray) -> np.ndarray:
    """H_perp = Z^T H Z   (Eq. 11, lines 88-92): the congruence transformation that turns
    H C = S C eps into the standard problem H_perp C_perp = C_perp eps when Z^T S Z = I."""
    return Z.T @ (H @ Z)


def final_residual_per_sqrt_n(S: np.ndarray, Z: np.ndarray) -> float:
    """||Z^T S Z - I||_F / sqrt(N), the figure north_star asks to report per mode."""
    return err_fro(residual(np.asarray(S, np.float64), np.asarray(Z, np.float64))) / math.sqrt(S.shape[0])
