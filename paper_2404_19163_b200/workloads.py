"""Seeded synthetic inputs (S, Z0) for the Z-refinement hot path.

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU
oracle.  It holds none of the method's arithmetic (no residual, no polynomial
update, no stopping test): it only builds symmetric positive definite overlap
matrices S and initial guesses Z0 with the shapes, spectra and structure of the
paper's workloads, as listed in BASELINE.json `configs` and SURVEY.md §8(d).

Citations:
  * problem statement  Z^T S Z = I, Z Z^T = S^-1          -- Eq. 10, line 85
  * convergence needs  ||Z0^T S Z0 - I||_2 < 1             -- Eq. 14
  * synthetic overlap  S~_ij = exp(-|i-j|/2) sin(i+1)      -- Eq. 39
  * initial guess      Z0 = S^-1/2 + alpha U, U~U(-.5,.5)  -- Eq. 40
  * ill-conditioned Ag561 matrix, eigenvalues 1e-5..1e1    -- Sec. V.D

Random draws always come from numpy's PCG64 (`default_rng(seed)`) on the CPU so
that they are reproducible across machines; the O(N^3) linear algebra of the
construction (QR, products) runs in FP64 with numpy on the CPU or, when a CUDA
`device` is passed, with torch on that device (same formulae).  Whatever is
produced, the SAME bytes are handed to the oracle and to the library.

"FP32 stored" (configs 2-4): the problem *is* the FP32-rounded matrix.  The
`Workload` then carries S and Z0 already rounded to FP32 and promoted back to
FP64 exactly (SURVEY.md §8(c) reading Q17), so oracle and library see the same
numbers in every precision mode.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

try:  # torch is only used for device-side construction of large inputs
    import torch
except Exception:  # pragma: no cover
    torch = None


@dataclasses.dataclass
class Workload:
    """One (S, Z0) problem instance. Arrays are FP64 numpy, C-contiguous."""

    name: str
    n: int
    S: np.ndarray                      # N x N symmetric positive definite
    Z0: np.ndarray                     # N x N initial guess
    lam: Optional[np.ndarray] = None   # spectrum used to build S (if spectral)
    Q: Optional[np.ndarray] = None     # eigenvectors used to build S (if spectral)
    alpha: Optional[float] = None      # Z0 = alpha * I when the start is a scaled identity
    fp32_stored: bool = False
    meta: dict = dataclasses.field(default_factory=dict)


# --------------------------------------------------------------------------
# small helpers (input construction only)
# --------------------------------------------------------------------------

def _use_torch(device) -> bool:
    return device is not None and torch is not None and str(device) != "cpu"


def geometric_grid(n: int, lam_min: float, lam_max: float) -> np.ndarray:
    """lam_i = lam_min * (lam_max/lam_min)^(i/(n-1)) -- "log-uniform" read as a
    deterministic geometric grid."""
    if n == 1:
        return np.array([lam_max], dtype=np.float64)
    i = np.arange(n, dtype=np.float64)
    return lam_min * (lam_max / lam_min) ** (i / (n - 1))


def haar_orthogonal(n: int, seed: int, device=None) -> np.ndarray:
    """Haar-distributed orthogonal matrix: QR of an N x N Gaussian with the
    sign of diag(R) folded into Q."""
    rng = np.random.default_rng(seed)
    G = rng.standard_normal((n, n))
    if _use_torch(device):
        g = torch.from_numpy(G).to(device)
        q, r = torch.linalg.qr(g)
        q = q * torch.sign(torch.diagonal(r)).unsqueeze(0)
        return np.ascontiguousarray(q.cpu().numpy())
    q, r = np.linalg.qr(G)
    q = q * np.sign(np.diag(r))[None, :]
    return np.ascontiguousarray(q)


def _matmul(a: np.ndarray, b: np.ndarray, device=None) -> np.ndarray:
    if _use_torch(device):
        return (torch.from_numpy(a).to(device) @ torch.from_numpy(b).to(device)).cpu().numpy()
    return a @ b


def spectral_matrix(Q: np.ndarray, d: np.ndarray, device=None) -> np.ndarray:
    """Q diag(d) Q^T, symmetrised."""
    M = _matmul(Q * d[None, :], np.ascontiguousarray(Q.T), device)
    return np.ascontiguousarray(0.5 * (M + M.T))


def lambda_max_power(S: np.ndarray, steps: int = 100, safety: float = 1.01) -> float:
    """Largest eigenvalue estimate by power iteration (start 1/sqrt(N), `steps`
    steps), inflated by `safety` so the estimate is an upper bound in practice
    (BASELINE.json config 1: "Z0 = I/sqrt(lambda_max(S)) from power iteration")."""
    n = S.shape[0]
    v = np.full(n, 1.0 / math.sqrt(n))
    lam = 0.0
    for _ in range(steps):
        w = S @ v
        lam = float(v @ w)
        nw = float(np.linalg.norm(w))
        if nw == 0.0:
            break
        v = w / nw
    return lam * safety


def spectral_norm_sym_power(apply, n: int, steps: int = 200, seed: int = 12345) -> float:
    """|lambda|_max of a symmetric operator given as a mat-vec closure."""
    rng = np.random.default_rng(seed)
    v = rng.standard_normal(n)
    v /= np.linalg.norm(v)
    lam = 0.0
    for _ in range(steps):
        w = apply(v)
        lam = float(np.linalg.norm(w))
        if lam == 0.0:
            break
        v = w / lam
    return lam


def round_fp32(a: np.ndarray) -> np.ndarray:
    """Round to FP32 and promote back to FP64 exactly ("FP32 stored")."""
    return np.ascontiguousarray(a.astype(np.float32).astype(np.float64))


def uniform_perturbation(n: int, seed: int) -> np.ndarray:
    """U_ij ~ U(-0.5, 0.5)  (Eq. 40)."""
    rng = np.random.default_rng(seed)
    return rng.random((n, n)) - 0.5


# --------------------------------------------------------------------------
# spectral family (configs 1, 3, 5 and the base of config 4)
# --------------------------------------------------------------------------

def spectral_workload(n: int, lam_min: float, lam_max: float, seed: int = 0, *,
                      fp32_stored: bool = False, device=None, name: str = "") -> Workload:
    """S = Q diag(lam) Q^T with Haar Q (seed) and a geometric-grid spectrum;
    Z0 = I / sqrt(lambda_hat), lambda_hat from power iteration on the S that is
    actually handed out (i.e. after FP32 rounding when fp32_stored)."""
    Q = haar_orthogonal(n, seed, device)
    lam = geometric_grid(n, lam_min, lam_max)
    S = spectral_matrix(Q, lam, device)
    if fp32_stored:
        S = round_fp32(S)
    lam_hat = lambda_max_power(S)
    alpha = 1.0 / math.sqrt(lam_hat)
    if fp32_stored:
        alpha = float(np.float32(alpha))
    Z0 = np.ascontiguousarray(alpha * np.eye(n))
    return Workload(name or f"spectral_n{n}_k{lam_max / lam_min:.0e}", n, S, Z0, lam=lam, Q=Q,
                    alpha=alpha, fp32_stored=fp32_stored,
                    meta={"lam_min": lam_min, "lam_max": lam_max, "seed": seed,
                          "lambda_hat": lam_hat})


def config1(device=None) -> Workload:
    """BASELINE.json configs[0]: N=256, FP64, kappa=100, Z0 = I/sqrt(lambda_max)."""
    return spectral_workload(256, 0.1, 10.0, seed=0, device=device, name="config1_n256_k1e2")


def config3(n: int = 4617, device=None) -> Workload:
    """BASELINE.json configs[2]: N=4617, lam in [1e-5, 1] (kappa=1e5), FP32 S,
    Z0 = I/sqrt(lambda_max).  Stands in for the Ag561 matrix."""
    return spectral_workload(n, 1e-5, 1.0, seed=0, fp32_stored=True, device=device,
                             name=f"config3_n{n}_k1e5")


def config5(n: int, device=None, fp32_stored: bool = False) -> Workload:
    """BASELINE.json configs[4]: sweep point, lam in [1e-3, 1], Z0 = I/sqrt(lambda_max),
    fixed 10 refinement iterations."""
    return spectral_workload(n, 1e-3, 1.0, seed=0, fp32_stored=fp32_stored, device=device,
                             name=f"config5_n{n}_k1e3")


# --------------------------------------------------------------------------
# config 2: banded-decay overlap
# --------------------------------------------------------------------------

def config2(n: int = 2048, seed: int = 0, lam_floor: float = 0.2) -> Workload:
    """BASELINE.json configs[1]: S_ij = exp(-0.5|i-j|)(1 + 0.05 u_ij), u ~ U(-1,1)
    symmetrised, S_ii = 1, shifted (only if needed) so lambda_min >= 0.2; FP32
    stored; Z0 = diag(S)^-1/2 * s with s = 1/sqrt(lambda_hat_max) (diag(S) is
    constant, so Z0 is a scaled identity)."""
    rng = np.random.default_rng(seed)
    u = rng.uniform(-1.0, 1.0, size=(n, n))
    u = 0.5 * (u + u.T)
    idx = np.arange(n)
    S = np.exp(-0.5 * np.abs(idx[:, None] - idx[None, :])) * (1.0 + 0.05 * u)
    np.fill_diagonal(S, 1.0)
    lam_min = float(np.linalg.eigvalsh(S)[0])
    shift = max(0.0, lam_floor - lam_min)
    if shift > 0.0:
        S = S + shift * np.eye(n)
    S = round_fp32(0.5 * (S + S.T))
    d = np.diag(S).copy()
    Dm = 1.0 / np.sqrt(d)
    lam_hat = lambda_max_power(S * Dm[:, None] * Dm[None, :])
    s = float(np.float32(1.0 / math.sqrt(lam_hat)))
    Z0 = round_fp32(np.diag(Dm * s))
    return Workload(f"config2_n{n}_banded", n, S, Z0, alpha=None, fp32_stored=True,
                    meta={"lam_min_before_shift": lam_min, "shift": shift, "seed": seed,
                          "lambda_hat": lam_hat})


# --------------------------------------------------------------------------
# config 4: warm start (MD / geometry-optimisation step)
# --------------------------------------------------------------------------

def config4(n: int = 8192, eps: float = 1e-3, seed_q: int = 0, seed_e: int = 1, *,
            fp32_stored: bool = True, device=None) -> Workload:
    """BASELINE.json configs[3], read as SURVEY.md §8(d) Q-D4 (the literal additive
    S0 + 1e-3 E violates Eq. 14): S0 = Q diag(lam) Q^T, lam in [1e-5, 1];
    E = symmetric Gaussian with unit-2-norm rows (re-symmetrised);
    S1 = S0^1/2 (I + eps E) S0^1/2  (SPD by construction, kappa unchanged);
    Z0 = S0^-1/2 = Q lam^-1/2 Q^T in FP64.  Then R0 = I - Z0^T S1 Z0 = -eps E
    up to rounding: a genuine "previous MD step" start."""
    Q = haar_orthogonal(n, seed_q, device)
    lam = geometric_grid(n, 1e-5, 1.0)
    rng = np.random.default_rng(seed_e)
    G = rng.standard_normal((n, n))
    E = (G + G.T) / math.sqrt(2.0)
    E /= np.linalg.norm(E, axis=1, keepdims=True)
    E = 0.5 * (E + E.T)
    Sh = spectral_matrix(Q, np.sqrt(lam), device)           # S0^{1/2}
    M = np.eye(n) + eps * E
    S1 = _matmul(_matmul(Sh, M, device), Sh, device)
    S1 = np.ascontiguousarray(0.5 * (S1 + S1.T))
    Z0 = spectral_matrix(Q, 1.0 / np.sqrt(lam), device)     # S0^{-1/2}
    if fp32_stored:
        S1 = round_fp32(S1)
        Z0 = round_fp32(Z0)
    return Workload(f"config4_n{n}_warm", n, S1, Z0, lam=lam, Q=Q, fp32_stored=fp32_stored,
                    meta={"eps": eps, "seed_q": seed_q, "seed_e": seed_e,
                          "R0_fro_nominal": eps * math.sqrt(n)})


# --------------------------------------------------------------------------
# the paper's own synthetic workload (Eq. 39 / Eq. 40)
# --------------------------------------------------------------------------

def paper_eq39(n: int, gamma: float = 0.5, device=None) -> tuple[np.ndarray, np.ndarray, np.ndarray]:
    """S~_ij = exp(-|i-j|/2) sin(i+1), 1<=i,j<=N (Eq. 39), read
    as symmetrised (S~ + S~^T)/2 because the printed form is not symmetric although
    the text calls it symmetric; S = S~ + (gamma - eps_1) I,
    gamma = 0.5.  Returns (S, eigenvalues, eigenvectors) -- the
    eigendecomposition is the paper's own route to S^-1/2 for Z0.
    With `device` (and N >= 4096) the two eigendecompositions of the CONSTRUCTION run in FP64 through
    torch.linalg on that device (minutes on the host at N = 16384); none of the method's arithmetic is here."""
    i = np.arange(1, n + 1, dtype=np.float64)
    St = np.exp(-np.abs(i[:, None] - i[None, :]) / 2.0) * np.sin(i + 1.0)[:, None]
    St = 0.5 * (St + St.T)
    if _use_torch(device) and n >= 4096:
        import torch
        eps1 = float(torch.linalg.eigvalsh(torch.from_numpy(St).to(device))[0].item())
        S = St + (gamma - eps1) * np.eye(n)
        S = np.ascontiguousarray(0.5 * (S + S.T))
        wt, Vt = torch.linalg.eigh(torch.from_numpy(S).to(device))
        w, V = wt.cpu().numpy(), np.ascontiguousarray(Vt.cpu().numpy())
        del wt, Vt
        return S, w, V
    eps1 = float(np.linalg.eigvalsh(St)[0])
    S = St + (gamma - eps1) * np.eye(n)
    S = np.ascontiguousarray(0.5 * (S + S.T))
    w, V = np.linalg.eigh(S)
    return S, w, V


def paper_workload(n: int, alpha: float = 0.005, seed: int = 0, *, fp32_stored: bool = True, device=None) -> Workload:
    """Eq. 39 overlap with Z0 = S^-1/2 + alpha U (Eq. 40): NON-symmetric start."""
    S, w, V = paper_eq39(n, device=device)
    Sinvh = spectral_matrix(V, 1.0 / np.sqrt(w), device)
    Z0 = Sinvh + alpha * uniform_perturbation(n, seed)
    if fp32_stored:
        S = round_fp32(S)
        Z0 = round_fp32(Z0)
    return Workload(f"paper_eq39_n{n}_a{alpha}", n, S, np.ascontiguousarray(Z0), lam=w, Q=V,
                    fp32_stored=fp32_stored, meta={"alpha_pert": alpha, "seed": seed})


def nonsymmetric_start(w: Workload, alpha: float, seed: int = 7) -> Workload:
    """Replace the start of a spectral workload by Z0 = S^-1/2 + alpha U (Eq. 40),
    with S^-1/2 = Q lam^-1/2 Q^T known from construction.  Needed because every
    Z0 ∝ I start keeps Z symmetric, which hides Z <-> Z^T mistakes."""
    assert w.Q is not None and w.lam is not None
    Sinvh = (w.Q / np.sqrt(w.lam)[None, :]) @ w.Q.T
    Z0 = Sinvh + alpha * uniform_perturbation(w.n, seed)
    if w.fp32_stored:
        Z0 = round_fp32(Z0)
    return dataclasses.replace(w, name=w.name + f"_nonsym{alpha}", Z0=np.ascontiguousarray(Z0),
                               alpha=None, meta={**w.meta, "alpha_pert": alpha, "seed_u": seed})


def random_spd_general(n: int, seed: int, kappa: float = 20.0, pert: float = 0.05,
                       fp32_stored: bool = False) -> Workload:
    """Small general-purpose parity case: spectral S with condition number kappa
    and a non-symmetric, non-commuting start Z0 = S^-1/2 (I + pert * G/sqrt(N)),
    G Gaussian.  ||R0||_2 ~ 2*pert."""
    Q = haar_orthogonal(n, seed)
    lam = geometric_grid(n, 1.0 / kappa, 1.0)
    S = spectral_matrix(Q, lam)
    rng = np.random.default_rng(seed + 1000)
    G = rng.standard_normal((n, n)) / math.sqrt(max(n, 1))
    Sinvh = (Q / np.sqrt(lam)[None, :]) @ Q.T
    Z0 = Sinvh @ (np.eye(n) + pert * G)
    if fp32_stored:
        S = round_fp32(S)
        Z0 = round_fp32(Z0)
    return Workload(f"general_n{n}_k{kappa:g}_s{seed}", n, S, np.ascontiguousarray(Z0), lam=lam, Q=Q,
                    fp32_stored=fp32_stored, meta={"pert": pert, "seed": seed})
