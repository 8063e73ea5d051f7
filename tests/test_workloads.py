"""The seeded generators produce valid instances of the problem the paper states:
S symmetric positive definite, ||Z0^T S Z0 - I||_2 < 1 (Eq. 14)."""
import numpy as np
import pytest

from paper_2404_19163_b200 import workloads as W


def _r0_norm2(w):
    X = w.Z0.T @ w.S @ w.Z0
    return float(np.linalg.norm(np.eye(w.n) - X, 2))


def _check(w, fp32):
    assert w.S.shape == (w.n, w.n) and w.Z0.shape == (w.n, w.n)
    assert w.S.dtype == np.float64 and w.Z0.dtype == np.float64
    assert np.array_equal(w.S, w.S.T)
    assert np.linalg.eigvalsh(w.S)[0] > 0
    assert _r0_norm2(w) < 1.0
    if fp32:
        assert np.array_equal(w.S, w.S.astype(np.float32).astype(np.float64))
        assert np.array_equal(w.Z0, w.Z0.astype(np.float32).astype(np.float64))


def test_config1():
    w = W.config1()
    _check(w, False)
    lam = np.linalg.eigvalsh(w.S)
    assert lam[0] == pytest.approx(0.1, rel=1e-9) and lam[-1] == pytest.approx(10.0, rel=1e-9)
    assert np.allclose(w.Q.T @ w.Q, np.eye(w.n), atol=1e-12)
    w2 = W.config1()
    assert np.array_equal(w.S, w2.S)          # seeded: bit-reproducible


def test_config2_small():
    w = W.config2(n=512)
    _check(w, True)
    assert np.all(np.diag(w.S) == 1.0) or w.meta["shift"] > 0
    assert np.linalg.eigvalsh(w.S)[0] >= 0.2 - 1e-6


def test_config3_small_and_config5():
    _check(W.config3(n=300), True)
    _check(W.config5(256), False)


def test_config4_small_is_a_warm_start():
    w = W.config4(n=256)
    _check(w, True)
    X = w.Z0.T @ w.S @ w.Z0
    r0f = np.linalg.norm(np.eye(w.n) - X)
    assert r0f < 5 * w.meta["R0_fro_nominal"] + 0.05
    assert not np.allclose(X, np.eye(w.n), atol=1e-6)


def test_paper_eq39_workload():
    w = W.paper_workload(256, alpha=0.005)
    _check(w, True)
    assert not np.allclose(w.Z0, w.Z0.T)
    lam = np.linalg.eigvalsh(w.S)
    assert lam[0] == pytest.approx(0.5, abs=1e-5)          # gamma = 0.5


def test_nonsymmetric_variants():
    w = W.nonsymmetric_start(W.spectral_workload(96, 1e-2, 1.0, seed=4), 0.01)
    _check(w, False)
    assert not np.allclose(w.Z0, w.Z0.T)
    g = W.random_spd_general(65, 3, kappa=100.0, pert=0.1, fp32_stored=True)
    _check(g, True)
    assert not np.allclose(g.Z0, g.Z0.T)
