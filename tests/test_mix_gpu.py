"""GPU parity of the FP64-master modes (include/zfac.h: ZFAC_MODE_F64_MIXED, ZFAC_MODE_F64_I8) against the oracle.

Both modes compute the residual to the FP64 level (F64_MIXED on the FP64 tensor pipe, F64_I8 from error-free int8 slices
on the INT8 tensor cores) and evaluate the update's correction in FP32-class arithmetic, added to the FP64 master.  The
oracle of that iteration is `O.refine(..., update_dtype=float32)` / `O.update_mixed` (pinned in
tests/test_oracle_refi_pins.py); against the all-FP64 oracle the result differs by the rounding of the correction,
~2^-22 ||R_0|| (a rotation of Z: any Z U is an inverse factor), so Z is held to 1e-6 there and what is unique -- the
invariant ||Z^T S Z - I||_F / sqrt(N) and Z Z^T = S^-1 -- to the FP64 level."""
import dataclasses
import math

import numpy as np
import pytest
import torch

from oracle import zfac_oracle as O
from paper_2404_19163_b200 import workloads as W

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
MIX = ["f64mix", "f64i8"]


def zb():
    from paper_2404_19163_b200 import binding
    return binding


def _rel(a, b):
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def _dev(a, dt=torch.float64):
    return torch.from_numpy(np.ascontiguousarray(a)).to(DEV, dt)


def run(w, mode, max_iter, stop, keep=(), options=None):
    b = zb()
    S, Z0 = _dev(w.S), _dev(w.Z0)
    with b.Zfac(w.n, mode, DEV) as zf:
        for k, v in (options or {}).items():
            zf.set_option(k, v)
        Z, it, err, fl = zf.refine(S, Z0, max_iter=max_iter, stop=stop)
        pk = {k: zf.peek(k).cpu().numpy() for k in keep}
        launches = zf.last_launch_count
    return Z.cpu().numpy(), it, err, fl, pk, launches


@pytest.mark.parametrize("mode", MIX)
@pytest.mark.parametrize("n", [96, 300, 700])
def test_residual_and_one_update_against_oracle(mode, n):
    """a1, a2, a3 to the FP64 level; one update against the oracle's mixed update."""
    b = zb()
    w = W.random_spd_general(n, seed=5 + n, kappa=200.0, pert=0.1, fp32_stored=False)
    Z, it, err, fl, pk, _ = run(w, mode, 0, b.ZFAC_STOP_FIXED, keep=[b.ZFAC_BUF_T, b.ZFAC_BUF_R, b.ZFAC_BUF_Z])
    A = w.S @ w.Z0
    R0 = O.residual(w.S, w.Z0)
    assert it == 0 and fl == b.ZFAC_R_MAXITER and len(err) == 1
    assert _rel(pk[b.ZFAC_BUF_T], A.T) < 1e-13                            # a1: T = (S Z)^T
    # a2: R = I - Z^T S Z; X ~ I is formed to ~1e-15 absolute, F64_I8 then stores R rounded to FP32 (6e-8 relative)
    tol_r = 1e-13 * math.sqrt(n) + (1e-7 * np.linalg.norm(R0) if mode == "f64i8" else 0.0)
    assert np.linalg.norm(pk[b.ZFAC_BUF_R] - R0) < tol_r
    assert err[0] == pytest.approx(O.err_fro(R0), rel=1e-7 if mode == "f64i8" else 1e-10)
    assert np.array_equal(Z, w.Z0) and np.array_equal(pk[b.ZFAC_BUF_Z], w.Z0)
    Z, it, err, fl, _, _ = run(w, mode, 1, b.ZFAC_STOP_FIXED)
    Zm = O.update_mixed(w.Z0, R0, np.float32)
    Zx = O.update_delta_form(w.Z0, R0)
    q = np.linalg.norm(0.5 * R0 + 0.375 * R0 @ R0, 2)
    print(f"[{mode} n={n}] one update: rel vs mixed oracle {_rel(Z, Zm):.2e}, vs FP64 oracle {_rel(Z, Zx):.2e} (||Q||_2 = {q:.2e})")
    assert it == 1 and len(err) == 2
    assert _rel(Z, Zx) < 4.0 * 2.0 ** -22 * q                             # the correction is FP32-class, the master FP64
    assert _rel(Z, Zm) < 4.0 * 2.0 ** -22 * q
    assert err[1] == pytest.approx(O.err_fro(O.residual(w.S, Z)), rel=1e-6, abs=1e-13 * math.sqrt(n))
    assert not np.allclose(Z, Z.T)


@pytest.mark.parametrize("mode", MIX)
@pytest.mark.parametrize("n", [1, 2, 17, 127, 128, 129, 255, 256, 257, 383, 700, 1100])
def test_full_run_reaches_the_fp64_level(mode, n):
    b = zb()
    w = W.random_spd_general(n, seed=300 + n, kappa=50.0, pert=0.1, fp32_stored=False)
    Z, it, err, fl, _, launches = run(w, mode, 40, b.ZFAC_STOP_PAPER)
    nat = O.refine(w.S, w.Z0, 40, O.STOP_PAPER)
    assert len(err) == it + 1
    if not (fl & b.ZFAC_R_STOPPED):
        assert fl == b.ZFAC_R_MAXITER and it == 40 and err[-1] <= 1e-300
        return
    ref = O.refine(w.S, w.Z0, it, O.STOP_FIXED)
    mix = O.refine(w.S, w.Z0, it, O.STOP_FIXED, update_dtype=np.float32)
    inv = O.final_residual_per_sqrt_n(w.S, Z)
    print(f"[{mode} n={n}] iters={it} (FP64 oracle stops at {nat.iters}) rel vs FP64 oracle {_rel(Z, ref.Z):.2e}, vs mixed oracle "
          f"{_rel(Z, mix.Z):.2e}; ||Z^T S Z - I||_F/sqrtN = {inv:.2e}; Err={np.array2string(err, precision=2)}")
    assert nat.iters <= it <= nat.iters + 2
    assert inv < 1e-12 * max(1.0, math.sqrt(n))
    assert _rel(Z, ref.Z) < 1e-6 and _rel(Z, mix.Z) < 1e-6
    assert _rel(Z @ Z.T, ref.Z @ ref.Z.T) < 1e-11
    for k in range(it + 1):
        if ref.err[k] > 1e-4:
            assert err[k] == pytest.approx(ref.err[k], rel=1e-4)
    assert err[it] == pytest.approx(O.err_fro(O.residual(w.S, Z)), rel=1e-2, abs=1e-13 * math.sqrt(n) + 1e-15)


@pytest.mark.parametrize("mode", MIX)
def test_ill_conditioned_kappa_1e5_and_unaligned_ld(mode):
    """kappa = 1e5 (the Ag561 stand-in of configs 3 / 4): the FP64-level residual is what makes the run converge where
    SPLIT16 stalls at ~1e-2; ld > n on every buffer."""
    b = zb()
    n = 770
    w = W.nonsymmetric_start(W.config3(n=n), alpha=2e-4)
    S64 = np.asarray(w.S, np.float64); Z64 = np.asarray(w.Z0, np.float64)
    Sb = torch.full((n, n + 3), float("nan"), dtype=torch.float64, device=DEV); Sb[:, :n] = _dev(S64)
    Zb0 = torch.full((n, n + 1), float("nan"), dtype=torch.float64, device=DEV); Zb0[:, :n] = _dev(Z64)
    out = torch.full((n, n + 5), -3.0, dtype=torch.float64, device=DEV)
    with b.Zfac(n, mode, DEV) as zf:
        Z, it, err, fl = zf.refine(Sb[:, :n], Zb0[:, :n], max_iter=40, stop=b.ZFAC_STOP_PAPER, out=out[:, :n])
    Z = Z.cpu().numpy()
    assert bool((out[:, n:] == -3.0).all())
    ref = O.refine(S64, Z64, it, O.STOP_FIXED)
    inv = O.final_residual_per_sqrt_n(S64, Z)
    print(f"[{mode} kappa=1e5 n={n}] iters={it} rel vs FP64 oracle {_rel(Z, ref.Z):.2e}; invariant {inv:.2e}; Err={np.array2string(err, precision=2)}")
    assert fl & b.ZFAC_R_STOPPED
    assert inv < 1e-10
    assert _rel(Z, ref.Z) < 1e-6


@pytest.mark.parametrize("high", MIX)
@pytest.mark.parametrize("low", ["split16", "hh16"])
def test_refi_into_the_fp64_master_modes(low, high):
    """Alg. 3 with the new refinement stage: low precision to its stop, then refinement steps whose residual is FP64-level.
    With max_iter = 0 the stage starts from FP64[Z0] and must match the oracle's mixed refinement steps."""
    b = zb()
    n = 520
    w = W.random_spd_general(n, seed=91, kappa=300.0, pert=0.1, fp32_stored=True)
    S, Z0 = _dev(w.S, torch.float32), _dev(w.Z0, torch.float32)
    with b.Zfac(n, low, DEV) as zl, b.Zfac(n, high, DEV) as zh:
        Z, it, err, fl = zl.refine_refi(zh, S, Z0, max_iter=0, refi_steps=2, final_check=True)
        assert Z.dtype == torch.float64 and it == 2 and (fl & b.ZFAC_R_REFINED) and len(err) == 4
        ora = O.refine(w.S, w.Z0, 2, O.STOP_FIXED, update_dtype=np.float32)
        assert _rel(Z.cpu().numpy(), ora.Z) < 1e-6
        assert err[1] == pytest.approx(ora.err[0], rel=1e-9)            # FP64[Z0]: the same residual
        assert np.allclose(err[1:], ora.err, rtol=2e-2, atol=1e-12)     # later ones carry the (different) FP32 roundings of the correction
        Z, it, err, fl = zl.refine_refi(zh, S, Z0, max_iter=30, refi_steps=2, final_check=True)
    Z = Z.cpu().numpy()
    k = it - 2
    inv = O.final_residual_per_sqrt_n(w.S, Z)
    print(f"[{low} -> {high}] low iters={k} Err={np.array2string(err, precision=2)} invariant={inv:.2e}")
    assert (fl & b.ZFAC_R_REFINED) and len(err) == it + 2 and inv < 1e-11
    assert err[-1] == pytest.approx(inv * math.sqrt(n), rel=1e-2, abs=1e-12)
    full = O.refine_with_refi(w.S, w.Z0, 30, low_dtype=np.float32, refi_steps=2, update_dtype=np.float32)
    assert _rel(Z @ Z.T, full.Z @ full.Z.T) < 1e-9


def test_i8_slice_count_sets_the_accuracy_and_nonfinite_input_is_reported():
    """ZFAC_OPT_I8_SLICES: s slices keep 7 s bits relative to the row maxima, so the floor of the residual scales like
    2^(-7 s); 8 slices are FP64-equivalent.  A NaN in the input cannot be sliced: it must still surface as
    ZFAC_R_NONFINITE (the other modes get that from the arithmetic itself)."""
    b = zb()
    n = 300
    w = W.random_spd_general(n, seed=17, kappa=100.0, pert=0.1, fp32_stored=False)
    floors = {}
    for s_ in (4, 6, 8):
        Z, it, err, fl, _, _ = run(w, "f64i8", 40, b.ZFAC_STOP_PAPER, options={"i8_slices": s_})
        floors[s_] = O.final_residual_per_sqrt_n(w.S, Z)
        assert fl & b.ZFAC_R_STOPPED
    print("[f64i8] invariant by slice count:", {k: f"{v:.2e}" for k, v in floors.items()})
    assert floors[8] < 1e-12 and floors[6] < 3e-9 and floors[4] < 3e-5
    assert floors[4] > 1e3 * floors[8]
    for mode in MIX:
        wb = W.Workload("nan", n, w.S, w.Z0.copy(), fp32_stored=False)
        wb.Z0[3, 4] = float("nan")
        Z, it, err, fl, _, _ = run(wb, mode, 10, b.ZFAC_STOP_PAPER)
        assert it == 0 and (fl & b.ZFAC_R_NONFINITE) and math.isnan(err[0]), mode
        ws = W.Workload("nanS", n, w.S.copy(), w.Z0, fp32_stored=False)
        ws.S[7, 7] = float("inf")
        Z, it, err, fl, _, _ = run(ws, mode, 10, b.ZFAC_STOP_PAPER)
        assert it == 0 and (fl & b.ZFAC_R_NONFINITE), mode


@pytest.mark.parametrize("mode", MIX)
def test_while_graph_and_determinism(mode):
    b = zb()
    n = 300
    w = W.random_spd_general(n, seed=23, kappa=40.0, pert=0.1, fp32_stored=False)
    S, Z0 = _dev(w.S), _dev(w.Z0)
    with b.Zfac(n, mode, DEV) as zf:
        Zd, itd, errd, fld = zf.refine(S, Z0, max_iter=25, stop=b.ZFAC_STOP_PAPER)
        Zd = Zd.clone()
        Z2, it2, err2, fl2 = zf.refine(S, Z0, max_iter=25, stop=b.ZFAC_STOP_PAPER)
        assert torch.equal(Zd, Z2) and np.array_equal(errd, err2)               # run-to-run determinism
        with b.ZfacLoopGraph(zf, S, Z0, max_iter=25, stop=b.ZFAC_STOP_PAPER) as lg:
            Zg, itg, errg, flg = lg.launch()
            assert itg == itd and flg == fld and np.array_equal(errg, errd) and torch.equal(Zg, Zd)
        with pytest.raises(b.ZfacError):
            zf.set_order(3)
        with pytest.raises(b.ZfacError):
            zf.congruence(S, Z0)


@pytest.mark.parametrize("mode", MIX)
def test_host_entry_point_and_float_inputs_match_the_device_entry_point_bitwise(mode):
    """zfac_refine_host in the FP64-master modes: the results of the first TWO updates are downloaded early, each behind
    its update (the master is updated in place: update n + 1 waits for the download of Z_n); whichever of them is the
    last update performed is the result, else the download at the end.  Runs that stop after 1, 2 and >= 3 updates,
    pinned and pageable, double and float (ZFAC_OPT_INPUT_F32) inputs, ld > n."""
    b = zb()
    n = 300
    w = W.random_spd_general(n, seed=55, kappa=30.0, pert=0.1, fp32_stored=True)
    lam, V = np.linalg.eigh(w.S)
    Zex = (V / np.sqrt(lam)) @ V.T
    G = np.random.default_rng(3).standard_normal((n, n)) / math.sqrt(n)
    starts = {"exact (1 update)": Zex, "close (2 updates)": W.round_fp32(Zex @ (np.eye(n) + 1e-3 * G)), "far (>= 3 updates)": w.Z0}
    seen = set()
    with b.Zfac(n, mode, DEV) as zf:
        for f32 in (0, 1):
            zf.set_option("input_f32", f32)
            idt = torch.float32 if f32 else torch.float64
            for name, Z0 in starts.items():
                Sd, Zd = _dev(w.S, idt), _dev(Z0, idt)
                Zref, itref, errref, flref = zf.refine(Sd, Zd, max_iter=30, stop=b.ZFAC_STOP_PAPER)
                Zref = Zref.cpu()
                seen.add(min(itref, 3))
                for pin in (True, False):
                    hS = torch.full((n, n + 2), float("nan"), dtype=idt); hS[:, :n] = torch.from_numpy(w.S).to(idt)
                    hZ0 = torch.from_numpy(np.ascontiguousarray(Z0)).to(idt)
                    hZ = torch.full((n, n + 3), -2.0, dtype=torch.float64)
                    if pin:
                        hS, hZ0, hZ = hS.pin_memory(), hZ0.pin_memory(), hZ.pin_memory()
                    _, it, err, fl = zf.refine_host(hS[:, :n], hZ0, hZ[:, :n], max_iter=30, stop=b.ZFAC_STOP_PAPER)
                    assert it == itref and fl == flref and np.array_equal(err, errref), (name, f32, pin)
                    assert torch.equal(hZ[:, :n], Zref), (name, f32, pin)
                    assert bool((hZ[:, n:] == -2.0).all())
        # float inputs promoted exactly: the same FP32-stored problem given as double gives the same bits
        zf.set_option("input_f32", 0)
        Za = zf.refine(_dev(w.S), _dev(w.Z0), max_iter=30, stop=b.ZFAC_STOP_PAPER)[0].clone()
        zf.set_option("input_f32", 1)
        Zb_ = zf.refine(_dev(w.S, torch.float32), _dev(w.Z0, torch.float32), max_iter=30, stop=b.ZFAC_STOP_PAPER)[0]
        assert torch.equal(Za, Zb_)
    assert seen == {1, 2, 3}
    with b.Zfac(n, "split16", DEV) as zs:
        with pytest.raises(b.ZfacError):
            zs.set_option("input_f32", 1)


# ------------------------------------------------------------------ full sizes, in the configuration bench.py times
def test_time_to_gate_path_config4_n8192_f64i8_float_inputs():
    """BASELINE configs[3] as `bench.py`'s `time_to_gate` runs it: N = 8192 warm start (kappa = 1e5), FP32-stored S and Z0 given
    as floats (ZFAC_OPT_INPUT_F32), mode F64_I8, paper stop rule.  Both gates of that figure against the oracle: Z within the
    split gate 1e-5 of the all-FP64 oracle run for the same number of updates (measured 7e-9: the FP32-class correction rotates
    Z by ~u sqrt(kappa) ||R_0||) and the invariant at the FP64 level; plus F64_MIXED on the same inputs (same update, DMMA
    residual): the two must agree with each other far below either gate."""
    b = zb()
    w = W.config4(n=8192, device=DEV)
    S32, Z32 = _dev(w.S, torch.float32), _dev(w.Z0, torch.float32)
    res = {}
    for mode in MIX:
        with b.Zfac(w.n, mode, DEV) as zf:
            zf.set_option("input_f32", 1)
            Z, it, err, fl = zf.refine(S32, Z32, max_iter=20, stop=b.ZFAC_STOP_PAPER)
            res[mode] = (Z.cpu().numpy(), it, err, fl)
    it = res["f64i8"][1]
    assert res["f64mix"][1] == it and 2 <= it <= 3
    ref = O.refine(w.S, w.Z0, it, O.STOP_FIXED)
    for mode in MIX:
        Z, _, err, fl = res[mode]
        rel = _rel(Z, ref.Z)
        inv = O.final_residual_per_sqrt_n(w.S, Z)
        print(f"[config4 N=8192 {mode}] iters={it} rel vs FP64 oracle={rel:.3e} ||Z^T S Z - I||_F/sqrtN={inv:.3e} "
              f"Err={np.array2string(err, precision=3)} oracle Err={np.array2string(ref.err, precision=3)}")
        assert fl & b.ZFAC_R_STOPPED
        assert rel <= 1e-5 and rel <= 1e-6                    # the split gate of bench.py, and the mode's own 1e-6
        assert inv <= 1e-10
        assert err[0] == pytest.approx(ref.err[0], rel=1e-6)
        # at the FP64 floor the reported Err carries the residual engine's own rounding (8 int8 slices / DMMA): within 2x
        assert 0.5 * inv * math.sqrt(w.n) <= err[it] <= 2.0 * inv * math.sqrt(w.n) + 1e-10
    assert _rel(res["f64i8"][0], res["f64mix"][0]) <= 1e-9


def test_config3_full_size_n4617_f64i8_padding_and_cold_start():
    """BASELINE configs[2]: N = 4617 (no tile multiple: identity padding of the FP64 master, of the int8 slices and of the
    operand pairs), kappa = 1e5, COLD start Z0 = I / sqrt(lambda_max): ~13 iterations whose early residuals are O(60) in the
    Frobenius norm (rscale < 1 in r_split) down to the FP64 floor.  Against the all-FP64 oracle for the same number of updates."""
    b = zb()
    w = W.config3()
    assert w.n == 4617
    # The paper's test alone fires when the FP32-class correction has brought Err to ~u32 sqrt(kappa) Err[n-1] (measured:
    # stop at n = 12 with 1.4e-9 per sqrt(N)); ZFAC_OPT_EXTRA_UPDATE answers that first firing with one more update -- the
    # refinement step of Alg. 3 built in -- which reaches the FP64 floor.
    Z0_, it0, err0, fl0, _, _ = run(w, "f64i8", 40, b.ZFAC_STOP_PAPER)
    inv0 = O.final_residual_per_sqrt_n(w.S, Z0_)
    print(f"[config3 N=4617 f64i8, paper test alone] iters={it0} invariant={inv0:.3e}")
    assert (fl0 & b.ZFAC_R_STOPPED) and not (fl0 & b.ZFAC_R_REFINED) and inv0 <= 1e-8
    Z, it, err, fl, _, _ = run(w, "f64i8", 40, b.ZFAC_STOP_PAPER, options={"extra_update": 1})
    assert it == it0 + 1 and (fl & b.ZFAC_R_REFINED) and np.array_equal(err[: it0 + 1], err0)
    nat = O.refine(w.S, w.Z0, 40, O.STOP_PAPER)
    ref = nat if it == nat.iters else O.refine(w.S, w.Z0, it, O.STOP_FIXED)
    rel = _rel(Z, ref.Z)
    inv = O.final_residual_per_sqrt_n(w.S, Z)
    print(f"[config3 N=4617 f64i8] iters={it} (FP64 oracle stops at {nat.iters}) rel={rel:.3e} invariant={inv:.3e} "
          f"trace={np.array2string(err, precision=3)}")
    # at the floor the stop index can differ by one between two correct implementations: the oracle's
    # Err[12] = 9.7e-11 passes its test against Err[11]^3 = 1.1e-9 by a factor 10 only
    assert fl & b.ZFAC_R_STOPPED and nat.iters - 1 <= it <= nat.iters + 2
    # Z itself is fixed up to an orthogonal factor only: 13 FP32-class corrections from a cold start leave a
    # rotation ~u32 sqrt(kappa) (measured rel 8.4e-5); the unique quantity Z Z^T = S^-1 is held to the FP64 level.
    zzt = _rel(Z @ Z.T, ref.Z @ ref.Z.T)
    print(f"[config3 N=4617 f64i8] rel of Z Z^T vs the oracle's: {zzt:.3e}")
    assert inv <= 1e-10 and zzt <= 1e-9 and rel <= 1e-3
    # the history tracks the FP64 one; during the slow phase (Err 63 -> 6, the small eigenvalues grow by 15/8 per update) the
    # 2^-22 rounding of each correction is carried along and amplified: measured 1.8e-4 at n = 9; the cubic phase then
    # triples the relative difference per update (1 % at n = 11, Err = 1.0e-3)
    for k in range(min(it, nat.iters) + 1):
        if nat.err[k] > 1e-3:
            assert err[k] == pytest.approx(nat.err[k], rel=1e-3 if nat.err[k] > 1.0 else 5e-2), k


@pytest.mark.parametrize("mode", MIX)
def test_extra_update_option_is_one_more_update_after_the_first_firing(mode):
    """ZFAC_OPT_EXTRA_UPDATE (include/zfac.h): with the paper's test, the run with the option is the run without it plus
    exactly ONE update and one residual -- same history up to the firing, flag ZFAC_R_REFINED, `iters` one larger -- and that
    update is the FP64-master update of the oracle (`update_mixed`) applied to the Z the plain run returned.  The option is
    refused outside the FP64-master modes; with ZFAC_STOP_FIXED it changes nothing; max_iter still bounds the run."""
    b = zb()
    w = W.spectral_workload(300, 1e-5, 1.0, seed=0)          # cold start, kappa = 1e5: the oracle's mixed run stops at 12 of 13
    Z0_, it0, err0, fl0, _, _ = run(w, mode, 40, b.ZFAC_STOP_PAPER)
    Z1_, it1, err1, fl1, _, _ = run(w, mode, 40, b.ZFAC_STOP_PAPER, options={"extra_update": 1})
    assert (fl0 & b.ZFAC_R_STOPPED) and not (fl0 & b.ZFAC_R_REFINED)
    assert it1 == it0 + 1 and (fl1 & b.ZFAC_R_STOPPED) and (fl1 & b.ZFAC_R_REFINED)
    assert np.array_equal(err1[: it0 + 1], err0) and len(err1) == it0 + 2
    Zm = O.update_mixed(Z0_, O.residual(w.S, Z0_), np.float32)
    assert _rel(Z1_, Zm) < 1e-12                                                       # the correction is ~1e-9 by now
    inv0, inv1 = O.final_residual_per_sqrt_n(w.S, Z0_), O.final_residual_per_sqrt_n(w.S, Z1_)
    print(f"[{mode} extra_update] iters {it0} -> {it1}, invariant {inv0:.2e} -> {inv1:.2e}")
    assert inv0 > 3e-11 and inv1 < 3e-12                     # the plain run stopped short of the FP64 floor; this one is there
    assert err1[-1] == pytest.approx(inv1 * math.sqrt(w.n), rel=0.5, abs=2e-13 * math.sqrt(w.n))
    # fixed count: the option is inert; max_iter = the plain stop index: the extra update does not fit and MAXITER is reported
    Zf0, itf0, errf0, flf0, _, _ = run(w, mode, 5, b.ZFAC_STOP_FIXED)
    Zf1, itf1, errf1, flf1, _, _ = run(w, mode, 5, b.ZFAC_STOP_FIXED, options={"extra_update": 1})
    assert itf0 == itf1 == 5 and flf0 == flf1 and np.array_equal(Zf0, Zf1) and np.array_equal(errf0, errf1)
    Zc, itc, errc, flc, _, _ = run(w, mode, it0, b.ZFAC_STOP_PAPER, options={"extra_update": 1})
    assert itc == it0 and (flc & b.ZFAC_R_MAXITER) and np.array_equal(Zc, Z0_)
    with b.Zfac(256, "split16", DEV) as zf:
        with pytest.raises(Exception):
            zf.set_option("extra_update", 1)
        assert zf.get_option("extra_update") == 0


@pytest.mark.parametrize("mode", MIX)
def test_final_check_option_skips_only_evaluations_whose_outcome_is_known(mode):
    """ZFAC_OPT_FINAL_CHECK = 0 (include/zfac.h).  (i) Warm start: the run ends by the test in both settings, with the same
    number of updates and the same Z bit for bit; the history is the same up to the last evaluated entry, Err[iters] is NaN,
    the flag ZFAC_R_NOCHECK is set (the skipped residual's kernels are still enqueued, they return at once).  The update that was not
    checked is the oracle's: Z against the oracle run for `iters` updates.  (ii) Cold start at kappa = 1e5: the last
    evaluated Err before the firing is 3e-4, its cube is far above 2^-53 sqrt(N): nothing is foregone, the run is the
    default run.  (iii) With ZFAC_OPT_EXTRA_UPDATE the evaluation after the extra update is the one skipped.  (iv) The WHILE
    graph and the host entry point follow.  (v) Refused outside the FP64-master modes."""
    b = zb()
    n = 300
    w = W.random_spd_general(n, seed=91, kappa=100.0, pert=0.02, fp32_stored=False)
    lam, V = np.linalg.eigh(w.S)
    G = np.random.default_rng(3).standard_normal((n, n)) / math.sqrt(n)
    w = dataclasses.replace(w, Z0=np.ascontiguousarray(((V / np.sqrt(lam)) @ V.T) @ (np.eye(n) + 1e-3 * G)))     # Err: 2e-2, 7e-8, floor
    Zd, itd, errd, fld, _, ld = run(w, mode, 30, b.ZFAC_STOP_PAPER)
    Zn, itn, errn, fln, _, ln = run(w, mode, 30, b.ZFAC_STOP_PAPER, options={"final_check": 0})
    print(f"[{mode} final_check=0] iters {itd} / {itn}, launches {ld} / {ln}, Err {errd} / {errn}")
    assert fld == b.ZFAC_R_STOPPED and fln == (b.ZFAC_R_STOPPED | b.ZFAC_R_NOCHECK)
    assert itn == itd and np.array_equal(Zn, Zd)
    assert len(errn) == itd + 1 and np.array_equal(errn[:itd], errd[:itd]) and np.isnan(errn[itd])
    assert errd[itd - 1] ** 3 < 2.0 ** -53 * math.sqrt(n)                 # why the last evaluation was foregone
    ref = O.refine(w.S, w.Z0, itn, O.STOP_FIXED)
    assert _rel(Zn, ref.Z) < 1e-8 and O.final_residual_per_sqrt_n(w.S, Zn) < 1e-12
    # (ii) cold start: nothing foregone
    wc = W.spectral_workload(300, 1e-5, 1.0, seed=0)
    Zc, itc, errc, flc, _, _ = run(wc, mode, 40, b.ZFAC_STOP_PAPER)
    Zc0, itc0, errc0, flc0, _, _ = run(wc, mode, 40, b.ZFAC_STOP_PAPER, options={"final_check": 0})
    assert itc0 == itc and flc0 == flc and np.array_equal(Zc0, Zc) and np.array_equal(errc0, errc)
    # (iii) with the extra update
    Ze, ite, erre, fle, _, _ = run(wc, mode, 40, b.ZFAC_STOP_PAPER, options={"extra_update": 1})
    Zx, itx, errx, flx, _, _ = run(wc, mode, 40, b.ZFAC_STOP_PAPER, options={"extra_update": 1, "final_check": 0})
    assert itx == ite == itc + 1 and np.array_equal(Zx, Ze)
    assert flx == (fle | b.ZFAC_R_NOCHECK) and (fle & b.ZFAC_R_REFINED)
    assert np.array_equal(errx[:ite], erre[:ite]) and np.isnan(errx[ite])
    # max_iter still bounds the run: the foregone update is not performed beyond it
    Zm, itm, errm, flm, _, _ = run(w, mode, itd - 1, b.ZFAC_STOP_PAPER, options={"final_check": 0})
    assert itm == itd - 1 and (flm & b.ZFAC_R_MAXITER) and not (flm & b.ZFAC_R_NOCHECK) and np.array_equal(errm, errd[:itd])
    # (iv) graph and host entry
    S, Z0 = _dev(w.S), _dev(w.Z0)
    with b.Zfac(n, mode, DEV) as zf:
        zf.set_option("final_check", 0)
        with b.ZfacLoopGraph(zf, S, Z0, max_iter=30, stop=b.ZFAC_STOP_PAPER) as lg:
            Zg, itg, errg, flg = lg.launch()
            assert itg == itn and flg == fln and np.array_equal(Zg.cpu().numpy(), Zn) and np.isnan(errg[itg])
        hS = torch.from_numpy(w.S).pin_memory(); hZ0 = torch.from_numpy(np.ascontiguousarray(w.Z0)).pin_memory()
        hZ = torch.empty((n, n), dtype=torch.float64).pin_memory()
        _, ith, errh, flh = zf.refine_host(hS, hZ0, hZ, max_iter=30, stop=b.ZFAC_STOP_PAPER)
        assert ith == itn and flh == fln and np.array_equal(hZ.numpy(), Zn)
        # a later call with the option back on is the default run again (State::last does not leak)
        zf.set_option("final_check", 1)
        Z1, it1, err1, fl1 = zf.refine(S, Z0, max_iter=30, stop=b.ZFAC_STOP_PAPER)
        assert it1 == itd and fl1 == fld and np.array_equal(err1, errd) and np.array_equal(Z1.cpu().numpy(), Zd)
    # (v)
    with b.Zfac(256, "f64", DEV) as zf:
        with pytest.raises(b.ZfacError):
            zf.set_option("final_check", 0)
        zf.set_option("final_check", 1)


def test_i8_cluster_option_is_scheduling_only():
    """ZFAC_OPT_I8_CLUSTER (include/zfac.h): a1 of F64_I8 on clusters of two CTA pairs that share the B slices by TMA
    multicast.  Same arithmetic per tile, exact FP64 sums: T, the history and Z are bit-identical to the default, for an
    even number of 256-row tiles (the cluster path), for an odd one (falls back to the pair kernel) and under
    ZFAC_OPT_MAX_PAIRS; refused outside F64_I8."""
    b = zb()
    for n, seed in ((1024, 5), (1500, 6), (700, 7)):          # padded to 1024 (4 tile rows), 1536 (6), 768 (3: fallback)
        w = W.random_spd_general(n, seed=seed, kappa=100.0, pert=0.05, fp32_stored=False)
        S, Z0 = _dev(w.S), _dev(w.Z0)
        with b.Zfac(n, "f64i8", DEV) as zf:
            ref = None
            for opts in ({"i8_cluster": 0}, {"i8_cluster": 1}, {"i8_cluster": 1, "max_pairs": 5}):
                for k, v in opts.items():
                    zf.set_option(k, v)
                Z, it, err, fl = zf.refine(S, Z0, max_iter=25, stop=b.ZFAC_STOP_PAPER)
                T = zf.peek(b.ZFAC_BUF_T)
                if ref is None:
                    ref = (Z.clone(), it, err.copy(), fl, T.clone())
                    assert O.final_residual_per_sqrt_n(w.S, Z.cpu().numpy()) < 1e-12
                else:
                    assert it == ref[1] and fl == ref[3], (n, opts)
                    assert torch.equal(Z, ref[0]) and torch.equal(T, ref[4]), (n, opts)
                    assert np.array_equal(err, ref[2]), (n, opts)        # a2's partial sums are stored per TILE: any grid gives the same Err
    with b.Zfac(256, "f64mix", DEV) as zf:
        with pytest.raises(b.ZfacError):
            zf.set_option("i8_cluster", 1)


@pytest.mark.parametrize("f32", [0, 1])
def test_f64i8_host_entry_point_with_the_banded_upload_is_bitwise_the_device_entry_point(f32):
    """zfac_refine_host in ZFAC_MODE_F64_I8 with pinned inputs and >= 4 tile rows: Z0 goes up first, S follows in row chunks,
    each chunk sliced and multiplied (the tile columns of T = W S^T that need its rows) as it arrives.  Same tiles, same
    arithmetic: Z, iters, Err[] and flags are the device entry point's bit for bit; with the option off as well."""
    b = zb()
    n = 1100                                                                  # padded to 1280: 5 tile rows, 5 upload chunks
    w = W.random_spd_general(n, seed=61, kappa=200.0, pert=0.05, fp32_stored=True)
    idt = torch.float32 if f32 else torch.float64
    with b.Zfac(n, "f64i8", DEV) as zf:
        zf.set_option("input_f32", f32)
        Sd, Zd = _dev(w.S, idt), _dev(w.Z0, idt)
        Zref, itref, errref, flref = zf.refine(Sd, Zd, max_iter=30, stop=b.ZFAC_STOP_PAPER)
        Zref = Zref.cpu()
        assert O.final_residual_per_sqrt_n(w.S, Zref.numpy()) < 1e-12
        hS = torch.full((n, n + 4), float("nan"), dtype=idt); hS[:, :n] = torch.from_numpy(w.S).to(idt)
        hS = hS.pin_memory()
        hZ0 = torch.from_numpy(np.ascontiguousarray(w.Z0)).to(idt).pin_memory()
        for overlap in (1, 0):
            zf.set_option("host_upload_overlap", overlap)
            hZ = torch.full((n, n), -2.0, dtype=torch.float64).pin_memory()
            _, it, err, fl = zf.refine_host(hS[:, :n], hZ0, hZ, max_iter=30, stop=b.ZFAC_STOP_PAPER)
            assert it == itref and fl == flref and np.array_equal(err, errref), overlap
            assert torch.equal(hZ, Zref), overlap


@pytest.mark.parametrize("n", [200, 900, 1400])
def test_i8_narrow_tiles_give_the_same_integers(n):
    """ZFAC_OPT_I8_NARROW: the INT8 kernels on 256 x 128 tiles (default up to padded order 1536).  Every element of T and R is
    the same exact integer sum whatever the tile: T, R and Z are bit-identical to the 256 x 256 tiles; Err[] agrees to the
    last bits (its partial sums are grouped by tile).  Also through the host entry point and with ZFAC_OPT_MAX_PAIRS."""
    b = zb()
    w = W.random_spd_general(n, seed=90 + n, kappa=100.0, pert=0.05, fp32_stored=False)
    S, Z0 = _dev(w.S), _dev(w.Z0)
    res = {}
    with b.Zfac(n, "f64i8", DEV) as zf:
        assert zf.get_option("i8_narrow") == -1
        for nar, pairs in ((0, 0), (1, 0), (-1, 0), (1, 3)):
            zf.set_option("i8_narrow", nar); zf.set_option("max_pairs", pairs)
            Z, it, err, fl = zf.refine(S, Z0, max_iter=25, stop=b.ZFAC_STOP_PAPER)
            res[(nar, pairs)] = (Z.clone(), it, err.copy(), fl, zf.peek(b.ZFAC_BUF_T).clone(), zf.peek(b.ZFAC_BUF_R).clone())
        zf.set_option("max_pairs", 0); zf.set_option("i8_narrow", 1)
        hS = torch.from_numpy(w.S).pin_memory(); hZ0 = torch.from_numpy(np.ascontiguousarray(w.Z0)).pin_memory()
        hZ = torch.empty((n, n), dtype=torch.float64).pin_memory()
        _, hit, herr, hfl = zf.refine_host(hS, hZ0, hZ, max_iter=25, stop=b.ZFAC_STOP_PAPER)
    ref = res[(0, 0)]
    assert O.final_residual_per_sqrt_n(w.S, ref[0].cpu().numpy()) < 1e-12
    for key in ((1, 0), (-1, 0), (1, 3)):
        r = res[key]
        assert r[1] == ref[1] and r[3] == ref[3], key
        assert torch.equal(r[0], ref[0]) and torch.equal(r[4], ref[4]) and torch.equal(r[5], ref[5]), key
        assert np.allclose(r[2], ref[2], rtol=1e-13, atol=0.0), key
    assert np.array_equal(res[(1, 0)][2], res[(-1, 0)][2]) and np.array_equal(res[(1, 0)][2], res[(1, 3)][2])   # same tiles: same Err bits
    assert hit == ref[1] and hfl == ref[3] and np.array_equal(herr, res[(1, 0)][2]) and torch.equal(hZ, ref[0].cpu())
