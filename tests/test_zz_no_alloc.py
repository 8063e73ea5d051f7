"""`zfac_residual_norm_noalloc` (include/zfac.h): the entry point that allocates nothing -- its scratch is a file-scope
device array of libzfac.so -- against the library's regular path and the oracle.

Collected last on purpose (file name): the suite runs with `pytest -x`, a failure here must not hide another test.
The GPU test passes alone in a fresh process and after the rest of the suite: it depends on nothing but its own inputs,
and the shared scratch array needs no particular contents at entry (the test shows that by interleaving sizes).
"""
import numpy as np
import pytest
import torch

from oracle import zfac_oracle as O
from paper_2404_19163_b200 import workloads as W

DEV = "cuda:0"
REL, ABS = 1e-10, 1e-12         # the F64 history tolerance of tests/test_parity_gpu.py (rel; ERR_ABS_MIN)


def zb():
    from paper_2404_19163_b200 import binding
    return binding


def _noalloc_err(b, S, Z, n, out):
    b.zfac_residual_norm_noalloc(S.data_ptr(), S.stride(0), Z.data_ptr(), Z.stride(0), n, out.data_ptr(),
                                 torch.cuda.current_stream(S.device).cuda_stream)


def _case(n, seed, pad):
    """(S, Z) on the device inside wider buffers (ld = n + pad; the margin is NaN: it must never be read)."""
    w = W.random_spd_general(n, seed=seed, kappa=50.0, pert=0.05, fp32_stored=False)
    S = torch.full((n, n + pad), float("nan"), dtype=torch.float64, device=DEV)
    Z = torch.full((n, n + pad), float("nan"), dtype=torch.float64, device=DEV)
    S[:, :n] = torch.from_numpy(w.S).to(DEV)
    Z[:, :n] = torch.from_numpy(w.Z0).to(DEV)
    return w, S, Z


@pytest.mark.gpu
def test_noalloc_residual_norm_matches_the_regular_path_on_calls_in_a_row():
    b = zb()
    out = torch.zeros(4, dtype=torch.float64, device=DEV)
    # sizes in this order on purpose: ragged (not a multiple of the 64-tile), the maximum, then small again -- the third and
    # fourth calls find the scratch full of the larger problems' T and partial sums
    cases = [(300, 11, 5), (b.ZFAC_NOALLOC_MAX_N, 12, 0), (130, 13, 3), (300, 11, 5), (1, 14, 2)]
    seen = {}
    for k, (n, seed, pad) in enumerate(cases):
        w, S, Z = _case(n, seed, pad)
        # the existing path: Alg. 2 with no update in FP64 mode returns Err[0] = ||I - Z0^T S Z0||_F (steps a1, a2, a3)
        with b.Zfac(n, "f64", DEV) as zf:
            _, it, err, fl = zf.refine(S[:, :n], Z[:, :n], max_iter=0, stop=b.ZFAC_STOP_FIXED)
        assert it == 0 and len(err) == 1
        torch.cuda.synchronize()
        free0, _ = torch.cuda.mem_get_info()
        slot = out[k % 4: k % 4 + 1]
        slot.fill_(-1.0)
        _noalloc_err(b, S, Z, n, slot)
        _noalloc_err(b, S, Z, n, out[(k + 1) % 4: (k + 1) % 4 + 1])          # two calls in a row, same stream
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        got, again = float(out[k % 4]), float(out[(k + 1) % 4])
        ora = O.err_fro(O.residual(w.S, w.Z0))
        print(f"[noalloc n={n}] Err = {got:.15e}  regular path {err[0]:.15e}  oracle {ora:.15e}")
        assert got == pytest.approx(err[0], rel=REL, abs=ABS)
        assert got == pytest.approx(ora, rel=REL, abs=ABS)
        assert again == got                                                      # deterministic, bit for bit
        if k > 0:                                                                # (the first launch may load the module)
            assert free1 == free0, "device memory was allocated or freed by the call"
        seen.setdefault((n, seed), []).append(got)
    assert seen[(300, 11)][0] == seen[(300, 11)][1]                              # stale scratch contents do not matter
    assert b.zfac_noalloc_last_error() == ""


@pytest.mark.gpu
def test_noalloc_in_place_of_the_history_of_a_refinement():
    """Err of every iterate of a short FP64 run, evaluated afterwards by the no-alloc entry point, is the run's history."""
    b = zb()
    n = 200
    w, S, Z = _case(n, 21, 0)
    out = torch.zeros(1, dtype=torch.float64, device=DEV)
    for k in (1, 2):
        with b.Zfac(n, "f64", DEV) as zf:
            Zk, it, err, fl = zf.refine(S, Z, max_iter=k, stop=b.ZFAC_STOP_FIXED)
            Zk = Zk.clone()
        _noalloc_err(b, S, Zk, n, out)
        torch.cuda.synchronize()
        assert float(out[0]) == pytest.approx(err[k], rel=1e-6, abs=1e-12 * np.sqrt(n))   # Err ~ 1e-4 .. 1e-12 here


def test_noalloc_rejects_sizes_beyond_the_maximum_with_a_clear_error():
    """Argument checks come before any CUDA call: they run without a GPU."""
    b = zb()
    with pytest.raises(b.ZfacError) as ei:
        b.zfac_residual_norm_noalloc(256, b.ZFAC_NOALLOC_MAX_N + 1, 256, b.ZFAC_NOALLOC_MAX_N + 1, b.ZFAC_NOALLOC_MAX_N + 1, 256)
    assert ei.value.status == b.ZFAC_E_INVALID
    assert "ZFAC_NOALLOC_MAX_N = 1024" in str(ei.value) and "exceeds" in str(ei.value)
    for args in ((0, 8, 256, 8, 8, 256), (256, 8, 256, 8, 0, 256), (256, 7, 256, 8, 8, 256), (256, 8, 256, 8, 8, 0)):
        with pytest.raises(b.ZfacError) as ei:
            b.zfac_residual_norm_noalloc(*args)
        assert ei.value.status == b.ZFAC_E_INVALID and b.zfac_noalloc_last_error() != ""
    # the header's constant and the binding's agree
    import os
    hdr = open(os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "include", "zfac.h")).read()
    assert f"#define ZFAC_NOALLOC_MAX_N {b.ZFAC_NOALLOC_MAX_N}" in hdr
