"""ctypes binding of libzfac.so -- the same names as include/zfac.h, argument marshalling only.

Every step of the path runs in the CUDA kernels of the library; nothing here computes.
PyTorch is used only for device memory (the workspace and the I/O tensors) and streams.
If the shared library is missing or cannot be loaded this module raises: there is no CPU
or PyTorch fallback path.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libzfac.so")

ZFAC_MODE_SPLIT16, ZFAC_MODE_TF32, ZFAC_MODE_F64, ZFAC_MODE_HH16, ZFAC_MODE_F64_MIXED, ZFAC_MODE_F64_I8 = 0, 1, 2, 3, 4, 5
ZFAC_STOP_PAPER, ZFAC_STOP_FIXED = 0, 1
ZFAC_OK, ZFAC_E_INVALID, ZFAC_E_UNSUPPORTED, ZFAC_E_WORKSPACE, ZFAC_E_CUDA = 0, 1, 2, 3, 4
ZFAC_R_STOPPED, ZFAC_R_MAXITER, ZFAC_R_NONFINITE, ZFAC_R_REFINED, ZFAC_R_RANGE, ZFAC_R_NOCHECK = 1, 2, 4, 8, 16, 32
ZFAC_BUF_T, ZFAC_BUF_R, ZFAC_BUF_Q, ZFAC_BUF_Z = 0, 1, 2, 3

(ZFAC_OPT_CHUNK_KB, ZFAC_OPT_CHUNK0_KB, ZFAC_OPT_HH_SQUARE, ZFAC_OPT_HH_SQUARE_ERR, ZFAC_OPT_PROMOTE_UPDATE, ZFAC_OPT_BAND,
 ZFAC_OPT_MAX_PAIRS, ZFAC_OPT_HOST_OVERLAP, ZFAC_OPT_HOST_UPLOAD_OVERLAP, ZFAC_OPT_HOST_A5_BANDS, ZFAC_OPT_I8_SLICES,
 ZFAC_OPT_INPUT_F32, ZFAC_OPT_EXTRA_UPDATE, ZFAC_OPT_FINAL_CHECK, ZFAC_OPT_I8_CLUSTER, ZFAC_OPT_NARROW_TILES, ZFAC_OPT_PDL, ZFAC_OPT_I8_NARROW) = range(18)
OPTIONS = {"chunk_kb": ZFAC_OPT_CHUNK_KB, "chunk0_kb": ZFAC_OPT_CHUNK0_KB, "hh_square": ZFAC_OPT_HH_SQUARE,
           "hh_square_err": ZFAC_OPT_HH_SQUARE_ERR, "promote_update": ZFAC_OPT_PROMOTE_UPDATE, "band": ZFAC_OPT_BAND,
           "max_pairs": ZFAC_OPT_MAX_PAIRS, "host_overlap": ZFAC_OPT_HOST_OVERLAP,
           "host_upload_overlap": ZFAC_OPT_HOST_UPLOAD_OVERLAP, "host_a5_bands": ZFAC_OPT_HOST_A5_BANDS,
           "i8_slices": ZFAC_OPT_I8_SLICES, "input_f32": ZFAC_OPT_INPUT_F32, "extra_update": ZFAC_OPT_EXTRA_UPDATE, "final_check": ZFAC_OPT_FINAL_CHECK, "i8_cluster": ZFAC_OPT_I8_CLUSTER, "narrow_tiles": ZFAC_OPT_NARROW_TILES, "pdl": ZFAC_OPT_PDL, "i8_narrow": ZFAC_OPT_I8_NARROW}

MODES = {"split16": ZFAC_MODE_SPLIT16, "tf32": ZFAC_MODE_TF32, "f64": ZFAC_MODE_F64, "hh16": ZFAC_MODE_HH16,
         "f64mix": ZFAC_MODE_F64_MIXED, "f64i8": ZFAC_MODE_F64_I8}
F64_ELT_MODES = (ZFAC_MODE_F64, ZFAC_MODE_F64_MIXED, ZFAC_MODE_F64_I8)

# symbols include/zfac.h declares (tests check that the library exports every one)
EXPORTS = [
    "zfac_workspace_bytes", "zfac_create", "zfac_refine", "zfac_refine_host", "zfac_refine_refi",
    "zfac_congruence", "zfac_peek",
    "zfac_last_launch_count", "zfac_padded_n", "zfac_destroy", "zfac_status_string",
    "zfac_last_cuda_error", "zfac_set_profile", "zfac_get_profile", "zfac_set_order", "zfac_get_order",
    "zfac_graph_create", "zfac_graph_launch", "zfac_graph_destroy",
    "zfac_set_option", "zfac_get_option", "zfac_refine_refi_host",
    "zfac_workspace_bytes_batched", "zfac_create_batched", "zfac_get_batch", "zfac_refine_batched",
    "zfac_residual_norm_noalloc", "zfac_noalloc_last_error",
]

_lib: Optional[ctypes.CDLL] = None


class ZfacError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = f"{where}: {zfac_status_string(status)}"
        if status == ZFAC_E_CUDA:
            msg += f" [{lib().zfac_last_cuda_error().decode()}]"
        super().__init__(msg)


def lib() -> ctypes.CDLL:
    """Load libzfac.so (built by paper_2404_19163_b200.build / __graft_entry__.build)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_2404_19163_b200.build` "
                           "(the CUDA extension is required; there is no fallback path)")
    L = ctypes.CDLL(LIB_PATH)
    vp, i64, sz, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_size_t, ctypes.c_int
    L.zfac_workspace_bytes.restype = sz
    L.zfac_workspace_bytes.argtypes = [i64, ci]
    L.zfac_padded_n.restype = i64
    L.zfac_padded_n.argtypes = [i64, ci]
    L.zfac_residual_norm_noalloc.restype = ci
    L.zfac_residual_norm_noalloc.argtypes = [vp, i64, vp, i64, i64, vp, vp]
    L.zfac_noalloc_last_error.restype = ctypes.c_char_p
    L.zfac_noalloc_last_error.argtypes = []
    L.zfac_create.restype = ci
    L.zfac_create.argtypes = [ctypes.POINTER(vp), i64, ci, vp, sz]
    L.zfac_refine.restype = ci
    L.zfac_refine.argtypes = [vp, vp, i64, vp, i64, vp, i64, ci, ci, vp, vp, vp, vp]
    L.zfac_refine_host.restype = ci
    L.zfac_refine_host.argtypes = [vp, vp, i64, vp, i64, vp, i64, ci, ci, vp, vp, vp, vp]
    L.zfac_refine_refi.restype = ci
    L.zfac_refine_refi.argtypes = [vp, vp, vp, i64, vp, i64, vp, i64, ci, ci, ci, vp, vp, vp, vp]
    L.zfac_refine_refi_host.restype = ci
    L.zfac_refine_refi_host.argtypes = [vp, vp, vp, i64, vp, i64, vp, i64, ci, ci, ci, vp, vp, vp, vp]
    L.zfac_set_option.restype = ci
    L.zfac_set_option.argtypes = [vp, ci, ctypes.c_double]
    L.zfac_get_option.restype = ci
    L.zfac_get_option.argtypes = [vp, ci, ctypes.POINTER(ctypes.c_double)]
    L.zfac_workspace_bytes_batched.restype = sz
    L.zfac_workspace_bytes_batched.argtypes = [i64, ci, ci]
    L.zfac_create_batched.restype = ci
    L.zfac_create_batched.argtypes = [ctypes.POINTER(vp), i64, ci, ci, vp, sz]
    L.zfac_get_batch.restype = ci
    L.zfac_get_batch.argtypes = [vp]
    L.zfac_refine_batched.restype = ci
    L.zfac_refine_batched.argtypes = [vp, vp, i64, i64, vp, i64, i64, vp, i64, i64, ci, ci, vp, vp, vp, vp]
    L.zfac_congruence.restype = ci
    L.zfac_congruence.argtypes = [vp, vp, i64, vp, i64, vp, i64, vp]
    L.zfac_peek.restype = ci
    L.zfac_peek.argtypes = [vp, ci, vp, i64, vp]
    L.zfac_last_launch_count.restype = ci
    L.zfac_last_launch_count.argtypes = [vp]
    L.zfac_destroy.restype = ci
    L.zfac_destroy.argtypes = [vp]
    L.zfac_status_string.restype = ctypes.c_char_p
    L.zfac_status_string.argtypes = [ci]
    L.zfac_last_cuda_error.restype = ctypes.c_char_p
    L.zfac_last_cuda_error.argtypes = []
    L.zfac_set_profile.restype = ci
    L.zfac_set_profile.argtypes = [vp, ci]
    L.zfac_get_profile.restype = ci
    L.zfac_get_profile.argtypes = [vp, vp, vp, ci]
    L.zfac_graph_create.restype = ci
    L.zfac_graph_create.argtypes = [vp, vp, i64, vp, i64, vp, i64, ci, ci, vp, vp, vp, ctypes.POINTER(vp)]
    L.zfac_graph_launch.restype = ci
    L.zfac_graph_launch.argtypes = [vp, vp]
    L.zfac_graph_destroy.restype = ci
    L.zfac_graph_destroy.argtypes = [vp]
    L.zfac_set_order.restype = ci
    L.zfac_set_order.argtypes = [vp, ci]
    L.zfac_get_order.restype = ci
    L.zfac_get_order.argtypes = [vp]
    _lib = L
    return L


# ---------------------------------------------------------------- 1:1 wrappers
def zfac_status_string(status: int) -> str:
    return lib().zfac_status_string(int(status)).decode()


def zfac_workspace_bytes(n: int, mode: int) -> int:
    return int(lib().zfac_workspace_bytes(int(n), int(mode)))


def zfac_padded_n(n: int, mode: int) -> int:
    return int(lib().zfac_padded_n(int(n), int(mode)))


ZFAC_NOALLOC_MAX_N = 1024


def zfac_noalloc_last_error() -> str:
    return lib().zfac_noalloc_last_error().decode()


def zfac_residual_norm_noalloc(d_S: int, lds: int, d_Z: int, ldz: int, n: int, d_err: int, stream: int = 0) -> None:
    """Err = ||I - Z^T S Z||_F (FP64) into *d_err; allocates nothing (scratch is a static device array of the library;
    n <= ZFAC_NOALLOC_MAX_N; overlapping calls race).  Raises ZfacError with the library's reason on failure."""
    st = lib().zfac_residual_norm_noalloc(ctypes.c_void_p(d_S), int(lds), ctypes.c_void_p(d_Z), int(ldz), int(n),
                                          ctypes.c_void_p(d_err), ctypes.c_void_p(stream))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_residual_norm_noalloc: " + zfac_noalloc_last_error())


def zfac_create(n: int, mode: int, d_workspace: int, nbytes: int) -> int:
    """Returns the opaque context handle (int). Raises ZfacError on failure."""
    h = ctypes.c_void_p()
    st = lib().zfac_create(ctypes.byref(h), int(n), int(mode), ctypes.c_void_p(d_workspace), int(nbytes))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_create")
    return h.value


def zfac_refine(ctx: int, d_S: int, lds: int, d_Z0: int, ldz0: int, d_Z: int, ldz: int, max_iter: int,
                stop: int, d_iters: int, d_err: int, d_flags: int, stream: int = 0) -> None:
    st = lib().zfac_refine(ctx, d_S, lds, d_Z0, ldz0, d_Z, ldz, int(max_iter), int(stop), d_iters, d_err,
                           d_flags, ctypes.c_void_p(stream))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_refine")


def zfac_refine_host(ctx: int, h_S: int, lds: int, h_Z0: int, ldz0: int, h_Z: int, ldz: int, max_iter: int,
                     stop: int, h_iters: int, h_err: int, h_flags: int, stream: int = 0) -> None:
    st = lib().zfac_refine_host(ctx, h_S, lds, h_Z0, ldz0, h_Z, ldz, int(max_iter), int(stop), h_iters, h_err,
                                h_flags, ctypes.c_void_p(stream))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_refine_host")


def zfac_refine_refi(low: int, f64: int, d_S: int, lds: int, d_Z0: int, ldz0: int, d_Z: int, ldz: int,
                     max_iter: int, refi_steps: int, final_check: int, d_iters: int, d_err: int, d_flags: int,
                     stream: int = 0) -> None:
    st = lib().zfac_refine_refi(low, f64, d_S, lds, d_Z0, ldz0, d_Z, ldz, int(max_iter), int(refi_steps),
                                int(final_check), d_iters, d_err, d_flags, ctypes.c_void_p(stream))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_refine_refi")


def zfac_refine_refi_host(low: int, high: int, h_S: int, lds: int, h_Z0: int, ldz0: int, h_Z: int, ldz: int,
                          max_iter: int, refi_steps: int, final_check: int, h_iters: int, h_err: int, h_flags: int,
                          stream: int = 0) -> None:
    st = lib().zfac_refine_refi_host(low, high, h_S, lds, h_Z0, ldz0, h_Z, ldz, int(max_iter), int(refi_steps),
                                     int(final_check), h_iters, h_err, h_flags, ctypes.c_void_p(stream))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_refine_refi_host")


def zfac_set_option(ctx: int, key: int, value: float) -> None:
    st = lib().zfac_set_option(ctx, int(key), float(value))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_set_option")


def zfac_get_option(ctx: int, key: int) -> float:
    v = ctypes.c_double(0.0)
    st = lib().zfac_get_option(ctx, int(key), ctypes.byref(v))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_get_option")
    return float(v.value)


def zfac_workspace_bytes_batched(n: int, mode: int, batch: int) -> int:
    return int(lib().zfac_workspace_bytes_batched(int(n), int(mode), int(batch)))


def zfac_create_batched(n: int, mode: int, batch: int, d_workspace: int, nbytes: int) -> int:
    h = ctypes.c_void_p()
    st = lib().zfac_create_batched(ctypes.byref(h), int(n), int(mode), int(batch), ctypes.c_void_p(d_workspace), int(nbytes))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_create_batched")
    return h.value


def zfac_get_batch(ctx: int) -> int:
    return int(lib().zfac_get_batch(ctx))


def zfac_refine_batched(ctx: int, d_S: int, lds: int, stride_S: int, d_Z0: int, ldz0: int, stride_Z0: int, d_Z: int,
                        ldz: int, stride_Z: int, max_iter: int, stop: int, d_iters: int, d_err: int, d_flags: int,
                        stream: int = 0) -> None:
    st = lib().zfac_refine_batched(ctx, d_S, lds, stride_S, d_Z0, ldz0, stride_Z0, d_Z, ldz, stride_Z, int(max_iter),
                                   int(stop), d_iters, d_err, d_flags, ctypes.c_void_p(stream))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_refine_batched")


def zfac_congruence(ctx: int, d_H: int, ldh: int, d_Z: int, ldz: int, d_out: int, ldo: int, stream: int = 0) -> None:
    st = lib().zfac_congruence(ctx, d_H, ldh, d_Z, ldz, d_out, ldo, ctypes.c_void_p(stream))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_congruence")


def zfac_peek(ctx: int, which: int, d_out: int, ld: int, stream: int = 0) -> None:
    st = lib().zfac_peek(ctx, int(which), d_out, int(ld), ctypes.c_void_p(stream))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_peek")


def zfac_last_launch_count(ctx: int) -> int:
    return int(lib().zfac_last_launch_count(ctx))


def zfac_graph_create(ctx: int, d_S: int, lds: int, d_Z0: int, ldz0: int, d_Z: int, ldz: int, max_iter: int,
                      stop: int, d_iters: int, d_err: int, d_flags: int) -> int:
    g = ctypes.c_void_p()
    st = lib().zfac_graph_create(ctx, d_S, lds, d_Z0, ldz0, d_Z, ldz, int(max_iter), int(stop), d_iters, d_err, d_flags,
                                 ctypes.byref(g))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_graph_create")
    return g.value


def zfac_graph_launch(graph: int, stream: int = 0) -> None:
    st = lib().zfac_graph_launch(graph, stream)
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_graph_launch")


def zfac_graph_destroy(graph: int) -> None:
    lib().zfac_graph_destroy(graph)


def zfac_set_order(ctx: int, m: int) -> None:
    """Order m of the refinement polynomial (2, 3, 4); see include/zfac.h."""
    st = lib().zfac_set_order(ctx, int(m))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_set_order")


def zfac_get_order(ctx: int) -> int:
    return int(lib().zfac_get_order(ctx))


def zfac_set_profile(ctx: int, enable: bool) -> None:
    st = lib().zfac_set_profile(ctx, int(bool(enable)))
    if st != ZFAC_OK:
        raise ZfacError(st, "zfac_set_profile")


def zfac_get_profile(ctx: int, cap: int = 1024):
    """[(step_id, iteration, ms), ...] for the GEMM kernels of the last call (stream must be synchronised)."""
    tags = (ctypes.c_int * cap)()
    ms = (ctypes.c_float * cap)()
    k = lib().zfac_get_profile(ctx, ctypes.addressof(tags), ctypes.addressof(ms), cap)
    return [(tags[i] & 15, tags[i] >> 4, float(ms[i])) for i in range(k)]


def zfac_destroy(ctx: int) -> None:
    lib().zfac_destroy(ctx)


# ---------------------------------------------------------------- convenience holder (marshalling only)
class Zfac:
    """Owns a torch uint8 workspace tensor and a zfac context for (n, mode) on the current device."""

    def __init__(self, n: int, mode: str | int, device: str | torch.device = "cuda",
                 workspace: Optional[torch.Tensor] = None):
        if not torch.cuda.is_available():
            raise RuntimeError("zfac needs a CUDA device (sm_100a); there is no CPU path")
        self.n = int(n)
        self.mode = MODES[mode] if isinstance(mode, str) else int(mode)
        self.dtype = torch.float64 if self.mode in F64_ELT_MODES else torch.float32
        self.in_dtype = self.dtype                      # element type of S and Z0 (float with ZFAC_OPT_INPUT_F32)
        self.device = torch.device(device)
        nbytes = zfac_workspace_bytes(self.n, self.mode)
        if nbytes == 0:
            raise ZfacError(ZFAC_E_INVALID, "zfac_workspace_bytes")
        if workspace is None:
            workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        elif (workspace.dtype != torch.uint8 or workspace.dim() != 1 or not workspace.is_contiguous()
              or workspace.device != self.device):
            # size and 256-byte alignment are the library's to check (ZFAC_E_WORKSPACE)
            raise ValueError("workspace: expected a contiguous 1-D uint8 tensor on the context's device")
        self.workspace = workspace                      # caller-owned memory (the C ABI's ownership rule)
        with torch.cuda.device(self.device):
            self.ctx = zfac_create(self.n, self.mode, self.workspace.data_ptr(), self.workspace.numel())

    def close(self) -> None:
        if getattr(self, "ctx", None):
            zfac_destroy(self.ctx)
            self.ctx = None
            self.workspace = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, t: torch.Tensor, name: str, dtype=None) -> None:
        dtype = dtype or self.dtype
        if t.dtype != dtype or t.dim() != 2 or t.shape[0] != self.n or t.shape[1] != self.n:
            raise ValueError(f"{name}: expected {self.n}x{self.n} {dtype}, got {tuple(t.shape)} {t.dtype}")
        if t.stride(1) != 1 or t.stride(0) < self.n:
            raise ValueError(f"{name}: must be row-major with unit column stride")

    def refine(self, S: torch.Tensor, Z0: torch.Tensor, max_iter: int = 40, stop: int = ZFAC_STOP_PAPER,
               out: Optional[torch.Tensor] = None, sync: bool = True):
        """Device tensors in, device tensors out: (Z, iters, err[0..iters], flags).
        With sync=False returns the raw device tensors (Z, d_iters, d_err, d_flags)."""
        self._check(S, "S", self.in_dtype); self._check(Z0, "Z0", self.in_dtype)
        Z = out if out is not None else torch.empty((self.n, self.n), dtype=self.dtype, device=S.device)
        self._check(Z, "Z")
        d_iters = torch.zeros(1, dtype=torch.int32, device=S.device)
        d_flags = torch.zeros(1, dtype=torch.int32, device=S.device)
        d_err = torch.full((max_iter + 1,), float("nan"), dtype=torch.float64, device=S.device)
        stream = torch.cuda.current_stream(S.device).cuda_stream
        zfac_refine(self.ctx, S.data_ptr(), S.stride(0), Z0.data_ptr(), Z0.stride(0), Z.data_ptr(), Z.stride(0),
                    max_iter, stop, d_iters.data_ptr(), d_err.data_ptr(), d_flags.data_ptr(), stream)
        if not sync:
            return Z, d_iters, d_err, d_flags
        torch.cuda.current_stream(S.device).synchronize()
        it = int(d_iters.item())
        return Z, it, d_err[: it + 1].cpu().numpy(), int(d_flags.item())

    def refine_host(self, S: torch.Tensor, Z0: torch.Tensor, Z: torch.Tensor, max_iter: int = 40,
                    stop: int = ZFAC_STOP_PAPER):
        """Host (pinned) tensors in and out, through zfac_refine_host."""
        for t, name, dt in ((S, "S", self.in_dtype), (Z0, "Z0", self.in_dtype), (Z, "Z", self.dtype)):
            self._check(t, name, dt)
            if t.is_cuda:
                raise ValueError(f"{name}: refine_host takes host tensors")
        iters = ctypes.c_int(0)
        flags = ctypes.c_int(0)
        err = np.full(max_iter + 1, np.nan, dtype=np.float64)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        with torch.cuda.device(self.device):
            zfac_refine_host(self.ctx, S.data_ptr(), S.stride(0), Z0.data_ptr(), Z0.stride(0), Z.data_ptr(),
                             Z.stride(0), max_iter, stop, ctypes.addressof(iters), err.ctypes.data,
                             ctypes.addressof(flags), stream)
        return Z, iters.value, err[: iters.value + 1], flags.value

    def set_option(self, key: str | int, value: float) -> None:
        """zfac_set_option; key by name (OPTIONS) or number."""
        k = OPTIONS[key] if isinstance(key, str) else int(key)
        zfac_set_option(self.ctx, k, value)
        if k == ZFAC_OPT_INPUT_F32:
            self.in_dtype = torch.float32 if int(value) else self.dtype

    def get_option(self, key: str | int) -> float:
        return zfac_get_option(self.ctx, OPTIONS[key] if isinstance(key, str) else int(key))

    def refine_refi(self, high: "Zfac", S: torch.Tensor, Z0: torch.Tensor, max_iter: int = 40, refi_steps: int = 1,
                    final_check: bool = True, out: Optional[torch.Tensor] = None, sync: bool = True):
        """Alg. 3: this (low-precision) context until its test fires, then `refi_steps` updates in the more precise
        context `high` (SPLIT16 or F64).  FP32 device tensors in, device tensor of `high`'s element type out:
        (Z, iters, err[...], flags)."""
        self._check(S, "S"); self._check(Z0, "Z0")
        Z = out if out is not None else torch.empty((self.n, self.n), dtype=high.dtype, device=S.device)
        self._check(Z, "Z", high.dtype)
        d_iters = torch.zeros(1, dtype=torch.int32, device=S.device)
        d_flags = torch.zeros(1, dtype=torch.int32, device=S.device)
        d_err = torch.full((max_iter + refi_steps + 2,), float("nan"), dtype=torch.float64, device=S.device)
        stream = torch.cuda.current_stream(S.device).cuda_stream
        zfac_refine_refi(self.ctx, high.ctx, S.data_ptr(), S.stride(0), Z0.data_ptr(), Z0.stride(0), Z.data_ptr(),
                         Z.stride(0), max_iter, refi_steps, int(final_check), d_iters.data_ptr(), d_err.data_ptr(),
                         d_flags.data_ptr(), stream)
        if not sync:
            return Z, d_iters, d_err, d_flags
        torch.cuda.current_stream(S.device).synchronize()
        it = int(d_iters.item())
        return Z, it, d_err[: it + 1 + int(final_check)].cpu().numpy(), int(d_flags.item())

    def refine_refi_host(self, high: "Zfac", S: torch.Tensor, Z0: torch.Tensor, Z: torch.Tensor, max_iter: int = 40,
                         refi_steps: int = 1, final_check: bool = True):
        """zfac_refine_refi_host: host (pinned) FP32 S, Z0 in, host Z of `high`'s element type out."""
        self._check(S, "S"); self._check(Z0, "Z0"); self._check(Z, "Z", high.dtype)
        for t, name in ((S, "S"), (Z0, "Z0"), (Z, "Z")):
            if t.is_cuda:
                raise ValueError(f"{name}: refine_refi_host takes host tensors")
        iters = ctypes.c_int(0)
        flags = ctypes.c_int(0)
        err = np.full(max_iter + refi_steps + 2, np.nan, dtype=np.float64)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        with torch.cuda.device(self.device):
            zfac_refine_refi_host(self.ctx, high.ctx, S.data_ptr(), S.stride(0), Z0.data_ptr(), Z0.stride(0), Z.data_ptr(),
                                  Z.stride(0), max_iter, refi_steps, int(final_check), ctypes.addressof(iters),
                                  err.ctypes.data, ctypes.addressof(flags), stream)
        return Z, iters.value, err[: iters.value + 1 + int(final_check)], flags.value

    def congruence(self, H: torch.Tensor, Z: torch.Tensor, out: Optional[torch.Tensor] = None) -> torch.Tensor:
        """H_perp = Z^T H Z (Eq. 11) on device tensors of the mode's element type."""
        self._check(H, "H"); self._check(Z, "Z")
        o = out if out is not None else torch.empty((self.n, self.n), dtype=self.dtype, device=H.device)
        self._check(o, "out")
        stream = torch.cuda.current_stream(H.device).cuda_stream
        zfac_congruence(self.ctx, H.data_ptr(), H.stride(0), Z.data_ptr(), Z.stride(0), o.data_ptr(), o.stride(0), stream)
        return o

    def peek(self, which: int) -> torch.Tensor:
        out = torch.empty((self.n, self.n), dtype=self.dtype, device=self.device)
        stream = torch.cuda.current_stream(self.device).cuda_stream
        zfac_peek(self.ctx, which, out.data_ptr(), out.stride(0), stream)
        torch.cuda.current_stream(self.device).synchronize()
        return out

    def set_profile(self, enable: bool) -> None:
        zfac_set_profile(self.ctx, enable)

    def set_order(self, m: int) -> None:
        zfac_set_order(self.ctx, m)

    @property
    def order(self) -> int:
        return zfac_get_order(self.ctx)

    def get_profile(self):
        return zfac_get_profile(self.ctx)

    @property
    def last_launch_count(self) -> int:
        return zfac_last_launch_count(self.ctx)


class ZfacBatched:
    """`batch` independent n x n problems refined by ONE launch sequence (zfac_create_batched / zfac_refine_batched):
    S, Z0, Z are [batch, n, n] device tensors (row-major problems, any batch stride).  Marshalling only."""

    def __init__(self, n: int, mode: str | int, batch: int, device: str | torch.device = "cuda"):
        if not torch.cuda.is_available():
            raise RuntimeError("zfac needs a CUDA device (sm_100a); there is no CPU path")
        self.n, self.batch, self.device = int(n), int(batch), torch.device(device)
        self.mode = MODES[mode] if isinstance(mode, str) else int(mode)
        self.dtype = torch.float32
        nbytes = zfac_workspace_bytes_batched(self.n, self.mode, self.batch)
        if nbytes == 0:
            raise ZfacError(ZFAC_E_INVALID, "zfac_workspace_bytes_batched")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
        with torch.cuda.device(self.device):
            self.ctx = zfac_create_batched(self.n, self.mode, self.batch, self.workspace.data_ptr(), self.workspace.numel())

    def close(self) -> None:
        if getattr(self, "ctx", None):
            zfac_destroy(self.ctx)
            self.ctx = None
            self.workspace = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_option(self, key: str | int, value: float) -> None:
        zfac_set_option(self.ctx, OPTIONS[key] if isinstance(key, str) else int(key), value)

    def set_order(self, m: int) -> None:
        zfac_set_order(self.ctx, m)

    def _check(self, t: torch.Tensor, name: str) -> None:
        if (t.dtype != self.dtype or t.dim() != 3 or t.shape[0] != self.batch or t.shape[1] != self.n or t.shape[2] != self.n
                or t.stride(2) != 1 or t.stride(1) < self.n or not t.is_cuda):
            raise ValueError(f"{name}: expected a [{self.batch}, {self.n}, {self.n}] {self.dtype} device tensor with unit column stride")

    def refine(self, S: torch.Tensor, Z0: torch.Tensor, max_iter: int = 40, stop: int = ZFAC_STOP_PAPER,
               out: Optional[torch.Tensor] = None, sync: bool = True):
        """sync=True: list of (Z_b, iters_b, err_b[0..iters_b], flags_b); sync=False: (Z, d_iters, d_err, d_flags)."""
        self._check(S, "S"); self._check(Z0, "Z0")
        Z = out if out is not None else torch.empty((self.batch, self.n, self.n), dtype=self.dtype, device=S.device)
        self._check(Z, "Z")
        d_iters = torch.zeros(self.batch, dtype=torch.int32, device=S.device)
        d_flags = torch.zeros(self.batch, dtype=torch.int32, device=S.device)
        d_err = torch.full((self.batch, max_iter + 1), float("nan"), dtype=torch.float64, device=S.device)
        stream = torch.cuda.current_stream(S.device).cuda_stream
        zfac_refine_batched(self.ctx, S.data_ptr(), S.stride(1), S.stride(0), Z0.data_ptr(), Z0.stride(1), Z0.stride(0),
                            Z.data_ptr(), Z.stride(1), Z.stride(0), max_iter, stop, d_iters.data_ptr(), d_err.data_ptr(),
                            d_flags.data_ptr(), stream)
        if not sync:
            return Z, d_iters, d_err, d_flags
        torch.cuda.current_stream(S.device).synchronize()
        its = d_iters.cpu().numpy(); fls = d_flags.cpu().numpy(); errs = d_err.cpu().numpy()
        return [(Z[b], int(its[b]), errs[b, : its[b] + 1], int(fls[b])) for b in range(self.batch)]

    @property
    def last_launch_count(self) -> int:
        return zfac_last_launch_count(self.ctx)


class ZfacBatch:
    """B independent n x n problems refined CONCURRENTLY: one context (own workspace) and one CUDA stream each.

    This is the scale-out the paper points to -- many graph-partitioned sub-problems, each solved densely
     -- on ONE GPU: `zfac_refine` is asynchronous on the caller's stream and contexts share no state,
    so at small n, where one problem's kernels cover 20-32 of the 148 SMs, the problems' kernels co-reside.  No
    kernel of the path changes; this holder only creates the contexts / streams and issues the calls (marshalling).
    Measured on B200, SPLIT16, 10 fixed updates: n = 1024, 1.57 ms per problem alone -> 0.30 ms with B >= 8
    (profiles/r1c_sweep.md)."""

    def __init__(self, n: int, mode: str | int, batch: int, device: str | torch.device = "cuda"):
        if batch < 1:
            raise ValueError("batch must be >= 1")
        self.n, self.batch, self.device = int(n), int(batch), torch.device(device)
        self.ctxs = [Zfac(n, mode, device) for _ in range(batch)]
        # each context sees one problem and would pick 256 x 128 tiles for it (ZFAC_OPT_NARROW_TILES = -1); together the
        # contexts fill the chip with wide tiles once batch x (padded n / 256)^2 exceeds 37 -- the library's own rule,
        # applied here to the whole set (measured, 16 streams at n = 1024: 301 TFLOP/s wide, 219 narrow)
        t = zfac_padded_n(self.n, self.ctxs[0].mode) // 256
        if self.ctxs[0].mode in (ZFAC_MODE_SPLIT16, ZFAC_MODE_HH16, ZFAC_MODE_TF32) and self.batch * t * t > 37:
            for c in self.ctxs:
                c.set_option("narrow_tiles", 0)
        self.streams = [torch.cuda.Stream(self.device) for _ in range(batch)]
        self.dtype = self.ctxs[0].dtype

    def close(self) -> None:
        for c in getattr(self, "ctxs", []):
            c.close()
        self.ctxs = []

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def set_order(self, m: int) -> None:
        for c in self.ctxs:
            c.set_order(m)

    def refine(self, S, Z0, max_iter: int = 40, stop: int = ZFAC_STOP_PAPER, out=None, sync: bool = True):
        """S, Z0: sequences of `batch` device tensors (or one tensor shared by every problem).  Problem i runs on
        stream i after whatever is pending on the current stream.  Returns a list of per-problem results in the
        format of `Zfac.refine` (sync=True: (Z, iters, err, flags); sync=False: raw device tensors -- the caller
        synchronises the streams, e.g. `wait()`)."""
        Ss = list(S) if isinstance(S, (list, tuple)) else [S] * self.batch
        Zs = list(Z0) if isinstance(Z0, (list, tuple)) else [Z0] * self.batch
        outs = list(out) if out is not None else [None] * self.batch
        if not (len(Ss) == len(Zs) == len(outs) == self.batch):
            raise ValueError(f"expected {self.batch} problems")
        cur = torch.cuda.current_stream(self.device)
        raw = []
        for c, st, s, z, o in zip(self.ctxs, self.streams, Ss, Zs, outs):
            st.wait_stream(cur)
            with torch.cuda.stream(st):
                raw.append(c.refine(s, z, max_iter=max_iter, stop=stop, out=o, sync=False))
        if not sync:
            return raw
        self.wait()
        res = []
        for Z, d_it, d_err, d_fl in raw:
            it = int(d_it.item())
            res.append((Z, it, d_err[: it + 1].cpu().numpy(), int(d_fl.item())))
        return res

    def wait(self) -> None:
        """Make the current stream wait for every problem's stream, then synchronise it."""
        cur = torch.cuda.current_stream(self.device)
        for st in self.streams:
            cur.wait_stream(st)
        cur.synchronize()


class ZfacGraph:
    """One `zfac_refine` call captured into a CUDA graph (include/zfac.h, "CUDA graphs") and replayed.

    The graph works on the tensors given here: write new S / Z0 contents INTO them (`S.copy_(...)`) and call
    `replay()`.  Marshalling only: capture uses torch's graph API around the same C-ABI call `Zfac.refine` makes."""

    def __init__(self, zf: Zfac, S: torch.Tensor, Z0: torch.Tensor, max_iter: int = 40, stop: int = ZFAC_STOP_PAPER,
                 out: Optional[torch.Tensor] = None):
        zf._check(S, "S"); zf._check(Z0, "Z0")
        self.zf, self.S, self.Z0, self.max_iter = zf, S, Z0, int(max_iter)
        self.Z = out if out is not None else torch.empty((zf.n, zf.n), dtype=zf.dtype, device=S.device)
        zf._check(self.Z, "Z")
        self.d_iters = torch.zeros(1, dtype=torch.int32, device=S.device)
        self.d_flags = torch.zeros(1, dtype=torch.int32, device=S.device)
        self.d_err = torch.full((self.max_iter + 1,), float("nan"), dtype=torch.float64, device=S.device)
        zf.set_profile(False)
        side = torch.cuda.Stream(S.device)
        side.wait_stream(torch.cuda.current_stream(S.device))
        self.graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(self.graph, stream=side):
            zfac_refine(zf.ctx, S.data_ptr(), S.stride(0), Z0.data_ptr(), Z0.stride(0), self.Z.data_ptr(),
                        self.Z.stride(0), self.max_iter, stop, self.d_iters.data_ptr(), self.d_err.data_ptr(),
                        self.d_flags.data_ptr(), torch.cuda.current_stream(S.device).cuda_stream)
        torch.cuda.current_stream(S.device).wait_stream(side)

    def replay(self, sync: bool = True):
        """Launch the captured call on the current stream.  sync=True: (Z, iters, err[0..iters], flags)."""
        self.graph.replay()
        if not sync:
            return self.Z, self.d_iters, self.d_err, self.d_flags
        torch.cuda.current_stream(self.S.device).synchronize()
        it = int(self.d_iters.item())
        return self.Z, it, self.d_err[: it + 1].cpu().numpy(), int(self.d_flags.item())


class ZfacLoopGraph:
    """The call as the library's own CUDA graph with a WHILE node (include/zfac.h, zfac_graph_*): it runs exactly as
    many iterations as the stop test allows -- no statically enqueued launches after the stop.  Bound to the tensors
    given here: write new S / Z0 contents INTO them and call `launch()`.  Marshalling only."""

    def __init__(self, zf: Zfac, S: torch.Tensor, Z0: torch.Tensor, max_iter: int = 40, stop: int = ZFAC_STOP_PAPER,
                 out: Optional[torch.Tensor] = None):
        zf._check(S, "S"); zf._check(Z0, "Z0")
        self.zf, self.S, self.Z0, self.max_iter = zf, S, Z0, int(max_iter)
        self.Z = out if out is not None else torch.empty((zf.n, zf.n), dtype=zf.dtype, device=S.device)
        zf._check(self.Z, "Z")
        self.d_iters = torch.zeros(1, dtype=torch.int32, device=S.device)
        self.d_flags = torch.zeros(1, dtype=torch.int32, device=S.device)
        self.d_err = torch.full((self.max_iter + 1,), float("nan"), dtype=torch.float64, device=S.device)
        with torch.cuda.device(S.device):
            self.graph = zfac_graph_create(zf.ctx, S.data_ptr(), S.stride(0), Z0.data_ptr(), Z0.stride(0),
                                           self.Z.data_ptr(), self.Z.stride(0), self.max_iter, stop,
                                           self.d_iters.data_ptr(), self.d_err.data_ptr(), self.d_flags.data_ptr())

    def close(self) -> None:
        if getattr(self, "graph", None):
            zfac_graph_destroy(self.graph)
            self.graph = None

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def launch(self, sync: bool = True):
        """Launch on the current stream.  sync=True: (Z, iters, err[0..iters], flags)."""
        zfac_graph_launch(self.graph, torch.cuda.current_stream(self.S.device).cuda_stream)
        if not sync:
            return self.Z, self.d_iters, self.d_err, self.d_flags
        torch.cuda.current_stream(self.S.device).synchronize()
        it = int(self.d_iters.item())
        return self.Z, it, self.d_err[: it + 1].cpu().numpy(), int(self.d_flags.item())

