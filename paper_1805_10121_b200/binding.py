"""Thin ctypes binding of libchase_filter.so (include/chase_filter.h): argument marshalling
only.  Every step of the path runs in the CUDA kernels behind the C ABI; torch is used for
device memory and streams.  There is no CPU fallback: a missing library raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np
import torch

from . import _build

CHASE_F32, CHASE_F64, CHASE_C64, CHASE_C128 = 0, 1, 2, 3
_DTYPE_CODE = {torch.float32: CHASE_F32, torch.float64: CHASE_F64,
               torch.complex64: CHASE_C64, torch.complex128: CHASE_C128}

EXPORTS = [
    "chase_filter", "chase_filter_ws", "chase_filter_host", "chase_filter_workspace_bytes",
    "chase_filter_scalars", "chase_filter_schedule", "chase_filter_kernel_path",
    "chase_filter_launch_count", "chase_fp64_peak_probe", "chase_filter_strerror", "chase_degrees",
    "chase_hemm", "chase_residuals", "chase_residuals_workspace_bytes", "chase_filter_step_plan",
    "chase_lanczos", "chase_lanczos_workspace_bytes", "chase_spectral_estimates", "chase_lanczos_ritz_vectors",
    "chase_hemm_rows", "chase_rows_barrier", "chase_rows_signal", "chase_rows_wait", "chase_rows_status",
    "chase_filter_rows_ws", "chase_filter_rows_hostsync_ws", "chase_ipc_export", "chase_ipc_open",
    "chase_ipc_close", "chase_residuals_static", "chase_scratch_cache_release",
    "chase_filter_host_open", "chase_filter_host_run", "chase_filter_host_close",
]
CHASE_STATIC_SCRATCH_BYTES = 48 << 20      # include/chase_filter.h
HOST_BARRIER_FN = ctypes.CFUNCTYPE(ctypes.c_int, ctypes.c_void_p)

_lib = None


class ChaseFilterError(RuntimeError):
    def __init__(self, code: int, msg: str):
        super().__init__(f"chase_filter error {code}: {msg}")
        self.code = code


def lib_path() -> str:
    """The in-tree library; CHASE_FILTER_LIB selects another build of the same sources."""
    return os.environ.get("CHASE_FILTER_LIB") or _build.LIB


def load() -> ctypes.CDLL:
    """Load the in-tree shared library; fail loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    path = lib_path()
    if not os.path.exists(path):
        raise ImportError(
            f"{path} is missing: build it with `python -m paper_1805_10121_b200._build` "
            "(or __graft_entry__.build()).  There is no CPU fallback.")
    lib = ctypes.CDLL(path)
    vp, i64, i32, dbl, sz = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int32, ctypes.c_double, ctypes.c_size_t
    lib.chase_filter_workspace_bytes.restype = sz
    lib.chase_filter_workspace_bytes.argtypes = [i64, i64, ctypes.c_int]
    lib.chase_filter_ws.restype = ctypes.c_int
    lib.chase_filter_ws.argtypes = [vp, i64, vp, i64, vp, dbl, dbl, dbl, ctypes.c_int, vp, sz, vp]
    lib.chase_filter.restype = ctypes.c_int
    lib.chase_filter.argtypes = [vp, i64, vp, i64, vp, dbl, dbl, dbl, ctypes.c_int, vp]
    lib.chase_filter_host.restype = ctypes.c_int
    lib.chase_filter_host.argtypes = [vp, i64, vp, i64, vp, dbl, dbl, dbl, ctypes.c_int, ctypes.c_int]
    lib.chase_filter_scalars.restype = ctypes.c_int
    lib.chase_filter_scalars.argtypes = [dbl, dbl, dbl, i32, vp, vp, vp]
    lib.chase_filter_schedule.restype = ctypes.c_int
    lib.chase_filter_schedule.argtypes = [vp, i64, vp]
    lib.chase_filter_kernel_path.restype = ctypes.c_int
    lib.chase_filter_kernel_path.argtypes = [i64, i64, ctypes.c_int]
    lib.chase_filter_launch_count.restype = i64
    lib.chase_filter_launch_count.argtypes = []
    lib.chase_fp64_peak_probe.restype = ctypes.c_int
    lib.chase_fp64_peak_probe.argtypes = [ctypes.c_int, ctypes.c_int, vp]
    lib.chase_degrees.restype = ctypes.c_int
    lib.chase_degrees.argtypes = [i64, vp, vp, dbl, dbl, dbl, i32, i32, vp, vp]
    lib.chase_hemm.restype = ctypes.c_int
    lib.chase_hemm.argtypes = [vp, i64, vp, vp, i64, dbl, dbl, dbl, ctypes.c_int, vp]
    lib.chase_residuals_workspace_bytes.restype = sz
    lib.chase_residuals_workspace_bytes.argtypes = [i64, i64, ctypes.c_int]
    lib.chase_residuals.restype = ctypes.c_int
    lib.chase_residuals.argtypes = [vp, i64, vp, i64, vp, vp, ctypes.c_int, vp, sz, vp]
    lib.chase_filter_host_open.restype = ctypes.c_int
    lib.chase_filter_host_open.argtypes = [vp, i64, i64, ctypes.c_int, ctypes.c_int, vp]
    lib.chase_filter_host_run.restype = ctypes.c_int
    lib.chase_filter_host_run.argtypes = [vp, vp, i64, vp, dbl, dbl, dbl]
    lib.chase_filter_host_close.restype = ctypes.c_int
    lib.chase_filter_host_close.argtypes = [vp]
    lib.chase_scratch_cache_release.restype = ctypes.c_int
    lib.chase_scratch_cache_release.argtypes = []
    lib.chase_residuals_static.restype = ctypes.c_int
    lib.chase_residuals_static.argtypes = [vp, i64, vp, i64, vp, vp, ctypes.c_int, vp]
    lib.chase_filter_step_plan.restype = ctypes.c_int
    lib.chase_filter_step_plan.argtypes = [i64, i64, ctypes.c_int, i32, vp, vp]
    lib.chase_lanczos_workspace_bytes.restype = sz
    lib.chase_lanczos_workspace_bytes.argtypes = [i64, i64, i32, ctypes.c_int]
    lib.chase_lanczos.restype = ctypes.c_int
    lib.chase_lanczos.argtypes = [vp, i64, vp, i64, i32, ctypes.c_int, vp, vp, vp, sz, vp]
    lib.chase_lanczos_ritz_vectors.restype = ctypes.c_int
    lib.chase_lanczos_ritz_vectors.argtypes = [vp, sz, i64, i64, i32, ctypes.c_int, i64, vp, vp, dbl, vp, i64, vp, i64,
                                               vp, vp, vp]
    lib.chase_spectral_estimates.restype = ctypes.c_int
    lib.chase_spectral_estimates.argtypes = [i32, i64, vp, vp, i64, dbl, dbl, vp, vp, vp]
    lib.chase_hemm_rows.restype = ctypes.c_int
    lib.chase_hemm_rows.argtypes = [vp, i64, i64, i64, vp, vp, i64, dbl, dbl, dbl, ctypes.c_int, i32, vp, vp]
    lib.chase_rows_barrier.restype = ctypes.c_int
    lib.chase_rows_barrier.argtypes = [vp, vp, i32, i32, ctypes.c_uint32, vp]
    lib.chase_rows_signal.restype = ctypes.c_int
    lib.chase_rows_signal.argtypes = [vp, vp, i32, i32, ctypes.c_uint32, vp]
    lib.chase_rows_wait.restype = ctypes.c_int
    lib.chase_rows_wait.argtypes = [vp, i32, ctypes.c_uint32, vp]
    lib.chase_rows_status.restype = ctypes.c_int
    lib.chase_rows_status.argtypes = [vp, i32, vp]
    lib.chase_filter_rows_ws.restype = ctypes.c_int
    lib.chase_filter_rows_ws.argtypes = [vp, i64, i64, i64, vp, i64, vp, dbl, dbl, dbl, ctypes.c_int, vp, sz,
                                         i32, i32, vp, vp, vp, vp, vp, vp]
    lib.chase_filter_rows_hostsync_ws.restype = ctypes.c_int
    lib.chase_filter_rows_hostsync_ws.argtypes = lib.chase_filter_rows_ws.argtypes + [HOST_BARRIER_FN, vp]
    lib.chase_ipc_export.restype = ctypes.c_int
    lib.chase_ipc_export.argtypes = [vp, vp, vp]
    lib.chase_ipc_open.restype = ctypes.c_int
    lib.chase_ipc_open.argtypes = [vp, vp]
    lib.chase_ipc_close.restype = ctypes.c_int
    lib.chase_ipc_close.argtypes = [vp]
    lib.chase_filter_strerror.restype = ctypes.c_char_p
    lib.chase_filter_strerror.argtypes = [ctypes.c_int]
    _lib = lib
    return lib


def chase_filter_strerror(code: int) -> str:
    return load().chase_filter_strerror(int(code)).decode()


def _check(code: int) -> None:
    if code != 0:
        raise ChaseFilterError(code, chase_filter_strerror(code))


def _degrees_array(degrees, ncols: int) -> np.ndarray:
    if isinstance(degrees, torch.Tensor):
        degrees = degrees.cpu().numpy()
    deg = np.ascontiguousarray(np.asarray(degrees, dtype=np.int32))
    if deg.shape != (ncols,):
        raise ValueError(f"degrees must have shape ({ncols},), got {deg.shape}")
    return deg


def _check_colmajor(x: torch.Tensor, name: str) -> None:
    if x.dim() != 2 or (x.shape[0] > 1 and x.stride(0) != 1) or \
            (x.shape[1] > 1 and x.stride(1) != x.shape[0]):
        raise ValueError(f"{name} must be column-major with ld = rows "
                         f"(shape {tuple(x.shape)}, strides {x.stride()})")


def _stream_ptr(stream: Optional[torch.cuda.Stream]) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def chase_filter_workspace_bytes(N: int, ncols: int, dtype: torch.dtype) -> int:
    return int(load().chase_filter_workspace_bytes(N, ncols, _DTYPE_CODE[dtype]))


def chase_filter_kernel_path(N: int, ncols: int, dtype: torch.dtype) -> int:
    return int(load().chase_filter_kernel_path(N, ncols, _DTYPE_CODE[dtype]))


def chase_filter_launch_count() -> int:
    return int(load().chase_filter_launch_count())


def chase_filter_ws(H: torch.Tensor, V: torch.Tensor, degrees, a: float, b: float, lambda1: float,
                    workspace: torch.Tensor, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """V[:, j] <- p_{degrees[j]}(H) V[:, j] in place (device tensors, column-major).
    `workspace`: any device tensor of >= chase_filter_workspace_bytes bytes.  Asynchronous."""
    lib = load()
    if not (H.is_cuda and V.is_cuda and workspace.is_cuda):
        raise ValueError("H, V and workspace must be CUDA tensors (there is no CPU path)")
    if H.dtype != V.dtype or H.dtype not in _DTYPE_CODE:
        raise ValueError("H and V must share a dtype in {f32, f64, c64, c128}")
    _check_colmajor(H, "H")
    _check_colmajor(V, "V")
    N, ncols = V.shape
    if H.shape != (N, N):
        raise ValueError("H must be N x N with N = V.shape[0]")
    deg = _degrees_array(degrees, ncols)
    ws_bytes = workspace.numel() * workspace.element_size()
    with torch.cuda.device(H.device):
        rc = lib.chase_filter_ws(H.data_ptr(), N, V.data_ptr(), ncols, deg.ctypes.data,
                                 float(a), float(b), float(lambda1), _DTYPE_CODE[H.dtype],
                                 workspace.data_ptr(), ws_bytes, _stream_ptr(stream))
    _check(rc)
    return V


def chase_filter(H: torch.Tensor, V: torch.Tensor, degrees, a: float, b: float, lambda1: float,
                 stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """Same as chase_filter_ws; scratch comes from cudaMallocAsync inside the library."""
    lib = load()
    if not (H.is_cuda and V.is_cuda):
        raise ValueError("H and V must be CUDA tensors (there is no CPU path)")
    if H.dtype != V.dtype or H.dtype not in _DTYPE_CODE:
        raise ValueError("H and V must share a dtype in {f32, f64, c64, c128}")
    _check_colmajor(H, "H")
    _check_colmajor(V, "V")
    N, ncols = V.shape
    if H.shape != (N, N):
        raise ValueError("H must be N x N with N = V.shape[0]")
    deg = _degrees_array(degrees, ncols)
    with torch.cuda.device(H.device):
        rc = lib.chase_filter(H.data_ptr(), N, V.data_ptr(), ncols, deg.ctypes.data,
                              float(a), float(b), float(lambda1), _DTYPE_CODE[H.dtype],
                              _stream_ptr(stream))
    _check(rc)
    return V


def chase_filter_host(H: torch.Tensor, V: torch.Tensor, degrees, a: float, b: float, lambda1: float,
                      device: int = 0) -> torch.Tensor:
    """HOST tensors in, result in V (host); H2D/D2H copies happen inside the C call."""
    lib = load()
    if H.is_cuda or V.is_cuda:
        raise ValueError("chase_filter_host takes host tensors")
    if H.dtype != V.dtype or H.dtype not in _DTYPE_CODE:
        raise ValueError("H and V must share a dtype in {f32, f64, c64, c128}")
    _check_colmajor(H, "H")
    _check_colmajor(V, "V")
    N, ncols = V.shape
    deg = _degrees_array(degrees, ncols)
    rc = lib.chase_filter_host(H.data_ptr(), N, V.data_ptr(), ncols, deg.ctypes.data,
                               float(a), float(b), float(lambda1), _DTYPE_CODE[H.dtype], int(device))
    _check(rc)
    return V


class HostFilter:
    """chase_filter_host_open / _run / _close: host tensors in and out like chase_filter_host, but H is uploaded
    once and stays on the device for every run() on this handle (a solve calls the filter hundreds of times)."""

    def __init__(self, H: torch.Tensor, max_ncols: int, device: int = 0):
        if H.is_cuda or H.dtype not in _DTYPE_CODE:
            raise ValueError("HostFilter takes a host tensor H of dtype f32, f64, c64 or c128")
        _check_colmajor(H, "H")
        if H.dim() != 2 or H.shape[0] != H.shape[1]:
            raise ValueError("H must be N x N")
        self.N, self.dtype, self.max_ncols = int(H.shape[0]), H.dtype, int(max_ncols)
        handle = ctypes.c_void_p()
        _check(load().chase_filter_host_open(H.data_ptr(), self.N, self.max_ncols, _DTYPE_CODE[H.dtype], int(device),
                                             ctypes.addressof(handle)))
        self._handle = handle

    def run(self, V: torch.Tensor, degrees, a: float, b: float, lambda1: float) -> torch.Tensor:
        if self._handle is None:
            raise ValueError("handle is closed")
        if V.is_cuda or V.dtype != self.dtype:
            raise ValueError("V must be a host tensor of H's dtype")
        _check_colmajor(V, "V")
        if V.shape[0] != self.N:
            raise ValueError("V must have N rows")
        ncols = int(V.shape[1])
        deg = _degrees_array(degrees, ncols)
        _check(load().chase_filter_host_run(self._handle, V.data_ptr(), ncols, deg.ctypes.data, float(a), float(b),
                                            float(lambda1)))
        return V

    def close(self) -> None:
        if self._handle is not None:
            h, self._handle = self._handle, None
            _check(load().chase_filter_host_close(h))

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()


def chase_filter_scalars(a: float, b: float, lambda1: float, m_max: int):
    """(alpha[0..m_max], beta[0..m_max], c); entry 0 unused."""
    alpha = np.zeros(m_max + 1)
    beta = np.zeros(m_max + 1)
    c = ctypes.c_double()
    _check(load().chase_filter_scalars(float(a), float(b), float(lambda1), int(m_max),
                                       alpha.ctypes.data, beta.ctypes.data, ctypes.addressof(c)))
    return alpha, beta, c.value


def chase_filter_schedule(degrees: Sequence[int]):
    """(m_max, offset[0..m_max]) with offset[k] = first active column of step k."""
    deg = np.ascontiguousarray(np.asarray(degrees, dtype=np.int32))
    lib = load()
    m_max = lib.chase_filter_schedule(deg.ctypes.data, deg.size, None)
    if m_max < 0:
        _check(m_max)
    offset = np.zeros(m_max + 1, dtype=np.int32)
    lib.chase_filter_schedule(deg.ctypes.data, deg.size, offset.ctypes.data)
    return m_max, offset


def chase_filter_step_plan(N: int, n_active: int, dtype: torch.dtype, sms: int = 148):
    """Work decomposition of one FP64 tensor-kernel launch: dict with tiles_m, tiles_n, tile_width,
    dp_tiles, sk_ctas, slabs_per_tile, grid, dp_rounds and sk_begin (numpy int32[sk_ctas + 1])."""
    out = np.zeros(9, dtype=np.int32)
    skb = np.zeros(161, dtype=np.int32)
    _check(load().chase_filter_step_plan(int(N), int(n_active), _DTYPE_CODE[dtype], int(sms), out.ctypes.data,
                                         skb.ctypes.data))
    keys = ("tiles_m", "tiles_n", "tile_width", "dp_tiles", "sk_ctas", "slabs_per_tile", "grid", "dp_rounds",
            "sk_first")
    plan = {k: int(v) for k, v in zip(keys, out)}
    plan["sk_begin"] = skb[: plan["sk_ctas"] + 1].copy()
    return plan


def chase_fp64_peak_probe(kind: int, iters: int = 4096) -> float:
    """GFLOP/s of the register-only probe (0: DFMA, 1: DMMA.8x8x4) on the current device."""
    g = ctypes.c_double()
    _check(load().chase_fp64_peak_probe(int(kind), int(iters), ctypes.addressof(g)))
    return g.value


def chase_degrees(resid, ritzv, tol: float, a: float, b: float, deg_extra: int = 2, deg_max: int = 36):
    """Alg. 5 + the sort of Alg. 1 l.15: (degrees sorted ascending [int32], perm [int64]) with
    degrees[i] belonging to original column perm[i]."""
    res = np.ascontiguousarray(np.asarray(resid, dtype=np.float64))
    rv = np.ascontiguousarray(np.asarray(ritzv, dtype=np.float64))
    if res.shape != rv.shape or res.ndim != 1:
        raise ValueError("resid and ritzv must be 1-D arrays of equal length")
    deg = np.zeros(res.size, dtype=np.int32)
    perm = np.zeros(res.size, dtype=np.int64)
    _check(load().chase_degrees(res.size, res.ctypes.data, rv.ctypes.data, float(tol), float(a), float(b),
                                int(deg_extra), int(deg_max), deg.ctypes.data, perm.ctypes.data))
    return deg, perm


def chase_hemm(H: torch.Tensor, X: torch.Tensor, Y: torch.Tensor, alpha: float = 1.0, beta: float = 0.0,
               shift: float = 0.0, stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """Y <- alpha (H - shift I) X + beta Y on the step kernels (device tensors, column-major)."""
    if not (H.is_cuda and X.is_cuda and Y.is_cuda):
        raise ValueError("H, X, Y must be CUDA tensors (there is no CPU path)")
    if not (H.dtype == X.dtype == Y.dtype) or H.dtype not in _DTYPE_CODE:
        raise ValueError("H, X, Y must share a dtype in {f32, f64, c64, c128}")
    for t, nm in ((H, "H"), (X, "X"), (Y, "Y")):
        _check_colmajor(t, nm)
    N, ncols = X.shape
    if H.shape != (N, N) or Y.shape != X.shape:
        raise ValueError("shape mismatch")
    with torch.cuda.device(H.device):
        _check(load().chase_hemm(H.data_ptr(), N, X.data_ptr(), Y.data_ptr(), ncols, float(alpha), float(beta),
                                 float(shift), _DTYPE_CODE[H.dtype], _stream_ptr(stream)))
    return Y


def chase_scratch_cache_release() -> None:
    """Frees the stream-K scratch buffers the library keeps for chase_hemm / the row-sharded calls."""
    _check(load().chase_scratch_cache_release())


def chase_residuals_workspace_bytes(N: int, ncols: int, dtype: torch.dtype) -> int:
    return int(load().chase_residuals_workspace_bytes(N, ncols, _DTYPE_CODE[dtype]))


def chase_residuals(H: torch.Tensor, V: torch.Tensor, ritzv, workspace: Optional[torch.Tensor] = None,
                    stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """resid[j] = ||H V[:,j] - ritzv[j] V[:,j]||_2 as a device float64 tensor [ncols]."""
    if not (H.is_cuda and V.is_cuda):
        raise ValueError("H and V must be CUDA tensors (there is no CPU path)")
    if H.dtype != V.dtype or H.dtype not in _DTYPE_CODE:
        raise ValueError("H and V must share a dtype in {f32, f64, c64, c128}")
    _check_colmajor(H, "H")
    _check_colmajor(V, "V")
    N, ncols = V.shape
    rv = np.ascontiguousarray(np.asarray(ritzv, dtype=np.float64))
    if rv.shape != (ncols,):
        raise ValueError("ritzv must have one entry per column")
    need = chase_residuals_workspace_bytes(N, ncols, H.dtype)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=H.device)
    resid = torch.empty(ncols, dtype=torch.float64, device=H.device)
    with torch.cuda.device(H.device):
        _check(load().chase_residuals(H.data_ptr(), N, V.data_ptr(), ncols, rv.ctypes.data, resid.data_ptr(),
                                      _DTYPE_CODE[H.dtype], workspace.data_ptr(),
                                      workspace.numel() * workspace.element_size(), _stream_ptr(stream)))
    return resid


def chase_residuals_static(H: torch.Tensor, V: torch.Tensor, ritzv, resid: torch.Tensor,
                           stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """chase_residuals for callers that may not allocate device memory (a plug-in inside an application
    whose pool owns the whole GPU, a process with a fixed HBM share, a loop that must stay out of the
    driver's allocator): the scratch is a 48 MiB static array inside libchase_filter.so, so this wrapper
    creates no tensor either -- the caller brings `resid` (device float64 [ncols]), which is also returned.
    Problems whose chase_residuals_workspace_bytes exceeds CHASE_STATIC_SCRATCH_BYTES raise ChaseFilterError
    (code -8).  All calls on one GPU share the array: keep them on one stream.  The first call on a device
    resolves the array's address; make it before any stream capture."""
    if not (H.is_cuda and V.is_cuda and resid.is_cuda):
        raise ValueError("H, V and resid must be CUDA tensors (there is no CPU path)")
    if H.dtype != V.dtype or H.dtype not in _DTYPE_CODE:
        raise ValueError("H and V must share a dtype in {f32, f64, c64, c128}")
    _check_colmajor(H, "H")
    _check_colmajor(V, "V")
    N, ncols = V.shape
    rv = np.ascontiguousarray(np.asarray(ritzv, dtype=np.float64))
    if rv.shape != (ncols,):
        raise ValueError("ritzv must have one entry per column")
    if resid.dtype != torch.float64 or resid.shape != (ncols,) or not resid.is_contiguous():
        raise ValueError("resid must be a contiguous float64 tensor with one entry per column")
    with torch.cuda.device(H.device):
        _check(load().chase_residuals_static(H.data_ptr(), N, V.data_ptr(), ncols, rv.ctypes.data, resid.data_ptr(),
                                             _DTYPE_CODE[H.dtype], _stream_ptr(stream)))
    return resid


def chase_lanczos_workspace_bytes(N: int, nruns: int, k: int, dtype: torch.dtype) -> int:
    return int(load().chase_lanczos_workspace_bytes(N, nruns, k, _DTYPE_CODE[dtype]))


def chase_lanczos(H: torch.Tensor, V0: torch.Tensor, k: int, workspace: Optional[torch.Tensor] = None,
                  stream: Optional[torch.cuda.Stream] = None):
    """k Lanczos steps for every column of V0 (Alg. 6 l.2 / l.8), coalesced into one HEMM per step.
    Returns host arrays (alpha[nruns, k], beta[nruns, k]); synchronises the stream."""
    if not (H.is_cuda and V0.is_cuda):
        raise ValueError("H and V0 must be CUDA tensors (there is no CPU path)")
    if H.dtype != V0.dtype or H.dtype not in _DTYPE_CODE:
        raise ValueError("H and V0 must share a dtype in {f32, f64, c64, c128}")
    _check_colmajor(H, "H")
    _check_colmajor(V0, "V0")
    N, nruns = V0.shape
    if H.shape != (N, N):
        raise ValueError("shape mismatch")
    need = chase_lanczos_workspace_bytes(N, nruns, k, H.dtype)
    if workspace is None:
        workspace = torch.empty(max(need, 16), dtype=torch.uint8, device=H.device)
    alpha = np.zeros((nruns, k), dtype=np.float64)
    beta = np.zeros((nruns, k), dtype=np.float64)
    with torch.cuda.device(H.device):
        _check(load().chase_lanczos(H.data_ptr(), N, V0.data_ptr(), nruns, int(k), _DTYPE_CODE[H.dtype],
                                    alpha.ctypes.data, beta.ctypes.data, workspace.data_ptr(),
                                    workspace.numel() * workspace.element_size(), _stream_ptr(stream)))
    return alpha, beta


def chase_lanczos_ritz_vectors(workspace: torch.Tensor, N: int, dtype: torch.dtype, alpha, beta, run: int,
                               mu_ne: float, Vhat: torch.Tensor, dst_cols,
                               stream: Optional[torch.cuda.Stream] = None):
    """Alg. 6 l.13: Ritz vectors of run `run` with Ritz value < mu_ne (ascending) into the columns
    dst_cols[i] of Vhat; `workspace` / alpha / beta come from the chase_lanczos call.  Returns the Ritz
    values written (numpy, length = number of vectors written <= len(dst_cols))."""
    if not (workspace.is_cuda and Vhat.is_cuda) or Vhat.dtype != dtype or dtype not in _DTYPE_CODE:
        raise ValueError("workspace and Vhat must be CUDA tensors, Vhat of the Lanczos dtype")
    _check_colmajor(Vhat, "Vhat")
    if Vhat.shape[0] != N:
        raise ValueError("Vhat must have N rows")
    a = np.ascontiguousarray(np.asarray(alpha, dtype=np.float64))
    b = np.ascontiguousarray(np.asarray(beta, dtype=np.float64))
    if a.ndim != 2 or a.shape != b.shape:
        raise ValueError("alpha and beta must be [nruns, k] arrays of equal shape")
    nruns, k = a.shape
    dst = np.ascontiguousarray(np.asarray(dst_cols, dtype=np.int64))
    count = ctypes.c_int64()
    vals = np.zeros(max(dst.size, 1), dtype=np.float64)
    with torch.cuda.device(Vhat.device):
        _check(load().chase_lanczos_ritz_vectors(
            workspace.data_ptr(), workspace.numel() * workspace.element_size(), int(N), int(nruns), int(k),
            _DTYPE_CODE[dtype], int(run), a.ctypes.data, b.ctypes.data, float(mu_ne), Vhat.data_ptr(),
            int(Vhat.shape[1]), dst.ctypes.data, int(dst.size), ctypes.addressof(count), vals.ctypes.data,
            _stream_ptr(stream)))
    return vals[: int(count.value)].copy()


def chase_spectral_estimates(alpha, beta, N: int, nev_nex: float, sigma: float = 0.25):
    """(b_sup, mu_1, mu_nev_nex) of Alg. 6 from the coefficients of 1 + n_vec Lanczos runs (host only);
    a single run gives (b_sup, None, None)."""
    a = np.ascontiguousarray(np.asarray(alpha, dtype=np.float64))
    b = np.ascontiguousarray(np.asarray(beta, dtype=np.float64))
    if a.ndim != 2 or a.shape != b.shape:
        raise ValueError("alpha and beta must be [nruns, k] arrays of equal shape")
    nruns, k = a.shape
    out = (ctypes.c_double * 3)()
    base = ctypes.addressof(out)
    _check(load().chase_spectral_estimates(int(k), int(nruns), a.ctypes.data, b.ctypes.data, int(N), float(nev_nex),
                                           float(sigma), base, base + 8, base + 16))
    return (out[0], None, None) if nruns == 1 else (out[0], out[1], out[2])


# ---------------------------------------------------------------------------------------------
# Row-sharded path (one process per GPU; H row block per rank, fused NVLink all-gather)
# ---------------------------------------------------------------------------------------------
def _ptr_array(ptrs: Sequence[int]):
    arr = (ctypes.c_void_p * max(len(ptrs), 1))()
    for i, p in enumerate(ptrs):
        arr[i] = int(p) if p else None
    return arr


def _check_rows(H_loc: torch.Tensor, N: int, row0: int):
    if not H_loc.is_cuda or H_loc.dtype not in _DTYPE_CODE:
        raise ValueError("H_loc must be a CUDA tensor of a supported dtype (there is no CPU path)")
    _check_colmajor(H_loc, "H_loc")
    nrows = H_loc.shape[0]
    if H_loc.shape[1] != N or row0 < 0 or row0 + nrows > N:
        raise ValueError("H_loc must be the nrows x N row block [row0, row0 + nrows) of H")
    return nrows


def chase_hemm_rows(H_loc: torch.Tensor, row0: int, X: torch.Tensor, Y: torch.Tensor, alpha: float = 1.0,
                    beta: float = 0.0, shift: float = 0.0, peer_Y: Sequence[int] = (),
                    stream: Optional[torch.cuda.Stream] = None) -> torch.Tensor:
    """Y[rows] <- alpha (H_loc X - shift X[rows]) + beta Y[rows]; the rows are also stored through the
    peer-mapped device pointers `peer_Y` (other ranks' Y buffers)."""
    N, ncols = X.shape
    nrows = _check_rows(H_loc, N, row0)
    if not (X.is_cuda and Y.is_cuda) or X.dtype != H_loc.dtype or Y.dtype != H_loc.dtype or Y.shape != X.shape:
        raise ValueError("X, Y must be CUDA tensors of H_loc's dtype and equal shape")
    _check_colmajor(X, "X")
    _check_colmajor(Y, "Y")
    arr = _ptr_array(peer_Y)
    with torch.cuda.device(H_loc.device):
        _check(load().chase_hemm_rows(H_loc.data_ptr(), N, int(row0), nrows, X.data_ptr(), Y.data_ptr(), ncols,
                                      float(alpha), float(beta), float(shift), _DTYPE_CODE[H_loc.dtype],
                                      len(peer_Y), arr, _stream_ptr(stream)))
    return Y


def _check_flags(flags: torch.Tensor, nranks: int) -> None:
    if not flags.is_cuda or flags.dtype != torch.int32 or flags.numel() < nranks + 1:
        raise ValueError("flags must be a CUDA int32 tensor with nranks + 1 entries (slots + status word)")


def chase_rows_barrier(flags: torch.Tensor, peer_flags: Sequence[int], rank: int, seq: int,
                       stream: Optional[torch.cuda.Stream] = None) -> None:
    """Inter-GPU barrier on `stream` over flag arrays in peer memory (see include/chase_filter.h)."""
    _check_flags(flags, len(peer_flags))
    arr = _ptr_array(peer_flags)
    with torch.cuda.device(flags.device):
        _check(load().chase_rows_barrier(flags.data_ptr(), arr, len(peer_flags), int(rank), int(seq) & 0xFFFFFFFF,
                                         _stream_ptr(stream)))


def chase_rows_signal(flags: torch.Tensor, peer_flags: Sequence[int], rank: int, seq: int,
                      stream: Optional[torch.cuda.Stream] = None) -> None:
    _check_flags(flags, len(peer_flags))
    arr = _ptr_array(peer_flags)
    with torch.cuda.device(flags.device):
        _check(load().chase_rows_signal(flags.data_ptr(), arr, len(peer_flags), int(rank), int(seq) & 0xFFFFFFFF,
                                        _stream_ptr(stream)))


def chase_rows_wait(flags: torch.Tensor, nranks: int, seq: int, stream: Optional[torch.cuda.Stream] = None) -> None:
    _check_flags(flags, nranks)
    with torch.cuda.device(flags.device):
        _check(load().chase_rows_wait(flags.data_ptr(), int(nranks), int(seq) & 0xFFFFFFFF, _stream_ptr(stream)))


def chase_rows_status(flags: torch.Tensor, nranks: int, stream: Optional[torch.cuda.Stream] = None) -> None:
    """Synchronises `stream`; raises ChaseFilterError(-7) if a barrier on these flags timed out."""
    _check_flags(flags, nranks)
    with torch.cuda.device(flags.device):
        _check(load().chase_rows_status(flags.data_ptr(), int(nranks), _stream_ptr(stream)))


def chase_filter_rows_ws(H_loc: torch.Tensor, row0: int, V: torch.Tensor, degrees, a: float, b: float,
                         lambda1: float, workspace: torch.Tensor, rank: int = 0, peer_V: Sequence[int] = (),
                         peer_W: Sequence[int] = (), flags: Optional[torch.Tensor] = None,
                         peer_flags: Sequence[int] = (), seq: int = 0,
                         stream: Optional[torch.cuda.Stream] = None, host_barrier=None) -> int:
    """Row-sharded filter; peer_V / peer_W / peer_flags hold one device pointer per rank (own entry
    ignored).  `host_barrier` (a callable returning 0) selects chase_filter_rows_hostsync_ws, for ranks
    that time-share one GPU.  Returns the advanced barrier sequence number."""
    N, ncols = V.shape
    nrows = _check_rows(H_loc, N, row0)
    if not V.is_cuda or V.dtype != H_loc.dtype:
        raise ValueError("V must be a CUDA tensor of H_loc's dtype")
    _check_colmajor(V, "V")
    deg = _degrees_array(degrees, ncols)
    nranks = max(len(peer_V), 1)
    if flags is not None:
        _check_flags(flags, nranks)
    seq_c = ctypes.c_uint32(int(seq) & 0xFFFFFFFF)
    args = [H_loc.data_ptr(), N, int(row0), nrows, V.data_ptr(), ncols, deg.ctypes.data, float(a), float(b),
            float(lambda1), _DTYPE_CODE[H_loc.dtype], workspace.data_ptr(),
            workspace.numel() * workspace.element_size(), nranks, int(rank),
            _ptr_array(peer_V) if len(peer_V) else None, _ptr_array(peer_W) if len(peer_W) else None,
            flags.data_ptr() if flags is not None else None,
            _ptr_array(peer_flags) if len(peer_flags) else None, ctypes.addressof(seq_c), _stream_ptr(stream)]
    with torch.cuda.device(H_loc.device):
        if host_barrier is None:
            _check(load().chase_filter_rows_ws(*args))
        else:
            # ctypes swallows an exception raised inside a callback and hands 0 (= success) to the C side, which
            # would then spin in the wait kernel for its whole timeout: report failure instead, keep the exception
            # and re-raise it once the C call has returned.
            raised = []

            def _barrier(_ctx):
                try:
                    return int(host_barrier() or 0)
                except BaseException as exc:           # noqa: BLE001 -- must not propagate into C
                    raised.append(exc)
                    return 1

            cb = HOST_BARRIER_FN(_barrier)
            rc = load().chase_filter_rows_hostsync_ws(*args, cb, None)
            if raised:
                raise raised[0]
            _check(rc)
    return int(seq_c.value)


def chase_ipc_export(t: torch.Tensor):
    """(64-byte handle, byte offset) of the CUDA allocation holding tensor `t` (for another process)."""
    h = ctypes.create_string_buffer(64)
    off = ctypes.c_int64()
    with torch.cuda.device(t.device):
        _check(load().chase_ipc_export(t.data_ptr(), h, ctypes.addressof(off)))
    return bytes(h.raw), int(off.value)


def chase_ipc_open(handle: bytes) -> int:
    """Maps a handle exported by another process on the current device; returns the base pointer."""
    base = ctypes.c_void_p()
    _check(load().chase_ipc_open(ctypes.c_char_p(handle), ctypes.addressof(base)))
    return int(base.value)


def chase_ipc_close(base: int) -> None:
    _check(load().chase_ipc_close(ctypes.c_void_p(base)))
