"""ctypes marshalling for libsagecal_b200.so.  No arithmetic of the method lives here."""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np
import torch

COH_FULL = 0
COH_SCALAR = 1
LM_COMPRESSED = 0
LM_DIRECT = 1
LM_FULLGN = 2
LM_PERCLUSTER = 3
WS_LM_PASS = 1
WS_CALIBRATE_FULLGN = 3
WS_CALIBRATE = 2

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_PKG, "libsagecal_b200.so")
_lib = None


class SagecalError(RuntimeError):
    def __init__(self, code: int, where: str):
        L = load_library()
        msg = L.sagecal_strerror(code).decode()
        extra = f" (cudaError {L.sagecal_last_cuda_error()})" if code == -3 else ""
        super().__init__(f"{where}: {msg}{extra} [code {code}]")
        self.code = code


def lib_path() -> str:
    return _LIB_PATH


def load_library():
    """dlopen the C-ABI library.  Raises if it has not been built: there is no fallback path."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(_LIB_PATH):
        raise ImportError(
            f"{_LIB_PATH} is missing: build it with `python -m paper_1910_13908_b200.build` "
            "(nvcc, sm_100a).  sagecal-b200 has no CPU or PyTorch fallback.")
    L = ctypes.CDLL(_LIB_PATH)
    i, d, vp, sz = ctypes.c_int, ctypes.c_double, ctypes.c_void_p, ctypes.c_size_t
    L.sagecal_strerror.restype = ctypes.c_char_p
    L.sagecal_strerror.argtypes = [i]
    L.sagecal_last_cuda_error.restype = i
    L.sagecal_version.restype = ctypes.c_char_p
    L.sagecal_workspace_bytes.restype = sz
    L.sagecal_workspace_bytes.argtypes = [i, i, i, i, i]
    L.sagecal_predict_workspace_bytes.restype = sz
    L.sagecal_predict_workspace_bytes.argtypes = [i, i]
    L.sagecal_predict_coherencies.restype = i
    L.sagecal_predict_coherencies.argtypes = [i, i, i, vp, d, vp, i, vp, vp, vp, vp, vp, vp, vp, vp, i, vp, i, vp, sz, vp]
    L.sagecal_predict_workspace_bytes_station.restype = sz
    L.sagecal_predict_workspace_bytes_station.argtypes = [i, i, i, i, i]
    L.sagecal_predict_set_form.restype = i
    L.sagecal_predict_set_form.argtypes = [i]
    L.sagecal_predict_static_bytes.restype = sz
    L.sagecal_predict_static_bytes.argtypes = []
    L.sagecal_predict_coherencies_static.restype = i
    L.sagecal_predict_coherencies_static.argtypes = [i, i, i, vp, d, vp, i, vp, vp, vp, vp, vp, vp, vp, vp, i, vp, i, vp]
    L.sagecal_predict_residual.restype = i
    L.sagecal_predict_residual.argtypes = [i, i, i, vp, d, vp, i, vp, vp, vp, vp, vp, vp, vp, vp, i, vp, vp, vp, vp, vp, sz, vp]
    L.sagecal_corrupt_subtract.restype = i
    L.sagecal_corrupt_subtract.argtypes = [i, i, i, i, i, vp, vp, vp, d, vp, vp, vp]
    L.sagecal_lm_cost_grad_jtj.restype = i
    L.sagecal_lm_cost_grad_jtj.argtypes = [i, i, i, vp, i, vp, vp, vp, vp, vp, vp, sz, vp]
    L.sagecal_sage_calibrate.restype = i
    L.sagecal_sage_calibrate.argtypes = [i, i, i, i, vp, i, vp, vp, vp, i, i, d, i, vp, vp, vp, sz, vp]
    L.sagecal_calibrate_interval_host.restype = i
    L.sagecal_calibrate_interval_host.argtypes = [i, i, i, vp, d, vp, i, vp, vp, vp, vp, vp, vp, vp, vp, i, vp, vp, vp,
                                                  i, i, d, i, vp, vp, vp]
    L.sagecal_calibrate_interval_host_async.restype = i
    L.sagecal_calibrate_interval_host_async.argtypes = L.sagecal_calibrate_interval_host.argtypes
    L.sagecal_host_sync.restype = i
    L.sagecal_host_sync.argtypes = [vp]
    L.sagecal_host_trim.restype = i
    L.sagecal_host_trim.argtypes = [vp]
    i64 = ctypes.c_int64
    L.sagecal_rows_workspace_bytes.restype = sz
    L.sagecal_rows_workspace_bytes.argtypes = [i, i]
    L.sagecal_rows_to_canonical.restype = i
    L.sagecal_rows_to_canonical.argtypes = [i, i, i, i64, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    L.sagecal_canonical_to_rows.restype = i
    L.sagecal_canonical_to_rows.argtypes = [i, i, i, i64, vp, vp, vp, vp]
    L.sagecal_apply_flags.restype = i
    L.sagecal_apply_flags.argtypes = [i, i, i, i, vp, i, vp, vp, vp]
    L.sagecal_launch_count.restype = ctypes.c_longlong
    L.sagecal_kernel_kinds.restype = i
    L.sagecal_kernel_kind_name.restype = ctypes.c_char_p
    L.sagecal_kernel_kind_name.argtypes = [i]
    L.sagecal_profile_enable.restype = i
    L.sagecal_profile_enable.argtypes = [ctypes.c_uint]
    L.sagecal_profile_read.restype = i
    L.sagecal_profile_read.argtypes = [vp, vp, vp]
    L.sagecal_profile_dfma_peak.restype = i
    L.sagecal_profile_dfma_peak.argtypes = [i, vp, vp, vp]
    L.sagecal_profile_dmma_peak.restype = i
    L.sagecal_profile_dmma_peak.argtypes = [i, vp, vp, vp]
    _lib = L
    return L


def launch_count() -> int:
    """sagecal_launch_count: kernels this process has launched through the library."""
    return int(load_library().sagecal_launch_count())


def kernel_kinds():
    L = load_library()
    return [L.sagecal_kernel_kind_name(k).decode() for k in range(L.sagecal_kernel_kinds())]


def profile_enable(kinds: Sequence[str] = ()) -> None:
    """sagecal_profile_enable: time every launch of the named kernel kinds with CUDA events (empty = off)."""
    names = kernel_kinds()
    mask = 0
    for k in kinds:
        mask |= 1 << names.index(k)
    _check(load_library().sagecal_profile_enable(mask), "sagecal_profile_enable")


def profile_read() -> dict:
    """sagecal_profile_read: {kind: dict(ms, timed, launches)}; waits for the recorded events."""
    L = load_library()
    names = kernel_kinds()
    ms = np.zeros(len(names), np.float64)
    timed = np.zeros(len(names), np.int64)
    launches = np.zeros(len(names), np.int64)
    _check(L.sagecal_profile_read(ms.ctypes.data, timed.ctypes.data, launches.ctypes.data), "sagecal_profile_read")
    return {n: dict(ms=float(ms[k]), timed=int(timed[k]), launches=int(launches[k])) for k, n in enumerate(names)}


def profile_dfma_peak(iters: int = 20000, stream=None) -> dict:
    """sagecal_profile_dfma_peak: the measured FP64 issue peak of the current device, dict(fma_per_s, ms)."""
    v = (ctypes.c_double * 2)()
    _check(load_library().sagecal_profile_dfma_peak(iters, ctypes.addressof(v), ctypes.addressof(v) + 8, _stream(stream)),
           "sagecal_profile_dfma_peak")
    return dict(fma_per_s=float(v[0]), ms=float(v[1]))


def profile_dmma_peak(iters: int = 4000, stream=None) -> dict:
    """sagecal_profile_dmma_peak: the measured FP64 tensor-core (DMMA) peak of the current device, dict(fma_per_s, ms)."""
    v = (ctypes.c_double * 2)()
    _check(load_library().sagecal_profile_dmma_peak(iters, ctypes.addressof(v), ctypes.addressof(v) + 8, _stream(stream)),
           "sagecal_profile_dmma_peak")
    return dict(fma_per_s=float(v[0]), ms=float(v[1]))


def version() -> str:
    return load_library().sagecal_version().decode()


def workspace_bytes(what: int, N: int, T: int, F: int, K: int = 1) -> int:
    return int(load_library().sagecal_workspace_bytes(what, N, T, F, K))


def _check(code: int, where: str):
    if code != 0:
        raise SagecalError(code, where)


def _stream(stream) -> int:
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


def _dev(t: Optional[torch.Tensor], dtype, name: str) -> Optional[int]:
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    return t.data_ptr()


def _workspace(nbytes: int, device) -> torch.Tensor:
    return torch.empty(max(int(nbytes), 256), dtype=torch.uint8, device=device)


def _rows(N: int, T: int) -> int:
    return T * (N * (N - 1) // 2)


def predict_coherencies(N: int, T: int, freqs: Sequence[float], f0: float, uvw: torch.Tensor,
                        cluster_offset: Sequence[int], src_l: torch.Tensor, src_m: torch.Tensor, src_I: torch.Tensor,
                        src_alpha: torch.Tensor, src_Q: Optional[torch.Tensor] = None,
                        src_U: Optional[torch.Tensor] = None, src_V: Optional[torch.Tensor] = None,
                        coh_format: int = COH_FULL, precision: int = 0, out: Optional[torch.Tensor] = None,
                        stream=None) -> torch.Tensor:
    """sagecal_predict_coherencies: coh [K, rows, F, 4] (COH_FULL) or [K, rows, F] (COH_SCALAR), complex128."""
    L = load_library()
    fr = np.ascontiguousarray(freqs, dtype=np.float64)
    co = np.ascontiguousarray(cluster_offset, dtype=np.int32)
    F, K, rows = int(fr.size), int(co.size) - 1, _rows(N, T)
    shape = (K, rows, F, 4) if coh_format == COH_FULL else (K, rows, F)
    if out is None:
        out = torch.empty(shape, dtype=torch.complex128, device=uvw.device)
    elif tuple(out.shape) != shape:
        raise ValueError(f"out: expected shape {shape}")
    if tuple(uvw.shape) != (rows, 3):
        raise ValueError(f"uvw: expected shape {(rows, 3)}")
    S = int(co[-1]) if co.size else 0
    for name, t in (("src_l", src_l), ("src_m", src_m), ("src_I", src_I), ("src_alpha", src_alpha),
                    ("src_Q", src_Q), ("src_U", src_U), ("src_V", src_V)):
        if t is not None and t.numel() != S:
            raise ValueError(f"{name}: expected {S} elements")
    wsb = int(L.sagecal_predict_workspace_bytes_station(N, T, F, K, S) if (src_Q is None and precision == 0)
              else L.sagecal_predict_workspace_bytes(F, S))
    ws = _workspace(wsb, uvw.device)
    f64 = torch.float64
    rc = L.sagecal_predict_coherencies(
        N, T, F, fr.ctypes.data, float(f0), _dev(uvw, f64, "uvw"), K, co.ctypes.data,
        _dev(src_l, f64, "src_l"), _dev(src_m, f64, "src_m"), _dev(src_I, f64, "src_I"),
        _dev(src_Q, f64, "src_Q"), _dev(src_U, f64, "src_U"), _dev(src_V, f64, "src_V"),
        _dev(src_alpha, f64, "src_alpha"), coh_format, _dev(out, torch.complex128, "out"), precision,
        ws.data_ptr(), wsb, _stream(stream))
    _check(rc, "sagecal_predict_coherencies")
    return out


def predict_set_form(form: int) -> None:
    """sagecal_predict_set_form: 0 = station form when the uvw allow it (default), 1 = always per baseline."""
    _check(load_library().sagecal_predict_set_form(int(form)), "sagecal_predict_set_form")


def predict_static_bytes() -> int:
    """sagecal_predict_static_bytes: size of the fixed device scratch of sagecal_predict_coherencies_static."""
    return int(load_library().sagecal_predict_static_bytes())


def predict_coherencies_static(N: int, T: int, freqs: Sequence[float], f0: float, uvw: torch.Tensor,
                               cluster_offset: Sequence[int], src_l: torch.Tensor, src_m: torch.Tensor,
                               src_I: torch.Tensor, src_alpha: torch.Tensor, out: torch.Tensor,
                               src_Q: Optional[torch.Tensor] = None, src_U: Optional[torch.Tensor] = None,
                               src_V: Optional[torch.Tensor] = None, coh_format: int = COH_FULL, precision: int = 0,
                               stream=None) -> torch.Tensor:
    """sagecal_predict_coherencies_static: the prediction with its scratch in a fixed device array of the library; the
    call allocates nothing, so `out` ([K, rows, F, 4] or [K, rows, F], complex128) is the caller's."""
    L = load_library()
    fr = np.ascontiguousarray(freqs, dtype=np.float64)
    co = np.ascontiguousarray(cluster_offset, dtype=np.int32)
    F, K, rows = int(fr.size), int(co.size) - 1, _rows(N, T)
    shape = (K, rows, F, 4) if coh_format == COH_FULL else (K, rows, F)
    if tuple(out.shape) != shape:
        raise ValueError(f"out: expected shape {shape}")
    if tuple(uvw.shape) != (rows, 3):
        raise ValueError(f"uvw: expected shape {(rows, 3)}")
    S = int(co[-1]) if co.size else 0
    for name, t in (("src_l", src_l), ("src_m", src_m), ("src_I", src_I), ("src_alpha", src_alpha),
                    ("src_Q", src_Q), ("src_U", src_U), ("src_V", src_V)):
        if t is not None and t.numel() != S:
            raise ValueError(f"{name}: expected {S} elements")
    f64 = torch.float64
    rc = L.sagecal_predict_coherencies_static(
        N, T, F, fr.ctypes.data, float(f0), _dev(uvw, f64, "uvw"), K, co.ctypes.data,
        _dev(src_l, f64, "src_l"), _dev(src_m, f64, "src_m"), _dev(src_I, f64, "src_I"),
        _dev(src_Q, f64, "src_Q"), _dev(src_U, f64, "src_U"), _dev(src_V, f64, "src_V"),
        _dev(src_alpha, f64, "src_alpha"), coh_format, _dev(out, torch.complex128, "out"), precision, _stream(stream))
    _check(rc, "sagecal_predict_coherencies_static")
    return out


def predict_residual(N: int, T: int, freqs: Sequence[float], f0: float, uvw: torch.Tensor,
                     cluster_offset: Sequence[int], src_l: torch.Tensor, src_m: torch.Tensor, src_I: torch.Tensor,
                     src_alpha: torch.Tensor, jones: torch.Tensor, vis: torch.Tensor,
                     src_Q: Optional[torch.Tensor] = None, src_U: Optional[torch.Tensor] = None,
                     src_V: Optional[torch.Tensor] = None, coh_format: int = COH_FULL,
                     out: Optional[torch.Tensor] = None, residual: Optional[torch.Tensor] = None, stream=None):
    """sagecal_predict_residual: the coherencies of all K clusters AND residual = vis - sum_k J_k C_k J_k^H in one pass.
    Returns (coh, residual)."""
    L = load_library()
    fr = np.ascontiguousarray(freqs, dtype=np.float64)
    co = np.ascontiguousarray(cluster_offset, dtype=np.int32)
    F, K, rows = int(fr.size), int(co.size) - 1, _rows(N, T)
    shape = (K, rows, F, 4) if coh_format == COH_FULL else (K, rows, F)
    c128 = torch.complex128
    if out is None:
        out = torch.empty(shape, dtype=c128, device=uvw.device)
    elif tuple(out.shape) != shape:
        raise ValueError(f"out: expected shape {shape}")
    if tuple(uvw.shape) != (rows, 3):
        raise ValueError(f"uvw: expected shape {(rows, 3)}")
    if vis.numel() != rows * F * 4 or jones.numel() != K * N * 4:
        raise ValueError("vis [rows,F,4] and jones [K,N,2,2] expected")
    if residual is None:
        residual = torch.empty((rows, F, 4), dtype=c128, device=uvw.device)
    elif residual.numel() != rows * F * 4:
        raise ValueError("residual: expected rows*F*4 elements")
    S = int(co[-1]) if co.size else 0
    for name, t in (("src_l", src_l), ("src_m", src_m), ("src_I", src_I), ("src_alpha", src_alpha),
                    ("src_Q", src_Q), ("src_U", src_U), ("src_V", src_V)):
        if t is not None and t.numel() != S:
            raise ValueError(f"{name}: expected {S} elements")
    wsb = int(L.sagecal_predict_workspace_bytes(F, S))
    ws = _workspace(wsb, uvw.device)
    f64 = torch.float64
    rc = L.sagecal_predict_residual(
        N, T, F, fr.ctypes.data, float(f0), _dev(uvw, f64, "uvw"), K, co.ctypes.data,
        _dev(src_l, f64, "src_l"), _dev(src_m, f64, "src_m"), _dev(src_I, f64, "src_I"),
        _dev(src_Q, f64, "src_Q"), _dev(src_U, f64, "src_U"), _dev(src_V, f64, "src_V"),
        _dev(src_alpha, f64, "src_alpha"), coh_format, _dev(out, c128, "out"), _dev(jones, c128, "jones"),
        _dev(vis, c128, "vis"), _dev(residual, c128, "residual"), ws.data_ptr(), wsb, _stream(stream))
    _check(rc, "sagecal_predict_residual")
    return out, residual


def _coh_check(coh: torch.Tensor, coh_format: int, K: int, rows: int, F: int, name="coh"):
    shape = (K, rows, F, 4) if coh_format == COH_FULL else (K, rows, F)
    if tuple(coh.shape) != shape:
        raise ValueError(f"{name}: expected shape {shape}, got {tuple(coh.shape)}")


def corrupt_subtract(N: int, T: int, F: int, coh: torch.Tensor, jones: torch.Tensor,
                     vis_in: Optional[torch.Tensor], sign: float = -1.0, cluster_mask: Optional[Sequence[int]] = None,
                     coh_format: int = COH_FULL, out: Optional[torch.Tensor] = None, stream=None) -> torch.Tensor:
    """sagecal_corrupt_subtract: out = vis_in + sign * sum_k J_p C_k J_q^H.  out may be vis_in (in place)."""
    L = load_library()
    K, rows = int(jones.shape[0]), _rows(N, T)
    c128 = torch.complex128
    if K:
        _coh_check(coh, coh_format, K, rows, F)
    if tuple(jones.shape[:2]) != (K, N) or jones.numel() != K * N * 4:
        raise ValueError("jones: expected shape [K, N, 2, 2]")
    if out is None:
        out = torch.empty((rows, F, 4), dtype=c128, device=jones.device)
    if out.numel() != rows * F * 4 or (vis_in is not None and vis_in.numel() != rows * F * 4):
        raise ValueError("vis: expected rows*F*4 elements")
    mask = None
    if cluster_mask is not None:
        mask = np.ascontiguousarray(cluster_mask, dtype=np.uint8)
        if mask.size != K:
            raise ValueError("cluster_mask: expected K entries")
    rc = L.sagecal_corrupt_subtract(N, T, F, K, coh_format, _dev(coh, c128, "coh") if K else None,
                                    _dev(jones, c128, "jones") if K else None,
                                    mask.ctypes.data if mask is not None else None, float(sign),
                                    _dev(vis_in, c128, "vis_in"), _dev(out, c128, "out"), _stream(stream))
    _check(rc, "sagecal_corrupt_subtract")
    return out


def lm_cost_grad_jtj(N: int, T: int, F: int, x: torch.Tensor, coh_k: torch.Tensor, jones_k: torch.Tensor,
                     coh_format: int = COH_FULL, stream=None):
    """sagecal_lm_cost_grad_jtj: returns (cost [1] f64, grad [N,2,2] c128, jtj [N,2,2] c128) device tensors."""
    L = load_library()
    rows = _rows(N, T)
    c128 = torch.complex128
    if x.numel() != rows * F * 4 or coh_k.numel() != rows * F * (4 if coh_format == COH_FULL else 1):
        raise ValueError("x / coh_k: wrong number of elements")
    if jones_k.numel() != N * 4:
        raise ValueError("jones_k: expected [N, 2, 2]")
    dev = x.device
    cost = torch.empty(1, dtype=torch.float64, device=dev)
    grad = torch.empty((N, 2, 2), dtype=c128, device=dev)
    jtj = torch.empty((N, 2, 2), dtype=c128, device=dev)
    wsb = workspace_bytes(WS_LM_PASS, N, T, F)
    ws = _workspace(wsb, dev)
    rc = L.sagecal_lm_cost_grad_jtj(N, T, F, _dev(x, c128, "x"), coh_format, _dev(coh_k, c128, "coh_k"),
                                    _dev(jones_k, c128, "jones_k"), cost.data_ptr(), grad.data_ptr(), jtj.data_ptr(),
                                    ws.data_ptr(), wsb, _stream(stream))
    _check(rc, "sagecal_lm_cost_grad_jtj")
    return cost, grad, jtj


def sage_calibrate(N: int, T: int, F: int, vis: Optional[torch.Tensor], coh: torch.Tensor, jones: torch.Tensor,
                   n_em: int, n_lm: int, tau: float = 1e-3, coh_format: int = COH_FULL,
                   residual: Optional[torch.Tensor] = None, trace: bool = True, workspace: Optional[torch.Tensor] = None,
                   lm_mode: int = LM_COMPRESSED, stream=None):
    """sagecal_sage_calibrate.  `jones` [K,N,2,2] is updated in place.  vis = None: `residual` (required then) already
    holds the initial residual written by predict_residual.
    Returns dict(jones, residual, cost_per_cluster [K], cost_trace [n_em*K+1] or None), all device tensors."""
    L = load_library()
    K, rows = int(jones.shape[0]), _rows(N, T)
    c128 = torch.complex128
    if K:
        _coh_check(coh, coh_format, K, rows, F)
    if vis is None and residual is None:
        raise ValueError("vis = None needs the residual predict_residual wrote")
    if vis is not None and vis.numel() != rows * F * 4:
        raise ValueError("vis: expected rows*F*4 elements")
    if residual is not None and residual.numel() != rows * F * 4:
        raise ValueError("residual: expected rows*F*4 elements")
    if jones.numel() != K * N * 4:
        raise ValueError("jones: expected [K, N, 2, 2]")
    dev = jones.device if vis is None else vis.device
    if residual is None:
        residual = torch.empty((rows, F, 4), dtype=c128, device=dev)
    cpc = torch.zeros(max(K, 1), dtype=torch.float64, device=dev)
    tr = torch.zeros(n_em * K + 1, dtype=torch.float64, device=dev) if trace else None
    wsb = workspace_bytes(WS_CALIBRATE_FULLGN if lm_mode == LM_FULLGN else WS_CALIBRATE, N, T, F, K)
    ws = workspace if workspace is not None else _workspace(wsb, dev)
    if ws.numel() < wsb:
        raise ValueError("workspace too small")
    rc = L.sagecal_sage_calibrate(N, T, F, K, _dev(vis, c128, "vis"), coh_format,
                                  _dev(coh, c128, "coh") if K else None, _dev(jones, c128, "jones") if K else None,
                                  _dev(residual, c128, "residual"), int(n_em), int(n_lm), float(tau), int(lm_mode),
                                  cpc.data_ptr(), tr.data_ptr() if tr is not None else None,
                                  ws.data_ptr(), ws.numel(), _stream(stream))
    _check(rc, "sagecal_sage_calibrate")
    return dict(jones=jones, residual=residual, cost_per_cluster=cpc[:K], cost_trace=tr)


def rows_to_canonical(N: int, T: int, F: int, ant1: torch.Tensor, ant2: torch.Tensor, tslot: torch.Tensor,
                      uvw_in: torch.Tensor, vis_in: torch.Tensor, flag_in: Optional[torch.Tensor] = None, stream=None):
    """sagecal_rows_to_canonical.  Returns dict(uvw [T*B,3], vis [T*B,F,4], flags [T*B,F] uint8,
    row_map [n] int64, status [4] int32), all device tensors."""
    L = load_library()
    n, rows = int(ant1.numel()), _rows(N, T)
    dev = vis_in.device
    i32, f64, c128, u8 = torch.int32, torch.float64, torch.complex128, torch.uint8
    if ant2.numel() != n or tslot.numel() != n or uvw_in.numel() != 3 * n or vis_in.numel() != n * F * 4:
        raise ValueError("row list: ant1/ant2/tslot [n], uvw_in [n,3], vis_in [n,F,4] expected")
    if flag_in is not None and flag_in.numel() != n * F:
        raise ValueError("flag_in: expected [n, F]")
    uvw = torch.empty((rows, 3), dtype=f64, device=dev)
    vis = torch.empty((rows, F, 4), dtype=c128, device=dev)
    flags = torch.empty((rows, F), dtype=u8, device=dev)
    row_map = torch.empty(max(n, 1), dtype=torch.int64, device=dev)
    status = torch.empty(4, dtype=i32, device=dev)
    wsb = int(L.sagecal_rows_workspace_bytes(N, T))
    ws = _workspace(wsb, dev)
    rc = L.sagecal_rows_to_canonical(N, T, F, n, _dev(ant1, i32, "ant1"), _dev(ant2, i32, "ant2"),
                                     _dev(tslot, i32, "tslot"), _dev(uvw_in, f64, "uvw_in"),
                                     _dev(vis_in, c128, "vis_in"), _dev(flag_in, u8, "flag_in"), uvw.data_ptr(),
                                     vis.data_ptr(), flags.data_ptr(), row_map.data_ptr(), status.data_ptr(),
                                     ws.data_ptr(), wsb, _stream(stream))
    _check(rc, "sagecal_rows_to_canonical")
    return dict(uvw=uvw, vis=vis, flags=flags, row_map=row_map[:n], status=status)


def canonical_to_rows(N: int, T: int, F: int, row_map: torch.Tensor, vis_canonical: torch.Tensor,
                      out: torch.Tensor, stream=None) -> torch.Tensor:
    """sagecal_canonical_to_rows: out[r] = the canonical slot of row r (Hermitian-transposed back for swapped rows);
    rows with row_map < 0 are left untouched."""
    L = load_library()
    n = int(row_map.numel())
    if vis_canonical.numel() != _rows(N, T) * F * 4 or out.numel() != n * F * 4:
        raise ValueError("vis_canonical [T*B,F,4] / out [n,F,4] expected")
    rc = L.sagecal_canonical_to_rows(N, T, F, n, _dev(row_map, torch.int64, "row_map"),
                                     _dev(vis_canonical, torch.complex128, "vis_canonical"),
                                     _dev(out, torch.complex128, "out"), _stream(stream))
    _check(rc, "sagecal_canonical_to_rows")
    return out


def apply_flags(N: int, T: int, F: int, flags: torch.Tensor, coh: Optional[torch.Tensor], vis: Optional[torch.Tensor],
                coh_format: int = COH_FULL, stream=None) -> None:
    """sagecal_apply_flags: zero the flagged samples of coh [K, ...] (all clusters) and of vis, in place."""
    L = load_library()
    rows = _rows(N, T)
    K = 0 if coh is None else int(coh.shape[0])
    if flags.numel() != rows * F:
        raise ValueError("flags: expected [T*B, F]")
    if K:
        _coh_check(coh, coh_format, K, rows, F)
    if vis is not None and vis.numel() != rows * F * 4:
        raise ValueError("vis: expected rows*F*4 elements")
    rc = L.sagecal_apply_flags(N, T, F, K, _dev(flags, torch.uint8, "flags"), coh_format,
                               _dev(coh, torch.complex128, "coh") if K else None,
                               _dev(vis, torch.complex128, "vis"), _stream(stream))
    _check(rc, "sagecal_apply_flags")


def _host(a, dtype, name):
    if a is None:
        return None, None
    if isinstance(a, torch.Tensor):
        if a.is_cuda or a.dtype != dtype or not a.is_contiguous():
            raise TypeError(f"{name}: expected a contiguous CPU tensor of dtype {dtype}")
        return a.data_ptr(), a
    raise TypeError(f"{name}: expected a CPU torch tensor (pinned memory recommended)")


def calibrate_interval_host(N: int, T: int, freqs: Sequence[float], f0: float, uvw: torch.Tensor,
                            cluster_offset: Sequence[int], src_l, src_m, src_I, src_alpha, vis: torch.Tensor,
                            jones: torch.Tensor, n_em: int, n_lm: int, tau: float = 1e-3, src_Q=None, src_U=None,
                            src_V=None, coh_format: int = COH_FULL, residual: Optional[torch.Tensor] = None,
                            cost_per_cluster: Optional[torch.Tensor] = None, lm_mode: int = LM_COMPRESSED, stream=None,
                            asynchronous: bool = False):
    """sagecal_calibrate_interval_host: predict + calibrate from HOST tensors (copies inside the call).
    `jones` (CPU, [K,N,2,2]) is updated in place; `residual` (CPU) is filled if given.
    asynchronous=True: sagecal_calibrate_interval_host_async -- returns once enqueued; every host tensor of the call
    (inputs and outputs) must stay alive and untouched until host_sync() (at most two intervals in flight)."""
    L = load_library()
    fr = np.ascontiguousarray(freqs, dtype=np.float64)
    co = np.ascontiguousarray(cluster_offset, dtype=np.int32)
    F, K = int(fr.size), int(co.size) - 1
    f64, c128 = torch.float64, torch.complex128
    if cost_per_cluster is None:
        cost_per_cluster = torch.zeros(K, dtype=f64)
    ptrs = [_host(t, f64, n)[0] for n, t in (("src_l", src_l), ("src_m", src_m), ("src_I", src_I), ("src_Q", src_Q),
                                            ("src_U", src_U), ("src_V", src_V), ("src_alpha", src_alpha))]
    fn = L.sagecal_calibrate_interval_host_async if asynchronous else L.sagecal_calibrate_interval_host
    rc = fn(
        N, T, F, fr.ctypes.data, float(f0), _host(uvw, f64, "uvw")[0], K, co.ctypes.data, *ptrs, coh_format,
        _host(vis, c128, "vis")[0], _host(jones, c128, "jones")[0], _host(residual, c128, "residual")[0],
        int(n_em), int(n_lm), float(tau), int(lm_mode), _host(cost_per_cluster, f64, "cost_per_cluster")[0], None,
        _stream(stream))
    _check(rc, "sagecal_calibrate_interval_host")
    return dict(jones=jones, residual=residual, cost_per_cluster=cost_per_cluster)


def host_trim(stream=None) -> None:
    """sagecal_host_trim: host_sync, then the arenas cached by the host entries go back to the device."""
    _check(load_library().sagecal_host_trim(_stream(stream)), "sagecal_host_trim")


def host_sync(stream=None) -> None:
    """sagecal_host_sync: waits for every interval the asynchronous host entry enqueued from this thread."""
    _check(load_library().sagecal_host_sync(_stream(stream)), "sagecal_host_sync")
