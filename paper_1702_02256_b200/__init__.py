"""paper_1702_02256_b200 -- B200-native SPIIR filtering (arXiv:1702.02256) behind a C ABI.

Thin Python binding of ``libspiir.so`` (see ``include/spiir.h``): argument marshalling only,
every step of the hot path runs in the CUDA kernels under ``csrc/``.  PyTorch supplies device
memory and streams.  There is no CPU fallback: if the library has not been built
(``python -m paper_1702_02256_b200.build``) every entry point raises.

Function names mirror the C ABI: ``spiir_plan_create`` / ``spiir_filter`` /
``spiir_resample_down`` / ``spiir_resample_up`` / ``spiir_mr_plan_create`` / ``spiir_mr_filter``.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libspiir.so")
_lib = None

SPIIR_OK, SPIIR_EINVAL, SPIIR_ENOMEM, SPIIR_ECUDA, SPIIR_EUNSUPPORTED, SPIIR_ESTATE = range(6)
SPIIR_DOWN2, SPIIR_UP2 = 0, 1

EXPORTS = (
    "spiir_plan_create", "spiir_filter", "spiir_plan_reset", "spiir_plan_destroy", "spiir_plan_launch_info",
    "spiir_plan_get_state", "spiir_plan_set_state", "spiir_kaiser_taps", "spiir_resamp_create",
    "spiir_resample_down", "spiir_resample_up", "spiir_resamp_reset", "spiir_resamp_destroy",
    "spiir_mr_plan_create", "spiir_mr_filter", "spiir_mr_plan_reset", "spiir_mr_plan_destroy",
    "spiir_mr_launches", "spiir_probe_fp32_peak", "spiir_host_layout", "spiir_host_geometry", "spiir_last_error", "spiir_version",
)


class SpiirError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        msg = lib().spiir_last_error().decode(errors="replace")
        super().__init__(f"{where} failed with status {status}: {msg}")


class _PlanOpts(ctypes.Structure):
    _fields_ = [("n_streams", ctypes.c_int), ("max_block", ctypes.c_int), ("time_chunks", ctypes.c_int),
                ("flags", ctypes.c_int)]


class _MrOpts(ctypes.Structure):
    _fields_ = [("n_streams", ctypes.c_int), ("max_block", ctypes.c_int), ("n_taps", ctypes.c_int),
                ("kaiser_beta", ctypes.c_double), ("cutoff", ctypes.c_double)]


def lib():
    """The loaded C-ABI library.  Raises if it has not been built: no fallback exists."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1702_02256_b200.build` "
                               "(there is no CPU or PyTorch fallback for the SPIIR hot path)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
        pvp = ctypes.POINTER(vp)
        L.spiir_plan_create.argtypes = [pvp, vp, vp, vp, ci, ci, ci, ctypes.POINTER(_PlanOpts)]
        L.spiir_filter.argtypes = [vp, vp, ci, vp, vp]
        L.spiir_plan_reset.argtypes = [vp, vp]
        L.spiir_plan_destroy.argtypes = [vp]
        L.spiir_plan_destroy.restype = None
        L.spiir_plan_launch_info.argtypes = [vp, ci, ctypes.POINTER(ci * 8)]
        L.spiir_plan_get_state.argtypes = [vp, vp, vp]
        L.spiir_plan_set_state.argtypes = [vp, vp, vp]
        L.spiir_kaiser_taps.argtypes = [ci, cd, cd, vp]
        L.spiir_resamp_create.argtypes = [pvp, ci, ci, cd, cd, ci, ci]
        L.spiir_resample_down.argtypes = [vp, vp, ci, vp, vp]
        L.spiir_resample_up.argtypes = [vp, vp, ci, vp, ci, vp]
        L.spiir_resamp_reset.argtypes = [vp, vp]
        L.spiir_resamp_destroy.argtypes = [vp]
        L.spiir_resamp_destroy.restype = None
        L.spiir_mr_plan_create.argtypes = [pvp, ci, ctypes.POINTER(ci), pvp, pvp, pvp, ctypes.POINTER(ci), ci,
                                           ctypes.POINTER(_MrOpts)]
        L.spiir_mr_filter.argtypes = [vp, vp, ci, vp, vp]
        L.spiir_mr_plan_reset.argtypes = [vp, vp]
        L.spiir_mr_plan_destroy.argtypes = [vp]
        L.spiir_mr_plan_destroy.restype = None
        L.spiir_mr_launches.argtypes = [vp, ci]
        L.spiir_probe_fp32_peak.argtypes = [ctypes.POINTER(cd)]
        L.spiir_host_layout.argtypes = [vp, vp, vp, ci, ci, ci, vp, vp, vp, ctypes.POINTER(ci * 4),
                                        ctypes.POINTER(cd)]
        L.spiir_host_geometry.argtypes = [ci, ci, ci, ci, ci, ci, ci, ci, ctypes.POINTER(ci * 8)]
        L.spiir_last_error.restype = ctypes.c_char_p
        L.spiir_version.restype = ctypes.c_char_p
        _lib = L
    return _lib


def _check(status: int, where: str) -> None:
    if status != SPIIR_OK:
        raise SpiirError(status, where)


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream)


def _bank_arrays(a1, b0, delays):
    a1 = np.ascontiguousarray(a1, dtype=np.complex64)
    b0 = np.ascontiguousarray(b0, dtype=np.complex64)
    d = np.ascontiguousarray(delays, dtype=np.int32)
    if a1.ndim != 2 or a1.shape != b0.shape or a1.shape != d.shape:
        raise ValueError("a1, b0, delays must all be [n_templates][n_filters]")
    return a1, b0, d


def version() -> str:
    return lib().spiir_version().decode()


def spiir_probe_fp32_peak() -> float:
    """TFLOP/s reached by a register-only FFMA loop on the current device (measurement aid)."""
    v = ctypes.c_double(0.0)
    _check(lib().spiir_probe_fp32_peak(ctypes.byref(v)), "spiir_probe_fp32_peak")
    return float(v.value)


def spiir_kaiser_taps(n_taps: int = 192, kaiser_beta: float = 5.0, cutoff: float = 0.25) -> np.ndarray:
    out = np.empty(n_taps, dtype=np.float32)
    _check(lib().spiir_kaiser_taps(n_taps, kaiser_beta, cutoff, out.ctypes.data), "spiir_kaiser_taps")
    return out


def spiir_host_layout(a1, b0, delays, avoid_conflicts: bool = True):
    """Host-only: the plan's filter permutation.  Returns dict(pos, coef, dly, F, LPT, G, conflict_degree)."""
    a1, b0, d = _bank_arrays(a1, b0, delays)
    T, Lf = a1.shape
    info = (ctypes.c_int * 4)()
    deg = ctypes.c_double()
    _check(lib().spiir_host_layout(a1.ctypes.data, b0.ctypes.data, d.ctypes.data, T, Lf, int(avoid_conflicts),
                                   None, None, None, ctypes.byref(info), ctypes.byref(deg)), "spiir_host_layout")
    nf = info[3]
    pos = np.empty(T * Lf, dtype=np.int32)
    coef = np.empty(nf * 4, dtype=np.float32)
    dly = np.empty(nf, dtype=np.int32)
    _check(lib().spiir_host_layout(a1.ctypes.data, b0.ctypes.data, d.ctypes.data, T, Lf, int(avoid_conflicts),
                                   pos.ctypes.data, coef.ctypes.data, dly.ctypes.data, ctypes.byref(info),
                                   ctypes.byref(deg)), "spiir_host_layout")
    return dict(pos=pos.reshape(T, Lf), coef=coef.reshape(-1, 4), dly=dly, F=info[0], LPT=info[1], G=info[2],
                conflict_degree=deg.value)


_INFO_KEYS = ("F", "lanes_per_template", "warps_per_cta", "grid", "time_chunks", "smem_bytes", "time_tile", "launches")


def spiir_host_geometry(n_templates, n_filters, n_streams, max_delay, n, time_chunks=0, n_sm=148,
                        smem_optin=232448):
    info = (ctypes.c_int * 8)()
    _check(lib().spiir_host_geometry(n_templates, n_filters, n_streams, max_delay, n, time_chunks, n_sm, smem_optin,
                                     ctypes.byref(info)), "spiir_host_geometry")
    return dict(zip(_INFO_KEYS, list(info)))


class Plan:
    """Single-rate SPIIR bank with carried state (spiir_plan_create / spiir_filter)."""

    def __init__(self, a1, b0, delays, rate_hz: int = 4096, n_streams: int = 1, max_block: int = 4096,
                 time_chunks: int = 0, flags: int = 0):
        a1, b0, d = _bank_arrays(a1, b0, delays)
        self.T, self.L = a1.shape
        self.S, self.max_block, self.rate_hz = int(n_streams), int(max_block), int(rate_hz)
        opts = _PlanOpts(self.S, self.max_block, int(time_chunks), int(flags))
        self._h = ctypes.c_void_p()
        _check(lib().spiir_plan_create(ctypes.byref(self._h), a1.ctypes.data, b0.ctypes.data, d.ctypes.data,
                                       self.T, self.L, self.rate_hz, ctypes.byref(opts)), "spiir_plan_create")

    def filter(self, x, out=None, stream=None):
        """x: CUDA float32 [n] or [S][n]; returns (or fills) CUDA complex64 [S][T][n]."""
        import torch
        if not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
            raise ValueError("x must be a contiguous CUDA float32 tensor")
        if x.dim() == 1:
            x = x[None, :]
        if x.shape[0] != self.S:
            raise ValueError("x must be [S][n]")
        n = int(x.shape[1])
        if out is None:
            out = torch.empty((self.S, self.T, n), dtype=torch.complex64, device=x.device)
        elif not (out.is_cuda and out.dtype == torch.complex64 and out.is_contiguous()
                  and out.numel() == self.S * self.T * n):
            raise ValueError("out must be a contiguous CUDA complex64 tensor of S*T*n elements")
        _check(lib().spiir_filter(self._h, x.data_ptr(), n, out.data_ptr(), _stream_ptr(stream)), "spiir_filter")
        return out

    def reset(self, stream=None) -> None:
        _check(lib().spiir_plan_reset(self._h, _stream_ptr(stream)), "spiir_plan_reset")

    def launch_info(self, n: int) -> dict:
        info = (ctypes.c_int * 8)()
        _check(lib().spiir_plan_launch_info(self._h, int(n), ctypes.byref(info)), "spiir_plan_launch_info")
        return dict(zip(_INFO_KEYS, list(info)))

    def get_state(self, stream=None):
        import torch
        y = torch.empty((self.S, self.T, self.L), dtype=torch.complex64, device="cuda")
        _check(lib().spiir_plan_get_state(self._h, y.data_ptr(), _stream_ptr(stream)), "spiir_plan_get_state")
        return y

    def set_state(self, y, stream=None) -> None:
        import torch
        if not (y.is_cuda and y.dtype == torch.complex64 and y.is_contiguous()
                and tuple(y.shape) == (self.S, self.T, self.L)):
            raise ValueError("y must be a contiguous CUDA complex64 [S][T][L] tensor")
        _check(lib().spiir_plan_set_state(self._h, y.data_ptr(), _stream_ptr(stream)), "spiir_plan_set_state")

    def close(self) -> None:
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Resampler:
    """One streaming x2 stage (spiir_resamp_create / spiir_resample_down / spiir_resample_up)."""

    def __init__(self, direction: str, n_rows: int, max_block: int, n_taps: int = 192, kaiser_beta: float = 5.0,
                 cutoff: float = 0.25):
        self.direction, self.rows, self.max_block = direction, int(n_rows), int(max_block)
        self._h = ctypes.c_void_p()
        _check(lib().spiir_resamp_create(ctypes.byref(self._h), {"down": SPIIR_DOWN2, "up": SPIIR_UP2}[direction],
                                         n_taps, kaiser_beta, cutoff, self.rows, self.max_block), "spiir_resamp_create")

    def down(self, u, out=None, stream=None):
        import torch
        if not (u.is_cuda and u.dtype == torch.float32 and u.is_contiguous()):
            raise ValueError("u must be a contiguous CUDA float32 tensor")
        if u.dim() == 1:
            u = u[None, :]
        n_in = int(u.shape[1])
        if out is None:
            out = torch.empty((self.rows, n_in // 2), dtype=torch.float32, device=u.device)
        _check(lib().spiir_resample_down(self._h, u.data_ptr(), n_in, out.data_ptr(), _stream_ptr(stream)),
               "spiir_resample_down")
        return out

    def up(self, v, out=None, accumulate: bool = False, stream=None):
        import torch
        if not (v.is_cuda and v.dtype == torch.complex64 and v.is_contiguous()):
            raise ValueError("v must be a contiguous CUDA complex64 tensor")
        if v.dim() == 1:
            v = v[None, :]
        n_in = int(v.shape[1])
        if out is None:
            if accumulate:
                raise ValueError("accumulate needs an output tensor")
            out = torch.empty((self.rows, 2 * n_in), dtype=torch.complex64, device=v.device)
        _check(lib().spiir_resample_up(self._h, v.data_ptr(), n_in, out.data_ptr(), int(bool(accumulate)),
                                       _stream_ptr(stream)), "spiir_resample_up")
        return out

    def reset(self, stream=None) -> None:
        _check(lib().spiir_resamp_reset(self._h, _stream_ptr(stream)), "spiir_resamp_reset")

    def close(self) -> None:
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_resamp_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class MultiratePlan:
    """Multirate SPIIR (spiir_mr_plan_create / spiir_mr_filter).  banks: highest rate first, each
    (a1, b0, delays) of shape [T][L_h]; rates_hz descending, each half of the previous."""

    def __init__(self, banks: Sequence, rates_hz: Sequence[int], n_streams: int = 1, max_block: Optional[int] = None,
                 n_taps: int = 192, kaiser_beta: float = 5.0, cutoff: float = 0.25):
        arrs = [_bank_arrays(*b) for b in banks]
        H = len(arrs)
        self.H, self.T, self.S = H, arrs[0][0].shape[0], int(n_streams)
        self.max_block = int(max_block if max_block is not None else rates_hz[0])
        vp = ctypes.c_void_p
        a1p = (vp * H)(*[a[0].ctypes.data for a in arrs])
        b0p = (vp * H)(*[a[1].ctypes.data for a in arrs])
        dp = (vp * H)(*[a[2].ctypes.data for a in arrs])
        nf = (ctypes.c_int * H)(*[a[0].shape[1] for a in arrs])
        rates = (ctypes.c_int * H)(*[int(r) for r in rates_hz])
        opts = _MrOpts(self.S, self.max_block, n_taps, kaiser_beta, cutoff)
        self._h = ctypes.c_void_p()
        _check(lib().spiir_mr_plan_create(ctypes.byref(self._h), H, rates, a1p, b0p, dp, nf, self.T,
                                          ctypes.byref(opts)), "spiir_mr_plan_create")

    def filter(self, x, out=None, stream=None):
        import torch
        if not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
            raise ValueError("x must be a contiguous CUDA float32 tensor")
        if x.dim() == 1:
            x = x[None, :]
        n = int(x.shape[1])
        if out is None:
            out = torch.empty((self.S, self.T, n), dtype=torch.complex64, device=x.device)
        _check(lib().spiir_mr_filter(self._h, x.data_ptr(), n, out.data_ptr(), _stream_ptr(stream)), "spiir_mr_filter")
        return out

    def launches(self, n: int) -> int:
        return int(lib().spiir_mr_launches(self._h, int(n)))

    def reset(self, stream=None) -> None:
        _check(lib().spiir_mr_plan_reset(self._h, _stream_ptr(stream)), "spiir_mr_plan_reset")

    def close(self) -> None:
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_mr_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
