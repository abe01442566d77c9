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
SPIIR_NOALLOC_SCRATCH_BYTES = 4 << 20

EXPORTS = (
    "spiir_plan_workspace_bytes", "spiir_plan_create", "spiir_plan_workspace_bytes_ragged", "spiir_plan_create_ragged",
    "spiir_filter", "spiir_plan_reset", "spiir_plan_destroy", "spiir_plan_launch_info",
    "spiir_plan_history_len", "spiir_plan_get_state", "spiir_plan_set_state", "spiir_kaiser_taps",
    "spiir_resamp_workspace_bytes", "spiir_resamp_create", "spiir_resample_down", "spiir_resample_up", "spiir_resamp_reset",
    "spiir_resamp_destroy", "spiir_resamp_history_len", "spiir_resamp_get_state", "spiir_resamp_set_state",
    "spiir_mr_workspace_bytes", "spiir_mr_plan_create", "spiir_mr_filter", "spiir_mr_plan_reset", "spiir_mr_plan_destroy",
    "spiir_mr_launches", "spiir_mr_plan_state_bytes", "spiir_mr_plan_get_state", "spiir_mr_plan_set_state",
    "spiir_assign_rates", "spiir_host_layout", "spiir_host_geometry", "spiir_host_lane_mapping",
    "spiir_pd_plan_create", "spiir_pd_filter", "spiir_pd_plan_reset", "spiir_pd_plan_destroy",
    "spiir_noalloc_scratch_need", "spiir_noalloc_setup", "spiir_filter_block_noalloc",
    "spiir_probe_fp32_peak", "spiir_probe_ffma2_operands", "spiir_last_error", "spiir_version",
)


class SpiirError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = int(status)
        msg = lib().spiir_last_error().decode(errors="replace")
        super().__init__(f"{where} failed with status {status}: {msg}")


class _PlanOpts(ctypes.Structure):
    _fields_ = [("n_streams", ctypes.c_int), ("max_block", ctypes.c_int), ("time_chunks", ctypes.c_int),
                ("flags", ctypes.c_int), ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t)]


class _ResampOpts(ctypes.Structure):
    _fields_ = [("max_block", ctypes.c_int), ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t),
                ("flags", ctypes.c_int)]


class _MrOpts(ctypes.Structure):
    _fields_ = [("n_streams", ctypes.c_int), ("max_block", ctypes.c_int),
                ("n_taps_down", ctypes.c_int), ("kaiser_beta_down", ctypes.c_double), ("cutoff_down", ctypes.c_double),
                ("n_taps_up", ctypes.c_int), ("kaiser_beta_up", ctypes.c_double), ("cutoff_up", ctypes.c_double),
                ("workspace", ctypes.c_void_p), ("workspace_bytes", ctypes.c_size_t)]


def lib():
    """The loaded C-ABI library.  Raises if it has not been built: no fallback exists."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise RuntimeError(f"{LIB_PATH} is missing: build it with `python -m paper_1702_02256_b200.build` "
                               "(there is no CPU or PyTorch fallback for the SPIIR hot path)")
        L = ctypes.CDLL(LIB_PATH)
        vp, ci, cd, sz = ctypes.c_void_p, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
        pvp = ctypes.POINTER(vp)
        L.spiir_plan_workspace_bytes.argtypes = [ci, ci, ci, ci, ci, ci]
        L.spiir_plan_workspace_bytes.restype = sz
        L.spiir_plan_workspace_bytes_ragged.argtypes = [vp, ci, ci, ci, ci, ci]
        L.spiir_plan_workspace_bytes_ragged.restype = sz
        L.spiir_plan_create.argtypes = [pvp, vp, vp, vp, ci, ci, ci, ctypes.POINTER(_PlanOpts)]
        L.spiir_plan_create_ragged.argtypes = [pvp, vp, vp, vp, vp, ci, ci, ctypes.POINTER(_PlanOpts)]
        L.spiir_filter.argtypes = [vp, vp, ci, vp, vp]
        L.spiir_plan_reset.argtypes = [vp, vp]
        L.spiir_plan_destroy.argtypes = [vp]
        L.spiir_plan_destroy.restype = None
        L.spiir_plan_launch_info.argtypes = [vp, ci, ctypes.POINTER(ci * 8)]
        L.spiir_plan_history_len.argtypes = [vp]
        L.spiir_plan_get_state.argtypes = [vp, vp, vp, vp]
        L.spiir_plan_set_state.argtypes = [vp, vp, vp, vp]
        L.spiir_kaiser_taps.argtypes = [ci, cd, cd, vp]
        L.spiir_resamp_workspace_bytes.argtypes = [ci, ci, ci]
        L.spiir_resamp_workspace_bytes.restype = sz
        L.spiir_resamp_create.argtypes = [pvp, ci, ci, cd, cd, ci, ctypes.POINTER(_ResampOpts)]
        L.spiir_resample_down.argtypes = [vp, vp, ci, vp, vp]
        L.spiir_resample_up.argtypes = [vp, vp, ci, vp, ci, vp]
        L.spiir_resamp_reset.argtypes = [vp, vp]
        L.spiir_resamp_destroy.argtypes = [vp]
        L.spiir_resamp_destroy.restype = None
        L.spiir_resamp_history_len.argtypes = [vp]
        L.spiir_resamp_get_state.argtypes = [vp, vp, vp]
        L.spiir_resamp_set_state.argtypes = [vp, vp, vp]
        L.spiir_mr_workspace_bytes.argtypes = [ci, ctypes.POINTER(ci), ctypes.POINTER(ci), ci, ctypes.POINTER(_MrOpts)]
        L.spiir_mr_workspace_bytes.restype = sz
        L.spiir_mr_plan_create.argtypes = [pvp, ci, ctypes.POINTER(ci), pvp, pvp, pvp, ctypes.POINTER(ci), ci,
                                           ctypes.POINTER(_MrOpts)]
        L.spiir_mr_filter.argtypes = [vp, vp, ci, vp, vp]
        L.spiir_mr_plan_reset.argtypes = [vp, vp]
        L.spiir_mr_plan_destroy.argtypes = [vp]
        L.spiir_mr_plan_destroy.restype = None
        L.spiir_mr_launches.argtypes = [vp, ci]
        L.spiir_mr_plan_state_bytes.argtypes = [vp]
        L.spiir_mr_plan_state_bytes.restype = sz
        L.spiir_mr_plan_get_state.argtypes = [vp, vp, vp]
        L.spiir_mr_plan_set_state.argtypes = [vp, vp, vp]
        L.spiir_assign_rates.argtypes = [vp, ci, ci, ctypes.POINTER(ci), ci, cd, vp]
        L.spiir_pd_plan_create.argtypes = [pvp, vp, vp, vp, ci, ci, ci]
        L.spiir_pd_filter.argtypes = [vp, vp, ci, vp, vp]
        L.spiir_pd_plan_reset.argtypes = [vp, vp]
        L.spiir_pd_plan_destroy.argtypes = [vp]
        L.spiir_pd_plan_destroy.restype = None
        L.spiir_noalloc_scratch_need.argtypes = [ci, ci, ci, ci]
        L.spiir_noalloc_scratch_need.restype = sz
        L.spiir_noalloc_setup.argtypes = []
        L.spiir_filter_block_noalloc.argtypes = [vp, vp, vp, ci, ci, vp, ci, ci, vp, vp]
        L.spiir_probe_fp32_peak.argtypes = [ctypes.POINTER(cd)]
        L.spiir_probe_ffma2_operands.argtypes = [ctypes.POINTER(cd * 4)]
        L.spiir_host_layout.argtypes = [vp, vp, vp, ci, ci, ci, vp, vp, vp, ctypes.POINTER(ci * 4),
                                        ctypes.POINTER(cd)]
        L.spiir_host_geometry.argtypes = [ci, ci, ci, ci, ci, ci, ci, ci, ctypes.POINTER(ci * 8)]
        L.spiir_host_lane_mapping.argtypes = [ci, ci, ctypes.POINTER(ci * 3)]
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


def spiir_probe_ffma2_operands() -> dict:
    """Cycles per packed FFMA2 warp-instruction when it reads 3 / 4 / 5 / 6 distinct register words (measurement aid)."""
    v = (ctypes.c_double * 4)()
    _check(lib().spiir_probe_ffma2_operands(ctypes.byref(v)), "spiir_probe_ffma2_operands")
    return {"words3": v[0], "words4": v[1], "words5": v[2], "words6": v[3]}


def spiir_kaiser_taps(n_taps: int = 192, kaiser_beta: float = 5.0, cutoff: float = 0.25) -> np.ndarray:
    out = np.empty(n_taps, dtype=np.float32)
    _check(lib().spiir_kaiser_taps(n_taps, kaiser_beta, cutoff, out.ctypes.data), "spiir_kaiser_taps")
    return out


def spiir_assign_rates(a1, base_rate_hz: int, rates_hz: Sequence[int], band_factor: float = 1.0) -> np.ndarray:
    """Rate index of every filter from its a1 (reading R8).  Host only."""
    a1 = np.ascontiguousarray(a1, dtype=np.complex64)
    rates = (ctypes.c_int * len(rates_hz))(*[int(r) for r in rates_hz])
    out = np.empty(a1.size, dtype=np.int32)
    _check(lib().spiir_assign_rates(a1.ctypes.data, a1.size, int(base_rate_hz), rates, len(rates_hz), float(band_factor),
                                    out.ctypes.data), "spiir_assign_rates")
    return out.reshape(a1.shape)


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


def spiir_host_lane_mapping(n_filters: int, n_templates: int = 1) -> dict:
    info = (ctypes.c_int * 3)()
    _check(lib().spiir_host_lane_mapping(int(n_filters), int(n_templates), ctypes.byref(info)), "spiir_host_lane_mapping")
    return {"F": info[0], "lanes_per_template": info[1], "warps_per_template": info[2]}


def _workspace(nbytes: int, device=None):
    """One torch tensor that the plan borrows for its lifetime: every device byte of a plan comes from PyTorch."""
    import torch
    if nbytes <= 0:
        raise SpiirError(SPIIR_EUNSUPPORTED, "workspace size query")
    return torch.empty(int(nbytes), dtype=torch.uint8, device=device or "cuda")


def _need(t, dtype, numel, what):
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.numel() == numel):
        raise ValueError(f"{what} must be a contiguous CUDA {dtype} tensor of {numel} elements")


class Plan:
    """Single-rate SPIIR bank with carried state (spiir_plan_create / spiir_filter).

    Uniform bank: ``Plan(a1, b0, delays)`` with [T][L] arrays.  Ragged bank (spiir_plan_create_ragged):
    ``Plan.ragged(a1_flat, b0_flat, delays_flat, filter_offsets)``.  The device workspace is a torch tensor."""

    def __init__(self, a1, b0, delays, rate_hz: int = 4096, n_streams: int = 1, max_block: int = 4096,
                 time_chunks: int = 0, flags: int = 0, _offsets=None):
        import torch
        self.S, self.max_block, self.rate_hz = int(n_streams), int(max_block), int(rate_hz)
        self.device = torch.device("cuda", torch.cuda.current_device()) if torch.cuda.is_available() else None
        self._h = ctypes.c_void_p()
        if _offsets is None:
            a1, b0, d = _bank_arrays(a1, b0, delays)
            self.T, self.L = a1.shape
            self.n_filters_total = self.T * self.L
            need = lib().spiir_plan_workspace_bytes(self.T, self.L, int(d.max(initial=0)), self.S, self.max_block, int(time_chunks))
            self._ws = _workspace(need) if need else None
            opts = _PlanOpts(self.S, self.max_block, int(time_chunks), int(flags),
                             self._ws.data_ptr() if self._ws is not None else None, need)
            _check(lib().spiir_plan_create(ctypes.byref(self._h), a1.ctypes.data, b0.ctypes.data, d.ctypes.data,
                                           self.T, self.L, self.rate_hz, ctypes.byref(opts)), "spiir_plan_create")
        else:
            a1 = np.ascontiguousarray(a1, dtype=np.complex64).ravel()
            b0 = np.ascontiguousarray(b0, dtype=np.complex64).ravel()
            d = np.ascontiguousarray(delays, dtype=np.int32).ravel()
            off = np.ascontiguousarray(_offsets, dtype=np.int32)
            if off.ndim != 1 or off.size < 2 or a1.size != off[-1] or b0.size != a1.size or d.size != a1.size:
                raise ValueError("ragged bank: flat arrays must have filter_offsets[-1] entries")
            self.T, self.L = off.size - 1, None
            self.n_filters_total = int(off[-1])
            need = lib().spiir_plan_workspace_bytes_ragged(off.ctypes.data, self.T, int(d.max(initial=0)), self.S, self.max_block,
                                                           int(time_chunks))
            self._ws = _workspace(need) if need else None
            opts = _PlanOpts(self.S, self.max_block, int(time_chunks), int(flags),
                             self._ws.data_ptr() if self._ws is not None else None, need)
            _check(lib().spiir_plan_create_ragged(ctypes.byref(self._h), a1.ctypes.data, b0.ctypes.data, d.ctypes.data,
                                                  off.ctypes.data, self.T, self.rate_hz, ctypes.byref(opts)),
                   "spiir_plan_create_ragged")
        self.history_len = int(lib().spiir_plan_history_len(self._h))

    @classmethod
    def ragged(cls, a1_flat, b0_flat, delays_flat, filter_offsets, **kw):
        return cls(a1_flat, b0_flat, delays_flat, _offsets=filter_offsets, **kw)

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
        else:
            _need(out, torch.complex64, self.S * self.T * n, "out")
        _check(lib().spiir_filter(self._h, x.data_ptr(), n, out.data_ptr(), _stream_ptr(stream)), "spiir_filter")
        return out

    def reset(self, stream=None) -> None:
        _check(lib().spiir_plan_reset(self._h, _stream_ptr(stream)), "spiir_plan_reset")

    def launch_info(self, n: int) -> dict:
        info = (ctypes.c_int * 8)()
        _check(lib().spiir_plan_launch_info(self._h, int(n), ctypes.byref(info)), "spiir_plan_launch_info")
        return dict(zip(_INFO_KEYS, list(info)))

    def get_state(self, stream=None):
        """(y, hist): filter state complex64 [S][T][L] (ragged: [S][total filters]) and the last history_len inputs."""
        import torch
        shape = (self.S, self.T, self.L) if self.L is not None else (self.S, self.n_filters_total)
        y = torch.empty(shape, dtype=torch.complex64, device=self.device)
        hist = torch.empty((self.S, self.history_len), dtype=torch.float32, device=self.device)
        _check(lib().spiir_plan_get_state(self._h, y.data_ptr(), hist.data_ptr() if self.history_len else None,
                                          _stream_ptr(stream)), "spiir_plan_get_state")
        return y, hist

    def set_state(self, y, hist, stream=None) -> None:
        import torch
        _need(y, torch.complex64, self.S * self.n_filters_total, "y")
        if self.history_len:
            _need(hist, torch.float32, self.S * self.history_len, "hist")
        _check(lib().spiir_plan_set_state(self._h, y.data_ptr(), hist.data_ptr() if self.history_len else None,
                                          _stream_ptr(stream)), "spiir_plan_set_state")

    def close(self) -> None:
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_plan_destroy(self._h)
            self._h = None
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Resampler:
    """One streaming x2 stage (spiir_resamp_create / spiir_resample_down / spiir_resample_up)."""

    def __init__(self, direction: str, n_rows: int, max_block: int, n_taps: int = 192, kaiser_beta: float = 5.0,
                 cutoff: float = 0.25, flags: int = 0):
        self.direction, self.rows, self.max_block = direction, int(n_rows), int(max_block)
        code = {"down": SPIIR_DOWN2, "up": SPIIR_UP2}[direction]
        need = lib().spiir_resamp_workspace_bytes(code, int(n_taps), self.rows)
        self._ws = _workspace(need) if need else None
        opts = _ResampOpts(self.max_block, self._ws.data_ptr() if self._ws is not None else None, need, int(flags))
        self._h = ctypes.c_void_p()
        _check(lib().spiir_resamp_create(ctypes.byref(self._h), code, n_taps, kaiser_beta, cutoff, self.rows,
                                         ctypes.byref(opts)), "spiir_resamp_create")
        self.history_len = int(lib().spiir_resamp_history_len(self._h))

    def down(self, u, out=None, stream=None):
        import torch
        if not (u.is_cuda and u.dtype == torch.float32 and u.is_contiguous()):
            raise ValueError("u must be a contiguous CUDA float32 tensor")
        if u.dim() == 1:
            u = u[None, :]
        if self.direction != "down" or u.shape[0] != self.rows or u.shape[1] % 2:
            raise ValueError("u must be [rows][even n_in] for a down stage")
        n_in = int(u.shape[1])
        if out is None:
            out = torch.empty((self.rows, n_in // 2), dtype=torch.float32, device=u.device)
        else:
            _need(out, torch.float32, self.rows * (n_in // 2), "out")
        _check(lib().spiir_resample_down(self._h, u.data_ptr(), n_in, out.data_ptr(), _stream_ptr(stream)),
               "spiir_resample_down")
        return out

    def up(self, v, out=None, accumulate: bool = False, stream=None):
        import torch
        if not (v.is_cuda and v.dtype == torch.complex64 and v.is_contiguous()):
            raise ValueError("v must be a contiguous CUDA complex64 tensor")
        if v.dim() == 1:
            v = v[None, :]
        if self.direction != "up" or v.shape[0] != self.rows:
            raise ValueError("v must be [rows][n_in] for an up stage")
        n_in = int(v.shape[1])
        if out is None:
            if accumulate:
                raise ValueError("accumulate needs an output tensor")
            out = torch.empty((self.rows, 2 * n_in), dtype=torch.complex64, device=v.device)
        else:
            _need(out, torch.complex64, self.rows * 2 * n_in, "out")
        _check(lib().spiir_resample_up(self._h, v.data_ptr(), n_in, out.data_ptr(), int(bool(accumulate)),
                                       _stream_ptr(stream)), "spiir_resample_up")
        return out

    def get_state(self, stream=None):
        import torch
        dt = torch.float32 if self.direction == "down" else torch.complex64
        h = torch.empty((self.rows, self.history_len), dtype=dt, device="cuda")
        _check(lib().spiir_resamp_get_state(self._h, h.data_ptr() if self.history_len else None, _stream_ptr(stream)),
               "spiir_resamp_get_state")
        return h

    def set_state(self, hist, stream=None) -> None:
        import torch
        dt = torch.float32 if self.direction == "down" else torch.complex64
        if self.history_len:
            _need(hist, dt, self.rows * self.history_len, "hist")
        _check(lib().spiir_resamp_set_state(self._h, hist.data_ptr() if self.history_len else None, _stream_ptr(stream)),
               "spiir_resamp_set_state")

    def reset(self, stream=None) -> None:
        _check(lib().spiir_resamp_reset(self._h, _stream_ptr(stream)), "spiir_resamp_reset")

    def close(self) -> None:
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_resamp_destroy(self._h)
            self._h = None
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class MultiratePlan:
    """Multirate SPIIR (spiir_mr_plan_create / spiir_mr_filter).  banks: highest rate first, each
    (a1, b0, delays) of shape [T][L_h]; rates_hz descending, each half of the previous.  n_taps / kaiser_beta /
    cutoff set both directions; the *_down / *_up arguments override one."""

    def __init__(self, banks: Sequence, rates_hz: Sequence[int], n_streams: int = 1, max_block: Optional[int] = None,
                 n_taps: int = 192, kaiser_beta: float = 5.0, cutoff: float = 0.25, n_taps_down=None, kaiser_beta_down=None,
                 cutoff_down=None, n_taps_up=None, kaiser_beta_up=None, cutoff_up=None):
        arrs = [_bank_arrays(*b) for b in banks]
        H = len(arrs)
        self.H, self.T, self.S = H, arrs[0][0].shape[0], int(n_streams)
        self.max_block = int(max_block if max_block is not None else rates_hz[0])
        vp = ctypes.c_void_p
        a1p = (vp * H)(*[a[0].ctypes.data for a in arrs])
        b0p = (vp * H)(*[a[1].ctypes.data for a in arrs])
        dp = (vp * H)(*[a[2].ctypes.data for a in arrs])
        nf = (ctypes.c_int * H)(*[a[0].shape[1] for a in arrs])
        dmax = (ctypes.c_int * H)(*[int(a[2].max(initial=0)) for a in arrs])
        rates = (ctypes.c_int * H)(*[int(r) for r in rates_hz])
        pick = lambda v, d: d if v is None else v
        opts = _MrOpts(self.S, self.max_block, int(pick(n_taps_down, n_taps)), float(pick(kaiser_beta_down, kaiser_beta)),
                       float(pick(cutoff_down, cutoff)), int(pick(n_taps_up, n_taps)), float(pick(kaiser_beta_up, kaiser_beta)),
                       float(pick(cutoff_up, cutoff)), None, 0)
        need = lib().spiir_mr_workspace_bytes(H, nf, dmax, self.T, ctypes.byref(opts))
        self._ws = _workspace(need) if need else None
        opts.workspace, opts.workspace_bytes = (self._ws.data_ptr() if self._ws is not None else None), need
        self._h = ctypes.c_void_p()
        _check(lib().spiir_mr_plan_create(ctypes.byref(self._h), H, rates, a1p, b0p, dp, nf, self.T,
                                          ctypes.byref(opts)), "spiir_mr_plan_create")

    def filter(self, x, out=None, stream=None):
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
        else:
            _need(out, torch.complex64, self.S * self.T * n, "out")
        _check(lib().spiir_mr_filter(self._h, x.data_ptr(), n, out.data_ptr(), _stream_ptr(stream)), "spiir_mr_filter")
        return out

    def launches(self, n: int) -> int:
        return int(lib().spiir_mr_launches(self._h, int(n)))

    def get_state(self, stream=None):
        """The whole resume state (every bank's y and history, every FIR history) as one uint8 device blob."""
        import torch
        blob = torch.empty(int(lib().spiir_mr_plan_state_bytes(self._h)), dtype=torch.uint8, device="cuda")
        _check(lib().spiir_mr_plan_get_state(self._h, blob.data_ptr(), _stream_ptr(stream)), "spiir_mr_plan_get_state")
        return blob

    def set_state(self, blob, stream=None) -> None:
        import torch
        _need(blob, torch.uint8, int(lib().spiir_mr_plan_state_bytes(self._h)), "blob")
        _check(lib().spiir_mr_plan_set_state(self._h, blob.data_ptr(), _stream_ptr(stream)), "spiir_mr_plan_set_state")

    def reset(self, stream=None) -> None:
        _check(lib().spiir_mr_plan_reset(self._h, _stream_ptr(stream)), "spiir_mr_plan_reset")

    def close(self) -> None:
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_mr_plan_destroy(self._h)
            self._h = None
        self._ws = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def filter_block_noalloc(a1, b0, delays, x, out=None, time_chunks: int = 0, stream=None):
    """spiir_filter_block_noalloc: one block from zero state, no plan, no workspace, no allocation inside the library
    (its scan scratch is a 4 MiB device array built into libspiir.so; calls that overlap on the GPU race on it).
    a1, b0: CUDA complex64 [T][L]; delays: CUDA int32 [T][L]; x: CUDA float32 [n]; returns (or fills) complex64 [T][n].
    Pass `out` to keep this wrapper allocation-free as well."""
    import torch
    for t, dt, name in ((a1, torch.complex64, "a1"), (b0, torch.complex64, "b0"), (delays, torch.int32, "delays"),
                        (x, torch.float32, "x")):
        if not (t.is_cuda and t.dtype == dt and t.is_contiguous()):
            raise ValueError(f"{name} must be a contiguous CUDA {dt} tensor")
    if a1.dim() != 2 or b0.shape != a1.shape or delays.shape != a1.shape or x.dim() != 1:
        raise ValueError("a1, b0, delays must be [T][L] and x [n]")
    T, L = int(a1.shape[0]), int(a1.shape[1])
    n = int(x.shape[0])
    if out is None:
        out = torch.empty((T, n), dtype=torch.complex64, device=x.device)
    else:
        _need(out, torch.complex64, T * n, "out")
    _check(lib().spiir_filter_block_noalloc(a1.data_ptr(), b0.data_ptr(), delays.data_ptr(), T, L, x.data_ptr(), n,
                                            int(time_chunks), out.data_ptr(), _stream_ptr(stream)), "spiir_filter_block_noalloc")
    return out


def noalloc_scratch_need(n_templates: int, n_filters: int, n: int, time_chunks: int = 0) -> int:
    return int(lib().spiir_noalloc_scratch_need(int(n_templates), int(n_filters), int(n), int(time_chunks)))


def noalloc_setup() -> None:
    _check(lib().spiir_noalloc_setup(), "spiir_noalloc_setup")


class PaperDesignPlan:
    """COMPARISON ONLY: the paper's own Maxwell kernel design on this GPU (spiir_pd_plan_create / spiir_pd_filter)."""

    def __init__(self, a1, b0, delays, max_block: int = 4096):
        a1, b0, d = _bank_arrays(a1, b0, delays)
        self.T, self.L = a1.shape
        self.max_block = int(max_block)
        self._h = ctypes.c_void_p()
        _check(lib().spiir_pd_plan_create(ctypes.byref(self._h), a1.ctypes.data, b0.ctypes.data, d.ctypes.data, self.T, self.L,
                                          self.max_block), "spiir_pd_plan_create")

    def filter(self, x, out=None, stream=None):
        import torch
        if not (x.is_cuda and x.dtype == torch.float32 and x.is_contiguous()):
            raise ValueError("x must be a contiguous CUDA float32 tensor")
        x = x.reshape(-1)
        n = int(x.numel())
        if out is None:
            out = torch.empty((1, self.T, n), dtype=torch.complex64, device=x.device)
        else:
            _need(out, torch.complex64, self.T * n, "out")
        _check(lib().spiir_pd_filter(self._h, x.data_ptr(), n, out.data_ptr(), _stream_ptr(stream)), "spiir_pd_filter")
        return out

    def reset(self, stream=None) -> None:
        _check(lib().spiir_pd_plan_reset(self._h, _stream_ptr(stream)), "spiir_pd_plan_reset")

    def close(self) -> None:
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_pd_plan_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
