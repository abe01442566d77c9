"""Float64 CPU oracle for the SPIIR hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes wrapper over ``oracle/spiir_oracle.c`` (plain C, double precision, written from
/root/reference/PAPER.md) plus the multirate composition of PAPER.md:75-77 written out in
numpy calls on those primitives.  Nothing here imports, links or shares code with
``paper_1702_02256_b200`` (the CUDA path); only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s ``cpu_baseline`` / ``--impl reference`` legs may import this package.

Pins: tests/test_oracle_pins.py (see the header of spiir_oracle.c).  No function here is
"parity unpinned"; the paper prints no worked numerical example, so all pins are closed
forms, library routines (scipy.signal.lfilter, numpy.convolve, numpy.kaiser), invariants
and brute force.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "spiir_oracle.c")
_SO = os.path.join(_HERE, "libspiir_oracle.so")
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (building the checker is not using it)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-fopenmp", "-std=c99", "-shared", "-fPIC",
                               "-o", _SO, _SRC, "-lm"])
    return _SO


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        vp, ci, dp = ctypes.c_void_p, ctypes.c_int, ctypes.POINTER(ctypes.c_double)
        lib.spiir_oracle_plan_create.argtypes = [ctypes.POINTER(vp), vp, vp, vp, ci, ci, ci]
        lib.spiir_oracle_filter.argtypes = [vp, vp, ci, vp]
        lib.spiir_oracle_plan_reset.argtypes = [vp]
        lib.spiir_oracle_plan_destroy.argtypes = [vp]
        lib.spiir_oracle_kaiser_taps.argtypes = [ci, ctypes.c_double, ctypes.c_double, vp, vp]
        lib.spiir_oracle_resamp_create.argtypes = [ctypes.POINTER(vp), ci, ci, vp, ci]
        lib.spiir_oracle_resamp_reset.argtypes = [vp]
        lib.spiir_oracle_resamp_destroy.argtypes = [vp]
        lib.spiir_oracle_down2.argtypes = [vp, vp, ci, vp]
        lib.spiir_oracle_up2.argtypes = [vp, vp, ci, vp, ci]
        lib.spiir_oracle_set_num_threads.argtypes = [ci]
        _lib = lib
    return _lib


def num_threads() -> int:
    return int(_load().spiir_oracle_num_threads())


def set_num_threads(n: int) -> None:
    _load().spiir_oracle_set_num_threads(int(n))


def _c64_as_f32_pairs(a) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.complex64)
    return a.view(np.float32)


class FilterOracle:
    """Streaming single-rate SPIIR bank, Eq. 7 + Eq. 8, float64.

    a1, b0: complex64 [T][L] (promoted exactly to complex128); delays int32 [T][L].
    ``filter(x)`` takes float32/float64 x of shape [n] or [S][n] and returns complex128
    z of shape [S][T][n]; consecutive calls continue one stream (state carried).
    """

    def __init__(self, a1, b0, delays, n_streams: int = 1):
        a1 = np.ascontiguousarray(a1, dtype=np.complex64)
        b0 = np.ascontiguousarray(b0, dtype=np.complex64)
        d = np.ascontiguousarray(delays, dtype=np.int32)
        if a1.ndim != 2 or a1.shape != b0.shape or a1.shape != d.shape:
            raise ValueError("a1, b0, delays must all be [T][L]")
        self.T, self.L, self.S = a1.shape[0], a1.shape[1], int(n_streams)
        self._h = ctypes.c_void_p()
        rc = _load().spiir_oracle_plan_create(ctypes.byref(self._h), a1.ctypes.data, b0.ctypes.data,
                                              d.ctypes.data, self.T, self.L, self.S)
        if rc != 0:
            raise ValueError("spiir_oracle_plan_create failed (negative delay or bad shape)")

    def filter(self, x) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.float64)
        if x.ndim == 1:
            x = x[None, :]
        if x.shape[0] != self.S:
            raise ValueError("x must be [S][n]")
        n = x.shape[1]
        z = np.empty((self.S, self.T, n), dtype=np.complex128)
        rc = _load().spiir_oracle_filter(self._h, x.ctypes.data, n, z.ctypes.data)
        if rc != 0:
            raise RuntimeError("spiir_oracle_filter failed")
        return z

    def reset(self) -> None:
        _load().spiir_oracle_plan_reset(self._h)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_oracle_plan_destroy(self._h)
            self._h = None


def kaiser_taps(n_taps: int = 192, beta: float = 5.0, cutoff: float = 0.25):
    """(h64, h32): the Kaiser-windowed-sinc low-pass of DESIGN.md O4 in double and rounded to float32."""
    h64 = np.empty(n_taps, dtype=np.float64)
    h32 = np.empty(n_taps, dtype=np.float32)
    if _load().spiir_oracle_kaiser_taps(n_taps, beta, cutoff, h64.ctypes.data, h32.ctypes.data) != 0:
        raise ValueError("bad tap parameters")
    return h64, h32


class ResampOracle:
    """One streaming x2 stage.  direction 'down': real rows [rows][n] -> [rows][n/2];
    'up': complex rows [rows][n] -> [rows][2n] (optionally accumulated into ``out``)."""

    def __init__(self, direction: str, n_rows: int, taps32=None, n_taps: int = 192,
                 beta: float = 5.0, cutoff: float = 0.25):
        if taps32 is None:
            taps32 = kaiser_taps(n_taps, beta, cutoff)[1]
        self.taps32 = np.ascontiguousarray(taps32, dtype=np.float32)
        self.direction, self.rows = direction, int(n_rows)
        self._h = ctypes.c_void_p()
        rc = _load().spiir_oracle_resamp_create(ctypes.byref(self._h), {"down": 0, "up": 1}[direction],
                                                self.taps32.size, self.taps32.ctypes.data, self.rows)
        if rc != 0:
            raise ValueError("spiir_oracle_resamp_create failed")

    def down(self, u) -> np.ndarray:
        u = np.ascontiguousarray(u, dtype=np.float64)
        if u.ndim == 1:
            u = u[None, :]
        assert u.shape[0] == self.rows and u.shape[1] % 2 == 0
        out = np.empty((self.rows, u.shape[1] // 2), dtype=np.float64)
        if _load().spiir_oracle_down2(self._h, u.ctypes.data, u.shape[1], out.ctypes.data) != 0:
            raise RuntimeError("spiir_oracle_down2 failed")
        return out

    def up(self, v, out=None) -> np.ndarray:
        v = np.ascontiguousarray(v, dtype=np.complex128)
        if v.ndim == 1:
            v = v[None, :]
        assert v.shape[0] == self.rows
        acc = out is not None
        if out is None:
            out = np.empty((self.rows, 2 * v.shape[1]), dtype=np.complex128)
        assert out.dtype == np.complex128 and out.flags.c_contiguous and out.shape == (self.rows, 2 * v.shape[1])
        if _load().spiir_oracle_up2(self._h, v.ctypes.data, v.shape[1], out.ctypes.data, int(acc)) != 0:
            raise RuntimeError("spiir_oracle_up2 failed")
        return out

    def reset(self) -> None:
        _load().spiir_oracle_resamp_reset(self._h)

    def __del__(self):
        if getattr(self, "_h", None) and _lib is not None:
            _lib.spiir_oracle_resamp_destroy(self._h)
            self._h = None


class MultirateOracle:
    """Multirate SPIIR of PAPER.md:75-77 (Fig. 1), O5, one stream per row of x.

    x_0 = x, x_h = down2(x_{h-1});  z_h = bank_h(x_h);  acc_{H-1} = z_{H-1};
    acc_{h-1} = z_{h-1} + up2(acc_h);  result acc_0 at the base rate.  All histories carried
    across calls.  banks: list over rates (highest first) of (a1, b0, delays), each [T][L_h].
    """

    def __init__(self, banks, n_streams: int = 1, n_taps: int = 192, beta: float = 5.0, cutoff: float = 0.25,
                 n_taps_down=None, beta_down=None, cutoff_down=None, n_taps_up=None, beta_up=None, cutoff_up=None):
        """n_taps / beta / cutoff: one filter for both directions (BASELINE.json configs[3]); the *_down /
        *_up arguments override it per direction (~100 dB / 384 taps down, ~60 dB / 32 taps up)."""
        self.H, self.S = len(banks), int(n_streams)
        self.T = np.asarray(banks[0][0]).shape[0]
        pick = lambda v, dflt: dflt if v is None else v
        taps_d = kaiser_taps(pick(n_taps_down, n_taps), pick(beta_down, beta), pick(cutoff_down, cutoff))[1]
        taps_u = kaiser_taps(pick(n_taps_up, n_taps), pick(beta_up, beta), pick(cutoff_up, cutoff))[1]
        self.filters = [FilterOracle(a1, b0, d, n_streams) for (a1, b0, d) in banks]
        self.downs = [ResampOracle("down", self.S, taps_d) for _ in range(self.H - 1)]
        self.ups = [ResampOracle("up", self.S * self.T, taps_u) for _ in range(self.H - 1)]

    def filter(self, x) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.float64)
        if x.ndim == 1:
            x = x[None, :]
        n = x.shape[1]
        assert n % (1 << (self.H - 1)) == 0, "block length must be divisible by 2^(H-1)"
        xs = [x]
        for h in range(1, self.H):
            xs.append(self.downs[h - 1].down(xs[h - 1]))
        zs = [self.filters[h].filter(xs[h]) for h in range(self.H)]          # [S][T][n / 2^h]
        acc = zs[self.H - 1]
        for h in range(self.H - 1, 0, -1):
            nxt = np.ascontiguousarray(zs[h - 1]).reshape(self.S * self.T, -1)
            self.ups[h - 1].up(acc.reshape(self.S * self.T, -1), out=nxt)   # nxt += up2(acc)
            acc = nxt.reshape(self.S, self.T, -1)
        return acc

    def reset(self) -> None:
        for o in self.filters + self.downs + self.ups:
            o.reset()
