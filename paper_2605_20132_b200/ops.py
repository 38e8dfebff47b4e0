"""Thin ctypes binding of include/filark_ops.h (argument marshalling only): streaming first-order
operators (running mean / de-mean / running AGC) and display decimation.  No CPU fallback."""
from __future__ import annotations

import ctypes
from typing import Optional

from .stream import FilarkError, _cur_stream, _ptr, load_library
from .workloads import CHANNEL_MAJOR, TIME_MAJOR

EMA_MODES = {"mean": 0, "demean": 1, "agc": 2}
DECIMATE_MODES = {"drop": 0, "peak": 1, "linear": 2}
_ready = False


def _lib():
    global _ready
    lib = load_library()
    if not _ready:
        vp, ll, ci = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int
        lib.filark_ema_create.restype = ci
        lib.filark_ema_create.argtypes = [ctypes.POINTER(vp), ci, ci, ci, ctypes.c_float, ci]
        lib.filark_ema_push.restype = ci
        lib.filark_ema_push.argtypes = [vp, vp, ll, vp, vp]
        lib.filark_ema_reset.restype = ci
        lib.filark_ema_reset.argtypes = [vp, vp]
        lib.filark_ema_destroy.restype = ci
        lib.filark_ema_destroy.argtypes = [vp]
        lib.filark_decimate.restype = ci
        lib.filark_decimate.argtypes = [vp, ci, ll, ll, ci, ci, ci, vp, vp]
        _ready = True
    return lib


class FilarkEma:
    """filark_ema_create / push / reset / destroy with torch CUDA tensors as buffers."""

    def __init__(self, n_ch: int, n_len: int, mode: str, eps: float = 0.0, layout: int = CHANNEL_MAJOR):
        self._lib = _lib()
        self._h = ctypes.c_void_p()
        self.n_ch, self.layout = int(n_ch), int(layout)
        st = self._lib.filark_ema_create(ctypes.byref(self._h), self.n_ch, int(n_len), EMA_MODES[mode], float(eps), self.layout)
        if st != 0:
            self._h = ctypes.c_void_p()
            raise FilarkError(st, "filark_ema_create")

    def push(self, d_in, d_out, stream: Optional[int] = None):
        n_c, n_t = (d_in.shape[0], d_in.shape[1]) if self.layout == CHANNEL_MAJOR else (d_in.shape[1], d_in.shape[0])
        if n_c != self.n_ch or d_out.shape != d_in.shape or not d_in.is_contiguous() or not d_out.is_contiguous():
            raise ValueError("chunks must be contiguous and of the stream's channel count")
        st = self._lib.filark_ema_push(self._h, _ptr(d_in), int(n_t), _ptr(d_out), _cur_stream() if stream is None else stream)
        if st != 0:
            raise FilarkError(st, "filark_ema_push")

    def reset(self, stream: Optional[int] = None):
        st = self._lib.filark_ema_reset(self._h, _cur_stream() if stream is None else stream)
        if st != 0:
            raise FilarkError(st, "filark_ema_reset")

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.filark_ema_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def decimate(d_in, mode: str, width: int, layout: int = CHANNEL_MAJOR, d_out=None, stream: Optional[int] = None):
    """filark_decimate on a dense 2-D float32 CUDA tensor; returns the [n_ch][width] / [width][n_ch] buffer."""
    import torch
    lib = _lib()
    if layout == CHANNEL_MAJOR:
        n_ch, n_t = d_in.shape
        shape, pitch = (n_ch, width), n_t
    else:
        n_t, n_ch = d_in.shape
        shape, pitch = (width, n_ch), n_ch
    if d_out is None:
        d_out = torch.empty(shape, dtype=torch.float32, device=d_in.device)
    st = lib.filark_decimate(_ptr(d_in), int(n_ch), int(n_t), int(pitch), int(layout), DECIMATE_MODES[mode], int(width),
                             _ptr(d_out), _cur_stream() if stream is None else stream)
    if st != 0:
        raise FilarkError(st, "filark_decimate")
    return d_out
