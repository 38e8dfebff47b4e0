"""Thin ctypes binding of include/filark_stream.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of csrc/; there is no CPU fallback: if
libfilark_stream.so is missing or fails to load, importing this module's functions raises.
torch is used for device memory and streams only.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

import numpy as np

from .build import LIB_PATH
from .workloads import CHANNEL_MAJOR, TIME_MAJOR

FLAG_NONE = 0
FLAG_SERIAL_SCAN = 1
FLAG_STRICT_ORDER = 2       # never overlap pushes, not even inside push_many (filark_stream.h, "Ordering")
FLAG_OVERLAP_PUSHES = 4     # the caller promises that nothing foreign lies between consecutive push calls
FLAG_TM_TRANSPOSE = 8       # time-major: always the transposing kernel (testing)
MAX_SECTIONS = 16

STATUS_NAMES = {0: "FILARK_OK", 1: "FILARK_ERR_INVALID_ARG", 2: "FILARK_ERR_UNSTABLE",
                3: "FILARK_ERR_ALLOC", 4: "FILARK_ERR_CUDA", 5: "FILARK_ERR_DEVICE_MISMATCH",
                6: "FILARK_ERR_ALIGNMENT", 7: "FILARK_ERR_TOO_LARGE"}

_lib = None
EVENT_DTYPE = np.dtype([("t_on", "<i8"), ("t_off", "<i8"), ("channel", "<i4"), ("peak", "<f4")])   # filark_event_t


class FilarkError(RuntimeError):
    def __init__(self, status: int, where: str, detail: str = ""):
        self.status = int(status)
        super().__init__(f"{where}: {STATUS_NAMES.get(self.status, self.status)} {detail}".strip())


def library_path() -> str:
    return LIB_PATH


def load_library():
    """Load the C-ABI library; fails loudly if it has not been built (no fallback)."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise FileNotFoundError(
            f"{LIB_PATH} is missing: build it with `python -m paper_2605_20132_b200.build` "
            "(there is no CPU fallback for the filark stream path)")
    lib = ctypes.CDLL(LIB_PATH)
    vp, ll, ci, cu = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_uint
    lib.filark_stream_create.restype = ci
    lib.filark_stream_create.argtypes = [ctypes.POINTER(vp), ci, vp, ci, ci, ci]
    lib.filark_stream_create_ex.restype = ci
    lib.filark_stream_create_ex.argtypes = [ctypes.POINTER(vp), ci, vp, ci, ci, ci, ci, cu]
    lib.filark_stream_push.restype = ci
    lib.filark_stream_push.argtypes = [vp, vp, ll, vp, vp, vp]
    lib.filark_stream_push_many.restype = ci
    lib.filark_stream_push_many.argtypes = [vp, ci, vp, vp, vp, vp, vp]
    lib.filark_stream_push_pitched.restype = ci
    lib.filark_stream_push_pitched.argtypes = [vp, vp, ll, ll, vp, vp, ll, vp]
    lib.filark_stream_push_host.restype = ci
    lib.filark_stream_push_host.argtypes = [vp, vp, ll, vp, vp, vp]
    lib.filark_stream_state_size.restype = ll
    lib.filark_stream_state_size.argtypes = [vp]
    lib.filark_stream_get_state.restype = ci
    lib.filark_stream_get_state.argtypes = [vp, vp, ll, vp]
    lib.filark_stream_set_state.restype = ci
    lib.filark_stream_set_state.argtypes = [vp, vp, ll, vp]
    lib.filark_stream_set_initial_condition.restype = ci
    lib.filark_stream_set_initial_condition.argtypes = [vp, vp, vp]
    lib.filark_stream_set_trigger.restype = ci
    lib.filark_stream_set_trigger.argtypes = [vp, ctypes.c_float, ctypes.c_float, ll, vp]
    lib.filark_stream_pop_events.restype = ci
    lib.filark_stream_pop_events.argtypes = [vp, vp, ll, ctypes.POINTER(ll), ctypes.POINTER(ll), vp]
    lib.filark_stream_zero_phase.restype = ci
    lib.filark_stream_zero_phase.argtypes = [vp, vp, ll, vp, vp]
    lib.filark_events_associate.restype = ci
    lib.filark_events_associate.argtypes = [vp, ll, ci, ll, vp, ll, ctypes.POINTER(ll)]
    lib.filark_stream_once_noalloc.restype = ci
    lib.filark_stream_once_noalloc.argtypes = [vp, ci, ci, ci, ci, vp, ci, ll, vp, vp, vp, ctypes.POINTER(ci)]
    lib.filark_stream_reset.restype = ci
    lib.filark_stream_reset.argtypes = [vp, vp]
    lib.filark_stream_destroy.restype = ci
    lib.filark_stream_destroy.argtypes = [vp]
    lib.filark_status_string.restype = ctypes.c_char_p
    lib.filark_status_string.argtypes = [ci]
    lib.filark_last_cuda_error.restype = ci
    lib.filark_last_cuda_error.argtypes = [vp]
    lib.filark_stream_launch_count.restype = ll
    lib.filark_stream_launch_count.argtypes = [vp]
    lib.filark_stream_samples_pushed.restype = ll
    lib.filark_stream_samples_pushed.argtypes = [vp]
    lib.filark_debug_design.restype = ci
    lib.filark_debug_design.argtypes = [vp, ci, vp, vp, vp]
    lib.filark_debug_push_geometry.restype = ci
    lib.filark_debug_push_geometry.argtypes = [ll, ci, ci, vp]
    lib.filark_debug_block_power.restype = ci
    lib.filark_debug_block_power.argtypes = [vp, ll, vp]
    _lib = lib
    return lib


def _ptr(t) -> Optional[int]:
    return None if t is None else int(t.data_ptr())


def _cur_stream() -> int:
    import torch
    try:        # the raw handle, without building a Stream object (a push is a few microseconds of host work)
        return int(torch._C._cuda_getCurrentRawStream(torch.cuda.current_device()))
    except Exception:
        return int(torch.cuda.current_stream().cuda_stream)


BOX_DTYPE = np.dtype([("t_on", "<i8"), ("t_off", "<i8"), ("ch_lo", "<i4"), ("ch_hi", "<i4"), ("peak", "<f4"),
                      ("n_events", "<i4")])   # filark_box_t


def associate_events(events, ch_gap: int = 1, t_gap: int = 0, cap: Optional[int] = None):
    """filark_events_associate: per-channel events (EVENT_DTYPE, as pop_events returns them) -> time-channel
    boxes (BOX_DTYPE); a host function.  Returns (boxes, number of boxes found)."""
    lib = load_library()
    ev = np.ascontiguousarray(events, dtype=EVENT_DTYPE)
    cap = ev.shape[0] if cap is None else int(cap)
    out = np.zeros(max(cap, 1), dtype=BOX_DTYPE)
    n = ctypes.c_longlong(0)
    st = lib.filark_events_associate(ev.ctypes.data if ev.shape[0] else None, ev.shape[0], int(ch_gap), int(t_gap),
                                     out.ctypes.data, cap, ctypes.byref(n))
    if st != 0:
        raise FilarkError(st, "filark_events_associate")
    return out[:min(cap, n.value)].copy(), int(n.value)


NOALLOC_MAX_CHANNELS = 16384      # FILARK_NOALLOC_MAX_CHANNELS


def once_noalloc(sos, sta_len: int, lta_len: int, d_in, d_filt=None, d_cf=None, layout: int = CHANNEL_MAJOR,
                 stream: Optional[int] = None):
    """filark_stream_once_noalloc: the whole path over one dense record from rest, no handle, no allocation
    (fixed scratch in the library's device image; at most NOALLOC_MAX_CHANNELS channels; calls that overlap
    on the GPU race on that scratch)."""
    import torch
    lib = load_library()
    sos = np.ascontiguousarray(np.asarray(sos, dtype=np.float64))
    if sos.ndim != 2 or sos.shape[1] != 6:
        raise ValueError("sos must be [n_sec][6]")
    for t in (d_in, d_filt, d_cf):
        if t is not None and (not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous() or t.dim() != 2):
            raise ValueError("buffers must be contiguous 2-D float32 CUDA tensors")
    n_ch, n_t = (d_in.shape[0], d_in.shape[1]) if layout == CHANNEL_MAJOR else (d_in.shape[1], d_in.shape[0])
    err = ctypes.c_int(0)
    st = lib.filark_stream_once_noalloc(sos.ctypes.data, int(sos.shape[0]), int(sta_len), int(lta_len), int(layout),
                                        _ptr(d_in), int(n_ch), int(n_t), _ptr(d_filt), _ptr(d_cf),
                                        _cur_stream() if stream is None else stream, ctypes.byref(err))
    if st != 0:
        raise FilarkError(st, "filark_stream_once_noalloc", f"(cudaError {err.value})" if st == 4 else "")


class PushBatch:
    """The marshalled arguments of one filark_stream_push_many call (pointer and length arrays);
    keeps the tensors alive.  Built once, enqueued any number of times."""

    def __init__(self, stream_obj: "FilarkStream", ins, filts=None, cfs=None):
        import torch
        n = len(ins)
        for seq in (filts, cfs):
            if seq is not None and len(seq) != n:
                raise ValueError("ins, filts and cfs must have the same length")
        for t in list(ins) + list(filts or []) + list(cfs or []):
            if t is not None and (not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous()):
                raise ValueError("buffers must be contiguous float32 CUDA tensors")
        self.n = n
        self.keep = (list(ins), list(filts) if filts is not None else None, list(cfs) if cfs is not None else None)
        self.n_t = (ctypes.c_longlong * n)(*[stream_obj._n_t(x) for x in ins])
        self.d_in = (ctypes.c_void_p * n)(*[_ptr(x) for x in ins])
        self.d_filt = None if filts is None else (ctypes.c_void_p * n)(*[_ptr(x) for x in filts])
        self.d_cf = None if cfs is None else (ctypes.c_void_p * n)(*[_ptr(x) for x in cfs])


class FilarkStream:
    """filark_stream_create / push / reset / destroy with torch CUDA tensors as buffers."""

    def __init__(self, n_ch: int, sos, sta_len: int, lta_len: int, layout: int = CHANNEL_MAJOR,
                 flags: int = FLAG_NONE):
        lib = load_library()
        sos = np.ascontiguousarray(np.asarray(sos, dtype=np.float64))
        if sos.ndim != 2 or sos.shape[1] != 6:
            raise ValueError("sos must be [n_sec][6]")
        self._lib = lib
        self._h = ctypes.c_void_p()
        self.n_ch, self.n_sec, self.layout = int(n_ch), int(sos.shape[0]), int(layout)
        st = lib.filark_stream_create_ex(ctypes.byref(self._h), self.n_ch, sos.ctypes.data,
                                         self.n_sec, int(sta_len), int(lta_len), self.layout,
                                         int(flags))
        if st != 0:
            self._h = ctypes.c_void_p()
            raise FilarkError(st, "filark_stream_create_ex")

    # -- helpers
    def _check(self, st: int, where: str):
        if st != 0:
            detail = ""
            if st == 4:
                detail = f"(cudaError {self._lib.filark_last_cuda_error(self._h)})"
            raise FilarkError(st, where, detail)

    def _n_t(self, x) -> int:
        if x.dim() != 2:
            raise ValueError("chunk must be 2-D")
        n_c, n_t = (x.shape[0], x.shape[1]) if self.layout == CHANNEL_MAJOR else (x.shape[1], x.shape[0])
        if n_c != self.n_ch:
            raise ValueError("chunk channel count does not match the stream")
        return int(n_t)

    # -- C ABI mirrors
    def push(self, d_in, d_filt=None, d_cf=None, stream: Optional[int] = None):
        """d_in/d_filt/d_cf: contiguous float32 CUDA tensors of identical 2-D shape."""
        import torch
        for t in (d_in, d_filt, d_cf):
            if t is not None and (not t.is_cuda or t.dtype != torch.float32 or not t.is_contiguous()):
                raise ValueError("buffers must be contiguous float32 CUDA tensors")
        n_t = self._n_t(d_in)
        st = self._lib.filark_stream_push(self._h, _ptr(d_in), n_t, _ptr(d_filt), _ptr(d_cf),
                                          _cur_stream() if stream is None else stream)
        self._check(st, "filark_stream_push")

    def push_many(self, ins, filts=None, cfs=None, stream: Optional[int] = None):
        """filark_stream_push_many: `ins` (and `filts`, `cfs`) are sequences of chunk tensors, or
        `ins` is a prepared PushBatch."""
        b = ins if isinstance(ins, PushBatch) else PushBatch(self, ins, filts, cfs)
        st = self._lib.filark_stream_push_many(self._h, b.n, b.d_in, b.n_t, b.d_filt, b.d_cf,
                                               _cur_stream() if stream is None else stream)
        self._check(st, "filark_stream_push_many")

    def push_pitched(self, d_in, n_t: int, in_pitch: int, d_filt, d_cf, out_pitch: int,
                     in_offset: int = 0, out_offset: int = 0, stream: Optional[int] = None):
        """Sub-view push: pointers are tensor base + offset (elements); pitches in elements."""
        pin = _ptr(d_in) + 4 * in_offset
        pf = None if d_filt is None else _ptr(d_filt) + 4 * out_offset
        pc = None if d_cf is None else _ptr(d_cf) + 4 * out_offset
        st = self._lib.filark_stream_push_pitched(self._h, pin, int(n_t), int(in_pitch), pf, pc,
                                                  int(out_pitch),
                                                  _cur_stream() if stream is None else stream)
        self._check(st, "filark_stream_push_pitched")

    def push_host(self, h_in, h_filt=None, h_cf=None, stream: Optional[int] = None):
        """Host (ideally pinned) float32 tensors/arrays; asynchronous on the stream."""
        n_t = self._n_t(h_in)
        st = self._lib.filark_stream_push_host(self._h, _ptr(h_in), n_t, _ptr(h_filt), _ptr(h_cf),
                                               _cur_stream() if stream is None else stream)
        self._check(st, "filark_stream_push_host")

    def reset(self, stream: Optional[int] = None):
        self._check(self._lib.filark_stream_reset(self._h, _cur_stream() if stream is None else stream),
                    "filark_stream_reset")

    def set_trigger(self, thr_on: float, thr_off: float, max_events: int = 1 << 20, stream: Optional[int] = None):
        self._check(self._lib.filark_stream_set_trigger(self._h, float(thr_on), float(thr_off), int(max_events),
                                                        _cur_stream() if stream is None else stream),
                    "filark_stream_set_trigger")
        self._ev_cap = int(max_events)

    def pop_events(self, stream: Optional[int] = None):
        """(events as a numpy record array (t_on, t_off, channel, peak), number dropped)."""
        cap = getattr(self, "_ev_cap", 0)
        out = np.zeros(max(cap, 1), dtype=EVENT_DTYPE)
        n, d = ctypes.c_longlong(0), ctypes.c_longlong(0)
        self._check(self._lib.filark_stream_pop_events(self._h, out.ctypes.data, cap, ctypes.byref(n), ctypes.byref(d),
                                                       _cur_stream() if stream is None else stream),
                    "filark_stream_pop_events")
        return out[:n.value].copy(), int(d.value)

    def zero_phase(self, d_in, d_out, stream: Optional[int] = None):
        """filark_stream_zero_phase: forward-backward filtering of a bounded window (carried state untouched)."""
        n_t = self._n_t(d_in)
        self._check(self._lib.filark_stream_zero_phase(self._h, _ptr(d_in), n_t, _ptr(d_out),
                                                       _cur_stream() if stream is None else stream),
                    "filark_stream_zero_phase")

    def get_state(self, stream: Optional[int] = None) -> bytes:
        """filark_stream_get_state: the documented state blob (host bytes)."""
        n = int(self._lib.filark_stream_state_size(self._h))
        buf = ctypes.create_string_buffer(n)
        self._check(self._lib.filark_stream_get_state(self._h, buf, n, _cur_stream() if stream is None else stream),
                    "filark_stream_get_state")
        return buf.raw

    def set_state(self, blob: bytes, stream: Optional[int] = None):
        self._check(self._lib.filark_stream_set_state(self._h, blob, len(blob), _cur_stream() if stream is None else stream),
                    "filark_stream_set_state")

    def set_initial_condition(self, x0, stream: Optional[int] = None):
        """x0: per-channel constant input level (scalar or [n_ch])."""
        a = np.ascontiguousarray(np.broadcast_to(np.asarray(x0, dtype=np.float32), (self.n_ch,)))
        self._check(self._lib.filark_stream_set_initial_condition(self._h, a.ctypes.data,
                                                                  _cur_stream() if stream is None else stream),
                    "filark_stream_set_initial_condition")

    def destroy(self):
        if getattr(self, "_h", None) is not None and self._h.value:
            self._lib.filark_stream_destroy(self._h)
            self._h = ctypes.c_void_p()

    close = destroy

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    @property
    def launch_count(self) -> int:
        return int(self._lib.filark_stream_launch_count(self._h))

    @property
    def samples_pushed(self) -> int:
        return int(self._lib.filark_stream_samples_pushed(self._h))


def push_host(stream_obj: FilarkStream, h_in, h_filt=None, h_cf=None):
    """Module-level alias of FilarkStream.push_host (the end-to-end call bench.py times)."""
    stream_obj.push_host(h_in, h_filt, h_cf)


# ---- host-only introspection (include/filark_debug.h) ----------------------------------------
def debug_design(sos):
    lib = load_library()
    sos = np.ascontiguousarray(np.asarray(sos, dtype=np.float64))
    n = sos.shape[0]
    kinds = np.zeros(n, dtype=np.int32)
    coefs = np.zeros((n, 9), dtype=np.float64)
    gain = ctypes.c_double(0.0)
    st = lib.filark_debug_design(sos.ctypes.data, n, kinds.ctypes.data, coefs.ctypes.data,
                                 ctypes.addressof(gain))
    if st != 0:
        raise FilarkError(st, "filark_debug_design")
    return kinds, coefs, float(gain.value)


def debug_push_geometry(n_t: int, r0: int = 0, force_L: int = 0):
    """dict(L, n_tiles, q_last, r1, vec4) of a channel-major push of n_t samples behind r0 waiting ones."""
    lib = load_library()
    out = np.zeros(5, dtype=np.int32)
    st = lib.filark_debug_push_geometry(int(n_t), int(r0), int(force_L), out.ctypes.data)
    if st != 0:
        raise FilarkError(st, "filark_debug_push_geometry")
    return dict(zip(("L", "n_tiles", "q_last", "r1", "vec4"), map(int, out)))


def debug_block_power(sos6, e: int):
    lib = load_library()
    sos6 = np.ascontiguousarray(np.asarray(sos6, dtype=np.float64))
    out = np.zeros(4, dtype=np.float64)
    st = lib.filark_debug_block_power(sos6.ctypes.data, int(e), out.ctypes.data)
    if st != 0:
        raise FilarkError(st, "filark_debug_block_power")
    return out.reshape(2, 2)
