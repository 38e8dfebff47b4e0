"""ctypes wrapper around oracle/filark_oracle.c (TEST INFRASTRUCTURE, not product code).

The arithmetic lives in the C file, which states the definition it follows
(SURVEY.md 8(c) readings R1-R18).  This module only builds
the shared object with gcc, marshals numpy arrays, and -- for the timed cpu_baseline
run -- splits the independent channels over host threads (ctypes drops the GIL).
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading
from concurrent.futures import ThreadPoolExecutor

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "filark_oracle.c")
_LIB = os.path.join(_HERE, "libfilark_oracle.so")
_lock = threading.Lock()
_lib = None

CHANNEL_MAJOR = 0  # chunk is [n_ch][n_t], time contiguous
TIME_MAJOR = 1     # chunk is [n_t][n_ch], channel contiguous


def oracle_lib_path() -> str:
    return _LIB


def build_oracle(force: bool = False) -> str:
    """Compile the oracle with gcc: no fast-math, no FMA contraction, plain -O2."""
    with _lock:
        if (not force and os.path.exists(_LIB)
                and os.path.getmtime(_LIB) >= os.path.getmtime(_SRC)):
            return _LIB
        cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-ffp-contract=off",
               "-fno-fast-math", "-o", _LIB, _SRC]
        subprocess.run(cmd, check=True, capture_output=True)
        return _LIB


def _load():
    global _lib
    if _lib is not None:
        return _lib
    build_oracle()
    lib = ctypes.CDLL(_LIB)
    vp, ll, ci = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int
    lib.filark_oracle_create.restype = vp
    lib.filark_oracle_create.argtypes = [ci, vp, ci, ci, ci]
    lib.filark_oracle_reset.restype = None
    lib.filark_oracle_reset.argtypes = [vp]
    lib.filark_oracle_destroy.restype = None
    lib.filark_oracle_destroy.argtypes = [vp]
    lib.filark_oracle_samples_seen.restype = ll
    lib.filark_oracle_samples_seen.argtypes = [vp]
    lib.filark_oracle_push_range.restype = ci
    lib.filark_oracle_push_range.argtypes = [vp, vp, ll, ll, ll, vp, vp, ci, ci]
    lib.filark_oracle_advance.restype = None
    lib.filark_oracle_advance.argtypes = [vp, ll]
    lib.filark_oracle_push.restype = ci
    lib.filark_oracle_push.argtypes = [vp, vp, ll, ll, ll, vp, vp]
    lib.filark_oracle_trace_f64.restype = ci
    lib.filark_oracle_trace_f64.argtypes = [vp, ci, vp, ll, vp, vp, vp]
    lib.filark_oracle_set_initial_condition.restype = ci
    lib.filark_oracle_set_initial_condition.argtypes = [vp, vp]
    lib.filark_oracle_state_doubles.restype = ll
    lib.filark_oracle_state_doubles.argtypes = [vp]
    lib.filark_oracle_get_state.restype = ci
    lib.filark_oracle_get_state.argtypes = [vp, vp, vp]
    lib.filark_oracle_set_state.restype = ci
    lib.filark_oracle_set_state.argtypes = [vp, vp, ll]
    lib.filark_oracle_decimate.restype = ci
    lib.filark_oracle_decimate.argtypes = [vp, ci, ll, ll, ll, ci, ci, vp, ll, ll]
    lib.filark_oracle_ema_create.restype = vp
    lib.filark_oracle_ema_create.argtypes = [ci, ci, ci, ctypes.c_double]
    lib.filark_oracle_ema_destroy.restype = None
    lib.filark_oracle_ema_destroy.argtypes = [vp]
    lib.filark_oracle_ema_push.restype = ci
    lib.filark_oracle_ema_push.argtypes = [vp, vp, ll, ll, ll, vp]
    lib.filark_oracle_trigger_create.restype = vp
    lib.filark_oracle_trigger_create.argtypes = [ci, ctypes.c_float, ctypes.c_float]
    lib.filark_oracle_trigger_destroy.restype = None
    lib.filark_oracle_trigger_destroy.argtypes = [vp]
    lib.filark_oracle_trigger_push.restype = ll
    lib.filark_oracle_trigger_push.argtypes = [vp, vp, ll, ll, ll, vp, ll]
    _lib = lib
    return lib


class Oracle:
    """Stateful float64 oracle stream: create -> push* -> reset, like the C ABI under test."""

    def __init__(self, n_ch: int, sos, sta_len: int, lta_len: int, layout: int = CHANNEL_MAJOR):
        lib = _load()
        sos = np.ascontiguousarray(np.asarray(sos, dtype=np.float64))
        if sos.ndim != 2 or sos.shape[1] != 6:
            raise ValueError("sos must be [n_sec][6]")
        self._lib = lib
        self.n_ch, self.n_sec = int(n_ch), int(sos.shape[0])
        self.sta_len, self.lta_len, self.layout = int(sta_len), int(lta_len), int(layout)
        self._h = lib.filark_oracle_create(self.n_ch, sos.ctypes.data, self.n_sec,
                                           self.sta_len, self.lta_len)
        if not self._h:
            raise ValueError("filark_oracle_create rejected its arguments")

    def close(self):
        if getattr(self, "_h", None):
            self._lib.filark_oracle_destroy(self._h)
            self._h = None

    __del__ = close

    def reset(self):
        self._lib.filark_oracle_reset(self._h)

    @property
    def samples_seen(self) -> int:
        return int(self._lib.filark_oracle_samples_seen(self._h))

    def _strides(self, n_t):
        return (n_t, 1) if self.layout == CHANNEL_MAJOR else (1, self.n_ch)

    def push(self, x: np.ndarray, want_filt=True, want_cf=True, threads: int = 1):
        """x: float32 dense chunk, [n_ch][n_t] (channel-major) or [n_t][n_ch] (time-major).
        Returns (filt, cf) float32 arrays of the same shape (None where not wanted)."""
        x = np.ascontiguousarray(x, dtype=np.float32)
        if x.ndim != 2:
            raise ValueError("chunk must be 2-D")
        n_t = x.shape[1] if self.layout == CHANNEL_MAJOR else x.shape[0]
        n_c = x.shape[0] if self.layout == CHANNEL_MAJOR else x.shape[1]
        if n_c != self.n_ch:
            raise ValueError("chunk channel count does not match the stream")
        filt = np.empty_like(x) if want_filt else None
        cf = np.empty_like(x) if want_cf else None
        sc, sn = self._strides(n_t)
        fp = filt.ctypes.data if filt is not None else None
        cp = cf.ctypes.data if cf is not None else None
        threads = max(1, min(int(threads), self.n_ch))
        if threads == 1:
            rc = self._lib.filark_oracle_push_range(self._h, x.ctypes.data, n_t, sc, sn, fp, cp,
                                                    0, self.n_ch)
            if rc:
                raise RuntimeError("oracle push failed")
        else:
            bounds = np.linspace(0, self.n_ch, threads + 1).astype(int)

            def work(i):
                return self._lib.filark_oracle_push_range(self._h, x.ctypes.data, n_t, sc, sn,
                                                          fp, cp, int(bounds[i]), int(bounds[i + 1]))
            with ThreadPoolExecutor(max_workers=threads) as ex:
                if any(ex.map(work, range(threads))):
                    raise RuntimeError("oracle push failed")
        self._lib.filark_oracle_advance(self._h, n_t)
        return filt, cf

    def set_initial_condition(self, x0):
        """Steady state for a constant input level x0[c] per channel (NEXT-2)."""
        x0 = np.ascontiguousarray(np.broadcast_to(np.asarray(x0, dtype=np.float64), (self.n_ch,)))
        if self._lib.filark_oracle_set_initial_condition(self._h, x0.ctypes.data):
            raise RuntimeError("oracle set_initial_condition failed")

    def get_state(self):
        """(state [n_ch][2 n_sec + 2] float64: z1,z2 per section, sta, lta; samples seen)."""
        out = np.empty((self.n_ch, 2 * self.n_sec + 2), dtype=np.float64)
        g = ctypes.c_longlong(0)
        if self._lib.filark_oracle_get_state(self._h, out.ctypes.data, ctypes.addressof(g)):
            raise RuntimeError("oracle get_state failed")
        return out, int(g.value)

    def set_state(self, state, g: int):
        state = np.ascontiguousarray(state, dtype=np.float64)
        assert state.shape == (self.n_ch, 2 * self.n_sec + 2)
        if self._lib.filark_oracle_set_state(self._h, state.ctypes.data, int(g)):
            raise RuntimeError("oracle set_state failed")

    def trace_f64(self, x: np.ndarray, channel: int = 0):
        """Double-precision input, one channel: returns (y, sta, lta) as float64 (for pins).
        Does not advance the warm-up counter."""
        x = np.ascontiguousarray(x, dtype=np.float64)
        y = np.empty_like(x); s = np.empty_like(x); l = np.empty_like(x)
        rc = self._lib.filark_oracle_trace_f64(self._h, int(channel), x.ctypes.data, x.size,
                                               y.ctypes.data, s.ctypes.data, l.ctypes.data)
        if rc:
            raise RuntimeError("oracle trace failed")
        return y, s, l


EVENT_DTYPE = np.dtype([("t_on", "<i8"), ("t_off", "<i8"), ("channel", "<i4"), ("peak", "<f4")])


class OracleTrigger:
    """On/off trigger with hysteresis on the CF, state carried across pushes (NEXT-1, reading R24)."""

    def __init__(self, n_ch: int, thr_on: float, thr_off: float, layout: int = CHANNEL_MAJOR):
        lib = _load()
        self._lib, self.n_ch, self.layout = lib, int(n_ch), int(layout)
        self._h = lib.filark_oracle_trigger_create(self.n_ch, float(thr_on), float(thr_off))
        if not self._h:
            raise ValueError("filark_oracle_trigger_create rejected its arguments")

    def push(self, cf: np.ndarray, cap: int = 1 << 20) -> np.ndarray:
        """cf: float32 chunk in the trigger's layout; returns the events this chunk closed."""
        cf = np.ascontiguousarray(cf, dtype=np.float32)
        n_t = cf.shape[1] if self.layout == CHANNEL_MAJOR else cf.shape[0]
        sc, sn = (n_t, 1) if self.layout == CHANNEL_MAJOR else (1, self.n_ch)
        out = np.zeros(cap, dtype=EVENT_DTYPE)
        n = self._lib.filark_oracle_trigger_push(self._h, cf.ctypes.data, n_t, sc, sn, out.ctypes.data, cap)
        if n < 0 or n > cap:
            raise RuntimeError("oracle trigger push failed or overflowed")
        return out[:n].copy()

    def close(self):
        if getattr(self, "_h", None):
            self._lib.filark_oracle_trigger_destroy(self._h)
            self._h = None

    __del__ = close


BOX_DTYPE = np.dtype([("t_on", "<i8"), ("t_off", "<i8"), ("ch_lo", "<i4"), ("ch_hi", "<i4"), ("peak", "<f4"),
                      ("n_events", "<i4")])


def oracle_associate(events: np.ndarray, ch_gap: int, t_gap: int) -> np.ndarray:
    """Per-channel trigger events -> time-channel-bounded events ("(t_on, t_off, channel
    range, peak cf) -- the monitor contract's actual output"; "a list of time-channel-bounded
    events", :132 "each described by a time and channel extent").  The paper gives no rule; reading R30 in
    DESIGN.md, written out as it is defined:

      two events are LINKED if their channels differ by at most ch_gap and their half-open intervals
      [t_on, t_off) come within t_gap samples of each other:  t_on1 < t_off2 + t_gap  and  t_on2 < t_off1 + t_gap
      (t_gap = 0: they overlap);
      a BOX is a connected component of the link graph: t_on = the smallest t_on, t_off = the largest t_off,
      [ch_lo, ch_hi] = the channel extent, peak = the largest peak, n_events = its size;
      boxes are listed in rising (t_on, ch_lo, t_off, ch_hi).

    The link matrix is built by comparing every pair; the components come from scipy's
    connected_components (a library primitive as one step)."""
    from scipy.sparse import csr_matrix
    from scipy.sparse.csgraph import connected_components
    ev = np.asarray(events, dtype=EVENT_DTYPE)
    n = ev.shape[0]
    if n == 0:
        return np.zeros(0, dtype=BOX_DTYPE)
    ch = ev["channel"].astype(np.int64); t0 = ev["t_on"].astype(np.int64); t1 = ev["t_off"].astype(np.int64)
    link = (np.abs(ch[:, None] - ch[None, :]) <= int(ch_gap)) & (t0[:, None] < t1[None, :] + int(t_gap)) & \
           (t0[None, :] < t1[:, None] + int(t_gap))
    n_box, label = connected_components(csr_matrix(link), directed=False)
    out = np.zeros(n_box, dtype=BOX_DTYPE)
    for b in range(n_box):
        m = ev[label == b]
        out[b] = (m["t_on"].min(), m["t_off"].max(), m["channel"].min(), m["channel"].max(), m["peak"].max(), m.shape[0])
    return out[np.lexsort((out["ch_hi"], out["t_off"], out["ch_lo"], out["t_on"]))]


def oracle_zero_phase(x: np.ndarray, sos) -> np.ndarray:
    """Zero-phase (forward-backward) filtering of a bounded window, channel-major x [n_ch][n_t]
    (PAPER.md:77 the display filter is "either a zero-phase or causal IIR filter ...
    applied only to the currently visible buffer").  Reading R29: the cascade run forward from the
    steady state of the window's first sample, the result reversed in time, run again from the steady
    state of ITS first sample, and reversed back -- no padding.  Built from the oracle's own steps."""
    x = np.ascontiguousarray(x, dtype=np.float32)
    n_ch = x.shape[0]
    fwd = Oracle(n_ch, sos, 1, 1)
    fwd.set_initial_condition(x[:, 0].astype(np.float64))
    y, _ = fwd.push(x, want_cf=False)
    fwd.close()
    r = np.ascontiguousarray(y[:, ::-1])
    bwd = Oracle(n_ch, sos, 1, 1)
    bwd.set_initial_condition(r[:, 0].astype(np.float64))
    z, _ = bwd.push(r, want_cf=False)
    bwd.close()
    return np.ascontiguousarray(z[:, ::-1])


DECIMATE_MODES = {"drop": 0, "peak": 1, "linear": 2}
EMA_MODES = {"mean": 0, "demean": 1, "agc": 2}


def oracle_decimate(x: np.ndarray, mode: str, width: int, layout: int = CHANNEL_MAJOR) -> np.ndarray:
    """Display decimation (NEXT-4, reading R25).  x: [n_ch][n_t] or [n_t][n_ch]; returns [n_ch][width] or [width][n_ch]."""
    lib = _load()
    x = np.ascontiguousarray(x, dtype=np.float32)
    if layout == CHANNEL_MAJOR:
        n_ch, n_t = x.shape
        out = np.empty((n_ch, width), dtype=np.float32)
        rc = lib.filark_oracle_decimate(x.ctypes.data, n_ch, n_t, n_t, 1, DECIMATE_MODES[mode], width, out.ctypes.data, width, 1)
    else:
        n_t, n_ch = x.shape
        out = np.empty((width, n_ch), dtype=np.float32)
        rc = lib.filark_oracle_decimate(x.ctypes.data, n_ch, n_t, 1, n_ch, DECIMATE_MODES[mode], width, out.ctypes.data, 1, n_ch)
    if rc:
        raise ValueError("filark_oracle_decimate rejected its arguments")
    return out


class OracleEma:
    """Streaming first-order operators (NEXT-3, reading R26): running mean, de-mean, running AGC."""

    def __init__(self, n_ch: int, n_len: int, mode: str, eps: float = 0.0, layout: int = CHANNEL_MAJOR):
        lib = _load()
        self._lib, self.n_ch, self.layout = lib, int(n_ch), int(layout)
        self._h = lib.filark_oracle_ema_create(self.n_ch, int(n_len), EMA_MODES[mode], float(eps))
        if not self._h:
            raise ValueError("filark_oracle_ema_create rejected its arguments")

    def push(self, x: np.ndarray) -> np.ndarray:
        x = np.ascontiguousarray(x, dtype=np.float32)
        n_t = x.shape[1] if self.layout == CHANNEL_MAJOR else x.shape[0]
        sc, sn = (n_t, 1) if self.layout == CHANNEL_MAJOR else (1, self.n_ch)
        out = np.empty_like(x)
        if self._lib.filark_oracle_ema_push(self._h, x.ctypes.data, n_t, sc, sn, out.ctypes.data):
            raise RuntimeError("oracle ema push failed")
        return out

    def close(self):
        if getattr(self, "_h", None):
            self._lib.filark_oracle_ema_destroy(self._h)
            self._h = None

    __del__ = close
