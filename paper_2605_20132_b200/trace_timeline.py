"""Per-warp device timeline of back-to-back pushes (tuning aid; DESIGN.md 6/7 quote its output).

    python -m paper_2605_20132_b200.trace_timeline [n_t] [pushes]

Builds csrc/filark_stream.cu with -DFK_TRACE into a library of its own (the product library has no
instrumentation), streams `pushes` chunks of cfg3's shape (6,000 channels x n_t samples, 8
sections) back to back and prints, from the %globaltimer stamps every warp leaves at fixed points
of filark_push_cm_kernel: the time between consecutive points (median, p10, p90) and the life of
a warp.  Points: 0 kernel entry, 1 control slot read, 7 first loads issued, 8 first tile landed,
2 dependents released, 3 tile in shared memory, 4 tile done, 5 work loop left, 6 exit.
"""
from __future__ import annotations

import collections
import ctypes
import os
import subprocess
import sys

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_PKG, "libfilark_stream_trace.so")


def build() -> str:
    src = os.path.join(_PKG, "csrc", "filark_stream.cu")
    cmd = ["nvcc", "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
           "-Xcompiler", "-fPIC", "-shared", "-DFK_TRACE", "-o", _LIB, src]
    subprocess.run(cmd, check=True)
    return _LIB


def main():
    import torch
    from . import stream as fstream
    from .workloads import CONFIGS, design_sos
    n_t = int(sys.argv[1]) if len(sys.argv) > 1 else 1500
    pushes = int(sys.argv[2]) if len(sys.argv) > 2 else 12
    if not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(os.path.join(_PKG, "csrc", "filark_kernels.cuh")):
        build()
    fstream.LIB_PATH = _LIB                      # the binding loads the instrumented build
    fstream._lib = None
    lib = fstream.load_library()
    lib.filark_trace_read.argtypes = [ctypes.c_void_p, ctypes.c_uint, ctypes.c_int]
    w = CONFIGS["cfg3"]
    sos = design_sos(w)
    xs = [torch.randn(w.n_ch, n_t, device="cuda") for _ in range(pushes)]
    fs = [torch.empty_like(x) for x in xs]
    cs = [torch.empty_like(x) for x in xs]
    s = fstream.FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len)
    for _ in range(2):
        for x, f, c in zip(xs, fs, cs):
            s.push(x, f, c)
    torch.cuda.synchronize()
    lib.filark_trace_read(None, 0, 1)
    for x, f, c in zip(xs, fs, cs):
        s.push(x, f, c)
    torch.cuda.synchronize()
    n_words = 16 * 4096 * 16 * 2
    buf = np.zeros(n_words, dtype=np.uint64)
    lib.filark_trace_read(buf.ctypes.data, n_words, 1)
    s.destroy()
    b = buf.reshape(-1, 2)
    b = b[b[:, 1] != 0]
    t = b[:, 0].astype(np.int64)
    m = b[:, 1]
    ep = (m >> np.uint64(48)).astype(int)
    gw = ((m >> np.uint64(32)) & np.uint64(0xFFFF)).astype(int)
    ev = (m & np.uint64(0x7FF)).astype(int)
    t = (t - t.min()) / 1000.0
    eps = sorted(set(ep.tolist()))
    starts = [t[(ep == e) & (ev == 0)].min() for e in eps]
    print(f"{len(eps)} pushes of {w.n_ch} x {n_t}; push period (first kernel entry to the next push's): "
          f"{np.median(np.diff(starts)):.1f} us")
    e = eps[len(eps) // 2]
    sel = np.where(ep == e)[0]
    per_warp = collections.defaultdict(list)
    for i in sel:
        per_warp[gw[i]].append((t[i], ev[i]))
    gaps = collections.defaultdict(list)
    life = collections.defaultdict(list)
    for v in per_warp.values():
        v.sort()
        for (ta, ea), (tb, eb) in zip(v, v[1:]):
            gaps[(ea, eb)].append(tb - ta)
        life[sum(1 for _, x in v if x == 4)].append(v[-1][0] - v[0][0])
    print("from -> to   count   median   p10   p90  (us)")
    for k in sorted(gaps):
        g = np.array(gaps[k])
        print(f"{k[0]:>4} -> {k[1]:<4} {len(g):6d} {np.median(g):8.2f} {np.percentile(g, 10):6.2f} {np.percentile(g, 90):6.2f}")
    for n, v in sorted(life.items()):
        print(f"warps with {n} tiles: {len(v)}, life median {np.median(v):.1f} us")


if __name__ == "__main__":
    main()
