"""B200-native fused SOS + STA/LTA stream path of FiLark's signal-processing layer.

Public names mirror the C ABI in include/filark_stream.h (argument marshalling only;
every step of the path runs in the sm_100a kernels of csrc/):

    from paper_2605_20132_b200 import FilarkStream
    s = FilarkStream(n_ch, sos, sta_len, lta_len, layout=CHANNEL_MAJOR)
    s.push(d_in, d_filt, d_cf)     # torch CUDA tensors, asynchronous on the current stream
    s.reset()

`workloads` (seeded synthetic inputs) is importable without the CUDA library; everything in
`stream` fails loudly if libfilark_stream.so is missing -- there is no CPU fallback.
"""
from .workloads import CHANNEL_MAJOR, TIME_MAJOR  # noqa: F401


def __getattr__(name):
    if name in ("FilarkStream", "FilarkError", "load_library", "library_path", "push_host"):
        from . import stream
        return getattr(stream, name)
    raise AttributeError(name)
