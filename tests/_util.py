"""Shared helpers of the GPU parity tests (tolerances of BASELINE.json north_star)."""
import numpy as np
import torch

from oracle import Oracle
from paper_2605_20132_b200.workloads import CHANNEL_MAJOR, TIME_MAJOR

# north_star: per-channel relative L2 <= 1e-4 and max abs <= 1e-3 x per-channel max |y|,
# applied to both outputs (reading R16).
REL_L2_TOL = 1e-4
MAX_ABS_TOL = 1e-3


def channel_errors(got: np.ndarray, ref: np.ndarray):
    """got/ref: [n_ch][n_t] float arrays.  Returns (worst rel-L2, worst max-abs / max|ref|)."""
    got = got.astype(np.float64); ref = ref.astype(np.float64)
    num = np.sqrt(((got - ref) ** 2).sum(axis=1))
    den = np.sqrt((ref ** 2).sum(axis=1))
    mx = np.abs(ref).max(axis=1)
    ma = np.abs(got - ref).max(axis=1)
    live = den > 0
    rel = np.where(live, num / np.where(live, den, 1.0), num)
    mrel = np.where(mx > 0, ma / np.where(mx > 0, mx, 1.0), ma)
    return float(rel.max()), float(mrel.max())


def assert_parity(got, ref, what=""):
    assert np.all(np.isfinite(got)), f"{what}: non-finite output"
    rel, mrel = channel_errors(got, ref)
    assert rel <= REL_L2_TOL, f"{what}: per-channel rel-L2 {rel:.3e} > {REL_L2_TOL}"
    assert mrel <= MAX_ABS_TOL, f"{what}: max-abs/max|y| {mrel:.3e} > {MAX_ABS_TOL}"
    return rel, mrel


def as_cm(a: np.ndarray, layout: int) -> np.ndarray:
    return a if layout == CHANNEL_MAJOR else np.ascontiguousarray(a.T)


def split(n_t, sizes):
    out, p, i = [], 0, 0
    while p < n_t:
        s = min(int(sizes[i % len(sizes)]), n_t - p)
        out.append((p, p + s)); p += s; i += 1
    return out


def run_gpu(stream, x_dev: torch.Tensor, layout: int, bounds, want_filt=True, want_cf=True):
    """Push the record chunk by chunk (dense per-chunk tensors); returns full filt, cf on device."""
    filt = torch.empty_like(x_dev) if want_filt else None
    cf = torch.empty_like(x_dev) if want_cf else None
    for a, b in bounds:
        if layout == CHANNEL_MAJOR:
            xin = x_dev[:, a:b].contiguous()
        else:
            xin = x_dev[a:b, :].contiguous()
        f = torch.empty_like(xin) if want_filt else None
        c = torch.empty_like(xin) if want_cf else None
        stream.push(xin, f, c)
        if layout == CHANNEL_MAJOR:
            if want_filt: filt[:, a:b] = f
            if want_cf: cf[:, a:b] = c
        else:
            if want_filt: filt[a:b, :] = f
            if want_cf: cf[a:b, :] = c
    torch.cuda.synchronize()
    return filt, cf


def run_oracle(x_cm: np.ndarray, sos, sta, lta, threads=8):
    """Whole-record oracle on a channel-major float32 array."""
    o = Oracle(x_cm.shape[0], sos, sta, lta, CHANNEL_MAJOR)
    f, c = o.push(np.ascontiguousarray(x_cm), threads=threads)
    o.close()
    return f, c
