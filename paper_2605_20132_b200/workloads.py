"""Seeded synthetic DAS workloads (BASELINE.json `configs`; recipe: SURVEY.md 8(d)).

This module serves BOTH the CUDA path (tests, bench.py) and the oracle (tests, cpu_baseline),
and therefore holds none of the method's arithmetic: no filtering, no STA/LTA, no scan.  It
produces (a) the input array x, (b) the `sos` design through the library routine
scipy.signal.butter (filter design is outside the C ABI, reading R3), (c) the push schedule.

The paper measures on OOI ocean-cable files that are not available; these
inputs stand in for them with the shapes of BASELINE.json `configs`:
  - N(0,1) white noise everywhere;
  - 1/f-coloured noise (strong low-frequency hydrodynamic noise);
  - Ricker arrivals with linear moveout across channels;
  - moving traffic/vessel-like sources.
Generators run on any torch device; the SAME tensor must be handed to both sides of a
comparison (CPU and CUDA random streams differ for the same seed).
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional

import numpy as np
import torch

CHANNEL_MAJOR = 0  # [n_ch][n_t], time contiguous (BASELINE.json configs[0])
TIME_MAJOR = 1     # [n_t][n_ch], channel contiguous (PAPER.md:160 dims='nt_nc')


@dataclasses.dataclass(frozen=True)
class Workload:
    name: str
    n_ch: int
    n_t: int
    fs: float
    order: int          # Butterworth prototype order N -> N bandpass sections (reading R2)
    band: tuple         # (lo_hz, hi_hz)
    sta_len: int        # samples (reading R12)
    lta_len: int
    chunk: int          # nominal push length in samples; 0 = random lengths (cfg5)
    seed: int
    n_ricker: int
    ricker_f: tuple     # (f_lo, f_hi) Hz, uniform
    aperture: float     # Gaussian channel aperture sigma (channels); 0 = all channels (cfg1)
    coloured: bool
    n_moving: int = 0
    chunk_seed: int = 0
    chunk_range: tuple = (0, 0)

    def scaled(self, n_ch: Optional[int] = None, n_t: Optional[int] = None) -> "Workload":
        """Same recipe at a smaller shape (parity cases the oracle finishes in seconds)."""
        n_ch, n_t = n_ch or self.n_ch, n_t or self.n_t
        frac = (n_ch * n_t) / float(self.n_ch * self.n_t)      # keep the event density
        n_r = self.n_ricker if self.aperture <= 0.0 else max(2, int(round(self.n_ricker * frac)))
        n_m = max(1, int(round(self.n_moving * frac))) if self.n_moving else 0
        return dataclasses.replace(self, n_ch=n_ch, n_t=n_t, n_ricker=n_r, n_moving=n_m,
                                   name=f"{self.name}[{n_ch}x{n_t}]")


# BASELINE.json configs[0..4] == SURVEY.md cfg 1..5
CONFIGS = {
    "cfg1": Workload("cfg1", 256, 10_000, 1000.0, 4, (1.0, 50.0), 50, 1000, 1000, 1001,
                     5, (25.0, 25.0), 0.0, False),
    "cfg2": Workload("cfg2", 2000, 60_000, 1000.0, 4, (2.0, 100.0), 50, 2000, 1000, 1002,
                     50, (10.0, 40.0), 100.0, True),
    "cfg3": Workload("cfg3", 6000, 90_000, 1500.0, 8, (1.0, 200.0), 150, 7500, 1500, 1003,
                     200, (10.0, 40.0), 100.0, True, n_moving=20),
    "cfg4": Workload("cfg4", 10_000, 100_000, 10_000.0, 4, (100.0, 2000.0), 100, 5000, 1000, 1004,
                     1000, (500.0, 500.0), 50.0, False),
    "cfg5": Workload("cfg5", 6000, 900_000, 1500.0, 8, (0.5, 100.0), 300, 15_000, 0, 1005,
                     2000, (10.0, 40.0), 100.0, True, chunk_seed=2005, chunk_range=(64, 6000)),
}


def design_sos(w: Workload) -> np.ndarray:
    """Digital Butterworth bandpass via the library routine (pre-warped bilinear transform).
    Returns float64 [n_sec][6] = b0 b1 b2 a0 a1 a2, n_sec == w.order (reading R2)."""
    from scipy.signal import butter
    sos = butter(w.order, [w.band[0], w.band[1]], btype="bandpass", fs=w.fs, output="sos")
    return np.ascontiguousarray(sos, dtype=np.float64)


def push_schedule(w: Workload, n_t: Optional[int] = None) -> List[int]:
    """Chunk lengths of the streamed run; their sum is n_t."""
    n_t = int(n_t if n_t is not None else w.n_t)
    if w.chunk > 0:
        out = [w.chunk] * (n_t // w.chunk)
        if n_t % w.chunk:
            out.append(n_t % w.chunk)
        return out
    rng = np.random.default_rng(w.chunk_seed)
    out, left = [], n_t
    lo, hi = w.chunk_range
    while left > 0:
        c = int(rng.integers(lo, hi + 1))
        c = min(c, left)
        out.append(c)
        left -= c
    return out


def _ricker(tau: torch.Tensor, f: float, amp: float) -> torch.Tensor:
    a = (math.pi * f) ** 2 * tau * tau
    return amp * (1.0 - 2.0 * a) * torch.exp(-a)


def _coloured_noise(n_ch: int, n_t: int, gen: torch.Generator, device) -> torch.Tensor:
    """Per channel: white Gaussian shaped by f^-1/2 (power ~ 1/f), DC bin zeroed, sigma = 1."""
    wn = torch.randn((n_ch, n_t), generator=gen, device=device, dtype=torch.float32)
    spec = torch.fft.rfft(wn, dim=1)
    k = torch.arange(spec.shape[1], device=device, dtype=torch.float32)
    shape = torch.where(k > 0, k.clamp(min=1.0).rsqrt(), torch.zeros_like(k))
    out = torch.fft.irfft(spec * shape, n=n_t, dim=1)
    out = out / out.std(dim=1, keepdim=True).clamp(min=1e-12)
    return out


def generate(w: Workload, device="cpu", layout: int = CHANNEL_MAJOR,
             ch_block: int = 1000) -> torch.Tensor:
    """Return the float32 record, [n_ch][n_t] (channel-major) or [n_t][n_ch] (time-major)."""
    device = torch.device(device)
    gen = torch.Generator(device=device)
    gen.manual_seed(w.seed)
    n_ch, n_t = w.n_ch, w.n_t
    x = torch.empty((n_ch, n_t), device=device, dtype=torch.float32)
    for c0 in range(0, n_ch, ch_block):
        c1 = min(n_ch, c0 + ch_block)
        blk = torch.randn((c1 - c0, n_t), generator=gen, device=device, dtype=torch.float32)
        if w.coloured:
            blk += _coloured_noise(c1 - c0, n_t, gen, device)
        x[c0:c1] = blk

    # event parameters from a host RNG so that they do not depend on the device
    rng = np.random.default_rng(w.seed + 7)
    ch = torch.arange(n_ch, device=device, dtype=torch.float32)
    if w.aperture <= 0.0:
        # cfg1: centres at samples 1500 + 1500k on channel 0, moveout +2 samples/channel
        for k in range(w.n_ricker):
            tc0 = 1500 + 1500 * k
            _add_ricker(x, w, tc0, 0.0, w.ricker_f[0], 2.0, 0.0, 5.0, ch)
    else:
        for _ in range(w.n_ricker):
            tc = float(rng.uniform(0, n_t))
            cc = float(rng.uniform(0, n_ch))
            f = float(rng.uniform(w.ricker_f[0], w.ricker_f[1]))
            mo = float(rng.uniform(-4.0, 4.0))
            _add_ricker(x, w, tc, cc, f, mo, w.aperture, 5.0, ch)
    for _ in range(w.n_moving):
        f = float(rng.uniform(5.0, 20.0))
        v = float(rng.uniform(0.5, 3.0)) * (1.0 if rng.uniform() < 0.5 else -1.0)
        t0 = int(rng.integers(0, max(1, n_t - 1)))
        c0 = 0.0 if v > 0 else float(n_ch - 1)
        _add_moving(x, w, t0, c0, v, f, 2.0, 10.0)
    if layout == TIME_MAJOR:
        return x.t().contiguous()
    return x


def _add_ricker(x, w, tc, cc, f, moveout, aperture, amp, ch):
    n_ch, n_t = x.shape
    half = int(math.ceil(1.6 / f * w.fs)) + 1          # Ricker support ~ +-1.5/f seconds
    if aperture > 0.0:
        c_lo = max(0, int(cc - 3.5 * aperture)); c_hi = min(n_ch, int(cc + 3.5 * aperture) + 1)
    else:
        c_lo, c_hi = 0, n_ch
    if c_hi <= c_lo:
        return
    chs = ch[c_lo:c_hi]
    centre = tc + moveout * (chs - cc)                                  # samples, per channel
    t_lo = max(0, int(centre.min().item()) - half); t_hi = min(n_t, int(centre.max().item()) + half + 1)
    if t_hi <= t_lo:
        return
    t = torch.arange(t_lo, t_hi, device=x.device, dtype=torch.float32)
    tau = (t[None, :] - centre[:, None]) / w.fs
    wav = _ricker(tau, f, amp)
    wav = torch.where(tau.abs() * f <= 1.6, wav, torch.zeros_like(wav))
    if aperture > 0.0:
        wav = wav * torch.exp(-0.5 * ((chs - cc) / aperture) ** 2)[:, None]
    x[c_lo:c_hi, t_lo:t_hi] += wav


def _add_moving(x, w, t0, c0, v, f, amp, sigma):
    n_ch, n_t = x.shape
    dur = int(min(n_t - t0, (n_ch - 1) / abs(v)))
    if dur <= 0:
        return
    t = torch.arange(t0, t0 + dur, device=x.device, dtype=torch.float32)
    centre = c0 + v * (t - t0)
    off = torch.arange(-40, 41, device=x.device, dtype=torch.float32)
    cidx = torch.round(centre)[:, None] + off[None, :]                   # [dur, 81]
    valid = (cidx >= 0) & (cidx < n_ch)
    val = amp * torch.sin(2.0 * math.pi * f * t / w.fs)[:, None] * \
        torch.exp(-0.5 * ((cidx - centre[:, None]) / sigma) ** 2)
    ci = cidx.clamp(0, n_ch - 1).long()
    ti = t.long()[:, None].expand_as(ci)
    x.index_put_((ci[valid], ti[valid]), val[valid], accumulate=True)


def checksum(x: torch.Tensor) -> float:
    """Cheap content fingerprint recorded beside measurements."""
    return float(x.double().abs().sum().item())


def channel_shard(n_ch: int, rank: int, world: int):
    """[lo, hi) channel range of `rank` when one record is sharded over `world` GPUs: channels are
    independent (no halo, no exchange step), so contiguous, balanced row ranges are all there is."""
    base, extra = divmod(int(n_ch), int(world))
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)
