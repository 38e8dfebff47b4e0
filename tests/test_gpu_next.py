"""GPU parity of the NEXT rows of SURVEY.md 8(f), through the C ABI, against the float64 oracle.
NEXT-2: other filter types on the same kernels (PAPER.md:109 low-pass / high-pass wrappers), state
export / import across handles, steady-state initial condition."""
import struct

import numpy as np
import pytest
import torch
from scipy import signal

from oracle import Oracle
from paper_2605_20132_b200.stream import FilarkError, FilarkStream
from paper_2605_20132_b200.workloads import CHANNEL_MAJOR, TIME_MAJOR, CONFIGS, design_sos, generate
from tests._util import assert_parity, run_gpu, run_oracle, split

pytestmark = pytest.mark.gpu

FILTERS = {
    "lowpass4": signal.butter(4, 0.08, "low", output="sos"),
    "highpass3": signal.butter(3, 0.2, "high", output="sos"),
    "lowpass_near_dc": signal.butter(4, 0.004, "low", output="sos"),        # poles next to z = 1, zeros at z = -1
    "highpass_near_dc": signal.butter(4, 0.002, "high", output="sos"),      # poles and zeros next to z = 1
    "bandstop": signal.butter(2, [0.1, 0.3], "bandstop", output="sos"),
    "cheby1_band": signal.cheby1(3, 1.0, [0.05, 0.2], "band", output="sos"),
}


@pytest.mark.parametrize("name", list(FILTERS))
@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
def test_other_filter_types(cuda_device, name, layout):
    sos = FILTERS[name]
    n_ch, n_t = 70, 20_000
    rng = np.random.default_rng(11)
    x = (rng.standard_normal((n_ch, n_t)) + 0.5).astype(np.float32)        # with a DC level
    ref_f, ref_c = run_oracle(x, sos, 40, 900)
    xd = torch.from_numpy(x if layout == CHANNEL_MAJOR else np.ascontiguousarray(x.T)).to(cuda_device)
    s = FilarkStream(n_ch, sos, 40, 900, layout)
    f, c = run_gpu(s, xd, layout, split(n_t, [1500, 4096, 333, 7000]))
    f = f.cpu().numpy(); c = c.cpu().numpy()
    if layout == TIME_MAJOR:
        f, c = f.T, c.T
    assert_parity(f, ref_f, f"{name} filt")
    assert_parity(c, ref_c, f"{name} cf")
    s.destroy()


@pytest.mark.parametrize("cut", [1536, 1234, 4001])
def test_state_export_import_round_trip(cuda_device, cut):
    """push A, export, import into a NEW handle, push B == the oracle's A || B; the cuts leave 0, 10
    and 17 raw samples waiting in the handle (L = 24), which the export runs over the state."""
    w = CONFIGS["cfg3"].scaled(n_ch=130, n_t=12_000)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    ref_f, ref_c = run_oracle(x.numpy(), sos, w.sta_len, w.lta_len)
    xd = x.to(cuda_device)
    a = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len)
    fa, ca = run_gpu(a, xd[:, :cut].contiguous(), CHANNEL_MAJOR, split(cut, [1000]))
    blob = a.get_state()
    magic, n_ch, n_sec, sta, lta, seen = struct.unpack_from("<8siiiiQ", blob, 0)
    assert (magic, n_ch, n_sec, sta, lta, seen) == (b"FKSTATE1", w.n_ch, 8, w.sta_len, w.lta_len, cut)
    assert len(blob) == 64 + w.n_ch * (2 * 8 + 2) * 8
    a.destroy()
    b = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len)
    b.set_state(blob)
    assert b.samples_pushed == cut
    fb, cb = run_gpu(b, xd[:, cut:].contiguous(), CHANNEL_MAJOR, split(w.n_t - cut, [1500, 700]))
    f = torch.cat([fa, fb], 1).cpu().numpy(); c = torch.cat([ca, cb], 1).cpu().numpy()
    assert_parity(f, ref_f, "round trip filt")
    assert_parity(c, ref_c, "round trip cf")
    # regression guard well inside the tolerance: the hand-over itself costs nothing visible
    d = np.abs(f[:, cut:cut + 200] - ref_f[:, cut:cut + 200]).max() / np.abs(ref_f).max()
    assert d < 2e-5, d
    # export right after import gives the state back (to rounding of the float state)
    st1 = np.frombuffer(blob, dtype=np.float64, offset=64)
    b2 = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len)
    b2.set_state(blob)
    st2 = np.frombuffer(b2.get_state(), dtype=np.float64, offset=64)
    assert np.allclose(st1, st2, rtol=2e-7, atol=1e-30)
    b.destroy(); b2.destroy()


def test_state_blob_is_checked(cuda_device):
    sos = FILTERS["lowpass4"]
    a = FilarkStream(8, sos, 10, 100)
    blob = a.get_state()
    other = FilarkStream(9, sos, 10, 100)
    with pytest.raises(FilarkError) as e:
        other.set_state(blob)
    assert e.value.status == 1
    with pytest.raises(FilarkError):
        a.set_state(blob[:100])
    bad = bytearray(blob); bad[0:8] = b"NOTSTATE"
    with pytest.raises(FilarkError):
        a.set_state(bytes(bad))
    a.destroy(); other.destroy()


@pytest.mark.parametrize("name", ["lowpass4", "lowpass_near_dc", "highpass_near_dc"])
def test_steady_state_initial_condition(cuda_device, name):
    """Input = a DC level per channel + noise.  With the steady-state condition for that level the
    start-up transient is gone, exactly as in the oracle with the same condition."""
    sos = FILTERS[name]
    n_ch, n_t = 64, 9_000
    rng = np.random.default_rng(21)
    level = rng.uniform(-50.0, 50.0, n_ch).astype(np.float32)
    x = (level[:, None] + 0.1 * rng.standard_normal((n_ch, n_t))).astype(np.float32)
    o = Oracle(n_ch, sos, 30, 600)
    o.set_initial_condition(level.astype(np.float64))
    ref_f, ref_c = o.push(x)
    o.close()
    s = FilarkStream(n_ch, sos, 30, 600)
    s.set_initial_condition(level)
    assert s.samples_pushed == 600
    f, c = run_gpu(s, torch.from_numpy(x).to(cuda_device), CHANNEL_MAJOR, split(n_t, [1500, 1001]))
    f = f.cpu().numpy(); c = c.cpu().numpy()
    # north-star tolerance plus the documented fp32 input-range term (a DC level D in the
    # input costs about 6e-8 D of absolute error per sample, here bounded by 5e-7 D): a high-pass
    # removes the level from the output but not from the arithmetic
    scale = np.abs(ref_f).max(1)
    assert (np.abs(f - ref_f).max(1) <= 1e-3 * scale + 5e-6 * np.abs(level)).all()
    num = np.sqrt(((f - ref_f).astype(np.float64) ** 2).sum(1)); den = np.sqrt((ref_f.astype(np.float64) ** 2).sum(1))
    assert (num <= 1e-4 * den + 5e-7 * np.abs(level) * np.sqrt(n_t)).all()
    assert_parity(c, ref_c, f"{name} cf with initial condition")
    s.destroy()
