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


# ---- NEXT-1: trigger / event emission on the CF ------------------------------------------------
from oracle import OracleTrigger  # noqa: E402


def _burst_record(n_ch, n_t, seed, n_bursts=60):
    """cfg3-shaped noise with short strong bursts at random (time, channel): the CF rises steeply
    through the thresholds (few ties) and falls back slowly."""
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=n_t)
    x = generate(w, device="cpu").numpy().copy()
    rng = np.random.default_rng(seed)
    for _ in range(n_bursts):
        c = int(rng.integers(0, n_ch)); t = int(rng.integers(8000, n_t - 400)); n = int(rng.integers(40, 300))
        x[c, t:t + n] += (rng.uniform(6.0, 15.0) * np.sin(2 * np.pi * rng.uniform(20, 120) / 1500.0 * np.arange(n))).astype(np.float32)
    return w, x


def _oracle_events(x, sos, w, thr_on, thr_off):
    ref_f, ref_c = run_oracle(x, sos, w.sta_len, w.lta_len)
    t = OracleTrigger(x.shape[0], thr_on, thr_off)
    ev = t.push(ref_c)
    t.close()
    return ref_c, np.sort(ev, order=["channel", "t_on"])


def _compare_events(got, ref, ref_cf, thr_on, thr_off, what):
    """Bit-exact (channel, t_on, t_off) away from threshold ties.  Tie rule (R24): an event
    boundary may differ between the two sides only where the oracle's cf is within 1e-4 (relative) of
    the threshold it is compared with at one of the two boundary samples."""
    got = np.sort(got, order=["channel", "t_on"])
    key = lambda e: (int(e["channel"]), int(e["t_on"]), int(e["t_off"]))
    gs, rs = {key(e): e for e in got}, {key(e): e for e in ref}
    assert len(rs) >= 20, f"{what}: only {len(rs)} events in the reference: the case tests nothing"
    same = set(gs) & set(rs)
    for k in same:
        assert abs(float(gs[k]["peak"]) - float(rs[k]["peak"])) <= 1e-4 * float(rs[k]["peak"]), (what, k)

    def tie(c, t, thr):
        return any(0 <= u < ref_cf.shape[1] and abs(float(ref_cf[c, u]) - thr) <= 1e-4 * thr for u in (t - 1, t, t + 1))
    odd = (set(gs) ^ set(rs))
    for c, a, b in odd:
        assert tie(c, a, thr_on) or tie(c, b, thr_off), f"{what}: event {(c, a, b)} differs away from a tie"
    assert len(odd) <= max(2, len(rs) // 10), f"{what}: {len(odd)} of {len(rs)} events differ"
    return len(same)


@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
@pytest.mark.parametrize("sizes,many", [([60_000], False), ([1500], False), ([1500], True), ([777, 4096, 33, 2500], True)])
def test_trigger_events_match_the_oracle(cuda_device, layout, sizes, many):
    thr_on, thr_off = 3.0, 1.5
    w, x = _burst_record(96, 60_000, 31)
    sos = design_sos(w)
    ref_cf, ref_ev = _oracle_events(x, sos, w, thr_on, thr_off)
    xd = torch.from_numpy(x if layout == CHANNEL_MAJOR else np.ascontiguousarray(x.T)).to(cuda_device)
    s = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len, layout)
    s.set_trigger(thr_on, thr_off, 10_000)
    bounds = split(w.n_t, sizes)
    cut = (lambda a, b: xd[:, a:b].contiguous()) if layout == CHANNEL_MAJOR else (lambda a, b: xd[a:b, :].contiguous())
    chunks = [cut(a, b) for a, b in bounds]
    cfs = [torch.empty_like(c) for c in chunks]
    if many:
        s.push_many(chunks, None, cfs)
    else:
        for c, o in zip(chunks, cfs):
            s.push(c, None, o)
    got, dropped = s.pop_events()
    assert dropped == 0
    n_same = _compare_events(got, ref_ev, ref_cf, thr_on, thr_off, f"layout {layout} {sizes} many={many}")
    assert n_same >= 20
    # the list is empty now; the same record again after reset gives the same events again
    again, _ = s.pop_events()
    assert len(again) == 0
    s.reset()
    s.push_many(chunks, None, cfs)
    got2, _ = s.pop_events()
    assert np.array_equal(np.sort(got2, order=["channel", "t_on"]), np.sort(got, order=["channel", "t_on"]))
    s.destroy()


def test_trigger_time_major_without_cf_output(cuda_device):
    """Time-major, events only (d_cf = NULL): only the warps whose tile matters to the trigger stage their cf --
    this used to wait at a CTA barrier for the others (found by `bench.py --layout tm`); watchdog by timeout."""
    thr_on, thr_off = 3.0, 1.5
    w, x = _burst_record(80, 30_000, 51, n_bursts=30)
    sos = design_sos(w)
    ref_cf, ref_ev = _oracle_events(x, sos, w, thr_on, thr_off)
    xd = torch.from_numpy(np.ascontiguousarray(x.T)).to(cuda_device)
    f = torch.empty_like(xd)
    s = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len, TIME_MAJOR)
    s.set_trigger(thr_on, thr_off, 10_000)
    chunks = [xd[a:b, :].contiguous() for a, b in split(w.n_t, [1500, 700, 4096])]
    s.push_many(chunks, [f[a:b, :] for a, b in split(w.n_t, [1500, 700, 4096])], None)
    done = torch.cuda.Event(); done.record()
    import time
    t0 = time.time()
    while not done.query():
        assert time.time() - t0 < 60.0, "the launch does not complete"
        time.sleep(0.01)
    got, dropped = s.pop_events()
    assert dropped == 0
    assert _compare_events(got, ref_ev, ref_cf, thr_on, thr_off, "time-major, no cf output") >= 10
    s.destroy()


def test_events_to_time_channel_boxes(cuda_device):
    """NEXT-1's output form: the events the trigger emitted on the GPU, associated into time-channel boxes by
    filark_events_associate, against the oracle's association of the same list (reading R30); and the boxes
    of the cfg3 recipe's moving sources do span channel ranges."""
    from oracle import oracle_associate
    from paper_2605_20132_b200.stream import associate_events
    w = CONFIGS["cfg3"].scaled(n_ch=400, n_t=45_000)
    sos = design_sos(w)
    xd = generate(w, device="cpu").to(cuda_device)
    s = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len)
    s.set_trigger(4.0, 2.0, 1 << 18)
    s.push(xd, None, torch.empty_like(xd))
    ev, dropped = s.pop_events()
    s.destroy()
    assert dropped == 0 and len(ev) > 50
    for ch_gap, t_gap in ((1, 0), (2, 75)):
        boxes, total = associate_events(ev, ch_gap, t_gap)
        ref = oracle_associate(ev, ch_gap, t_gap)
        assert total == ref.shape[0] and sorted(map(tuple, boxes.tolist())) == sorted(map(tuple, ref.tolist()))
        assert boxes["n_events"].sum() == len(ev)
    assert total < len(ev) and (boxes["ch_hi"] - boxes["ch_lo"]).max() >= 3       # arrivals seen on neighbouring channels merge


def test_trigger_without_cf_output_and_list_overflow(cuda_device):
    """Events only (d_cf = NULL, filt kept): same events; a short list drops and counts the rest;
    thr_on = thr_off = 0 switches the trigger off; a pop with too little room consumes nothing."""
    thr_on, thr_off = 3.0, 1.5
    w, x = _burst_record(64, 40_000, 41, n_bursts=40)
    sos = design_sos(w)
    ref_cf, ref_ev = _oracle_events(x, sos, w, thr_on, thr_off)
    xd = torch.from_numpy(x).to(cuda_device)
    f = torch.empty_like(xd)
    s = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len)
    s.set_trigger(thr_on, thr_off, 5000)
    s.push(xd, f, None)
    got, dropped = s.pop_events()
    _compare_events(got, ref_ev, ref_cf, thr_on, thr_off, "events only")
    n_all = len(got)
    s.reset(); s.set_trigger(thr_on, thr_off, 7)
    s.push(xd, f, None)
    s._ev_cap = 3
    with pytest.raises(FilarkError):
        s.pop_events()                                       # room for 3, 7 pending: nothing consumed
    s._ev_cap = 7
    got, dropped = s.pop_events()
    assert len(got) == 7 and dropped == n_all - 7
    s.reset(); s.set_trigger(0.0, 0.0, 0)
    s.push(xd, f, None)
    got, dropped = s.pop_events()
    assert len(got) == 0 and dropped == 0
    for bad in ((2.0, 3.0, 10), (-1.0, 0.5, 10), (3.0, 1.0, 0)):
        with pytest.raises(FilarkError):
            s.set_trigger(*bad)
    s.destroy()


# ---- NEXT-3: streaming first-order operators; NEXT-4: display decimation -------------------------
from oracle import OracleEma, oracle_decimate  # noqa: E402
from paper_2605_20132_b200.ops import FilarkEma, decimate  # noqa: E402


@pytest.mark.parametrize("mode", ["mean", "demean", "agc"])
@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
@pytest.mark.parametrize("n_len", [1, 40, 5000])
def test_ema_operators(cuda_device, mode, layout, n_len):
    """Running mean / de-mean / running AGC against the oracle, pushed in ragged chunks (the state is
    carried; tiles of 512 samples, so the chunk lengths cover several tiles and ragged tails)."""
    n_ch, n_t = 150, 12_345
    rng = np.random.default_rng(n_len)
    x = (rng.standard_normal((n_ch, n_t)) * 2.0 + 0.7).astype(np.float32)
    eps = 1e-3 if mode == "agc" else 0.0
    o = OracleEma(n_ch, n_len, mode, eps)
    ref = o.push(x)
    o.close()
    xd = torch.from_numpy(x if layout == CHANNEL_MAJOR else np.ascontiguousarray(x.T)).to(cuda_device)
    h = FilarkEma(n_ch, n_len, mode, eps, layout)
    outs = []
    for a, b in split(n_t, [4096, 1, 511, 512, 513, 3000]):
        xin = (xd[:, a:b] if layout == CHANNEL_MAJOR else xd[a:b, :]).contiguous()
        y = torch.empty_like(xin)
        h.push(xin, y)
        outs.append(y)
    got = torch.cat(outs, 1 if layout == CHANNEL_MAJOR else 0).cpu().numpy()
    if layout == TIME_MAJOR:
        got = got.T
    # (north-star bounds relative to the scale of the data the operator works on: de-mean with N = 1 is
    # identically zero in the oracle)
    num = np.sqrt(((got - ref).astype(np.float64) ** 2).sum(1))
    den = np.maximum(np.sqrt((ref.astype(np.float64) ** 2).sum(1)), np.sqrt((x.astype(np.float64) ** 2).sum(1)) * 1e-2)
    assert (num <= 2e-5 * den).all(), (num / den).max()
    assert np.abs(got - ref).max() <= 1e-3 * max(np.abs(ref).max(), 1e-2 * np.abs(x).max())
    # reset: the same record again gives the same output bit for bit; in place is allowed
    h.reset()
    xin = xd.clone()
    h.push(xin, xin)
    again = xin.cpu().numpy()
    if layout == TIME_MAJOR:
        again = again.T
    assert np.abs(again - ref).max() <= 1e-3 * max(np.abs(ref).max(), 1e-2 * np.abs(x).max())
    h.destroy()


@pytest.mark.parametrize("mode", ["mean", "demean", "agc"])
@pytest.mark.parametrize("n_ch", [100, 64, 4])
def test_ema_time_major_aligned_rows(cuda_device, mode, n_ch):
    """Time-major with a channel count that is a multiple of four: the rows arrive through the cp.async ring
    (n_ch = 100: the last block of 32 channels is partial; 64: complete blocks; 4: one 16-byte piece per row);
    chunk lengths around the tile of 256 rows, one chunk in place."""
    n_t, n_len = 3_000, 300
    rng = np.random.default_rng(n_ch)
    x = (rng.standard_normal((n_ch, n_t)) * 2.0 + 0.7).astype(np.float32)
    eps = 1e-3 if mode == "agc" else 0.0
    o = OracleEma(n_ch, n_len, mode, eps)
    ref = o.push(x)
    o.close()
    xd = torch.from_numpy(np.ascontiguousarray(x.T)).to(cuda_device)
    h = FilarkEma(n_ch, n_len, mode, eps, TIME_MAJOR)
    outs = []
    for i, (a, b) in enumerate(split(n_t, [256, 255, 257, 1, 768, 513, 950])):
        xin = xd[a:b, :].contiguous()
        y = xin if i == 4 else torch.empty_like(xin)
        h.push(xin, y)
        outs.append(y)
    got = torch.cat(outs, 0).cpu().numpy().T
    num = np.sqrt(((got - ref).astype(np.float64) ** 2).sum(1))
    den = np.maximum(np.sqrt((ref.astype(np.float64) ** 2).sum(1)), np.sqrt((x.astype(np.float64) ** 2).sum(1)) * 1e-2)
    assert (num <= 2e-5 * den).all(), (num / den).max()
    assert np.abs(got - ref).max() <= 1e-3 * max(np.abs(ref).max(), 1e-2 * np.abs(x).max())
    h.destroy()


@pytest.mark.parametrize("mode", ["drop", "peak", "linear"])
@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
@pytest.mark.parametrize("n_t,width", [(90_000, 2048), (1500, 2048), (2048, 2048), (100_003, 777), (33, 1)])
def test_display_decimation(cuda_device, mode, layout, n_t, width):
    """drop and peak are selections: bit-exact; linear within fp32 rounding of the oracle's double."""
    n_ch = 97
    rng = np.random.default_rng(n_t + width)
    x = rng.standard_normal((n_ch, n_t)).astype(np.float32)
    x[:, ::7] = np.round(x[:, ::7])                                    # equal magnitudes: the first one wins
    xl = x if layout == CHANNEL_MAJOR else np.ascontiguousarray(x.T)
    ref = oracle_decimate(xl, mode, width, layout)
    got = decimate(torch.from_numpy(xl).to(cuda_device), mode, width, layout).cpu().numpy()
    if mode == "linear":
        assert np.abs(got - ref).max() <= 1e-5 * max(1.0, np.abs(ref).max())
    else:
        assert np.array_equal(got, ref)


def test_decimation_of_the_stream_outputs_and_argument_checks(cuda_device):
    """The step behind S7 in the viewer: the filtered tile and its CF go to a
    2048-column display buffer; pitched input (a window of a longer record); bad arguments."""
    w = CONFIGS["cfg3"].scaled(n_ch=64, n_t=30_000)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    s = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len)
    xd = x.to(cuda_device); f = torch.empty_like(xd); c = torch.empty_like(xd)
    s.push(xd, f, c)
    env = decimate(f, "peak", 2048)
    torch.cuda.synchronize()
    assert np.array_equal(env.cpu().numpy(), oracle_decimate(f.cpu().numpy(), "peak", 2048))
    # a window [5000, 25000) of every channel: pitch = the record's row length
    from paper_2605_20132_b200.ops import _lib, DECIMATE_MODES
    out = torch.empty((w.n_ch, 512), device=cuda_device)
    st = _lib().filark_decimate(f.data_ptr() + 4 * 5000, w.n_ch, 20_000, w.n_t, 0, DECIMATE_MODES["drop"], 512, out.data_ptr(), None)
    assert st == 0
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), oracle_decimate(f[:, 5000:25_000].cpu().numpy(), "drop", 512))
    for bad in (dict(n_t=0), dict(width=0), dict(mode=7), dict(layout=3), dict(pitch=10)):
        a = dict(n_t=20_000, width=512, mode=0, layout=0, pitch=w.n_t); a.update(bad)
        assert _lib().filark_decimate(f.data_ptr(), w.n_ch, a["n_t"], a["pitch"], a["layout"], a["mode"], a["width"], out.data_ptr(), None) == 1
    assert _lib().filark_decimate(f.data_ptr(), w.n_ch, 20_000, w.n_t, 0, 0, 512, f.data_ptr() + 4096, None) == 1     # overlap
    s.destroy()


# ---- NEXT-2: zero-phase window mode -------------------------------------------------------------
from oracle import oracle_zero_phase  # noqa: E402


@pytest.mark.parametrize("name", ["lowpass4", "highpass3", "cfg3"])
@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
def test_zero_phase_window(cuda_device, name, layout):
    """Forward-backward filtering of a visible window against the oracle's composition;
    the stream's own carried state is not touched."""
    sos = FILTERS[name] if name != "cfg3" else design_sos(CONFIGS["cfg3"])
    n_ch, n_t = 80, 8_191
    rng = np.random.default_rng(17)
    x = (rng.standard_normal((n_ch, n_t)) + rng.uniform(-3, 3, (n_ch, 1))).astype(np.float32)
    ref = oracle_zero_phase(x, sos)
    xl = x if layout == CHANNEL_MAJOR else np.ascontiguousarray(x.T)
    xd = torch.from_numpy(xl).to(cuda_device)
    s = FilarkStream(n_ch, sos, 40, 900, layout)
    f0 = torch.empty_like(xd); c0 = torch.empty_like(xd)
    s.push(xd, f0, c0)                                    # the stream is somewhere in its record
    out = torch.empty_like(xd)
    s.zero_phase(xd, out)
    s.zero_phase(xd[:5000].contiguous() if layout == TIME_MAJOR else xd[:, :5000].contiguous(),
                 torch.empty((5000, n_ch) if layout == TIME_MAJOR else (n_ch, 5000), device=cuda_device))   # a smaller window reuses the temporaries
    got = out.cpu().numpy()
    got = got.T if layout == TIME_MAJOR else got
    scale = np.maximum(np.abs(ref).max(1), 1e-2 * np.abs(x).max(1))
    assert (np.abs(got - ref).max(1) <= 1e-3 * scale).all()
    num = np.sqrt(((got - ref).astype(np.float64) ** 2).sum(1)); den = np.sqrt((ref.astype(np.float64) ** 2).sum(1))
    assert (num <= 1e-4 * den + 5e-7 * np.abs(x).max(1) * np.sqrt(n_t)).all(), (num / den).max()
    # the stream goes on as if nothing had happened
    f1 = torch.empty_like(xd); c1 = torch.empty_like(xd)
    s.push(xd, f1, c1)
    s2 = FilarkStream(n_ch, sos, 40, 900, layout)
    g0 = torch.empty_like(xd); g1 = torch.empty_like(xd); d0 = torch.empty_like(xd); d1 = torch.empty_like(xd)
    s2.push(xd, g0, d0); s2.push(xd, g1, d1)
    torch.cuda.synchronize()
    assert torch.equal(f1, g1) and torch.equal(c1, d1)
    s.destroy(); s2.destroy()
