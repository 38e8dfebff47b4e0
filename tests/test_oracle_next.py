"""CPU pins of the oracle's NEXT-2 additions (steady-state initial condition, state export/import):
SURVEY.md 8(f), PAPER.md:255 ("a short transient determined by ... the initial condition"), :109,
:169 (state carried across chunk, file -- and here process -- boundaries).  None of the expected
values comes from the CUDA path."""
import numpy as np
import pytest
from scipy import signal

from oracle import Oracle
from paper_2605_20132_b200.workloads import CONFIGS, design_sos


def _designs():
    return {
        "cfg3 band-pass": design_sos(CONFIGS["cfg3"]),
        "low-pass": signal.butter(4, 0.08, "low", output="sos"),
        "high-pass": signal.butter(3, 0.2, "high", output="sos"),
        "a0 != 1": signal.butter(2, 0.3, "low", output="sos") * np.array([2.0, 2.0, 2.0, 2.0, 2.0, 2.0]),
    }


@pytest.mark.parametrize("name", list(_designs()))
def test_steady_state_condition_is_scipys_sosfilt_zi(name):
    """The library idiom `sosfilt(sos, x, zi=sosfilt_zi(sos) * x0)`: state of the step response."""
    sos = _designs()[name]
    x0 = np.array([3.0, -1.5, 0.0, 1000.0])
    o = Oracle(4, sos, 5, 40)
    o.set_initial_condition(x0)
    st, g = o.get_state()
    zi = signal.sosfilt_zi(sos / sos[:, 3:4])                  # [n_sec][2], for a unit step
    # scipy's zi of section k is for a unit step INTO THE CASCADE: it already includes the DC gain of
    # the sections in front of it
    for c in range(4):
        assert np.allclose(st[c, :2 * sos.shape[0]].reshape(-1, 2), zi * x0[c], rtol=1e-9, atol=1e-9 * (1 + abs(x0[c])))
    assert g == 40
    o.close()


def test_constant_input_from_steady_state_has_no_transient():
    """Closed form: with the steady-state condition a constant input gives the constant H(1) x0 from
    the first sample on, the averages sit at (H(1) x0)^2 and cf = 1 at once (the warm-up is over)."""
    sos = signal.butter(4, 0.08, "low", output="sos")
    h1 = np.prod(sos[:, :3].sum(1) / sos[:, 3:].sum(1))
    x0 = np.array([2.5, -4.0])
    o = Oracle(2, sos, 7, 50)
    o.set_initial_condition(x0)
    x = np.repeat(x0[:, None], 300, axis=1).astype(np.float32)
    f, c = o.push(x)
    assert np.allclose(f, (h1 * x0)[:, None], rtol=1e-6)
    assert np.allclose(c, 1.0, rtol=1e-6)
    # from rest the same input has a transient: the condition matters
    o2 = Oracle(2, sos, 7, 50)
    f2, _ = o2.push(x)
    assert np.abs(f2[:, 0] - h1 * x0).max() > 0.5
    o.close(); o2.close()


def test_state_round_trip_is_bit_identical():
    """push A, export, import into a fresh oracle, push B == push A || B, bit for bit."""
    w = CONFIGS["cfg3"]
    sos = design_sos(w)
    rng = np.random.default_rng(3)
    x = rng.standard_normal((3, 5000)).astype(np.float32)
    whole = Oracle(3, sos, 20, 300)
    fw, cw = whole.push(x)
    a = Oracle(3, sos, 20, 300)
    fa, ca = a.push(x[:, :1234])
    st, g = a.get_state()
    assert g == 1234 and st.shape == (3, 2 * sos.shape[0] + 2)
    b = Oracle(3, sos, 20, 300)
    b.set_state(st, g)
    fb, cb = b.push(x[:, 1234:])
    assert np.array_equal(np.concatenate([fa, fb], 1), fw)
    assert np.array_equal(np.concatenate([ca, cb], 1), cw)
    for o in (whole, a, b):
        o.close()


def test_lowpass_and_highpass_match_scipy():
    """The operator is any SOS cascade (PAPER.md:109 names band-pass, low-pass and high-pass wrappers)."""
    rng = np.random.default_rng(5)
    x = rng.standard_normal((2, 3000)).astype(np.float32)
    for sos in (signal.butter(4, 0.08, "low", output="sos"), signal.butter(3, 0.2, "high", output="sos")):
        o = Oracle(2, sos, 10, 100)
        f, _ = o.push(x)
        ref = signal.sosfilt(sos, x.astype(np.float64), axis=1)
        assert np.abs(f - ref).max() <= 2e-7 * np.abs(ref).max() + 1e-7
        o.close()


# ---- NEXT-1: on/off trigger on the CF (reading R24) -------------------------------------------
from oracle import OracleTrigger  # noqa: E402


def _ramp_cf():
    """Hand-built CF of 3 channels with transitions at known indices."""
    n = 400
    cf = np.zeros((3, n), dtype=np.float32)
    # channel 0: rises through thr_on = 4 at 100 (value 4.0 exactly counts: >=), peak 9 at 130, falls
    # below thr_off = 2 at 180; a bump between the thresholds at 220..240 must not trigger
    cf[0, 100:180] = 4.0; cf[0, 130] = 9.0; cf[0, 179] = 2.0            # 2.0 is NOT below thr_off
    cf[0, 180] = 1.99
    cf[0, 220:240] = 3.0
    # channel 1: two events; between them cf dips to 2.5 (between the thresholds): stays on
    cf[1, 50:90] = 5.0; cf[1, 60:70] = 2.5; cf[1, 90] = 0.5
    cf[1, 300:310] = 7.5
    # channel 2: on at the very last sample: no event yet
    cf[2, n - 1] = 100.0
    return cf


def test_trigger_hand_built_ramps():
    cf = _ramp_cf()
    t = OracleTrigger(3, 4.0, 2.0)
    ev = t.push(cf)
    got = [(int(e["channel"]), int(e["t_on"]), int(e["t_off"]), float(e["peak"])) for e in ev]
    assert got == [(0, 100, 180, 9.0), (1, 50, 90, 5.0), (1, 300, 310, 7.5)]
    # the event of channel 2 closes in the next push, with the index where it began
    ev2 = t.push(np.zeros((3, 10), dtype=np.float32))
    assert [(int(e["channel"]), int(e["t_on"]), int(e["t_off"]), float(e["peak"])) for e in ev2] == [(2, 399, 400, 100.0)]
    t.close()


@pytest.mark.parametrize("sizes", [[400], [1] * 400, [100, 80, 1, 219], [179, 1, 1, 219], [129, 2, 269]])
def test_trigger_is_chunk_invariant(sizes):
    """Events that straddle push boundaries: any chunking gives the same events."""
    cf = _ramp_cf()
    whole = OracleTrigger(3, 4.0, 2.0)
    ref = np.sort(whole.push(cf), order=["t_on", "channel"])
    t = OracleTrigger(3, 4.0, 2.0)
    parts, p = [], 0
    for s in sizes:
        parts.append(t.push(cf[:, p:p + s])); p += s
    got = np.sort(np.concatenate(parts), order=["t_on", "channel"])
    assert np.array_equal(got, ref)
    whole.close(); t.close()


def test_trigger_layouts_agree_and_arguments_are_checked():
    from oracle.oracle import TIME_MAJOR
    cf = _ramp_cf()
    a = OracleTrigger(3, 4.0, 2.0)
    b = OracleTrigger(3, 4.0, 2.0, TIME_MAJOR)
    ea = np.sort(a.push(cf), order=["t_on", "channel"])
    eb = np.sort(b.push(np.ascontiguousarray(cf.T)), order=["t_on", "channel"])
    assert np.array_equal(ea, eb)
    for bad in ((0.0, 0.0), (2.0, 3.0), (4.0, 0.0)):
        with pytest.raises(ValueError):
            OracleTrigger(3, *bad)
    a.close(); b.close()


def test_trigger_against_brute_force_on_random_cf():
    """Independent restatement: intervals of a run-length encoding of the hysteresis state computed
    with numpy (forward fill of the last decisive sample)."""
    rng = np.random.default_rng(9)
    cf = np.abs(rng.standard_normal((5, 3000))).astype(np.float32) * 2.0
    thr_on, thr_off = np.float32(3.5), np.float32(1.0)
    t = OracleTrigger(5, float(thr_on), float(thr_off))
    ev = np.sort(t.push(cf), order=["channel", "t_on"])
    exp = []
    for c in range(5):
        dec = np.where(cf[c] >= thr_on, 1, np.where(cf[c] < thr_off, 0, -1))       # decisive samples
        idx = np.where(dec >= 0, np.arange(dec.size), -1)
        last = np.maximum.accumulate(idx)
        state = np.where(last >= 0, dec[np.maximum(last, 0)], 0)                 # state AFTER each sample
        prev = np.r_[0, state[:-1]]
        ons = np.flatnonzero((prev == 0) & (state == 1)); offs = np.flatnonzero((prev == 1) & (state == 0))
        for a, b in zip(ons, offs):
            exp.append((c, a, b, cf[c, a:b].max()))
    assert len(ev) == len(exp) and len(exp) > 10
    for e, (c, a, b, pk) in zip(ev, exp):
        assert (int(e["channel"]), int(e["t_on"]), int(e["t_off"])) == (c, a, b) and e["peak"] == pk
    t.close()


# ---- NEXT-4: display decimation (reading R25) --------------------------------------------------
from oracle import OracleEma, oracle_decimate  # noqa: E402
from oracle.oracle import TIME_MAJOR as _TM  # noqa: E402


def test_decimate_small_worked_example():
    """10 samples to 4 columns: columns [0,2) [2,5) [5,7) [7,10)."""
    x = np.array([[1, -3, 2, 2, -2, 0.5, -0.5, 4, -9, 9]], dtype=np.float32)
    assert oracle_decimate(x, "drop", 4).tolist() == [[1.0, 2.0, 0.5, 4.0]]
    assert oracle_decimate(x, "peak", 4).tolist() == [[-3.0, 2.0, 0.5, -9.0]]         # first of equal magnitudes
    lin = oracle_decimate(x, "linear", 4)[0]
    assert np.allclose(lin, [1.0, 2.0, -0.5, 9.0])                                      # positions 0, 3, 6, 9
    assert np.allclose(oracle_decimate(x, "linear", 3)[0], [1.0, (-2 + 0.5) / 2, 9.0])  # positions 0, 4.5, 9


@pytest.mark.parametrize("n_t,width", [(1000, 128), (2048, 2048), (100, 300), (90_000, 2048), (7, 1)])
def test_decimate_against_numpy(n_t, width):
    rng = np.random.default_rng(n_t + width)
    x = rng.standard_normal((3, n_t)).astype(np.float32)
    a = (np.arange(width + 1, dtype=np.int64) * n_t) // width
    lo, hi = a[:-1], np.maximum(a[1:], a[:-1] + 1)
    assert np.array_equal(oracle_decimate(x, "drop", width), x[:, lo])
    pk = oracle_decimate(x, "peak", width)
    for c in range(3):
        for j in (0, width // 3, width - 1):
            seg = x[c, lo[j]:hi[j]]
            assert pk[c, j] == seg[np.argmax(np.abs(seg))]
    assert (np.abs(pk) >= np.abs(x[:, lo])).all()                       # the envelope is never below the dropped sample
    ref = np.stack([np.interp(np.linspace(0, n_t - 1, width) if width > 1 else [0.0], np.arange(n_t), x[c].astype(np.float64)) for c in range(3)])
    assert np.allclose(oracle_decimate(x, "linear", width), ref, rtol=1e-6, atol=1e-6)
    # time-major input gives the transposed result
    for mode in ("drop", "peak", "linear"):
        assert np.array_equal(oracle_decimate(np.ascontiguousarray(x.T), mode, width, _TM).T, oracle_decimate(x, mode, width))


# ---- NEXT-3: streaming first-order operators (reading R26) ------------------------------------
def test_ema_operators_against_lfilter_and_closed_forms():
    rng = np.random.default_rng(2)
    x = (rng.standard_normal((2, 4000)) * 3.0 + 1.5).astype(np.float32)
    N = 40
    m = signal.lfilter([1.0 / N], [1.0, -(1.0 - 1.0 / N)], x.astype(np.float64), axis=1)
    o = OracleEma(2, N, "mean"); assert np.allclose(o.push(x), m, rtol=1e-6, atol=1e-7); o.close()
    o = OracleEma(2, N, "demean"); assert np.allclose(o.push(x), x - m, rtol=1e-5, atol=1e-6); o.close()
    ma = signal.lfilter([1.0 / N], [1.0, -(1.0 - 1.0 / N)], np.abs(x.astype(np.float64)), axis=1)
    o = OracleEma(2, N, "agc", 1e-3); assert np.allclose(o.push(x), x / (ma + 1e-3), rtol=1e-5); o.close()
    # closed form: a constant input c gives m[n] = c (1 - (1 - 1/N)^(n+1))
    c = np.full((1, 300), 2.5, dtype=np.float32)
    o = OracleEma(1, N, "mean")
    assert np.allclose(o.push(c)[0], 2.5 * (1 - (1 - 1 / N) ** (np.arange(300) + 1)), rtol=1e-6); o.close()
    # AGC of a scaled input: the output does not change (eps = 0) once the average is non-zero
    o1, o2 = OracleEma(2, N, "agc"), OracleEma(2, N, "agc")
    assert np.allclose(o1.push(x), o2.push(8.0 * x), rtol=1e-6); o1.close(); o2.close()


@pytest.mark.parametrize("mode", ["mean", "demean", "agc"])
def test_ema_operators_are_chunk_invariant_bitwise(mode):
    rng = np.random.default_rng(4)
    x = rng.standard_normal((3, 2000)).astype(np.float32)
    a = OracleEma(3, 25, mode, 1e-6); whole = a.push(x); a.close()
    b = OracleEma(3, 25, mode, 1e-6)
    parts, p = [], 0
    for s in [1, 2, 3, 500, 31, 1463]:
        parts.append(b.push(x[:, p:p + s])); p += s
    b.close()
    assert np.array_equal(np.concatenate(parts, 1), whole)


# ---- NEXT-2: zero-phase display-filter mode (reading R29) -------------------------------------
from oracle import oracle_zero_phase  # noqa: E402


@pytest.mark.parametrize("name", ["low-pass", "high-pass", "cfg3 band-pass"])
def test_zero_phase_is_scipys_sosfiltfilt_without_padding(name):
    sos = _designs()[name]
    rng = np.random.default_rng(12)
    x = (rng.standard_normal((3, 4000)) + 2.0).astype(np.float32)
    got = oracle_zero_phase(x, sos)
    ref = signal.sosfiltfilt(sos, x.astype(np.float64), axis=1, padtype=None)
    # (the intermediate signal is rounded to float32 once in the oracle: outputs of the path are float32)
    assert np.abs(got - ref).max() <= 5e-6 * max(1.0, np.abs(ref).max())


def test_zero_phase_commutes_with_time_reversal():
    """Zero phase: filtering the time-reversed window gives the time-reversed output up to the edge
    effects of the two initial conditions -- exactly so for a window that starts and ends at rest."""
    sos = signal.butter(4, 0.1, "low", output="sos")
    x = np.zeros((1, 6000), dtype=np.float32)
    x[0, 2500:3500] = np.hanning(1000).astype(np.float32)
    a = oracle_zero_phase(x, sos)
    b = oracle_zero_phase(np.ascontiguousarray(x[:, ::-1]), sos)[:, ::-1]
    assert np.abs(a - b).max() <= 1e-5
    # no delay: the output of a symmetric pulse is symmetric about the same centre
    assert np.abs(a[0, 2000:4000] - a[0, 2000:4000][::-1]).max() <= 1e-2 * a.max()


# ---- NEXT-1, second half: per-channel events -> time-channel boxes (reading R30) ----------------------
import os  # noqa: E402

from oracle import BOX_DTYPE, EVENT_DTYPE, oracle_associate  # noqa: E402


def _read_associate_golden():
    ev, boxes = [], {"B": [], "C": [], "D": []}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "associate_small.txt")):
        f = line.split()
        if not f or f[0] == "#":
            continue
        if f[0] == "E":
            ev.append((int(f[1]), int(f[2]), int(f[3]), float(f[4])))
        else:
            boxes[f[0]].append((int(f[1]), int(f[2]), int(f[3]), int(f[4]), float(f[5]), int(f[6])))
    return np.array(ev, dtype=EVENT_DTYPE), {k: np.array(v, dtype=BOX_DTYPE) for k, v in boxes.items()}


def test_associate_worked_example():
    """The hand-derived fixture (tests/golden/associate_small.txt), three settings of the two gaps."""
    ev, want = _read_associate_golden()
    for key, (cg, tg) in {"B": (1, 0), "C": (2, 0), "D": (1, 60)}.items():
        got = oracle_associate(ev, cg, tg)
        assert got.tolist() == want[key].tolist(), key
        # the order of the input does not matter
        assert oracle_associate(ev[::-1], cg, tg).tolist() == want[key].tolist()


def _associate_brute(ev, ch_gap, t_gap):
    """Union-find in plain Python loops over every pair (tiny inputs only)."""
    n = len(ev)
    parent = list(range(n))

    def find(i):
        while parent[i] != i:
            i = parent[i]
        return i
    for i in range(n):
        for j in range(i):
            a, b = ev[i], ev[j]
            if abs(int(a["channel"]) - int(b["channel"])) <= ch_gap and a["t_on"] < b["t_off"] + t_gap and b["t_on"] < a["t_off"] + t_gap:
                parent[find(i)] = find(j)
    groups = {}
    for i in range(n):
        groups.setdefault(find(i), []).append(i)
    out = []
    for idx in groups.values():
        m = ev[idx]
        out.append((int(m["t_on"].min()), int(m["t_off"].max()), int(m["channel"].min()), int(m["channel"].max()),
                    float(m["peak"].max()), len(idx)))
    return sorted(out, key=lambda b: (b[0], b[2], b[1], b[3]))


def _random_events(rng, n, n_ch, t_max, dur):
    t_on = rng.integers(0, t_max, n)
    ev = np.zeros(n, dtype=EVENT_DTYPE)
    ev["t_on"] = t_on; ev["t_off"] = t_on + rng.integers(1, dur, n)
    ev["channel"] = rng.integers(0, n_ch, n); ev["peak"] = rng.random(n).astype(np.float32) * 10
    return ev


@pytest.mark.parametrize("seed", range(6))
def test_associate_equals_pairwise_union_find(seed):
    rng = np.random.default_rng(seed)
    ev = _random_events(rng, 60, 12, 400, 60)
    for cg, tg in ((0, 0), (1, 0), (1, 25), (3, 5)):
        got = oracle_associate(ev, cg, tg)
        assert [tuple(b) for b in got.tolist()] == _associate_brute(ev, cg, tg)


def test_associate_invariants_and_special_cases():
    rng = np.random.default_rng(42)
    ev = _random_events(rng, 500, 40, 5000, 80)
    boxes = oracle_associate(ev, 1, 0)
    assert boxes["n_events"].sum() == ev.shape[0]                       # every event in exactly one box
    assert np.all(boxes["t_on"] < boxes["t_off"]) and np.all(boxes["ch_lo"] <= boxes["ch_hi"])
    for e in ev:                                                        # ... and inside some box of at least its peak
        inside = (boxes["t_on"] <= e["t_on"]) & (e["t_off"] <= boxes["t_off"]) & (boxes["ch_lo"] <= e["channel"]) & \
                 (e["channel"] <= boxes["ch_hi"]) & (boxes["peak"] >= e["peak"])
        assert inside.any()
    # gaps so large that everything is linked: one box, the bounding box of all events
    one = oracle_associate(ev, 1000, 10**9)
    assert one.shape[0] == 1 and one[0]["n_events"] == 500
    assert (one[0]["t_on"], one[0]["t_off"], one[0]["ch_lo"], one[0]["ch_hi"]) == \
           (ev["t_on"].min(), ev["t_off"].max(), ev["channel"].min(), ev["channel"].max())
    assert one[0]["peak"] == ev["peak"].max()
    # larger gaps only merge: the number of boxes never grows
    assert oracle_associate(ev, 2, 0).shape[0] <= boxes.shape[0] and oracle_associate(ev, 1, 50).shape[0] <= boxes.shape[0]
    # events that cannot be linked (one per channel, channels two apart): the identity
    lone = np.zeros(5, dtype=EVENT_DTYPE)
    lone["t_on"] = 10; lone["t_off"] = 20; lone["channel"] = np.arange(5) * 2; lone["peak"] = 1.0
    b = oracle_associate(lone, 1, 0)
    assert b.shape[0] == 5 and np.all(b["n_events"] == 1) and b["ch_lo"].tolist() == [0, 2, 4, 6, 8]
    # touching intervals do not overlap (half-open): [10, 20) and [20, 30) on adjacent channels
    two = np.zeros(2, dtype=EVENT_DTYPE)
    two["t_on"] = [10, 20]; two["t_off"] = [20, 30]; two["channel"] = [3, 4]; two["peak"] = 1.0
    assert oracle_associate(two, 1, 0).shape[0] == 2 and oracle_associate(two, 1, 1).shape[0] == 1
    assert oracle_associate(np.zeros(0, dtype=EVENT_DTYPE), 1, 0).shape[0] == 0
