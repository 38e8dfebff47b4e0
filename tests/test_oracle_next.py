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
