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
