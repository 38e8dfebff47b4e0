"""Pins for the float64 oracle (oracle/filark_oracle.c) against things other than itself.

The paper prints no worked numerical example, so every pin comes from
the mathematics of the operator PAPER.md:109, 121, 255 names (cascaded SOS, causal,
sample-wise, state carried exactly) and of the CF BASELINE.json north_star names
(recursive STA/LTA): closed forms, invariants, library special cases, brute force.
Each pin is chosen so that a plausible mistake (dropped term, wrong sign, swapped b/a,
off-by-one in the state delay, STA/LTA swapped, warm-up miscounted) fails at least one.
"""
import os

import numpy as np
import pytest
from scipy import signal

from oracle import Oracle
from oracle.oracle import CHANNEL_MAJOR, TIME_MAJOR
from paper_2605_20132_b200.workloads import CONFIGS, design_sos

IDENT = np.array([[1.0, 0, 0, 1.0, 0, 0]])
RNG = np.random.default_rng(12345)


def _trace(sos, x, sta=1, lta=1):
    o = Oracle(1, sos, sta, lta)
    y, s, l = o.trace_f64(np.asarray(x, dtype=np.float64))
    o.close()
    return y, s, l


def _impulse(n):
    x = np.zeros(n); x[0] = 1.0
    return x


# --------------------------------------------------------------------------- single biquad
def _g_complex(r, th, n):
    k = np.arange(n)
    return r ** k * np.sin((k + 1) * th) / np.sin(th)


@pytest.mark.parametrize("r,th", [(0.9, 0.3), (0.999, 0.01), (0.5, 2.5), (0.99999, 0.004)])
def test_impulse_closed_form_complex_poles(r, th):
    """h[n] = b0 g[n] + b1 g[n-1] + b2 g[n-2], g[n] = r^n sin((n+1)th)/sin(th) (textbook)."""
    n = 400
    b = np.array([0.7, -0.3, 0.45])
    a1, a2 = -2 * r * np.cos(th), r * r
    g = _g_complex(r, th, n)
    h = b[0] * g
    h[1:] += b[1] * g[:-1]
    h[2:] += b[2] * g[:-2]
    y, _, _ = _trace(np.array([[*b, 1.0, a1, a2]]), _impulse(n))
    assert np.max(np.abs(y - h)) <= 1e-12 * np.max(np.abs(h)) * max(1.0, 1 / (1 - r) * 1e-2)


def test_impulse_closed_form_real_and_double_poles():
    n = 200
    k = np.arange(n)
    p1, p2 = 0.8, -0.35
    g = (p1 ** (k + 1) - p2 ** (k + 1)) / (p1 - p2)
    y, _, _ = _trace(np.array([[1.0, 0, 0, 1.0, -(p1 + p2), p1 * p2]]), _impulse(n))
    assert np.allclose(y, g, rtol=1e-12, atol=1e-15)
    p = 0.6
    g = (k + 1) * p ** k
    y, _, _ = _trace(np.array([[1.0, 0, 0, 1.0, -2 * p, p * p]]), _impulse(n))
    assert np.allclose(y, g, rtol=1e-12, atol=1e-15)


def test_numerator_taps_and_delay():
    """Pure FIR section: output is exactly b0 x[n] + b1 x[n-1] + b2 x[n-2] (catches state-delay
    off-by-one and swapped b1/b2)."""
    x = RNG.standard_normal(50)
    b = np.array([0.25, -1.5, 3.0])
    y, _, _ = _trace(np.array([[*b, 1.0, 0.0, 0.0]]), x)
    ref = b[0] * x
    ref[1:] += b[1] * x[:-1]
    ref[2:] += b[2] * x[:-2]
    assert np.allclose(y, ref, rtol=0, atol=1e-14)


def test_a0_normalisation():
    """Reading R5: coefficients are divided by a0 once; scaling a row changes nothing."""
    sos = design_sos(CONFIGS["cfg1"])
    x = RNG.standard_normal(500)
    y0, _, _ = _trace(sos, x)
    sos2 = sos.copy(); sos2[1] *= 4.0; sos2[3] *= -0.5      # exact powers of two
    y1, _, _ = _trace(sos2, x)
    assert np.array_equal(y0, y1)


# --------------------------------------------------------------------------- bandpass cascade
def _freq_resp(sos, w):
    z = np.exp(-1j * w)
    h = np.ones_like(z)
    for s in sos:
        h = h * (s[0] + s[1] * z + s[2] * z * z) / (s[3] + s[4] * z + s[5] * z * z)
    return h


@pytest.mark.parametrize("name", list(CONFIGS))
def test_design_is_butterworth_bandpass(name):
    """Reading R2/R3: N sections, |H|^2 = 1/2 at both edges, |H(0)| = |H(pi)| = 0, max gain 1."""
    w = CONFIGS[name]
    sos = design_sos(w)
    assert sos.shape == (w.order, 6)
    edges = 2 * np.pi * np.array(w.band) / w.fs
    assert np.allclose(np.abs(_freq_resp(sos, edges)) ** 2, 0.5, rtol=1e-9)
    assert np.abs(_freq_resp(sos, np.array([0.0, np.pi]))).max() < 1e-9
    grid = np.linspace(edges[0], edges[1], 2001)
    assert abs(np.abs(_freq_resp(sos, grid)).max() - 1.0) < 1e-9


@pytest.mark.parametrize("name,settle", [("cfg1", 30000), ("cfg2", 15000), ("cfg4", 4000)])
def test_zero_gain_at_dc_and_nyquist(name, settle):
    """Constant input and alternating +-1 decay to zero through the bandpass cascade."""
    sos = design_sos(CONFIGS[name])
    y, _, _ = _trace(sos, np.ones(settle))
    assert np.abs(y[-200:]).max() < 1e-6 * np.abs(y).max()
    alt = np.where(np.arange(settle) % 2 == 0, 1.0, -1.0)
    y, _, _ = _trace(sos, alt)
    assert np.abs(y[-200:]).max() < 1e-6 * max(np.abs(y).max(), 1e-3)


@pytest.mark.parametrize("name,f_hz", [("cfg1", 20.0), ("cfg1", 50.0), ("cfg2", 2.0), ("cfg4", 700.0)])
def test_steady_state_sinusoid_matches_transfer_function(name, f_hz):
    """After the transient, a sinusoid comes out scaled by |H| and shifted by arg H, with H
    evaluated from the sos polynomials (independent of the recurrence)."""
    w = CONFIGS[name]
    sos = design_sos(w)
    n = 60000
    om = 2 * np.pi * f_hz / w.fs
    t = np.arange(n)
    y, _, _ = _trace(sos, np.cos(om * t))
    h = _freq_resp(sos, np.array([om]))[0]
    ref = np.abs(h) * np.cos(om * t + np.angle(h))
    assert np.max(np.abs(y[-2000:] - ref[-2000:])) < 1e-7


def test_linearity():
    sos = design_sos(CONFIGS["cfg3"])
    x1, x2 = RNG.standard_normal(3000), RNG.standard_normal(3000)
    al, be = 0.37, -2.25
    y1, _, _ = _trace(sos, x1)
    y2, _, _ = _trace(sos, x2)
    y12, _, _ = _trace(sos, al * x1 + be * x2)
    assert np.max(np.abs(y12 - (al * y1 + be * y2))) < 1e-11 * np.max(np.abs(y12))


# --------------------------------------------------------------------------- brute force
def test_brute_force_expanded_difference_equation():
    """n <= 64, 2 sections: multiply out the section polynomials and evaluate the 4th-order
    difference equation directly (no states), in extended precision."""
    sos = np.array([[0.2, 0.4, 0.2, 1.0, -1.2, 0.5],
                    [1.0, -2.0, 1.0, 2.0, -2.4, 1.3]])
    b = np.convolve(sos[0, :3], sos[1, :3]).astype(np.longdouble)
    a = np.convolve(sos[0, 3:], sos[1, 3:]).astype(np.longdouble)
    x = RNG.standard_normal(64)
    y = np.zeros(64, dtype=np.longdouble)
    for n in range(64):
        acc = np.longdouble(0)
        for k in range(5):
            if n - k >= 0:
                acc += b[k] * np.longdouble(x[n - k])
        for k in range(1, 5):
            if n - k >= 0:
                acc -= a[k] * y[n - k]
        y[n] = acc / a[0]
    got, _, _ = _trace(sos, x)
    assert np.max(np.abs(got - y.astype(np.float64))) < 1e-13 * np.max(np.abs(got))


def test_brute_force_convolution_with_closed_form_impulse_response():
    r, th = 0.93, 0.7
    n = 64
    g = _g_complex(r, th, n)
    h = 1.0 * g
    h[1:] += -1.0 * g[:-1]                         # b = [1, -1, 0]
    x = RNG.standard_normal(n)
    ref = np.array([sum(h[k] * x[m - k] for k in range(m + 1)) for m in range(n)])
    y, _, _ = _trace(np.array([[1.0, -1.0, 0.0, 1.0, -2 * r * np.cos(th), r * r]]), x)
    assert np.allclose(y, ref, rtol=1e-12, atol=1e-14)


# --------------------------------------------------------------------------- library special cases
@pytest.mark.parametrize("name", list(CONFIGS))
def test_matches_scipy_sosfilt(name):
    sos = design_sos(CONFIGS[name])
    x = RNG.standard_normal(5000)
    y, _, _ = _trace(sos, x)
    ref = signal.sosfilt(sos, x)
    assert np.max(np.abs(y - ref)) < 1e-10 * np.max(np.abs(ref))


def test_averages_match_scipy_lfilter():
    x = RNG.standard_normal(4000)
    ns, nl = 37, 911
    _, s, l = _trace(IDENT, x, ns, nl)
    e = x * x
    for got, n in ((s, ns), (l, nl)):
        c = 1.0 / n
        ref = signal.lfilter([c], [1.0, -(1.0 - c)], e)
        assert np.max(np.abs(got - ref)) < 1e-12 * np.max(np.abs(ref))


# --------------------------------------------------------------------------- STA / LTA
def test_cf_closed_form_constant_energy():
    """e == 1: sta[n] = 1 - (1-1/Ns)^(n+1); cf = sta/lta once g >= lta_len, 0 before (R10)."""
    ns, nl, n = 20, 300, 2000
    o = Oracle(1, IDENT, ns, nl)
    x = np.where(np.arange(n) % 3 == 0, -1.0, 1.0).astype(np.float32)[None, :]
    _, cf = o.push(x)
    k = np.arange(n)
    sta = 1 - (1 - 1 / ns) ** (k + 1)
    lta = 1 - (1 - 1 / nl) ** (k + 1)
    ref = np.where(k >= nl, sta / lta, 0.0)
    assert np.all(cf[0, :nl] == 0.0)
    assert cf[0, nl] != 0.0
    assert np.max(np.abs(cf[0] - ref)) < 2e-7


def test_cf_energy_step_closed_form_and_bound():
    """From steady state E0, a step to E1: cf(k) = (E0 as^k + E1(1-as^k))/(E0 al^k + E1(1-al^k))
    with k counted from the first stepped sample (inclusive); 0 <= cf <= lta_len/sta_len."""
    ns, nl = 150, 7500
    a0, a1 = 1.0, 10.0
    n0, n1 = 120000, 4000
    x = np.concatenate([np.full(n0, a0), np.full(n1, a1)]).astype(np.float32)[None, :]
    o = Oracle(1, IDENT, ns, nl)
    _, cf = o.push(x)
    k = np.arange(1, n1 + 1)
    al_s, al_l = 1 - 1 / ns, 1 - 1 / nl
    e0, e1 = a0 * a0, a1 * a1
    ref = (e0 * al_s ** k + e1 * (1 - al_s ** k)) / (e0 * al_l ** k + e1 * (1 - al_l ** k))
    assert np.max(np.abs(cf[0, n0:] - ref)) < 5e-6 * ref.max()
    assert cf.min() >= 0.0 and cf.max() <= nl / ns
    assert ref.max() > 15.0          # the step is actually seen as a trigger-sized CF


def test_cf_scale_invariance_is_bit_identical():
    w = CONFIGS["cfg1"]
    sos = design_sos(w)
    x = RNG.standard_normal((2, 4000)).astype(np.float32)
    o = Oracle(2, sos, w.sta_len, w.lta_len)
    f1, c1 = o.push(x)
    o.reset()
    f2, c2 = o.push(x * np.float32(8.0))
    assert np.array_equal(c1, c2)
    assert np.array_equal(f1 * np.float32(8.0), f2)


def test_dead_channel_gives_zero():
    w = CONFIGS["cfg1"]
    o = Oracle(2, design_sos(w), w.sta_len, w.lta_len)
    x = np.zeros((2, 3000), dtype=np.float32)
    x[1] = RNG.standard_normal(3000)
    f, c = o.push(x)
    assert np.all(f[0] == 0) and np.all(c[0] == 0)
    assert np.all(np.isfinite(c)) and c[1, w.lta_len:].max() > 0


def test_sta_and_lta_are_not_swapped():
    """After an amplitude increase the CF rises above 1 (STA reacts faster than LTA)."""
    o = Oracle(1, IDENT, 10, 200)
    x = np.concatenate([np.ones(5000), 3 * np.ones(50)]).astype(np.float32)[None, :]
    _, cf = o.push(x)
    assert abs(cf[0, 4999] - 1.0) < 1e-6 and cf[0, -1] > 3.0


def test_filt_is_float32_rounding_of_the_double_output():
    sos = design_sos(CONFIGS["cfg2"])
    x = RNG.standard_normal(2000).astype(np.float32)
    o = Oracle(1, sos, 50, 2000)
    f, _ = o.push(x[None, :])
    y, _, _ = _trace(sos, x.astype(np.float64))
    assert np.array_equal(f[0], y.astype(np.float32))


# --------------------------------------------------------------------------- chunk contract
def _chunks(n, sizes):
    out, p, i = [], 0, 0
    while p < n:
        s = min(sizes[i % len(sizes)], n - p)
        out.append((p, p + s)); p += s; i += 1
    return out


@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
@pytest.mark.parametrize("sizes", [[1000], [1], [1, 2, 3, 31, 32, 33, 97, 500], [7, 4096]])
def test_chunked_equals_whole_bit_identical(layout, sizes):
    """any chunking gives the whole-record output -- bit-identical here."""
    w = CONFIGS["cfg1"]
    sos = design_sos(w)
    n_ch, n_t = 3, 2600
    x = RNG.standard_normal((n_ch, n_t)).astype(np.float32)
    xs = x if layout == CHANNEL_MAJOR else np.ascontiguousarray(x.T)
    o = Oracle(n_ch, sos, w.sta_len, w.lta_len, layout)
    fw, cw = o.push(xs)
    o.reset()
    assert o.samples_seen == 0
    fp, cp = [], []
    for a, b in _chunks(n_t, sizes):
        blk = xs[:, a:b] if layout == CHANNEL_MAJOR else xs[a:b, :]
        f, c = o.push(blk)
        fp.append(f); cp.append(c)
    ax = 1 if layout == CHANNEL_MAJOR else 0
    assert np.array_equal(np.concatenate(fp, axis=ax), fw)
    assert np.array_equal(np.concatenate(cp, axis=ax), cw)
    assert o.samples_seen == n_t


def test_layouts_agree_and_threads_agree():
    w = CONFIGS["cfg2"]
    sos = design_sos(w)
    x = RNG.standard_normal((5, 3000)).astype(np.float32)
    oc = Oracle(5, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR)
    ot = Oracle(5, sos, w.sta_len, w.lta_len, TIME_MAJOR)
    fc, cc = oc.push(x)
    ft, ct = ot.push(np.ascontiguousarray(x.T), threads=3)
    assert np.array_equal(fc, ft.T) and np.array_equal(cc, ct.T)


def test_reset_restores_the_just_created_state():
    w = CONFIGS["cfg1"]
    sos = design_sos(w)
    x = RNG.standard_normal((2, 1500)).astype(np.float32)
    o = Oracle(2, sos, w.sta_len, w.lta_len)
    f1, c1 = o.push(x)
    o.push(x)
    o.reset()
    f2, c2 = o.push(x)
    assert np.array_equal(f1, f2) and np.array_equal(c1, c2)


def test_empty_push_is_a_no_op():
    o = Oracle(2, IDENT, 2, 4)
    f, c = o.push(np.zeros((2, 0), dtype=np.float32))
    assert f.shape == (2, 0) and o.samples_seen == 0


def test_create_rejects_bad_arguments():
    for args in [(0, IDENT, 1, 2), (1, IDENT, 0, 2), (1, IDENT, 3, 2),
                 (1, np.array([[1.0, 0, 0, 0.0, 0, 0]]), 1, 2)]:
        with pytest.raises(ValueError):
            Oracle(*args)


# --------------------------------------------------------------------------- stored fixture
def test_golden_fixture_regression():
    """tests/golden/oracle_small.txt was written by tests/golden/make_golden.py, which calls
    only oracle/.  It freezes the oracle's arithmetic: a later change must be deliberate."""
    path = os.path.join(os.path.dirname(__file__), "golden", "oracle_small.txt")
    from tests.golden.make_golden import golden_case
    sos, sta, lta, x = golden_case()
    tab = np.loadtxt(path)
    o = Oracle(x.shape[0], sos, sta, lta)
    f, c = o.push(x)
    got = np.stack([x.ravel(), f.ravel(), c.ravel()], axis=1)
    assert np.array_equal(got.astype(np.float32), tab.astype(np.float32))


# --------------------------------------------------------------------------- the fused path as a whole
@pytest.mark.parametrize("name", ["cfg1", "cfg3", "cfg5"])
def test_fused_path_matches_the_scipy_composition(name):
    """The whole path (cascade -> energy of the UNROUNDED output -> two averages -> ratio with the
    warm-up and the guard, state carried over ragged pushes) against the same chain built from
    library routines: scipy.signal.sosfilt, then lfilter for each average.  Pins the composition,
    not only its parts: order of the steps, which signal is squared, which average divides which,
    where the warm-up counter starts, what a chunk boundary does."""
    w = CONFIGS[name]
    sos = design_sos(w)
    sta, lta = 40, 700                      # short enough for the warm-up to end inside the record
    rng = np.random.default_rng(2024)
    n_ch, n_t = 3, 6000
    x = rng.standard_normal((n_ch, n_t)).astype(np.float32)
    x[1] *= 1e-3
    x[2, 2500:] = 0.0                       # a channel that dies: the averages decay, the guard never trips
    o = Oracle(n_ch, sos, sta, lta)
    fs, cs, p = [], [], 0
    for c in [1, 999, 1500, 7, 2048, 1445]:
        f, cf = o.push(np.ascontiguousarray(x[:, p:p + c]))
        fs.append(f); cs.append(cf); p += c
    o.close()
    assert p == n_t
    filt, cf = np.concatenate(fs, 1), np.concatenate(cs, 1)
    for ch in range(n_ch):
        y = signal.sosfilt(sos, x[ch].astype(np.float64))
        e = y * y
        s = signal.lfilter([1.0 / sta], [1.0, -(1.0 - 1.0 / sta)], e)
        l = signal.lfilter([1.0 / lta], [1.0, -(1.0 - 1.0 / lta)], e)
        ref_cf = np.where((np.arange(n_t) >= lta) & (l > 1e-30), s / np.where(l > 1e-30, l, 1.0), 0.0)
        assert np.max(np.abs(filt[ch] - y)) <= 1e-6 * np.max(np.abs(y))            # float32 rounding of y
        assert np.all(cf[ch, :lta] == 0.0) and cf[ch, lta] != 0.0                  # warm-up: exactly lta_len zeros
        assert np.max(np.abs(cf[ch] - ref_cf)) <= 2e-6 * np.max(np.abs(ref_cf))
