"""CPU tests of the library's host side: the C-ABI .so loads and exports every declared symbol,
the state-space rewrite of each section is equivalent to the section it replaces, the float64
block powers are right, and the tiling of a push covers every sample exactly once.
No compute call is made (no GPU here)."""
import ctypes
import os
import re

import numpy as np
import pytest
from scipy import signal

from paper_2605_20132_b200 import build as fbuild
from paper_2605_20132_b200.workloads import CONFIGS, design_sos, push_schedule

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    fbuild.build_library()
    from paper_2605_20132_b200 import stream
    return stream


def _declared_symbols():
    names = []
    for hdr in ("filark_stream.h", "filark_debug.h", "filark_ops.h"):
        text = open(os.path.join(ROOT, "include", hdr)).read()
        text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
        names += re.findall(r"\b(filark_[a-z_0-9]+)\s*\(", text)
    return sorted(set(names))


def test_library_exports_every_declared_symbol(lib):
    cdll = ctypes.CDLL(lib.library_path())
    names = _declared_symbols()
    assert {"filark_stream_create", "filark_stream_push", "filark_stream_reset"} <= set(names)
    for n in names:
        assert hasattr(cdll, n), f"{n} declared in include/ but not exported"


def test_status_strings(lib):
    l = lib.load_library()
    for code in range(8):
        assert l.filark_status_string(code)


def _simulate(kinds, coefs, gain, x):
    """float64 simulation of the state-space cascade the kernels run."""
    v = gain * np.asarray(x, dtype=np.float64)
    for k in range(len(kinds)):
        A = coefs[k, :4].reshape(2, 2); B = coefs[k, 4:6]; C = coefs[k, 6:8]; D = coefs[k, 8]
        s = np.zeros(2); y = np.empty_like(v)
        for n in range(v.size):
            y[n] = C @ s + D * v[n]
            s = A @ s + B * v[n]
        v = y
    return v


@pytest.mark.parametrize("name", list(CONFIGS))
def test_state_space_rewrite_equals_sosfilt(lib, name):
    sos = design_sos(CONFIGS[name])
    kinds, coefs, gain = lib.debug_design(sos)
    x = np.random.default_rng(3).standard_normal(1500)
    ref = signal.sosfilt(sos, x)
    got = _simulate(kinds, coefs, gain, x)
    assert np.max(np.abs(got - ref)) < 1e-9 * np.max(np.abs(ref))
    # poles next to z = 1 must be in the delta form (all these designs have zeros at z = 1 there),
    # the rest in direct form II
    for k, s in enumerate(sos):
        assert kinds[k] == (2 if 1 + s[4] / s[3] + s[5] / s[3] < 0.05 else 0)


def test_rewrite_handles_odd_sections(lib):
    sos = np.array([[0.0, 1.0, 0.0, 1.0, -1.9, 0.9025 + 1e-4],     # b0 = 0, complex poles near z=1
                    [2.0, 0.5, 0.0, 2.0, -1.0, 0.0],               # first order, a0 != 1
                    [1.0, 0.0, 0.0, 1.0, 0.0, 0.0],                # identity
                    [0.3, 0.1, 0.2, 1.0, -1.6, 0.64],              # double real pole 0.8 (near z = 1, no zero there)
                    [1.0, 2.0, 1.0, 1.0, -1.95, 0.9512],           # complex poles near z = 1, zeros at z = -1
                    [1.0, -1.0, 0.0, 1.0, -0.999, 0.0],            # first-order high-pass, real pole near z = 1
                    [0.5, 0.3, 0.5, 1.0, 1.9, 0.9125]])            # complex poles near z = -1
    kinds, coefs, gain = lib.debug_design(sos)
    assert list(kinds) == [1, 0, 0, 3, 3, 2, 4]
    x = np.random.default_rng(4).standard_normal(400)
    ref = signal.sosfilt(sos / sos[:, 3:4], x)       # scipy wants a0 == 1
    got = _simulate(kinds, coefs, gain, x)
    assert np.max(np.abs(got - ref)) < 1e-10 * np.max(np.abs(ref))


def test_unstable_and_invalid_sections_are_rejected(lib):
    with pytest.raises(lib.FilarkError) as e:
        lib.debug_design(np.array([[1.0, 0, 0, 1.0, -2.0, 1.0]]))       # double pole at z = 1
    assert e.value.status == 2
    with pytest.raises(lib.FilarkError) as e:
        lib.debug_design(np.array([[1.0, 0, 0, 1.0, 0.0, -1.1]]))
    assert e.value.status == 2
    with pytest.raises(lib.FilarkError) as e:
        lib.debug_design(np.array([[1.0, 0, 0, 0.0, 0.5, 0.1]]))        # a0 = 0
    assert e.value.status == 1
    with pytest.raises(lib.FilarkError) as e:
        lib.debug_design(np.array([[np.nan, 0, 0, 1.0, 0.5, 0.1]]))
    assert e.value.status == 1


@pytest.mark.parametrize("e", [0, 1, 31, 32, 1024, 32768])
def test_block_powers_match_numpy(lib, e):
    sos = design_sos(CONFIGS["cfg5"])
    kinds, coefs, _ = lib.debug_design(sos)
    for k in range(sos.shape[0]):
        A = coefs[k, :4].reshape(2, 2)
        ref = np.linalg.matrix_power(A, e)
        got = lib.debug_block_power(sos[k], e)
        assert np.max(np.abs(got - ref)) < 1e-9 * max(1.0, np.abs(ref).max())


def test_push_geometry_covers_every_sample_once(lib):
    """Stream-aligned slots: a sequence of pushes advances the state over every sample exactly
    once, whatever the chunking, and what does not fill a slot waits for the next push."""
    lens = set(range(1, 70)) | {1000, 1023, 1024, 1025, 1500, 1530, 2047, 2048, 6000, 90000, 99991, 900000}
    lens |= set(push_schedule(CONFIGS["cfg5"])[:50])
    for n_t in sorted(lens):
        for force in (0, 8, 16, 24):
            for r0 in (0, 1, 4, 7, 23, 47):
                g = lib.debug_push_geometry(n_t, r0, force)
                L = g["L"]
                assert L in (8, 16, 24) and (force == 0 or L == force)
                total = r0 + n_t
                n_full, r1 = divmod(total, L)
                assert g["r1"] == r1 and 0 <= r1 < L
                slots = n_full + (1 if r1 else 0)
                assert g["n_tiles"] == (slots + 63) // 64 >= 1
                assert g["q_last"] == n_full - 64 * (g["n_tiles"] - 1) and 0 <= g["q_last"] <= 64
                assert g["vec4"] == (1 if r0 % 4 == 0 else 0)
    # a chunked stream: the state has moved over exactly (pushed - waiting) samples after every push
    rng = np.random.default_rng(5)
    for force in (0, 8, 16, 24):
        r0, pushed, advanced = 0, 0, 0
        for n_t in rng.integers(1, 4000, size=200).tolist():
            g = lib.debug_push_geometry(n_t, r0, force)
            advanced += (64 * (g["n_tiles"] - 1) + g["q_last"]) * g["L"]
            pushed += n_t
            r0 = g["r1"]
            assert advanced + r0 == pushed and r0 < 24
    # the cheapest variant for the configs' chunk lengths puts the whole chunk in one tile
    assert lib.debug_push_geometry(1500)["L"] == 24 and lib.debug_push_geometry(1500)["n_tiles"] == 1
    assert lib.debug_push_geometry(1000)["L"] == 16 and lib.debug_push_geometry(1000)["n_tiles"] == 1


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    from paper_2605_20132_b200 import stream
    monkeypatch.setattr(stream, "_lib", None)
    monkeypatch.setattr(stream, "LIB_PATH", str(tmp_path / "nope.so"))
    with pytest.raises(FileNotFoundError):
        stream.load_library()
