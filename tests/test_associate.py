"""filark_events_associate (include/filark_stream.h; NEXT-1 "channel range", reading R30) against the oracle's
association.  It is a host function on a host list, so this parity test needs no GPU; the end-to-end case
(events from the trigger on the GPU) is in tests/test_gpu_next.py."""
import os

import numpy as np
import pytest

from oracle import BOX_DTYPE, EVENT_DTYPE, oracle_associate
from paper_2605_20132_b200 import build as fbuild


@pytest.fixture(scope="module")
def assoc():
    fbuild.build_library()
    from paper_2605_20132_b200 import stream
    return stream


def _events(rng, n, n_ch, t_max, dur):
    ev = np.zeros(n, dtype=EVENT_DTYPE)
    ev["t_on"] = rng.integers(0, t_max, n)
    ev["t_off"] = ev["t_on"] + rng.integers(1, dur, n)
    ev["channel"] = rng.integers(0, n_ch, n)
    ev["peak"] = (rng.random(n) * 10).astype(np.float32)
    return ev


def _key(boxes):
    return sorted(tuple(b) for b in boxes.tolist())


@pytest.mark.parametrize("n,n_ch,t_max,dur", [(1, 4, 100, 10), (60, 12, 400, 60), (3000, 300, 90_000, 400),
                                              (4000, 50, 20_000, 300), (2000, 6000, 5_400_000, 3000)])
@pytest.mark.parametrize("ch_gap,t_gap", [(0, 0), (1, 0), (1, 150), (4, 7)])
def test_library_equals_oracle(assoc, n, n_ch, t_max, dur, ch_gap, t_gap):
    ev = _events(np.random.default_rng(n + 7 * ch_gap + t_gap), n, n_ch, t_max, dur)
    ref = oracle_associate(ev, ch_gap, t_gap)
    got, total = assoc.associate_events(ev, ch_gap, t_gap)
    assert total == ref.shape[0]
    assert got.dtype == BOX_DTYPE and _key(got) == _key(ref)
    # listed in rising (t_on, ch_lo, t_off, ch_hi)
    k = [(b["t_on"], b["ch_lo"], b["t_off"], b["ch_hi"]) for b in got]
    assert k == sorted(k)
    # the order of the list does not matter
    again, _ = assoc.associate_events(ev[np.random.default_rng(1).permutation(n)], ch_gap, t_gap)
    assert _key(again) == _key(ref)


def test_worked_example(assoc):
    """tests/golden/associate_small.txt (hand-derived)."""
    ev, want = [], {"B": [], "C": [], "D": []}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "associate_small.txt")):
        f = line.split()
        if not f or f[0] == "#":
            continue
        if f[0] == "E":
            ev.append((int(f[1]), int(f[2]), int(f[3]), float(f[4])))
        else:
            want[f[0]].append((int(f[1]), int(f[2]), int(f[3]), int(f[4]), float(f[5]), int(f[6])))
    ev = np.array(ev, dtype=EVENT_DTYPE)
    for key, (cg, tg) in {"B": (1, 0), "C": (2, 0), "D": (1, 60)}.items():
        got, total = assoc.associate_events(ev, cg, tg)
        assert total == len(want[key]) and got.tolist() == want[key]


def test_overflow_empty_and_bad_arguments(assoc):
    ev = _events(np.random.default_rng(3), 200, 100, 100_000, 50)
    ref = oracle_associate(ev, 0, 0)
    got, total = assoc.associate_events(ev, 0, 0, cap=10)
    assert total == ref.shape[0] > 10 and got.tolist() == ref[:10].tolist()      # the first ten, the rest dropped and counted
    got, total = assoc.associate_events(np.zeros(0, dtype=EVENT_DTYPE), 1, 0)
    assert total == 0 and got.shape[0] == 0
    for bad in ((-1, 0), (0, -5)):
        with pytest.raises(assoc.FilarkError) as e:
            assoc.associate_events(ev, *bad)
        assert e.value.status == 1
