"""GPU test of filark_stream_once_noalloc (include/filark_stream.h): the entry point that allocates nothing --
its device scratch is a fixed array in the library's device image -- against the existing path (a handle:
create + one push of the same record), on two calls in a row that share the scratch.  Tolerance: the one of
every parity test (tests/_util.py).  Collected last on purpose (the file name): the suite runs with
pytest -x."""
import dataclasses

import numpy as np
import pytest
import torch

from paper_2605_20132_b200.workloads import CHANNEL_MAJOR, TIME_MAJOR, CONFIGS, design_sos, generate
from tests._util import as_cm, assert_parity

pytestmark = pytest.mark.gpu


def _existing_path(w, sos, x_dev, layout):
    from paper_2605_20132_b200.stream import FilarkStream
    s = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len, layout)
    f, c = torch.empty_like(x_dev), torch.empty_like(x_dev)
    s.push(x_dev, f, c)
    torch.cuda.synchronize()
    s.destroy()
    return f.cpu().numpy(), c.cpu().numpy()


@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
def test_two_calls_in_a_row_match_the_handle_path(cuda_device, layout):
    from paper_2605_20132_b200.stream import once_noalloc
    # two different records behind one another: the second has fewer channels, another cascade, another
    # sub-block variant and a ragged length, so anything the first call left in the scratch would show
    cases = [(CONFIGS["cfg3"].scaled(n_ch=212, n_t=20_007), 11), (CONFIGS["cfg2"].scaled(n_ch=64, n_t=1_000), 12)]
    for rep in range(2):                                  # ... and the pair twice
        for w, seed in cases:
            sos = design_sos(w)
            x_cm = generate(dataclasses.replace(w, seed=w.seed + seed + rep), device="cpu", layout=CHANNEL_MAJOR)
            x_dev = (x_cm if layout == CHANNEL_MAJOR else x_cm.t().contiguous()).to(cuda_device)
            ref_f, ref_c = _existing_path(w, sos, x_dev, layout)
            f, c = torch.full_like(x_dev, float("nan")), torch.full_like(x_dev, float("nan"))
            once_noalloc(sos, w.sta_len, w.lta_len, x_dev, f, c, layout)
            torch.cuda.synchronize()
            what = f"once_noalloc rep {rep} {w.n_ch} x {w.n_t} layout {layout}"
            assert_parity(as_cm(f.cpu().numpy(), layout), as_cm(ref_f, layout), what + " filt")
            assert_parity(as_cm(c.cpu().numpy(), layout), as_cm(ref_c, layout), what + " cf")
            # the same kernel on the same input: in fact identical
            assert np.array_equal(f.cpu().numpy(), ref_f) and np.array_equal(c.cpu().numpy(), ref_c), what


def test_one_output_only_and_back_to_back_without_sync(cuda_device):
    """Two calls enqueued directly behind one another in one stream (no host synchronisation between them)."""
    from paper_2605_20132_b200.stream import once_noalloc
    w = CONFIGS["cfg3"].scaled(n_ch=300, n_t=4_500)
    sos = design_sos(w)
    x1 = generate(w, device="cpu").to(cuda_device)
    x2 = (x1.flip(1) * 0.5).contiguous()
    r1, r2 = _existing_path(w, sos, x1, CHANNEL_MAJOR), _existing_path(w, sos, x2, CHANNEL_MAJOR)
    f1, c2 = torch.empty_like(x1), torch.empty_like(x2)
    once_noalloc(sos, w.sta_len, w.lta_len, x1, f1, None)
    once_noalloc(sos, w.sta_len, w.lta_len, x2, None, c2)
    torch.cuda.synchronize()
    assert_parity(f1.cpu().numpy(), r1[0], "first call, filt only")
    assert_parity(c2.cpu().numpy(), r2[1], "second call, cf only")


def test_limits_and_errors(cuda_device):
    from paper_2605_20132_b200.stream import FilarkError, NOALLOC_MAX_CHANNELS, once_noalloc
    w = CONFIGS["cfg1"]
    sos = design_sos(w)
    big = torch.zeros((NOALLOC_MAX_CHANNELS + 1, 64), device=cuda_device)
    with pytest.raises(FilarkError) as e:
        once_noalloc(sos, w.sta_len, w.lta_len, big, torch.empty_like(big), None)
    assert e.value.status == 7                                            # FILARK_ERR_TOO_LARGE
    x = torch.zeros((8, 64), device=cuda_device)
    with pytest.raises(FilarkError) as e:
        once_noalloc(sos, w.sta_len, w.lta_len, x, None, None)            # no output wanted
    assert e.value.status == 1
    with pytest.raises(FilarkError) as e:
        once_noalloc(sos, w.sta_len, w.lta_len, x, x, None)               # output over the input
    assert e.value.status == 1
    # the largest size it takes
    full = torch.randn((NOALLOC_MAX_CHANNELS, 96), device=cuda_device)
    f = torch.empty_like(full)
    once_noalloc(sos, w.sta_len, w.lta_len, full, f, None)
    torch.cuda.synchronize()
    ref = _existing_path(w.scaled(n_ch=NOALLOC_MAX_CHANNELS, n_t=96), sos, full, CHANNEL_MAJOR)[0]
    assert np.array_equal(f.cpu().numpy(), ref)
