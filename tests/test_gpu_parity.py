"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by element,
on the same seeded inputs.  Tolerance: BASELINE.json north_star (tests/_util.py)."""
import numpy as np
import pytest
import torch

from paper_2605_20132_b200.workloads import (CHANNEL_MAJOR, TIME_MAJOR, CONFIGS, design_sos,
                                              generate, push_schedule)
from tests._util import as_cm, assert_parity, channel_errors, run_gpu, run_oracle, split

pytestmark = pytest.mark.gpu


def _stream(w, layout=CHANNEL_MAJOR, flags=0):
    from paper_2605_20132_b200.stream import FilarkStream
    return FilarkStream(w.n_ch, design_sos(w), w.sta_len, w.lta_len, layout, flags)


def _case(w, cuda_device, layout):
    x_cm = generate(w, device="cpu", layout=CHANNEL_MAJOR)
    ref_f, ref_c = run_oracle(x_cm.numpy(), design_sos(w), w.sta_len, w.lta_len)
    x_dev = (x_cm if layout == CHANNEL_MAJOR else x_cm.t().contiguous()).to(cuda_device)
    return x_dev, ref_f, ref_c


def _check(filt, cf, ref_f, ref_c, layout, what):
    r1 = assert_parity(as_cm(filt.cpu().numpy(), layout), ref_f, what + " filt")
    r2 = assert_parity(as_cm(cf.cpu().numpy(), layout), ref_c, what + " cf")
    return r1, r2


# ------------------------------------------------------------------ configs[0]: full size
@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
def test_cfg1_whole_and_chunked(cuda_device, layout):
    w = CONFIGS["cfg1"]
    x_dev, ref_f, ref_c = _case(w, cuda_device, layout)
    s = _stream(w, layout)
    f, c = run_gpu(s, x_dev, layout, [(0, w.n_t)])
    _check(f, c, ref_f, ref_c, layout, "cfg1 whole")
    s.reset()
    f2, c2 = run_gpu(s, x_dev, layout, split(w.n_t, [w.chunk]))
    _check(f2, c2, ref_f, ref_c, layout, "cfg1 chunked")
    # chunked vs whole on the GPU itself, same tolerance
    assert_parity(as_cm(f2.cpu().numpy(), layout), as_cm(f.cpu().numpy(), layout), "gpu chunked vs whole filt")
    assert_parity(as_cm(c2.cpu().numpy(), layout), as_cm(c.cpu().numpy(), layout), "gpu chunked vs whole cf")
    s.destroy()


# ------------------------------------------------------------------ configs[1..4]: scaled shapes
SCALED = [("cfg2", 96, 60_000), ("cfg3", 64, 90_000), ("cfg4", 80, 100_000), ("cfg5", 40, 300_000)]


@pytest.mark.parametrize("name,n_ch,n_t", SCALED)
def test_scaled_configs_channel_major(cuda_device, name, n_ch, n_t):
    w = CONFIGS[name].scaled(n_ch=n_ch, n_t=n_t)
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w)
    f, c = run_gpu(s, x_dev, CHANNEL_MAJOR, [(0, n_t)])
    _check(f, c, ref_f, ref_c, CHANNEL_MAJOR, f"{name} whole")
    s.reset()
    sched = push_schedule(w)
    bounds = split(n_t, sched)
    f, c = run_gpu(s, x_dev, CHANNEL_MAJOR, bounds)
    _check(f, c, ref_f, ref_c, CHANNEL_MAJOR, f"{name} in {len(bounds)} pushes")
    s.destroy()


@pytest.mark.parametrize("flags", [0, 8], ids=["lanes", "transpose"])
@pytest.mark.parametrize("name,n_ch,n_t", [("cfg3", 48, 30_000), ("cfg5", 33, 60_000), ("cfg3", 100, 9_000)])
def test_scaled_configs_time_major(cuda_device, name, n_ch, n_t, flags):
    """Both time-major kernels: one channel per lane (filark_kernels_tr.cuh, the default) and the transposing
    one (FILARK_FLAG_TM_TRANSPOSE = 8; what a handle with a trigger set runs)."""
    w = CONFIGS[name].scaled(n_ch=n_ch, n_t=n_t)
    x_dev, ref_f, ref_c = _case(w, cuda_device, TIME_MAJOR)
    s = _stream(w, TIME_MAJOR, flags)
    f, c = run_gpu(s, x_dev, TIME_MAJOR, split(n_t, push_schedule(w)))
    _check(f, c, ref_f, ref_c, TIME_MAJOR, f"{name} time-major")
    s.reset()
    f, c = run_gpu(s, x_dev, TIME_MAJOR, [(0, n_t)])
    _check(f, c, ref_f, ref_c, TIME_MAJOR, f"{name} time-major whole")
    s.destroy()


# ------------------------------------------------------------------ chunking fuzz / ragged tails
FUZZ = [[1], [2, 3], [31, 32, 33], [1, 2, 3, 31, 32, 33, 97, 499, 1021, 1024, 1025, 2047, 4099],
        [7919], [1023, 1], [4096, 5], "random"]


@pytest.mark.parametrize("n_ch", [1, 31, 33, 70])
@pytest.mark.parametrize("seed", [0, 1, 2])
def test_time_major_schedules_fuzz(cuda_device, n_ch, seed):
    """The time-major kernel with one channel per lane on schedules of odd chunk lengths through push_many (one
    launch: samples that do not fill a slot wait for the next chunk in shared memory; tiles of 768 rows; chunks
    shorter than a slot; a block of channels that is not full), then a second schedule on the same handle."""
    rng = np.random.default_rng(100 * n_ch + seed)
    pool = [1, 5, 23, 24, 25, 47, 700, 767, 768, 769, 1500, 3000]
    sizes = rng.choice(pool, size=40).tolist()
    n_t = 12_000
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=n_t)
    x_dev, ref_f, ref_c = _case(w, cuda_device, TIME_MAJOR)
    s = _stream(w, TIME_MAJOR)
    bounds = split(n_t, sizes)
    half = len(bounds) // 2
    f, c = torch.empty_like(x_dev), torch.empty_like(x_dev)
    for part in (bounds[:half], bounds[half:]):
        ins = [x_dev[a:b, :].contiguous() for a, b in part]
        fo, co = [torch.empty_like(t) for t in ins], [torch.empty_like(t) for t in ins]
        s.push_many(ins, fo, co)
        for (a, b), tf, tc in zip(part, fo, co):
            f[a:b, :] = tf; c[a:b, :] = tc
    torch.cuda.synchronize()
    _check(f, c, ref_f, ref_c, TIME_MAJOR, f"time-major fuzz n_ch={n_ch} {sizes[:8]}")
    s.destroy()


@pytest.mark.parametrize("sizes", FUZZ, ids=[str(s) for s in FUZZ])
def test_chunking_fuzz(cuda_device, sizes):
    w = CONFIGS["cfg3"].scaled(n_ch=9, n_t=13_007 if sizes != [1] else 700)
    if sizes == "random":
        sizes = np.random.default_rng(99).integers(1, 3000, size=64).tolist()
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w)
    f, c = run_gpu(s, x_dev, CHANNEL_MAJOR, split(w.n_t, sizes))
    _check(f, c, ref_f, ref_c, CHANNEL_MAJOR, f"fuzz {sizes[:6]}")
    s.destroy()


def test_aligned_chunks_behind_an_odd_sample_count(cuda_device):
    """Chunks whose rows are 16-byte aligned take the kernel build without the unrolled shifted paths; when the
    handle's sample count is odd by then, their tiles are shifted all the same (compact loop of that build).
    Chunks with odd lengths take the other build."""
    w = CONFIGS["cfg3"].scaled(n_ch=11, n_t=16_000)
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w)
    f, c = run_gpu(s, x_dev, CHANNEL_MAJOR, split(w.n_t, [1501, 1500, 1500, 7, 1500, 3000, 2, 1536, 1537]))
    _check(f, c, ref_f, ref_c, CHANNEL_MAJOR, "aligned chunks, odd count")
    s.destroy()


@pytest.mark.parametrize("L", [8, 16, 24])
@pytest.mark.parametrize("n_t", [13_007, 6_144, 1_500, 777])
def test_every_kernel_variant(cuda_device, L, n_t):
    """Each compiled sub-block length on ragged and exact pushes (flags force the variant)."""
    w = CONFIGS["cfg5"].scaled(n_ch=7, n_t=n_t)
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w, CHANNEL_MAJOR, flags=L << 8)
    f, c = run_gpu(s, x_dev, CHANNEL_MAJOR, split(w.n_t, [2048, 1500, 64 * L, 64 * L - 1, 64 * L + 1, 5, 1, 3001]))
    _check(f, c, ref_f, ref_c, CHANNEL_MAJOR, f"L={L} n_t={n_t}")
    s.destroy()


def test_serial_diagnostic_kernel(cuda_device):
    w = CONFIGS["cfg2"].scaled(n_ch=40, n_t=20_000)
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w, CHANNEL_MAJOR, flags=1)
    f, c = run_gpu(s, x_dev, CHANNEL_MAJOR, split(w.n_t, [999]))
    _check(f, c, ref_f, ref_c, CHANNEL_MAJOR, "serial kernel")
    s.destroy()


# ------------------------------------------------------------------ degenerate inputs
def test_dead_channel_dc_offset_and_spike(cuda_device):
    w = CONFIGS["cfg1"].scaled(n_ch=6, n_t=9000)
    x = generate(w).numpy().copy()
    x[0] = 0.0                       # dead channel -> filt = cf = 0 exactly
    x[1] += 1000.0                   # DC offset (fp32 dynamic range)
    x[2, 4000] += 1e4                # single huge spike
    x[3] *= 1e-12                    # tiny amplitudes
    ref_f, ref_c = run_oracle(x, design_sos(w), w.sta_len, w.lta_len)
    s = _stream(w)
    f, c = run_gpu(s, torch.from_numpy(x).to(cuda_device), CHANNEL_MAJOR, split(w.n_t, [1000]))
    f, c = f.cpu().numpy(), c.cpu().numpy()
    assert np.all(f[0] == 0) and np.all(c[0] == 0)
    for ch in (2, 3, 4, 5):
        assert_parity(f[ch:ch + 1], ref_f[ch:ch + 1], f"ch{ch} filt")
        assert_parity(c[ch:ch + 1], ref_c[ch:ch + 1], f"ch{ch} cf")
    # DC offset 1000: absolute error ~ 6e-8 * 1000 on an O(1) band-passed signal after the transient
    rel, _ = channel_errors(f[1:2], ref_f[1:2])
    assert rel < 1e-3
    assert np.all(c >= 0) and c.max() <= w.lta_len / w.sta_len * (1 + 1e-5)
    s.destroy()


def test_warmup_and_reset(cuda_device):
    w = CONFIGS["cfg1"].scaled(n_ch=4, n_t=3000)
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w)
    f, c = run_gpu(s, x_dev, CHANNEL_MAJOR, split(w.n_t, [300]))
    c_np = c.cpu().numpy()
    assert np.all(c_np[:, :w.lta_len] == 0) and np.all(c_np[:, w.lta_len] > 0)
    assert s.samples_pushed == w.n_t
    s.reset()
    f2, c2 = run_gpu(s, x_dev, CHANNEL_MAJOR, split(w.n_t, [300]))
    assert torch.equal(f, f2) and torch.equal(c, c2)      # same launches -> bit-identical
    s.destroy()


def test_optional_outputs_and_empty_push(cuda_device):
    w = CONFIGS["cfg2"].scaled(n_ch=5, n_t=5000)
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w)
    bounds = split(w.n_t, [1234])
    f, _ = run_gpu(s, x_dev, CHANNEL_MAJOR, bounds, want_cf=False)
    s.reset()
    s.push(x_dev[:, :0].contiguous(), torch.empty((5, 0), device=cuda_device),
           torch.empty((5, 0), device=cuda_device))          # n_t = 0: no-op
    assert s.samples_pushed == 0
    _, c = run_gpu(s, x_dev, CHANNEL_MAJOR, bounds, want_filt=False)
    assert_parity(f.cpu().numpy(), ref_f, "filt only")
    assert_parity(c.cpu().numpy(), ref_c, "cf only (state still advances without filt)")
    s.destroy()


def test_pitched_push_on_subviews(cuda_device):
    """Push column windows of a whole channel-major record without packing them."""
    w = CONFIGS["cfg4"].scaled(n_ch=12, n_t=7000)
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w)
    filt = torch.zeros_like(x_dev); cf = torch.zeros_like(x_dev)
    for a, b in split(w.n_t, [1000, 333]):
        s.push_pitched(x_dev, b - a, w.n_t, filt, cf, w.n_t, in_offset=a, out_offset=a)
    torch.cuda.synchronize()
    _check(filt, cf, ref_f, ref_c, CHANNEL_MAJOR, "pitched")
    s.destroy()


def test_error_codes(cuda_device):
    from paper_2605_20132_b200.stream import FilarkError, FilarkStream
    w = CONFIGS["cfg1"].scaled(n_ch=4, n_t=64)
    sos = design_sos(w)
    for bad in [dict(n_ch=0), dict(sta_len=0), dict(lta_len=10, sta_len=20), dict(layout=7), dict(flags=16), dict(flags=7 << 8), dict(flags=32 << 8)]:
        kw = dict(n_ch=4, sos=sos, sta_len=5, lta_len=50, layout=0, flags=0); kw.update(bad)
        with pytest.raises(FilarkError) as e:
            FilarkStream(**kw)
        assert e.value.status == 1
    with pytest.raises(FilarkError) as e:
        FilarkStream(4, np.array([[1.0, 0, 0, 1.0, -2.1, 1.1]]), 5, 50)
    assert e.value.status == 2
    s = FilarkStream(4, sos, 5, 50)
    x = torch.zeros((4, 64), device=cuda_device)
    with pytest.raises(FilarkError) as e:
        s.push(x, None, None)                         # both outputs NULL
    assert e.value.status == 1
    with pytest.raises(FilarkError) as e:
        s.push(x, x, None)                            # in-place rejected
    assert e.value.status == 1
    big = torch.zeros((4 * 64 + 1,), device=cuda_device)
    with pytest.raises(FilarkError) as e:             # misaligned pointer (2 bytes off)
        s._check(s._lib.filark_stream_push(s._h, big.data_ptr() + 2, 64, x.data_ptr(), None, None), "push")
    assert e.value.status == 6
    s.destroy()


def test_cuda_graph_capture_replays_with_carried_state(cuda_device):
    """A captured push has no host-side mutable arguments: replaying it streams the record."""
    w = CONFIGS["cfg1"].scaled(n_ch=8, n_t=6000)
    x_dev, ref_f, ref_c = _case(w, cuda_device, CHANNEL_MAJOR)
    s = _stream(w)
    chunk = 1000
    xin = torch.empty((8, chunk), device=cuda_device); f = torch.empty_like(xin); c = torch.empty_like(xin)
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        xin.copy_(x_dev[:, :chunk]); s.push(xin, f, c); s.reset()      # warm-up outside capture
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            s.push(xin, f, c)
    outs_f, outs_c = [], []
    for a, b in split(w.n_t, [chunk]):
        xin.copy_(x_dev[:, a:b]); g.replay()
        outs_f.append(f.clone()); outs_c.append(c.clone())
    torch.cuda.synchronize()
    _check(torch.cat(outs_f, 1), torch.cat(outs_c, 1), ref_f, ref_c, CHANNEL_MAJOR, "graph replay")
    s.destroy()


def test_push_host_end_to_end(cuda_device):
    w = CONFIGS["cfg2"].scaled(n_ch=16, n_t=8000)
    x = generate(w)
    ref_f, ref_c = run_oracle(x.numpy(), design_sos(w), w.sta_len, w.lta_len)
    s = _stream(w)
    fs, cs = [], []
    for a, b in split(w.n_t, [2000]):
        hin = x[:, a:b].contiguous().pin_memory()
        hf = torch.empty_like(hin).pin_memory(); hc = torch.empty_like(hin).pin_memory()
        s.push_host(hin, hf, hc)
        torch.cuda.synchronize()
        fs.append(hf.clone()); cs.append(hc.clone())
    assert_parity(torch.cat(fs, 1).numpy(), ref_f, "push_host filt")
    assert_parity(torch.cat(cs, 1).numpy(), ref_c, "push_host cf")
    s.destroy()


@pytest.mark.parametrize("sizes", [[0], [1500], [700, 333, 1501, 64]])
def test_all_section_forms(cuda_device, sizes):
    """A cascade that needs every section form of csrc/design.hpp (b0 = 0, first order, identity,
    double real pole, poles near z = 1 with and without zeros there, poles near z = -1): the
    general kernel, not the one built for Butterworth-type cascades only."""
    from paper_2605_20132_b200.stream import FilarkStream, debug_design
    sos = np.array([[0.0, 1.0, 0.0, 1.0, -1.9, 0.9025 + 1e-4],
                    [2.0, 0.5, 0.0, 2.0, -1.0, 0.0],
                    [1.0, 0.0, 0.0, 1.0, 0.0, 0.0],
                    [0.3, 0.1, 0.2, 1.0, -1.6, 0.64],
                    [1.0, 2.0, 1.0, 1.0, -1.95, 0.9512],
                    [1.0, -1.0, 0.0, 1.0, -0.999, 0.0],
                    [0.5, 0.3, 0.5, 1.0, 1.9, 0.9125]])
    assert set(debug_design(sos)[0]) == {0, 1, 2, 3, 4}
    n_ch, n_t = 37, 20_000
    x = torch.from_numpy(np.random.default_rng(11).standard_normal((n_ch, n_t)).astype(np.float32))
    ref_f, ref_c = run_oracle(x.numpy(), sos, 40, 900)
    s = FilarkStream(n_ch, sos, 40, 900)
    f, c = run_gpu(s, x.to(cuda_device), CHANNEL_MAJOR, [(0, n_t)] if sizes == [0] else split(n_t, sizes))
    _check(f, c, ref_f, ref_c, CHANNEL_MAJOR, f"all section forms {sizes}")
    s.destroy()


@pytest.mark.parametrize("layout", [CHANNEL_MAJOR, TIME_MAJOR])
def test_no_write_outside_the_chunk(cuda_device, layout):
    """Outputs are windows of canary-filled buffers at odd offsets and pitches (rows start at every
    alignment, chunks of odd lengths): everything outside the windows must still hold the canary
    afterwards (compute-sanitizer is not available on the GPU pool), everything inside must match
    the oracle."""
    w = CONFIGS["cfg4"].scaled(n_ch=19, n_t=4321)
    x_cm = generate(w, device="cpu", layout=CHANNEL_MAJOR)
    ref_f, ref_c = run_oracle(x_cm.numpy(), design_sos(w), w.sta_len, w.lta_len)
    s = _stream(w, layout)
    canary = 12345.0
    got_f = np.zeros((w.n_ch, w.n_t), np.float32); got_c = np.zeros_like(got_f)
    p = 0
    for k, c in enumerate([1501, 7, 1024, 333, 1, 1455]):
        blk = x_cm[:, p:p + c]
        rows, cols = (w.n_ch, c) if layout == CHANNEL_MAJOR else (c, w.n_ch)
        pitch_in, pitch_out = cols + 3 + (k % 3), cols + 5 + (k % 2)
        off_in, off_out = 1 + k % 4, 2 + (k * 3) % 5
        xin = torch.full((off_in + rows * pitch_in + 9,), 777.0, device=cuda_device)
        src = (blk if layout == CHANNEL_MAJOR else blk.t()).contiguous().to(cuda_device)
        xin[off_in:off_in + rows * pitch_in].view(rows, pitch_in)[:, :cols] = src
        bf = torch.full((off_out + rows * pitch_out + 9,), canary, device=cuda_device)
        bc = torch.full_like(bf, canary)
        s.push_pitched(xin, c, pitch_in, bf, bc, pitch_out, in_offset=off_in, out_offset=off_out)
        torch.cuda.synchronize()
        for buf, got in ((bf, got_f), (bc, got_c)):
            h = buf.cpu().numpy()
            body = h[off_out:off_out + rows * pitch_out].reshape(rows, pitch_out)
            assert np.all(h[:off_out] == canary) and np.all(h[off_out + rows * pitch_out:] == canary), "wrote outside the buffer window"
            assert np.all(body[:, cols:] == canary), "wrote into the gap between rows"
            win = body[:, :cols]
            got[:, p:p + c] = win if layout == CHANNEL_MAJOR else win.T
        p += c
    assert p == w.n_t
    assert_parity(got_f, ref_f, "canary windows filt")
    assert_parity(got_c, ref_c, "canary windows cf")
    s.destroy()
