"""GPU: consecutive pushes of a handle overlap on the device where the library knows what lies
between them (FILARK_FLAG_OVERLAP_PUSHES, filark_stream_push_many; include/filark_stream.h,
"Ordering"; csrc/filark_kernels.cuh).  Back-to-back pushes with nothing between them in the stream must give
bit-identical outputs to the same pushes under FILARK_FLAG_STRICT_ORDER (every push an ordinary
dependent launch) and match the float64 oracle; pushes whose buffers clash with the ones before
them, and pushes of another handle in the same stream, must be ordered like any stream work."""
import numpy as np
import pytest
import torch

from paper_2605_20132_b200.stream import FLAG_OVERLAP_PUSHES, FLAG_STRICT_ORDER, FilarkStream

OV = FLAG_OVERLAP_PUSHES
from paper_2605_20132_b200.workloads import CHANNEL_MAJOR, CONFIGS, design_sos, generate
from tests._util import assert_parity, run_oracle, split

pytestmark = pytest.mark.gpu


def _back_to_back(s, chunks, outs_f, outs_c):
    """Nothing but pushes goes into the stream: this is the case in which they overlap."""
    for x, f, c in zip(chunks, outs_f, outs_c):
        s.push(x, f, c)


def _alloc(chunks):
    return [torch.empty_like(x) for x in chunks], [torch.empty_like(x) for x in chunks]


@pytest.mark.parametrize("n_ch,n_t,sizes", [
    (3000, 12_000, [1500]),                 # the bench's push shape: 16-byte path, r0 alternates 0 / 12
    (2500, 9_000, [700, 333, 1501, 64]),    # ragged: 4-byte path, hist crosses pushes
    (2000, 9_000, [1500, 100, 1000, 7]),    # the variant changes from push to push: r0 >= L of the next one
    (6000, 6_000, [1000]),                  # more channels than resident warps
    (700, 40_000, [16_000, 8_000]),         # several segments per channel and push
])
def test_overlapped_equals_strict_order_and_oracle(cuda_device, n_ch, n_t, sizes):
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=n_t)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    xd = x.to(cuda_device)
    chunks = [xd[:, a:b].contiguous() for a, b in split(n_t, sizes)]
    res = {}
    for flags in (OV, FLAG_STRICT_ORDER):
        s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, flags)
        of, oc = _alloc(chunks)
        for rep in range(3):                               # reset + replay: counters start over
            torch.cuda.synchronize()
            _back_to_back(s, chunks, of, oc)
            torch.cuda.synchronize()
            if rep < 2:
                s.reset()
        res[flags] = (torch.cat(of, 1).cpu().numpy(), torch.cat(oc, 1).cpu().numpy())
        s.destroy()
    assert np.array_equal(res[OV][0], res[FLAG_STRICT_ORDER][0]), "filt differs from strict order"
    assert np.array_equal(res[OV][1], res[FLAG_STRICT_ORDER][1]), "cf differs from strict order"
    pick = np.unique(np.r_[0, 1, n_ch // 3, n_ch // 2, n_ch - 2, n_ch - 1,
                           np.random.default_rng(5).integers(0, n_ch, 26)])
    ref_f, ref_c = run_oracle(x.numpy()[pick], sos, w.sta_len, w.lta_len)
    assert_parity(res[OV][0][pick], ref_f, "overlapped filt")
    assert_parity(res[OV][1][pick], ref_c, "overlapped cf")


@pytest.mark.parametrize("n_ch,n_t,sizes", [(3001, 9_000, [1500]), (1000, 7_000, [700, 333, 1501, 64])])
def test_time_major_overlapped_equals_strict_order_and_oracle(cuda_device, n_ch, n_t, sizes):
    """The same for time-major chunks ([n_t][n_ch]; the last group of 16 channels is partial)."""
    from paper_2605_20132_b200.workloads import TIME_MAJOR
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=n_t)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    xd = x.t().contiguous().to(cuda_device)
    chunks = [xd[a:b, :].contiguous() for a, b in split(n_t, sizes)]
    res = {}
    for flags in (OV, FLAG_STRICT_ORDER):
        s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, TIME_MAJOR, flags)
        of, oc = _alloc(chunks)
        for rep in range(2):
            torch.cuda.synchronize()
            _back_to_back(s, chunks, of, oc)
            torch.cuda.synchronize()
            if rep < 1:
                s.reset()
        res[flags] = (torch.cat(of, 0).t().contiguous().cpu().numpy(), torch.cat(oc, 0).t().contiguous().cpu().numpy())
        s.destroy()
    assert np.array_equal(res[OV][0], res[FLAG_STRICT_ORDER][0]), "filt differs from strict order"
    assert np.array_equal(res[OV][1], res[FLAG_STRICT_ORDER][1]), "cf differs from strict order"
    pick = np.unique(np.r_[0, 15, 16, n_ch - 17, n_ch - 1, np.random.default_rng(6).integers(0, n_ch, 20)])
    ref_f, ref_c = run_oracle(x.numpy()[pick], sos, w.sta_len, w.lta_len)
    assert_parity(res[OV][0][pick], ref_f, "time-major overlapped filt")
    assert_parity(res[OV][1][pick], ref_c, "time-major overlapped cf")


def test_long_run_of_overlapped_pushes(cuda_device):
    """200 pushes in flight behind each other: counters, slot parity and the in-flight bound."""
    n_ch, chunk, n_push = 1200, 252, 200
    w = CONFIGS["cfg4"].scaled(n_ch=n_ch, n_t=chunk * n_push)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    xd = x.to(cuda_device)
    chunks = [xd[:, a:b].contiguous() for a, b in split(w.n_t, [chunk])]
    s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, OV)
    of, oc = _alloc(chunks)
    _back_to_back(s, chunks, of, oc)
    torch.cuda.synchronize()
    assert s.launch_count == n_push
    pick = np.arange(0, n_ch, 97)
    ref_f, ref_c = run_oracle(x.numpy()[pick], sos, w.sta_len, w.lta_len)
    assert_parity(torch.cat(of, 1).cpu().numpy()[pick], ref_f, "200 pushes filt")
    assert_parity(torch.cat(oc, 1).cpu().numpy()[pick], ref_c, "200 pushes cf")
    s.destroy()


def test_clashing_buffers_are_ordered(cuda_device):
    """(a) every push writes the SAME output buffers; (b) a push reads what the push before it
    wrote.  Both must behave as plain stream order says."""
    n_ch, chunk, n_push = 2400, 1500, 6
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=chunk * n_push)
    sos = design_sos(w)
    xd = generate(w, device="cpu").to(cuda_device)
    chunks = [xd[:, a:b].contiguous() for a, b in split(w.n_t, [chunk])]
    # reference: strict order, separate buffers
    s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, FLAG_STRICT_ORDER)
    of, oc = _alloc(chunks)
    _back_to_back(s, chunks, of, oc)
    torch.cuda.synchronize()
    s.destroy()
    # (a) one pair of output buffers for all pushes: the last push must win everywhere
    s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, OV)
    f1 = torch.empty_like(chunks[0]); c1 = torch.empty_like(chunks[0])
    for xk in chunks:
        s.push(xk, f1, c1)
    torch.cuda.synchronize()
    assert torch.equal(f1, of[-1]) and torch.equal(c1, oc[-1])
    s.destroy()
    # (b) second handle-free chain: push k + 1 filters the filt output of push k again
    for flags in (OV, FLAG_STRICT_ORDER):
        s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, flags)
        bufs = [chunks[0]] + [torch.empty_like(chunks[0]) for _ in range(n_push)]
        for k in range(n_push):
            s.push(bufs[k], bufs[k + 1], None)
        torch.cuda.synchronize()
        if flags == OV:
            got = [b.clone() for b in bufs[1:]]
        else:
            for a, b in zip(got, bufs[1:]):
                assert torch.equal(a, b), "a push read its input before the push before it had written it"
        s.destroy()


def test_two_handles_chained_in_one_stream(cuda_device):
    """Handle B filters what handle A wrote, push by push, in one stream: B's pushes follow A's
    pushes directly and must still see A's output complete."""
    n_ch, chunk, n_push = 2400, 1500, 5
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=chunk * n_push)
    sos = design_sos(w)
    xd = generate(w, device="cpu").to(cuda_device)
    chunks = [xd[:, a:b].contiguous() for a, b in split(w.n_t, [chunk])]
    out = {}
    for flags in (OV, FLAG_STRICT_ORDER):
        a = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, flags)
        b = FilarkStream(n_ch, sos[:2], w.sta_len, w.lta_len, CHANNEL_MAJOR, flags)
        fa, _ = _alloc(chunks); fb, cb = _alloc(chunks)
        for k in range(n_push):
            a.push(chunks[k], fa[k], None)
            b.push(fa[k], fb[k], cb[k])
        torch.cuda.synchronize()
        out[flags] = (torch.cat(fb, 1), torch.cat(cb, 1))
        a.destroy(); b.destroy()
    assert torch.equal(out[OV][0], out[FLAG_STRICT_ORDER][0])
    assert torch.equal(out[OV][1], out[FLAG_STRICT_ORDER][1])


def test_graph_of_back_to_back_pushes(cuda_device):
    """Several pushes captured into ONE graph (programmatic edges between them), replayed."""
    n_ch, chunk, per_graph, n_rep = 2000, 1500, 4, 3
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=chunk * per_graph * n_rep)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    xd = x.to(cuda_device)
    s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, OV)
    xin = [torch.empty((n_ch, chunk), device=cuda_device) for _ in range(per_graph)]
    of, oc = _alloc(xin)
    side = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        s.push(xin[0], of[0], oc[0]); s.reset()             # warm-up outside capture
        torch.cuda.synchronize()
        with torch.cuda.graph(g, stream=side):
            for k in range(per_graph):
                s.push(xin[k], of[k], oc[k])
    got_f, got_c = [], []
    for r in range(n_rep):
        for k in range(per_graph):
            a = (r * per_graph + k) * chunk
            xin[k].copy_(xd[:, a:a + chunk])
        g.replay()
        torch.cuda.synchronize()
        got_f += [t.clone() for t in of]; got_c += [t.clone() for t in oc]
    pick = np.arange(0, n_ch, 131)
    ref_f, ref_c = run_oracle(x.numpy()[pick], sos, w.sta_len, w.lta_len)
    assert_parity(torch.cat(got_f, 1).cpu().numpy()[pick], ref_f, "graph of pushes filt")
    assert_parity(torch.cat(got_c, 1).cpu().numpy()[pick], ref_c, "graph of pushes cf")
    s.destroy()


def test_push_many_equals_separate_pushes(cuda_device):
    """filark_stream_push_many == the same pushes one call at a time, bit for bit (same sub-block
    length L everywhere), for a schedule with ragged and zero-length chunks, NULL output arrays and
    single NULL outputs; the chunks share no buffer, so one launch serves them all."""
    L24 = 24 << 8
    n_ch, sizes = 2600, [1500, 1500, 64, 0, 1501, 3000, 7, 1500]
    n_t = sum(sizes)
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=n_t)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    xd = x.to(cuda_device)
    chunks, p = [], 0
    for c in sizes:
        chunks.append(xd[:, p:p + c].contiguous()); p += c
    ref = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, FLAG_STRICT_ORDER | L24)
    rf, rc = _alloc(chunks)
    for a, f, c in zip(chunks, rf, rc):
        ref.push(a, f, c)
    torch.cuda.synchronize()
    ref.destroy()
    for flags in (L24, OV | L24):
        s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, CHANNEL_MAJOR, flags)
        of, oc = _alloc(chunks)
        for rep in range(2):
            s.push_many(chunks, of, oc)
            torch.cuda.synchronize()
            assert s.launch_count == rep + 1
            for a, b in zip(of + oc, rf + rc):
                assert torch.equal(a, b)
            s.reset()
        # only one output wanted: a NULL array, and NULL entries
        of2, _ = _alloc(chunks)
        s.push_many(chunks, of2, None)
        oc2 = [torch.empty_like(t) for t in chunks]
        s.reset()
        s.push_many(chunks, [None if i % 2 else f for i, f in enumerate(of)], oc2)
        torch.cuda.synchronize()
        for a, b in zip(of2 + oc2, rf + rc):
            assert torch.equal(a, b)
        s.destroy()
    pick = np.arange(0, n_ch, 211)
    ref_f, ref_c = run_oracle(x.numpy()[pick], sos, w.sta_len, w.lta_len)
    assert_parity(torch.cat(rf, 1).cpu().numpy()[pick], ref_f, "push_many filt")
    assert_parity(torch.cat(rc, 1).cpu().numpy()[pick], ref_c, "push_many cf")


def test_default_pushes_see_foreign_producers(cuda_device):
    """Default flags: a push behaves like any kernel in its stream.  Here another kernel (a torch
    copy, then an in-place scale) produces every push's input right before the push and a third
    consumes its output right after it; nothing may be read early or late."""
    n_ch, chunk, n_push = 3000, 1500, 8
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=chunk * n_push)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    xd = x.to(cuda_device)
    s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len)
    xin = torch.empty((n_ch, chunk), device=cuda_device)
    f = torch.empty_like(xin); c = torch.empty_like(xin)
    got_f, got_c = [], []
    for k in range(n_push):
        xin.copy_(xd[:, k * chunk:(k + 1) * chunk] * 0.5)      # producer kernels of this push's input
        xin.mul_(2.0)
        s.push(xin, f, c)
        got_f.append(f.clone()); got_c.append(c.clone())       # consumer kernels of its outputs
    torch.cuda.synchronize()
    pick = np.arange(0, n_ch, 173)
    ref_f, ref_c = run_oracle(x.numpy()[pick], sos, w.sta_len, w.lta_len)
    assert_parity(torch.cat(got_f, 1).cpu().numpy()[pick], ref_f, "default-order filt")
    assert_parity(torch.cat(got_c, 1).cpu().numpy()[pick], ref_c, "default-order cf")
    s.destroy()


def _wait_for(event, seconds, what):
    """Poll instead of synchronising: a device that no longer makes progress fails the test
    instead of blocking the process in the driver."""
    import time
    t0 = time.time()
    while not event.query():
        assert time.time() - t0 < seconds, f"{what}: the device made no progress for {seconds} s"
        time.sleep(0.01)


@pytest.mark.parametrize("layout_name", ["cm", "tm"])
def test_two_handles_on_two_streams_multi_segment(cuda_device, layout_name):
    """Two handles push long chunks (several segments per channel: work items that wait for each
    other inside a push) on two streams at the same time, so that each grid is only partially
    resident.  Work items are claimed in rising order by resident warps, so the waits always end
    (csrc/filark_kernels.cuh, "Work items"); the outputs equal those of the handles run alone."""
    from paper_2605_20132_b200.workloads import TIME_MAJOR
    layout = CHANNEL_MAJOR if layout_name == "cm" else TIME_MAJOR
    n_ch, n_t, n_push = 900, 30_000, 3
    w = CONFIGS["cfg3"].scaled(n_ch=n_ch, n_t=n_t * n_push)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    xd = x.to(cuda_device) if layout == CHANNEL_MAJOR else x.t().contiguous().to(cuda_device)
    cut = (lambda a, b: xd[:, a:b].contiguous()) if layout == CHANNEL_MAJOR else (lambda a, b: xd[a:b, :].contiguous())
    chunks = [cut(k * n_t, (k + 1) * n_t) for k in range(n_push)]
    # alone
    s = FilarkStream(n_ch, sos, w.sta_len, w.lta_len, layout, OV)
    rf, rc = _alloc(chunks)
    _back_to_back(s, chunks, rf, rc)
    torch.cuda.synchronize()
    s.destroy()
    # together, several rounds
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    hs = [FilarkStream(n_ch, sos, w.sta_len, w.lta_len, layout, OV) for _ in streams]
    outs = [_alloc(chunks) for _ in streams]
    for rnd in range(4):
        torch.cuda.synchronize()
        evs = []
        for k in range(n_push):
            for st, h, (of, oc) in zip(streams, hs, outs):
                with torch.cuda.stream(st):
                    h.push(chunks[k], of[k], oc[k])
        for st in streams:
            ev = torch.cuda.Event()
            ev.record(st)
            evs.append(ev)
        for ev in evs:
            _wait_for(ev, 60.0, "two handles on two streams")
        for of, oc in outs:
            for a, b in zip(of + oc, rf + rc):
                assert torch.equal(a, b)
        for st, h in zip(streams, hs):
            with torch.cuda.stream(st):
                h.reset()
    for h in hs:
        h.destroy()


def test_second_device_in_one_process():
    """Kernel attributes (dynamic shared memory opt-in) are per device: a handle on a second GPU of
    the same process must launch as the first one does.  Skipped with fewer than two GPUs."""
    if not torch.cuda.is_available() or torch.cuda.device_count() < 2:
        pytest.skip("needs two CUDA devices")
    w = CONFIGS["cfg3"].scaled(n_ch=300, n_t=4_000)
    sos = design_sos(w)
    x = generate(w, device="cpu")
    ref_f, ref_c = run_oracle(x.numpy(), sos, w.sta_len, w.lta_len)
    for dev in (0, 1):
        with torch.cuda.device(dev):
            xd = x.to(f"cuda:{dev}")
            s = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len)
            f = torch.empty_like(xd); c = torch.empty_like(xd)
            s.push(xd, f, c)
            torch.cuda.synchronize()
            assert_parity(f.cpu().numpy(), ref_f, f"device {dev} filt")
            assert_parity(c.cpu().numpy(), ref_c, f"device {dev} cf")
    # destroy with ANOTHER device current
    with torch.cuda.device(0):
        s.destroy()
