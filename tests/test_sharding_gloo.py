"""The N > 1 path of bench.py on CPU: the fused path shards by channel with no exchange step
(DESIGN.md 9), so the only multi-rank logic is the partition of the channel axis and the
max-over-ranks reduction of the timing.  World size 2, gloo."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2605_20132_b200.workloads import CONFIGS, channel_shard, design_sos, generate


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import Oracle
    w = CONFIGS["cfg1"].scaled(n_ch=37, n_t=3000)
    x = generate(w).numpy()
    lo, hi = channel_shard(w.n_ch, rank, world)
    o = Oracle(hi - lo, design_sos(w), w.sta_len, w.lta_len)
    f, c = o.push(np.ascontiguousarray(x[lo:hi])); o.close()
    # gather the shards (a check only: the data path itself has no collective)
    parts = [None] * world
    dist.all_gather_object(parts, (lo, hi, f, c))
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)                      # bench.py's max-over-ranks timing
    if rank == 0:
        out.put((parts, float(t.item())))
    dist.barrier()
    dist.destroy_process_group()


def test_channel_shards_reassemble_to_the_whole_record():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    parts, tmax = q.get(timeout=180)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert tmax == 2.0
    from oracle import Oracle
    w = CONFIGS["cfg1"].scaled(n_ch=37, n_t=3000)
    x = generate(w).numpy()
    o = Oracle(w.n_ch, design_sos(w), w.sta_len, w.lta_len)
    f, c = o.push(x); o.close()
    parts.sort(key=lambda t: t[0])
    assert parts[0][0] == 0 and parts[-1][1] == w.n_ch and parts[0][1] == parts[1][0]
    assert np.array_equal(np.concatenate([p[2] for p in parts]), f)       # channels are independent: bit-identical
    assert np.array_equal(np.concatenate([p[3] for p in parts]), c)


def test_channel_shard_partition_properties():
    for n_ch in (1, 2, 7, 256, 6000, 10_000):
        for world in (1, 2, 3, 4, 8):
            cuts = [channel_shard(n_ch, r, world) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n_ch
            assert all(a[1] == b[0] for a, b in zip(cuts, cuts[1:]))
            sizes = [hi - lo for lo, hi in cuts]
            assert max(sizes) - min(sizes) <= 1
