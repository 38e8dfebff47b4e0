"""Small end-to-end case for compute-sanitizer runs (one tool per run):

    compute-sanitizer --tool memcheck  python tests/sanitizer_case.py
    compute-sanitizer --tool racecheck python tests/sanitizer_case.py

Streams a 40-channel record in ragged pushes through both layouts (every staging path: 16-byte
and 4-byte, history, partial slots, several tiles and segments) and checks parity with the oracle."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from oracle import Oracle  # noqa: E402
from paper_2605_20132_b200.stream import FilarkStream  # noqa: E402
from paper_2605_20132_b200.workloads import CHANNEL_MAJOR, TIME_MAJOR, CONFIGS, design_sos, generate  # noqa: E402


def main():
    w = CONFIGS["cfg3"].scaled(n_ch=40, n_t=9000)
    sos = design_sos(w)
    x = generate(w)
    o = Oracle(w.n_ch, sos, w.sta_len, w.lta_len)
    ref_f, ref_c = o.push(x.numpy()); o.close()
    for layout in (CHANNEL_MAJOR, TIME_MAJOR):
        xd = (x if layout == CHANNEL_MAJOR else x.t().contiguous()).cuda()
        s = FilarkStream(w.n_ch, sos, w.sta_len, w.lta_len, layout)
        fs, cs, p = [], [], 0
        for c in [1500, 1500, 1024, 37, 1, 2048, 2890]:
            xin = (xd[:, p:p + c] if layout == CHANNEL_MAJOR else xd[p:p + c, :]).contiguous()
            f = torch.empty_like(xin); q = torch.empty_like(xin)
            s.push(xin, f, q); fs.append(f); cs.append(q); p += c
        torch.cuda.synchronize()
        dim = 1 if layout == CHANNEL_MAJOR else 0
        f = torch.cat(fs, dim).cpu().numpy(); q = torch.cat(cs, dim).cpu().numpy()
        if layout == TIME_MAJOR:
            f, q = f.T, q.T
        for got, ref in ((f, ref_f), (q, ref_c)):
            d = got.astype(np.float64) - ref
            rel = np.sqrt((d * d).sum(1)) / np.maximum(np.sqrt((ref.astype(np.float64) ** 2).sum(1)), 1e-300)
            assert rel.max() <= 1e-4, rel.max()
        s.destroy()
    print("sanitizer case ok")


if __name__ == "__main__":
    main()
