"""Writes tests/golden/oracle_small.txt from the oracle ALONE (imports only oracle/ and numpy).

The paper (arxiv 2605.20132) prints no worked numerical example for its stateful SOS IIR
operator and never defines STA/LTA, so there is no paper value to
store.  This fixture is a regression freeze of the float64 oracle on a tiny hand-made case
(2 channels x 48 samples, two sections, sta 3 / lta 8); the oracle itself is pinned to closed
forms and library routines in tests/test_oracle_pins.py.

Run:  python -m tests.golden.make_golden      (from the repo root)
"""
import os

import numpy as np


def golden_case():
    sos = np.array([[0.5, 1.0, 0.5, 1.0, -0.9, 0.41],       # complex poles 0.45 +- 0.455i
                    [1.0, -2.0, 1.0, 2.0, -3.2, 1.3]])      # a0 != 1; poles 0.8 +- 0.1i
    n_t = 48
    t = np.arange(n_t)
    x = np.stack([np.sin(0.37 * t) + 0.25 * ((t * 7) % 5 - 2),
                  np.where(t == 5, 4.0, 0.0) - 0.125 * (t % 3)]).astype(np.float32)
    return sos, 3, 8, x


def main():
    from oracle import Oracle
    sos, sta, lta, x = golden_case()
    o = Oracle(x.shape[0], sos, sta, lta)
    f, c = o.push(x)
    out = np.stack([x.ravel(), f.ravel(), c.ravel()], axis=1)
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_small.txt")
    np.savetxt(path, out, fmt="%.9e",
               header="x filt cf  (row = channel*48 + sample); written by make_golden.py from oracle/ only")
    print("wrote", path)


if __name__ == "__main__":
    main()
