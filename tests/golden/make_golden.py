"""Writes tests/golden/oracle_cfg0_samples.txt from the CPU oracle ONLY (never from the CUDA path).

The paper prints no waveform or likelihood value (Fig. 1 is an image without numbers, Fig. 2's
posterior depends on its code and sampler seed), so there is no paper-printed
golden value to store.  This fixture is a regression guard of the oracle itself: config 0's recipe
(BASELINE.json:configs[0]) at 24 fixed sample indices of walkers 0 and 5, plus logL of walkers 1..3
against walker 0's noise-less spectrum at a reduced length.  Run:  python tests/golden/make_golden.py
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)
from oracle.oracle import Oracle                      # noqa: E402
from paper_2311_17174_b200 import workloads as W      # noqa: E402

IDX = np.array([0, 1, 2, 255, 256, 257, 1000, 4095, 4096, 10000, 20000, 30000, 32767, 32768, 40000, 50000,
                60000, 65000, 65279, 65280, 65281, 65533, 65534, 65535], dtype=np.int64)


def compute():
    o = Oracle()
    cfg = W.CONFIGS[0]
    P = W.draw_params(cfg)
    rows = []
    for k in (0, 5):
        hI, hII, st = o.waveform(P[k], cfg.N, cfg.dt, cfg.n_max, idx=IDX)
        for i, a, b in zip(IDX, hI, hII):
            rows.append(("h", k, int(i), a, b))
    small = W.scaled(cfg, K=4, N=1 << 12)
    psd = W.lisa_psd_barack_cutler(small.N, small.dt)
    hI, hII, _ = o.waveform(P[0], small.N, small.dt, small.n_max)
    D = np.stack([o.rfft(hI), o.rfft(hII)])
    logL, st = o.loglike_batch(P[:4], small.N, small.dt, small.n_max, D, psd)
    for k in range(4):
        rows.append(("logL", k, small.N, logL[k], float(st[k])))
    return rows


def main():
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_cfg0_samples.txt")
    with open(path, "w") as f:
        f.write("# written by tests/golden/make_golden.py from oracle/ only; config 0 recipe, seed 0\n")
        f.write("# kind walker index value_a value_b   (h: h_I h_II at sample index; logL: logL status at N=index)\n")
        for kind, k, i, a, b in compute():
            f.write(f"{kind} {k} {i} {a!r} {b!r}\n".replace("np.float64(", "").replace(")", ""))


if __name__ == "__main__":
    main()
