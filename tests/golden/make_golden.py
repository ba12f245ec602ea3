"""Writes tests/golden/oracle_regression.txt from the ORACLE ONLY (oracle/ + dd_workloads/).

    python tests/golden/make_golden.py

Each line: case name, number of outputs, sum of outputs, sum of (index+1)*value mod 2^61-1.
These values guard the oracle against accidental change; they pin nothing by themselves
(the pins are in tests/test_oracle_pins.py).  Nothing here touches the CUDA path.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
sys.path.insert(0, ROOT)

import dd_workloads as W  # noqa: E402
import oracle  # noqa: E402

M61 = (1 << 61) - 1


def checksum(a: np.ndarray) -> tuple[int, int, int]:
    flat = np.asarray(a, dtype=np.int64).ravel()
    s = int(flat.sum())
    w = 0
    idx = np.arange(1, flat.size + 1, dtype=object)
    w = int((idx * flat.astype(object)).sum() % M61)
    return flat.size, s, w


def cases():
    yield "cfg1", W.CONFIGS[1]
    yield "cfg2-r", W.CONFIGS[2].reduced(nsamps=3000, ndm=40, nchans=128)
    yield "cfg4-r", W.CONFIGS[4].reduced(nsamps=2500, ndm=24, nchans=96)


def run_case(cfg: W.Config) -> np.ndarray:
    tab = oracle.delay_table(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.dm_list())
    pulses = W.make_pulses(cfg, lambda idx: tab[idx])
    packed, stride = W.gen_packed(cfg, int(tab.max()), pulses)
    return oracle.dedisperse(packed[0].numpy(), cfg.nbits, cfg.nsamps, tab)


def main():
    out = os.path.join(os.path.dirname(os.path.abspath(__file__)), "oracle_regression.txt")
    with open(out, "w") as f:
        f.write("# written by tests/golden/make_golden.py (oracle only); columns: case n sum weighted_sum_mod_2^61-1\n")
        for name, cfg in cases():
            n, s, w = checksum(run_case(cfg))
            f.write(f"{name} {n} {s} {w}\n")
    print(open(out).read())


if __name__ == "__main__":
    main()
