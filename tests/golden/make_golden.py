"""Writes tests/golden/cfg{K}_reff.txt: oracle R_eff for the parity pairs of workload K.

Calls ONLY `oracle/` (and the seeded input generator).  Nothing here ever comes from the CUDA path.
Pairs: the full cross product for workloads 1-2, the seeded 4096-pair sample (pdn_inputs.sample_pairs,
reading G21) for workloads 3-5.  Each line: `bump_index load_index R_eff` with R_eff printed by
repr() (round-trips the FP64 value).  Header lines start with '#'.

Usage:  python tests/golden/make_golden.py 1 2 3 [--workers W]
"""
import argparse
import os
import sys
import time

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, os.path.dirname(os.path.dirname(HERE)))

import pdn_inputs as P                                           # noqa: E402
from oracle.reff_oracle import Oracle, reff_pairs_forked          # noqa: E402


def pairs_for(cfg, net):
    if cfg <= 2:
        bi, li = np.meshgrid(np.arange(net.m), np.arange(net.nl), indexing="ij")
        return bi.ravel().astype(np.int32), li.ravel().astype(np.int32)
    return P.sample_pairs(net, 4096, seed=0, cfg=cfg)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("cfgs", type=int, nargs="+")
    ap.add_argument("--workers", type=int, default=os.cpu_count())
    a = ap.parse_args()
    for cfg in a.cfgs:
        net = P.make_config(cfg, seed=0)
        t0 = time.time()
        o = Oracle(net)
        t1 = time.time()
        bi, li = pairs_for(cfg, net)
        r = reff_pairs_forked(o, bi, li, a.workers)
        t2 = time.time()
        path = os.path.join(HERE, f"cfg{cfg}_reff.txt")
        with open(path, "w") as f:
            f.write(f"# workload {cfg} of BASELINE.json configs, seed 0; oracle/reff_oracle.py (Eq. 2, PAPER.md:40-43)\n")
            f.write(f"# factor {t1 - t0:.1f} s, {bi.size} pairs in {t2 - t1:.1f} s on {a.workers} forked workers\n")
            f.write("# bump_index load_index R_eff_ohm\n")
            for i, j, v in zip(bi, li, r):
                f.write(f"{int(i)} {int(j)} {float(v)!r}\n")
        print(f"cfg{cfg}: factor {t1 - t0:.1f}s pairs {t2 - t1:.1f}s -> {path}", flush=True)


if __name__ == "__main__":
    main()
