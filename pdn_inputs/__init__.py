"""Seeded synthetic 3D-IC PDN inputs (shared by the oracle tests, the GPU tests and bench.py).

This module holds NONE of the method's arithmetic: it only draws resistor networks.  It is the
one piece of code both the CPU oracle (`oracle/`) and the CUDA path (`paper_2607_05818_b200/`)
are fed from, so that random-number order cannot diverge between them.

Network model (PAPER.md:71, 81, 104 -- resistor-network model of stacked 2D PDNs joined by TSVs;
Table I PAPER.md:87-102 for m, n, d, p, Rt):

  * d tiers; tier 0 = top (bumps, the paper's die_1), tier d-1 = bottom (loads, die_d).
  * tier t is an N x N node mesh; node (y, x); edge conductances in siemens
        gx[t][y][x] joins (y,x)-(y,x+1)   (last column is padding, always 0)
        gy[t][y][x] joins (y,x)-(y+1,x)   (last row    is padding, always 0)
    0 means "segment absent".
  * interface i joins tier i and tier i+1 through p_i TSVs; TSV k sits at one site (y,x) used in
    both tiers and has resistance Rt[i][k] ohm.
  * m bumps are nodes of tier 0, n loads are nodes of tier d-1.

The five workloads are the synthetic stand-ins for the paper's proprietary benchmarks D1-D9
 named by BASELINE.json `configs`; conventions G14-G21 of SURVEY.md 8(c).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List

import numpy as np


@dataclass
class Network:
    """A stacked-mesh resistor network.  All arrays are numpy, float64 / int32."""
    n: int                                  # mesh is n x n nodes per tier
    gx: List[np.ndarray]                    # per tier, (n, n) float64, last column 0
    gy: List[np.ndarray]                    # per tier, (n, n) float64, last row 0
    tsv_site: List[np.ndarray]              # per interface, (p_i, 2) int32 rows (y, x)
    tsv_r: List[np.ndarray]                 # per interface, (p_i,) float64 ohm
    bumps: np.ndarray                       # (m, 2) int32 rows (y, x) on tier 0
    loads: np.ndarray                       # (nl, 2) int32 rows (y, x) on tier d-1
    name: str = ""
    meta: dict = field(default_factory=dict)

    @property
    def d(self) -> int:
        return len(self.gx)

    @property
    def m(self) -> int:
        return int(self.bumps.shape[0])

    @property
    def nl(self) -> int:
        return int(self.loads.shape[0])


# ----------------------------------------------------------------------------- helpers

def _planes(n: int, rx, ry):
    """Conductance planes from per-segment RESISTANCES rx, ry of shape (n, n); pads are zeroed."""
    gx = 1.0 / np.asarray(rx, dtype=np.float64)
    gy = 1.0 / np.asarray(ry, dtype=np.float64)
    gx = np.array(np.broadcast_to(gx, (n, n)), dtype=np.float64)
    gy = np.array(np.broadcast_to(gy, (n, n)), dtype=np.float64)
    gx[:, n - 1] = 0.0
    gy[n - 1, :] = 0.0
    return gx, gy


def _jitter_planes(rng, n: int, r_x: float, r_y: float, lo=0.9, hi=1.1):
    """Segment resistance r * U[lo,hi] (G20: the jitter multiplies the RESISTANCE). gx drawn first."""
    ux = rng.uniform(lo, hi, size=(n, n))
    uy = rng.uniform(lo, hi, size=(n, n))
    return _planes(n, r_x * ux, r_y * uy)


def _distinct_sites(rng, n: int, count: int) -> np.ndarray:
    """`count` distinct uniformly random nodes of an n x n mesh (sampling without replacement)."""
    flat = rng.choice(n * n, size=count, replace=False)
    return np.stack([flat // n, flat % n], axis=1).astype(np.int32)


class _UnionFind:
    def __init__(self, size: int):
        self.p = np.arange(size, dtype=np.int64)

    def find(self, a: int) -> int:
        p = self.p
        while p[a] != a:
            p[a] = p[p[a]]
            a = p[a]
        return a

    def union(self, a: int, b: int) -> bool:
        ra, rb = self.find(a), self.find(b)
        if ra == rb:
            return False
        self.p[rb] = ra
        return True


def _labels(n: int, gx: np.ndarray, gy: np.ndarray) -> np.ndarray:
    """Connected-component label of every node of one tier (edges with g > 0)."""
    from scipy.sparse import coo_matrix
    from scipy.sparse.csgraph import connected_components
    idx = np.arange(n * n).reshape(n, n)
    mx = gx[:, : n - 1] > 0
    my = gy[: n - 1, :] > 0
    rows = np.concatenate([idx[:, : n - 1][mx], idx[: n - 1, :][my]])
    cols = np.concatenate([idx[:, 1:][mx], idx[1:, :][my]])
    a = coo_matrix((np.ones(rows.size), (rows, cols)), shape=(n * n, n * n))
    _, lab = connected_components(a, directed=False)
    return lab


def _remove_segments_keep_connected(rng, n: int, gx: np.ndarray, gy: np.ndarray, prob: float) -> int:
    """G17: drop each segment with probability `prob`; then, while the tier has more than one
    component, restore (in index order: all gx then all gy) removed segments that join two
    different components.  Returns the number of restored segments.  Modifies gx, gy in place."""
    kx = rng.uniform(size=(n, n)) < prob
    ky = rng.uniform(size=(n, n)) < prob
    kx[:, n - 1] = False
    ky[n - 1, :] = False
    gx0, gy0 = gx.copy(), gy.copy()
    gx[kx] = 0.0
    gy[ky] = 0.0
    lab = _labels(n, gx, gy)
    ncomp = int(lab.max()) + 1
    restored = 0
    if ncomp > 1:
        uf = _UnionFind(ncomp)
        lab2 = lab.reshape(n, n)
        for (y, x) in np.argwhere(kx):
            if uf.union(int(lab2[y, x]), int(lab2[y, x + 1])):
                gx[y, x] = gx0[y, x]
                restored += 1
        for (y, x) in np.argwhere(ky):
            if uf.union(int(lab2[y, x]), int(lab2[y + 1, x])):
                gy[y, x] = gy0[y, x]
                restored += 1
    return restored


# ----------------------------------------------------------------------------- the five workloads

CONFIGS = {
    # cfg: d, n, p per interface, m bumps, n loads, tsv nominal ohm
    1: dict(d=2, n=32, p=16, m=4, nl=16, rt=0.05),
    2: dict(d=3, n=128, p=64, m=32, nl=256, rt=0.05),
    3: dict(d=4, n=512, p=256, m=256, nl=1024, rt=0.03),
    4: dict(d=4, n=1024, p=512, m=1024, nl=1024, rt=0.04),
    5: dict(d=8, n=1024, p=512, m=2048, nl=2048, rt=0.05),
}


def make_config(cfg: int, seed: int = 0) -> Network:
    """Workload `cfg` in 1..5 of BASELINE.json `configs` (recipe: SURVEY.md 8(d), G14-G21).

    RNG: numpy.random.default_rng([seed, cfg]); draw order: tiers in order (gx, gy, then the
    removal masks of config 4), interfaces in order (sites then Rt), bumps, loads."""
    c = CONFIGS[cfg]
    d, n, p = c["d"], c["n"], c["p"]
    rng = np.random.default_rng([seed, cfg])
    gxs, gys, meta = [], [], {"cfg": cfg, "seed": seed}
    restored = 0
    for t in range(d):
        if cfg == 1:
            gx, gy = _jitter_planes(rng, n, 1.0, 1.0)
        elif cfg == 2:
            gx, gy = _jitter_planes(rng, n, 0.5 * (t + 1), 0.5 * (t + 1))
        elif cfg == 3:
            gx, gy = _jitter_planes(rng, n, 0.2 * (t + 1), 0.2 * (t + 1))
        elif cfg == 4:
            gx, gy = _jitter_planes(rng, n, 1.0, 3.0)
            restored += _remove_segments_keep_connected(rng, n, gx, gy, 0.005)
        else:
            gx, gy = _jitter_planes(rng, n, 0.1 * (t + 1), 0.1 * (t + 1))
        gxs.append(gx)
        gys.append(gy)
    meta["restored_segments"] = restored

    centres = None
    if cfg == 4:   # G19: 8 cluster centres shared by all interfaces, drawn before the interfaces
        centres = rng.uniform(0, n, size=(8, 2))
    sites, rts = [], []
    for i in range(d - 1):
        if cfg == 3:      # G18: 16x16 lattice, pitch 32, centres 16+32k, integer jitter in [-4,4]
            ky, kx = np.meshgrid(np.arange(16), np.arange(16), indexing="ij")
            jy = rng.integers(-4, 5, size=(16, 16))
            jx = rng.integers(-4, 5, size=(16, 16))
            s = np.stack([(16 + 32 * ky + jy).ravel(), (16 + 32 * kx + jx).ravel()], axis=1)
        elif cfg == 4:    # G19: 64 sites per centre, sigma 40, round, clip, redraw duplicates
            seen, rows = set(), []
            for cy, cx in centres:
                got = 0
                while got < p // 8:
                    y = int(np.clip(np.rint(rng.normal(cy, 40.0)), 0, n - 1))
                    x = int(np.clip(np.rint(rng.normal(cx, 40.0)), 0, n - 1))
                    if (y, x) in seen:
                        continue
                    seen.add((y, x))
                    rows.append((y, x))
                    got += 1
            s = np.array(rows)
        else:
            s = _distinct_sites(rng, n, p)
        sites.append(np.ascontiguousarray(s, dtype=np.int32))
        rts.append(c["rt"] * rng.uniform(0.8, 1.2, size=p))
    bumps = _distinct_sites(rng, n, c["m"])
    loads = _distinct_sites(rng, n, c["nl"])
    return Network(n=n, gx=gxs, gy=gys, tsv_site=sites, tsv_r=rts, bumps=bumps, loads=loads,
                   name=f"cfg{cfg}", meta=meta)


def sample_pairs(net: Network, count: int = 4096, seed: int = 0, cfg: int = 0):
    """G21: i.i.d. uniform (bump index, load index) pairs from default_rng([seed, cfg, 1])."""
    rng = np.random.default_rng([seed, cfg, 1])
    bi = rng.integers(0, net.m, size=count).astype(np.int32)
    li = rng.integers(0, net.nl, size=count).astype(np.int32)
    return bi, li


# ----------------------------------------------------------------------------- small test networks

def make_uniform(d: int, n: int, r_x: float = 1.0, r_y: float = 1.0, rt: float = 0.05,
                 tsv_sites=None, bumps=None, loads=None) -> Network:
    """Identical uniform tiers (x-segments r_x ohm, y-segments r_y ohm); explicit site lists."""
    gxs, gys = [], []
    for _ in range(d):
        gx, gy = _planes(n, np.full((n, n), r_x), np.full((n, n), r_y))
        gxs.append(gx)
        gys.append(gy)
    if tsv_sites is None:
        tsv_sites = [np.array([[0, 0]])] * (d - 1)
    sites = [np.ascontiguousarray(s, dtype=np.int32).reshape(-1, 2) for s in tsv_sites]
    rts = [np.full(s.shape[0], float(rt)) for s in sites]
    bumps = np.ascontiguousarray(bumps if bumps is not None else [[0, 0]], dtype=np.int32).reshape(-1, 2)
    loads = np.ascontiguousarray(loads if loads is not None else [[n - 1, n - 1]], dtype=np.int32).reshape(-1, 2)
    return Network(n=n, gx=gxs, gy=gys, tsv_site=sites, tsv_r=rts, bumps=bumps, loads=loads,
                   name=f"uniform{d}x{n}")


def make_random(seed: int, d: int, n: int, p: int, m: int, nl: int, r_lo=0.5, r_hi=2.0,
                rt_lo=0.02, rt_hi=0.2, drop: float = 0.0, aniso: float = 1.0) -> Network:
    """Small random stack for property tests: segment resistance U[r_lo,r_hi] (y-segments scaled by
    `aniso`), optional random segment removal keeping tiers connected, p distinct TSV sites per
    interface, m bumps, nl loads (distinct within each list)."""
    rng = np.random.default_rng([seed, d, n, p])
    gxs, gys = [], []
    for _ in range(d):
        gx, gy = _jitter_planes(rng, n, 1.0, aniso, r_lo, r_hi)
        if drop > 0:
            _remove_segments_keep_connected(rng, n, gx, gy, drop)
        gxs.append(gx)
        gys.append(gy)
    sites = [_distinct_sites(rng, n, p) for _ in range(d - 1)]
    rts = [rng.uniform(rt_lo, rt_hi, size=p) for _ in range(d - 1)]
    return Network(n=n, gx=gxs, gy=gys, tsv_site=sites, tsv_r=rts,
                   bumps=_distinct_sites(rng, n, m), loads=_distinct_sites(rng, n, nl),
                   name=f"rand{seed}_{d}x{n}")
