"""CPU FP64 oracle for bump-load effective resistances of a stacked-mesh PDN.

TEST INFRASTRUCTURE ONLY.  Only `tests/`, `__graft_entry__.smoke()` and bench.py's `cpu_baseline` /
`--impl reference` legs may import this file.  It shares no code with the CUDA path and never sees
a per-tier quantity: it works on the Laplacian of the WHOLE 3D network.

What it computes (the definition the method reaches exactly, up to rounding):

    R_eff(b, l) = (e_b - e_l)^T  G^+  (e_b - e_l)                       PAPER.md:40-43, Eq. (2)

"inject a unit current (e.g., 1A) and measure the resulting voltage difference between the two
nodes", on the bare resistor graph G of all tier segments and all TSVs (nothing is
grounded, no other bump is tied to a supply: reading G11 of DESIGN.md).

How (the paper's golden flow: Cholesky-type sparse direct factorisation, then
forward/backward substitution, serial, ONE PAIR AT A TIME):

  1. number nodes globally  id = t*N*N + y*N + x ; assemble G (CSC, FP64): every segment / TSV of
     conductance g between u, v adds  G_uu += g, G_vv += g, G_uv -= g, G_vu -= g.
  2. check the graph is connected.
  3. ground the LAST node (delete its row and column => SPD matrix) and factor once with SuperLU
     (symmetric mode, no pivoting) -- the only sparse direct solver in the image.
  4. per pair: rhs = e_b - e_l (grounded row dropped), v = solve(rhs), ONE step of iterative
     refinement (r = rhs - Gg v ; v += solve(r)), R = v_b - v_l  (v of the grounded node is 0).
  5. tiny graphs: `reff_dense_pinv` evaluates Eq. (2) literally with numpy.linalg.pinv.
  6. `node_voltages` / `load_voltages`: the operating point behind Eq. (4) from KCL directly
     (G v = i with the bump as the reference), for the same-side / voltage extension of the path.

Pins (tests/test_oracle_pins.py, all independent of this file's arithmetic): series / parallel
chains, n-segment line = n*r, 2x2 grid (3r/4 adjacent, r diagonal), Wu's closed form Eq. (3)
PAPER.md:49 on uniform meshes, the separable 3D product-graph closed form, Foster's theorem,
symmetry, triangle inequality, scaling, Rayleigh monotonicity, brute-force pinv on tiny graphs; for the
voltages: the series-chain closed form and the identity of Eq. (4) itself.
"""
from __future__ import annotations

import numpy as np
import scipy.sparse as sp
from scipy.sparse.csgraph import connected_components
from scipy.sparse.linalg import splu


def edge_list(net):
    """All resistors of the 3D network as (u, v, g) arrays with global node ids (step 1)."""
    n, d = net.n, net.d
    idx = np.arange(n * n, dtype=np.int64).reshape(n, n)
    us, vs, gs = [], [], []
    for t in range(d):
        off = t * n * n
        gx, gy = net.gx[t], net.gy[t]
        mx = gx[:, : n - 1] > 0
        my = gy[: n - 1, :] > 0
        us += [off + idx[:, : n - 1][mx], off + idx[: n - 1, :][my]]
        vs += [off + idx[:, 1:][mx], off + idx[1:, :][my]]
        gs += [gx[:, : n - 1][mx], gy[: n - 1, :][my]]
    for i in range(d - 1):
        s = net.tsv_site[i].astype(np.int64)
        loc = s[:, 0] * n + s[:, 1]
        us.append(i * n * n + loc)
        vs.append((i + 1) * n * n + loc)
        gs.append(1.0 / np.asarray(net.tsv_r[i], dtype=np.float64))
    return np.concatenate(us), np.concatenate(vs), np.concatenate(gs).astype(np.float64)


def laplacian_from_edges(nn: int, u, v, g) -> sp.csc_matrix:
    """Weighted graph Laplacian of any resistor list (parallel resistors add)."""
    u = np.asarray(u, dtype=np.int64)
    v = np.asarray(v, dtype=np.int64)
    g = np.asarray(g, dtype=np.float64)
    rows = np.concatenate([u, v, u, v])
    cols = np.concatenate([u, v, v, u])
    vals = np.concatenate([g, g, -g, -g])
    return sp.coo_matrix((vals, (rows, cols)), shape=(nn, nn)).tocsc()


def laplacian(net) -> sp.csc_matrix:
    """Weighted graph Laplacian G of the whole 3D network (step 1)."""
    u, v, g = edge_list(net)
    return laplacian_from_edges(net.d * net.n * net.n, u, v, g)


def node_ids(net):
    """Global ids of the bumps (tier 0) and of the loads (tier d-1)."""
    n = net.n
    b = net.bumps[:, 0].astype(np.int64) * n + net.bumps[:, 1]
    l = (net.d - 1) * n * n + net.loads[:, 0].astype(np.int64) * n + net.loads[:, 1]
    return b, l


class Oracle:
    """Factor once (steps 1-3), then `reff(b, l)` one pair at a time (step 4)."""

    def __init__(self, net, _G=None):
        self.net = net
        self.G = laplacian(net) if _G is None else _G
        nn = self.G.shape[0]
        ncomp, _ = connected_components(self.G, directed=False)
        if ncomp != 1:
            raise ValueError(f"network is not connected ({ncomp} components)")
        self.nn = nn
        self.Gg = self.G[: nn - 1, : nn - 1].tocsc()       # ground the last node
        self.lu = splu(self.Gg, permc_spec="MMD_AT_PLUS_A", diag_pivot_thresh=0.0,
                       options=dict(SymmetricMode=True))
        if net is not None:
            self.bump_id, self.load_id = node_ids(net)

    @classmethod
    def from_edges(cls, nn: int, u, v, g) -> "Oracle":
        """Oracle of an arbitrary resistor list (used by the chain pins); only `reff_nodes`."""
        return cls(None, _G=laplacian_from_edges(nn, u, v, g))

    def reff_nodes(self, a: int, b: int) -> float:
        """R_eff between two global node ids (Eq. 2 via one grounded solve + one refinement)."""
        if a == b:
            return 0.0
        g = self.nn - 1
        rhs = np.zeros(g)
        if a != g:
            rhs[a] += 1.0
        if b != g:
            rhs[b] -= 1.0
        v = self.lu.solve(rhs)
        r = rhs - self.Gg @ v
        v += self.lu.solve(r)
        va = v[a] if a != g else 0.0
        vb = v[b] if b != g else 0.0
        return float(va - vb)

    def node_voltages(self, src: int, v_src: float, sinks, currents) -> np.ndarray:
        """Voltages at the `sinks` when node `src` is held at `v_src` and sink k draws `currents[k]` amperes out
        of the network (which enter at `src`): the DC operating point the paper's Eq. (4)
        expresses through effective resistances.  Computed here from its definition -- KCL, G v = i, one
        grounded solve + one refinement step -- without any effective resistance."""
        g = self.nn - 1
        sinks = np.asarray(sinks, dtype=np.int64)
        currents = np.asarray(currents, dtype=np.float64)
        inj = np.zeros(self.nn)
        np.add.at(inj, sinks, -currents)
        inj[src] += currents.sum()
        rhs = inj[:g]
        v = self.lu.solve(rhs)
        v += self.lu.solve(rhs - self.Gg @ v)
        full = np.append(v, 0.0)                      # the grounded node sits at 0
        return v_src + (full[sinks] - full[src])

    def load_voltages(self, bump_idx: int, currents, v_bump: float) -> np.ndarray:
        """Voltage of every load when bump `bump_idx` is the only supply (at v_bump) and load k draws currents[k]."""
        return self.node_voltages(int(self.bump_id[bump_idx]), v_bump, self.load_id, currents)

    def reff_same_side(self, side: int) -> np.ndarray:
        """R_eff between all pairs of bumps (side 0) or loads (side 1), one pair at a time (Eq. 2)."""
        ids = self.bump_id if side == 0 else self.load_id
        out = np.zeros((ids.size, ids.size))
        for i in range(ids.size):
            for j in range(i + 1, ids.size):
                out[i, j] = out[j, i] = self.reff_nodes(int(ids[i]), int(ids[j]))
        return out

    def reff(self, bump_idx: int, load_idx: int) -> float:
        return self.reff_nodes(int(self.bump_id[bump_idx]), int(self.load_id[load_idx]))

    def reff_pairs(self, bump_idx, load_idx) -> np.ndarray:
        return np.array([self.reff(int(i), int(j)) for i, j in zip(bump_idx, load_idx)])

    def reff_all(self) -> np.ndarray:
        """Full m x n cross product, still one pair at a time."""
        out = np.empty((self.net.m, self.net.nl))
        for i in range(self.net.m):
            for j in range(self.net.nl):
                out[i, j] = self.reff(i, j)
        return out


def reff_dense_pinv(net) -> np.ndarray:
    """Eq. (2) literally, via numpy.linalg.pinv of the dense Laplacian (tiny graphs only)."""
    G = laplacian(net).toarray()
    Gp = np.linalg.pinv(G, hermitian=True)
    b, l = node_ids(net)
    dg = np.diag(Gp)
    return dg[b][:, None] + dg[l][None, :] - 2.0 * Gp[np.ix_(b, l)]


# ---------------------------------------------------------------------------------------------
# Sample production for the large workloads: the factorisation is shared by forked workers, each
# of which still evaluates ONE PAIR AT A TIME with `Oracle.reff` (no change to the arithmetic).
_FORK_ORACLE = None


def _fork_chunk(args):
    bi, li = args
    return _FORK_ORACLE.reff_pairs(bi, li)


def reff_pairs_forked(oracle: Oracle, bump_idx, load_idx, workers: int) -> np.ndarray:
    """`oracle.reff_pairs` split over `workers` forked processes (copy-on-write factor)."""
    import multiprocessing as mp
    global _FORK_ORACLE
    bump_idx = np.asarray(bump_idx)
    load_idx = np.asarray(load_idx)
    if workers <= 1 or bump_idx.size < 2 * workers:
        return oracle.reff_pairs(bump_idx, load_idx)
    _FORK_ORACLE = oracle
    chunks = [(b, l) for b, l in zip(np.array_split(bump_idx, workers * 4),
                                     np.array_split(load_idx, workers * 4)) if b.size]
    with mp.get_context("fork").Pool(workers) as pool:
        parts = pool.map(_fork_chunk, chunks)
    _FORK_ORACLE = None
    return np.concatenate(parts)
