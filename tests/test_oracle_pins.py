"""Pins of the CPU oracle (oracle/reff_oracle.py) to what the paper and the mathematics fix.

None of these retype the oracle's formula or re-call its solver: every expected value is a closed
form, an invariant, or a brute-force definition.  A dropped term, a wrong sign or index, a
transposed plane (gx/gy), a mis-numbered tier or a mis-placed TSV fails at least one of them.
"""
import math

import numpy as np
import pytest

import pdn_inputs as P
from oracle.reff_oracle import Oracle, edge_list, laplacian, reff_dense_pinv

from closed_forms import wu_mesh_reff, product_graph_reff


def single_tier(n, rx=1.0, ry=1.0):
    """d = 1 network (no TSVs): pins on one mesh go through `Oracle.reff_nodes`."""
    net = P.make_uniform(1, n, rx, ry, tsv_sites=[])
    return net


# ------------------------------------------------------------------ textbook chains (general graphs)

def test_series_chain_n_segments_is_n_r():
    for nseg, r in [(1, 2.0), (7, 0.3), (40, 1.25)]:
        u = np.arange(nseg)
        o = Oracle.from_edges(nseg + 1, u, u + 1, np.full(nseg, 1.0 / r))
        assert o.reff_nodes(0, nseg) == pytest.approx(nseg * r, rel=1e-13)
        assert o.reff_nodes(2 % (nseg + 1), 2 % (nseg + 1)) == 0.0
        if nseg >= 5:
            assert o.reff_nodes(1, 4) == pytest.approx(3 * r, rel=1e-13)


def test_parallel_resistors_is_r_over_k():
    for k, r in [(2, 1.0), (5, 3.0)]:
        o = Oracle.from_edges(2, np.zeros(k, int), np.ones(k, int), np.full(k, 1.0 / r))
        assert o.reff_nodes(0, 1) == pytest.approx(r / k, rel=1e-14)
    # unequal: 1 || 2 || 4 ohm = 4/7
    o = Oracle.from_edges(2, [0, 0, 0], [1, 1, 1], [1.0, 0.5, 0.25])
    assert o.reff_nodes(1, 0) == pytest.approx(4.0 / 7.0, rel=1e-14)


def test_series_parallel_ladder():
    # 0 -1ohm- 1 ; 1 =(2ohm || 2ohm)= 2 ; 2 -3ohm- 3   => 1 + 1 + 3
    o = Oracle.from_edges(4, [0, 1, 1, 2], [1, 2, 2, 3], [1.0, 0.5, 0.5, 1.0 / 3.0])
    assert o.reff_nodes(0, 3) == pytest.approx(5.0, rel=1e-14)


def test_stack_of_1x1_tiers_is_sum_of_tsv_resistances():
    # d tiers of one node each, one TSV per interface: a chain through the tiers
    net = P.make_uniform(4, 1, rt=0.0, tsv_sites=[[[0, 0]]] * 3, bumps=[[0, 0]], loads=[[0, 0]])
    net.tsv_r = [np.array([0.5]), np.array([0.25]), np.array([2.0])]
    assert Oracle(net).reff(0, 0) == pytest.approx(2.75, rel=1e-14)


# ------------------------------------------------------------------ mesh assembly

def test_2x2_grid():
    r = 1.7
    o = Oracle(single_tier(2, r, r))
    # nodes: 0=(0,0) 1=(0,1) 2=(1,0) 3=(1,1); a 4-cycle: adjacent r*3r/(4r), opposite 2r*2r/(4r)
    assert o.reff_nodes(0, 1) == pytest.approx(0.75 * r, rel=1e-14)
    assert o.reff_nodes(0, 2) == pytest.approx(0.75 * r, rel=1e-14)
    assert o.reff_nodes(0, 3) == pytest.approx(1.0 * r, rel=1e-14)
    assert o.reff_nodes(1, 2) == pytest.approx(1.0 * r, rel=1e-14)


def test_2x2_grid_distinguishes_gx_from_gy():
    # x-segments 1 ohm, y-segments 3 ohm: cycle 1,3,1,3. (0,0)-(0,1): 1 || 7 = 7/8; (0,0)-(1,0): 3 || 5 = 15/8
    o = Oracle(single_tier(2, 1.0, 3.0))
    assert o.reff_nodes(0, 1) == pytest.approx(7.0 / 8.0, rel=1e-14)
    assert o.reff_nodes(0, 2) == pytest.approx(15.0 / 8.0, rel=1e-14)
    assert o.reff_nodes(0, 3) == pytest.approx(2.0, rel=1e-14)


def test_comb_tree_path_lengths():
    # rows joined only through column 0: a tree, so R = sum of resistances along the unique path
    n, rx, ry = 6, 0.5, 2.0
    net = single_tier(n, rx, ry)
    net.gy[0][:, 1:] = 0.0
    o = Oracle(net)
    a = 0 * n + (n - 1)          # (0, n-1)
    b = (n - 1) * n + (n - 1)    # (n-1, n-1)
    assert o.reff_nodes(a, b) == pytest.approx(2 * (n - 1) * rx + (n - 1) * ry, rel=1e-13)
    c = 2 * n + 3                # (2, 3)
    assert o.reff_nodes(a, c) == pytest.approx((n - 1) * rx + 2 * ry + 3 * rx, rel=1e-13)


@pytest.mark.parametrize("n,rx,ry", [(4, 1.0, 1.0), (7, 1.0, 1.0), (6, 0.7, 2.3), (16, 2.0, 0.5)])
def test_wu_closed_form_eq3_uniform_mesh(n, rx, ry):
    """PAPER.md:49 Eq. (3) [Wu 2004] on a uniform n x n tier, reading G1."""
    o = Oracle(single_tier(n, rx, ry))
    rng = np.random.default_rng(n)
    for _ in range(12):
        y1, x1, y2, x2 = rng.integers(0, n, size=4)
        if (y1, x1) == (y2, x2):
            continue
        want = wu_mesh_reff(n, n, rx, ry, x1, y1, x2, y2)
        got = o.reff_nodes(int(y1 * n + x1), int(y2 * n + x2))
        assert got == pytest.approx(want, rel=1e-11)


def test_edge_count_and_laplacian_rows():
    net = P.make_random(3, d=3, n=5, p=4, m=2, nl=3)
    u, v, g = edge_list(net)
    assert u.size == 3 * 2 * 5 * 4 + 2 * 4          # 2*n*(n-1) segments per tier + TSVs
    assert np.all(g > 0)
    G = laplacian(net)
    assert abs(G.sum(axis=0)).max() < 1e-12 and abs(G - G.T).max() < 1e-15
    # TSV k of interface i joins the SAME site of tier i and tier i+1
    n = net.n
    for i in range(2):
        for k in range(4):
            y, x = net.tsv_site[i][k]
            a, b = i * n * n + y * n + x, (i + 1) * n * n + y * n + x
            assert G[a, b] == pytest.approx(-1.0 / net.tsv_r[i][k])


# ------------------------------------------------------------------ 3D stacks

def test_single_tsv_series_law():
    """One TSV per interface: tiers are in series (Eq. 5 with a single current path):
    R = sum_t R^t(entry, exit) + sum Rt, every intra-tier term from Eq. (3)."""
    n, rx, ry = 6, 1.3, 0.8
    sites = [[[1, 4]], [[5, 0]], [[2, 2]]]
    net = P.make_uniform(4, n, rx, ry, tsv_sites=sites, bumps=[[0, 0], [3, 5]], loads=[[5, 5], [0, 1]])
    net.tsv_r = [np.array([0.11]), np.array([0.07]), np.array([0.2])]
    o = Oracle(net)
    for bi, (by, bx) in enumerate(net.bumps):
        for li, (ly, lx) in enumerate(net.loads):
            hops = [(by, bx)] + [tuple(s[0]) for s in sites] + [(ly, lx)]
            # tier t is entered at hops[t] and left at hops[t+1]
            want = sum(r[0] for r in net.tsv_r)
            for t in range(4):
                (y1, x1), (y2, x2) = hops[t], hops[t + 1]
                if (y1, x1) != (y2, x2):
                    want += wu_mesh_reff(n, n, rx, ry, x1, y1, x2, y2)
            assert o.reff(bi, li) == pytest.approx(want, rel=1e-11)


@pytest.mark.parametrize("d,n,rx,ry,rt", [(2, 3, 1.0, 1.0, 0.5), (3, 4, 0.6, 1.9, 0.05), (4, 5, 1.0, 3.0, 0.2)])
def test_separable_product_graph_closed_form(d, n, rx, ry, rt):
    """Identical uniform tiers with a TSV at EVERY node and uniform Rt: the path-graph product
    P_n x P_n x P_d, whose Laplacian is diagonalised by DCT-II modes."""
    all_sites = np.array([[y, x] for y in range(n) for x in range(n)])
    bumps = [[0, 0], [n - 1, 1]]
    loads = [[n - 1, n - 1], [1, 0], [0, 0]]
    net = P.make_uniform(d, n, rx, ry, rt=rt, tsv_sites=[all_sites] * (d - 1), bumps=bumps, loads=loads)
    o = Oracle(net)
    for bi, (by, bx) in enumerate(bumps):
        for li, (ly, lx) in enumerate(loads):
            want = product_graph_reff(n, n, d, rx, ry, rt, (bx, by, 0), (lx, ly, d - 1))
            assert o.reff(bi, li) == pytest.approx(want, rel=1e-11)


@pytest.mark.parametrize("seed,d,n,p", [(0, 2, 4, 3), (1, 3, 5, 4), (2, 4, 6, 5), (3, 2, 8, 1)])
def test_bruteforce_pinv_on_tiny_random_stacks(seed, d, n, p):
    net = P.make_random(seed, d=d, n=n, p=p, m=3, nl=4, drop=0.1, aniso=2.5)
    got = Oracle(net).reff_all()
    want = reff_dense_pinv(net)
    # independent brute force: solve the KCL system with lstsq instead of pinv
    G = laplacian(net).toarray()
    b_id = net.bumps[:, 0] * n + net.bumps[:, 1]
    l_id = (d - 1) * n * n + net.loads[:, 0] * n + net.loads[:, 1]
    for i, a in enumerate(b_id):
        for j, b in enumerate(l_id):
            rhs = np.zeros(G.shape[0])
            rhs[a] += 1
            rhs[b] -= 1
            v = np.linalg.lstsq(G, rhs, rcond=None)[0]
            assert got[i, j] == pytest.approx(v[a] - v[b], rel=1e-9)
    assert np.allclose(got, want, rtol=1e-10, atol=0)


def test_foster_theorem():
    """sum over resistors of g_e * R_eff(e) = #nodes - 1 (Foster 1949)."""
    for seed, d, n, p in [(5, 2, 6, 3), (6, 3, 6, 4), (7, 4, 6, 2)]:
        net = P.make_random(seed, d=d, n=n, p=p, m=1, nl=1, drop=0.05)
        o = Oracle(net)
        u, v, g = edge_list(net)
        total = sum(ge * o.reff_nodes(int(a), int(b)) for a, b, ge in zip(u, v, g))
        assert total == pytest.approx(d * n * n - 1, rel=1e-11)


def test_symmetry_triangle_scaling():
    net = P.make_random(11, d=3, n=6, p=3, m=2, nl=2)
    o = Oracle(net)
    rng = np.random.default_rng(0)
    nn = 3 * 36
    for _ in range(20):
        a, b, c = rng.choice(nn, size=3, replace=False)
        rab, rba = o.reff_nodes(int(a), int(b)), o.reff_nodes(int(b), int(a))
        assert rab == pytest.approx(rba, rel=1e-12)
        rac, rcb = o.reff_nodes(int(a), int(c)), o.reff_nodes(int(c), int(b))
        assert rab <= rac + rcb + 1e-12 and rab > 0
    # all resistances x c  =>  every R_eff x c
    c = 3.5
    net2 = P.make_random(11, d=3, n=6, p=3, m=2, nl=2)
    net2.gx = [g / c for g in net2.gx]
    net2.gy = [g / c for g in net2.gy]
    net2.tsv_r = [r * c for r in net2.tsv_r]
    assert np.allclose(Oracle(net2).reff_all(), c * o.reff_all(), rtol=1e-12)


def test_rayleigh_monotonicity_added_tsv_and_segment():
    net = P.make_random(21, d=3, n=6, p=2, m=4, nl=4, drop=0.1)
    base = Oracle(net).reff_all()
    # add a TSV to interface 0 at a free site
    used = {tuple(s) for s in net.tsv_site[0]}
    free = next((y, x) for y in range(6) for x in range(6) if (y, x) not in used)
    net.tsv_site[0] = np.vstack([net.tsv_site[0], [free]]).astype(np.int32)
    net.tsv_r[0] = np.append(net.tsv_r[0], 0.05)
    more = Oracle(net).reff_all()
    assert np.all(more <= base * (1 + 1e-12)) and np.any(more < base * (1 - 1e-6))
    # strengthen a segment
    net.gx[1][2, 2] += 5.0
    more2 = Oracle(net).reff_all()
    assert np.all(more2 <= more * (1 + 1e-12))


def test_disconnected_network_is_rejected():
    net = single_tier(4)
    net.gx[0][:, 1] = 0.0
    net.gy[0][:, :] = 0.0
    with pytest.raises(ValueError):
        Oracle(net)


def test_forked_sampler_equals_serial():
    from oracle.reff_oracle import reff_pairs_forked
    net = P.make_config(1)
    o = Oracle(net)
    bi, li = P.sample_pairs(net, 40, cfg=1)
    assert np.array_equal(reff_pairs_forked(o, bi, li, 2), o.reff_pairs(bi, li))


# ----------------------------------------------------------------------------------------- Eq. (4) voltages
def test_node_voltages_on_a_series_chain_closed_form():
    """Chain 0-1-...-n of r-ohm segments, node 0 held at v0, node k draws I_k: the segment (j-1, j) carries the
    current of all loads at or beyond j, so v_j = v0 - r * sum_{s=1..j} sum_{k>=s} I_k."""
    from oracle.reff_oracle import Oracle
    n, r, v0 = 9, 0.37, 1.2
    u = np.arange(n); v = np.arange(1, n + 1)
    o = Oracle.from_edges(n + 1, u, v, np.full(n, 1.0 / r))
    sinks = np.array([2, 5, 9, 7])
    cur = np.array([0.3, 1.1, 0.05, 0.7])
    got = o.node_voltages(0, v0, sinks, cur)
    full_i = np.zeros(n + 1); full_i[sinks] = cur
    want = []
    for j in sinks:
        drop = sum(r * full_i[s:].sum() for s in range(1, j + 1))
        want.append(v0 - drop)
    assert np.allclose(got, want, rtol=1e-12, atol=0)


def test_eq4_identity_between_voltages_and_effective_resistances():
    """PAPER.md:60-65, Eq. (4): v_j = v_b - 1/2 sum_k I_k (R_bj + R_bk - R_jk).  The left side comes from KCL
    (node_voltages), the right side from per-pair effective resistances: two independent routes in the oracle."""
    from oracle.reff_oracle import Oracle
    net = P.make_random(5, d=3, n=6, p=3, m=2, nl=5, drop=0.05)
    o = Oracle(net)
    cur = np.array([0.2, 0.9, 0.0, 1.3, 0.4])
    RLL = o.reff_same_side(1)
    for b in range(net.m):
        Rb = np.array([o.reff(b, k) for k in range(net.nl)])
        want = 0.9 - 0.5 * ((Rb[:, None] + Rb[None, :] - RLL) * cur[None, :]).sum(axis=1)
        assert np.allclose(o.load_voltages(b, cur, 0.9), want, rtol=1e-11, atol=1e-13)
    # same-side resistances against the dense pseudo-inverse
    from oracle.reff_oracle import laplacian, node_ids
    Gp = np.linalg.pinv(laplacian(net).toarray(), hermitian=True)
    _, l = node_ids(net)
    dg = np.diag(Gp)
    assert np.allclose(RLL, dg[l][:, None] + dg[l][None, :] - 2 * Gp[np.ix_(l, l)], rtol=1e-9, atol=1e-12)
