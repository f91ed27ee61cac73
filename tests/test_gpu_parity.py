"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element.

Tolerance (BASELINE.json north_star): per pair |R_gpu - R_oracle| / R_oracle, max <= 1e-6 and
mean <= 1e-8.  Workloads 1-2: the full cross product; workloads 3-5: the seeded 4096-pair sample.
Expected values for the five workloads are the oracle's, stored under tests/golden/ by
tests/golden/make_golden.py (which calls only oracle/); small cases run the oracle live.
"""
import os

import numpy as np
import pytest

import pdn_inputs as P

pytestmark = pytest.mark.gpu

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")
MAX_REL, MEAN_REL = 1e-6, 1e-8


def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    return torch


def load_golden(cfg):
    path = os.path.join(GOLDEN, f"cfg{cfg}_reff.txt")
    if not os.path.exists(path):
        pytest.skip(f"{path} not generated yet (tests/golden/make_golden.py {cfg})")
    a = np.loadtxt(path, comments="#")
    return a[:, 0].astype(np.int32), a[:, 1].astype(np.int32), a[:, 2]


def check(got, want):
    rel = np.abs(got - want) / want
    assert np.all(np.isfinite(got))
    assert rel.max() <= MAX_REL, f"max rel err {rel.max():.3e}"
    assert rel.mean() <= MEAN_REL, f"mean rel err {rel.mean():.3e}"
    return rel


def gpu_all_pairs(net, **kw):
    torch = torch_cuda()
    from paper_2607_05818_b200 import Pdn
    pdn = Pdn.from_network(net, device="cuda:0", **kw)
    out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
    pdn.reff(out)
    st = pdn.stats()
    pdn.close()
    return out.cpu().numpy().reshape(net.m, net.nl), st


@pytest.mark.parametrize("cfg", [1, 2])
def test_workload_full_cross_product(cfg):
    bi, li, want = load_golden(cfg)
    net = P.make_config(cfg, seed=0)
    got, st = gpu_all_pairs(net)
    rel = check(got[bi, li], want)
    print(f"cfg{cfg}: max {rel.max():.2e} mean {rel.mean():.2e} iters {st['pcg_iters_max']}")


@pytest.mark.parametrize("cfg", [1, 2, 3, 4])
def test_precond_f32_meets_the_same_tolerance(cfg):
    """Opt-in PDN_PRECOND_F32 (multigrid sweeps in FP32 registers; CG operator, residuals, solutions FP64):
    same tolerance against the oracle, at most two PCG iterations more than the FP64 preconditioner, and it
    agrees with the default path far inside the tolerance."""
    from paper_2607_05818_b200 import PDN_PRECOND_F32
    bi, li, want = load_golden(cfg)
    net = P.make_config(cfg, seed=0)
    got32, st32 = gpu_all_pairs(net, flags=PDN_PRECOND_F32)
    rel = check(got32[bi, li], want)
    got64, st64 = gpu_all_pairs(net)
    assert st32["pcg_iters_max"] <= st64["pcg_iters_max"] + 2
    assert np.abs(got32 - got64).max() / got64.min() <= 1e-7
    print(f"cfg{cfg} f32 preconditioner: max {rel.max():.2e} mean {rel.mean():.2e} iters {st32['pcg_iters_max']} (f64: {st64['pcg_iters_max']})")


@pytest.mark.parametrize("seed,aniso", [(3, 1.0), (4, 3.0), (5, 40.0)])
def test_precond_f32_random_stacks_against_live_oracle(seed, aniso):
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import PDN_PRECOND_F32
    net = P.make_random(seed, d=3, n=150, p=12, m=5, nl=7, drop=0.01, aniso=aniso)
    got, _ = gpu_all_pairs(net, flags=PDN_PRECOND_F32, rtol=1e-10)
    check(got, Oracle(net).reff_all())


@pytest.mark.parametrize("cfg", [3, 4, 5])
def test_workload_sampled_pairs(cfg):
    """Full-size workloads in the launch configuration bench.py times; pair-list mode of pdn_reff."""
    torch = torch_cuda()
    from paper_2607_05818_b200 import Pdn
    bi, li, want = load_golden(cfg)
    net = P.make_config(cfg, seed=0)
    sbi, sli = P.sample_pairs(net, 4096, seed=0, cfg=cfg)
    assert np.array_equal(sbi, bi) and np.array_equal(sli, li)
    pdn = Pdn.from_network(net, device="cuda:0")
    out = torch.empty(bi.size, dtype=torch.float64, device="cuda:0")
    pdn.reff(out, torch.from_numpy(bi).cuda(), torch.from_numpy(li).cuda())
    rel = check(out.cpu().numpy(), want)
    # the full cross product agrees with the gathered list
    full = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
    pdn.reff(full)
    full = full.cpu().numpy().reshape(net.m, net.nl)
    assert np.allclose(full[bi, li], out.cpu().numpy(), rtol=1e-12, atol=0)   # summation order differs
    st = pdn.stats()
    pdn.close()
    print(f"cfg{cfg}: max {rel.max():.2e} mean {rel.mean():.2e} iters {st['pcg_iters_max']} "
          f"stencil {st['ms_stencil']:.0f} ms dense {st['ms_dense']:.1f} ms")


@pytest.mark.parametrize("seed,d,n,p,m,nl,kw", [
    (0, 2, 2, 1, 1, 1, {}),                 # smallest legal mesh (single level)
    (1, 3, 3, 2, 2, 3, {}),
    (2, 2, 4, 3, 4, 4, {}),                 # n = 4: the mesh is its own coarsest level
    (3, 4, 5, 4, 3, 3, {}),                 # first two-level size, odd
    (4, 3, 7, 5, 4, 6, dict(drop=0.1)),
    (5, 2, 8, 6, 5, 5, dict(aniso=3.0)),
    (6, 3, 13, 7, 6, 4, dict(drop=0.08, aniso=2.0)),   # odd sizes on every level: 13, 7, 4
    (7, 2, 33, 9, 8, 8, {}),                # one node more than a tile: ragged tail
    (8, 4, 40, 11, 5, 9, dict(drop=0.05)),
    (9, 2, 70, 16, 6, 7, dict(aniso=0.25)), # several tiles + ragged tail
    (10, 3, 100, 5, 3, 12, dict(drop=0.02, aniso=3.0)),
])
@pytest.mark.parametrize("rtol", [None, 1e-10], ids=["default_rtol", "rtol1e-10"])
def test_random_stacks_against_live_oracle(seed, d, n, p, m, nl, kw, rtol):
    """`default_rtol`: no rtol argument at all -- the library's default stopping rule (rtol 1e-8 for TSV sources,
    1e-5 for bump / load sources) must meet the north_star tolerance away from the five workloads too."""
    from oracle.reff_oracle import Oracle
    net = P.make_random(seed, d=d, n=n, p=p, m=m, nl=nl, **kw)
    want = Oracle(net).reff_all()
    got, _ = gpu_all_pairs(net, **({} if rtol is None else dict(rtol=rtol)))
    check(got, want)


def test_strongly_heterogeneous_conductances_converge_and_match():
    """Four decades of segment resistance and 10 % removed segments: far from the BASELINE workloads, but the
    solver must still converge (well below the iteration cap) and match the oracle."""
    from oracle.reff_oracle import Oracle
    net = P.make_random(7, d=2, n=150, p=10, m=4, nl=5, r_lo=0.01, r_hi=100.0, drop=0.1)
    got, st = gpu_all_pairs(net)
    assert st["pcg_iters_max"] < 120
    check(got, Oracle(net).reff_all())


@pytest.mark.parametrize("rtol", [None, 1e-10], ids=["default_rtol", "rtol1e-10"])
@pytest.mark.parametrize("nu", [1, 2, 3, 4])
def test_every_smoother_depth(nu, rtol):
    from oracle.reff_oracle import Oracle
    net = P.make_random(20 + nu, d=2, n=45, p=6, m=4, nl=4, drop=0.03)
    got, st = gpu_all_pairs(net, nu=nu, **({} if rtol is None else dict(rtol=rtol)))
    check(got, Oracle(net).reff_all())


def test_small_rhs_batches_and_host_planes_give_same_answer():
    torch = torch_cuda()
    from paper_2607_05818_b200 import Pdn
    net = P.make_config(1, seed=0)
    ref, _ = gpu_all_pairs(net)
    got, _ = gpu_all_pairs(net, rhs_batch=3)          # ragged batches: 16 = 5*3 + 1, 4 = 3 + 1
    assert np.allclose(got, ref, rtol=1e-8, atol=0)
    pdn = Pdn.from_network(net)                       # numpy planes => PDN_TIERS_ON_HOST
    out = np.empty(net.m * net.nl)
    pdn.reff_host(out)
    assert np.allclose(out.reshape(net.m, net.nl), ref, rtol=1e-8, atol=0)
    bi = np.array([3, 0, 2], dtype=np.int32)
    li = np.array([15, 7, 0], dtype=np.int32)
    out3 = np.empty(3)
    pdn.reff_host(out3, bi, li)
    assert np.allclose(out3, out.reshape(net.m, net.nl)[bi, li], rtol=1e-12, atol=0)   # summation order differs
    pdn.close()


@pytest.mark.parametrize("fast_path", [True, False])
def test_port_matrix_matches_wu_closed_form(fast_path):
    """S1 pin: on a uniform tier the intra-die R_jk = Z_jj + Z_kk - 2 Z_jk from the GPU port matrix
    must equal PAPER.md:49 Eq. (3) -- both for the spectral fast path (uniform.cuh: Eq. 3 as two dense
    contractions) and for the numerical multigrid-PCG path forced onto the same tier."""
    from closed_forms import wu_mesh_reff
    from paper_2607_05818_b200 import PDN_NO_UNIFORM_FAST_PATH, Pdn
    torch_cuda()
    n, rx, ry = 24, 0.8, 1.7
    sites = [np.array([[1, 2], [20, 5], [11, 11], [23, 23], [0, 17]])]
    bumps = np.array([[3, 3], [9, 21]])
    loads = np.array([[5, 5]])
    net = P.make_uniform(2, n, rx, ry, rt=0.1, tsv_sites=sites, bumps=bumps, loads=loads)
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-11, flags=0 if fast_path else PDN_NO_UNIFORM_FAST_PATH)
    Z = pdn.port_matrix(0)
    assert pdn.stats()["n_uniform_tiers"] == (2 if fast_path else 0)
    pdn.close()
    pts = [tuple(s) for s in sites[0]] + [tuple(b) for b in bumps]
    assert Z.shape == (7, 7)
    for j in range(7):
        for k in range(5):                      # column must be a TSV port (bump-bump entries are not computed)
            if j == k:
                continue
            (y1, x1), (y2, x2) = pts[j], pts[k]
            want = wu_mesh_reff(n, n, rx, ry, x1, y1, x2, y2)
            got = Z[j, j] + Z[k, k] - 2 * Z[j, k]
            assert got == pytest.approx(want, rel=1e-11 if fast_path else 1e-8)
    assert np.isnan(Z[5, 6]) and np.isnan(Z[6, 5])


@pytest.mark.parametrize("d,n,rx,ry", [(2, 45, 1.0, 1.0), (3, 64, 0.5, 2.0), (4, 130, 1.3, 0.4)])
def test_uniform_stacks_fast_path_against_live_oracle(d, n, rx, ry):
    """End to end on uniform tiers: the Eq. (3) fast path and the numerical path both match the oracle, and
    each other; a stack with one jittered tier takes the fast path only on the uniform ones."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import PDN_NO_UNIFORM_FAST_PATH
    rng = np.random.default_rng([d, n])
    sites = [P._distinct_sites(rng, n, 7) for _ in range(d - 1)]
    net = P.make_uniform(d, n, rx, ry, rt=0.07, tsv_sites=sites, bumps=P._distinct_sites(rng, n, 5),
                         loads=P._distinct_sites(rng, n, 6))
    want = Oracle(net).reff_all()
    fast, st = gpu_all_pairs(net)
    assert st["n_uniform_tiers"] == d and st["pcg_iters_max"] == 0
    rel = check(fast, want)
    assert rel.max() < 1e-10                  # the closed form is exact up to rounding
    slow, st2 = gpu_all_pairs(net, flags=PDN_NO_UNIFORM_FAST_PATH, rtol=1e-10)
    assert st2["n_uniform_tiers"] == 0 and st2["pcg_iters_max"] > 0
    check(slow, want)
    net.gx[1], net.gy[1] = P._jitter_planes(rng, n, rx, ry)          # tier 1 no longer uniform
    mixed, st3 = gpu_all_pairs(net, rtol=1e-10)
    assert st3["n_uniform_tiers"] == d - 1
    check(mixed, Oracle(net).reff_all())


def test_port_matrix_of_a_nonuniform_tier_matches_the_dense_pseudo_inverse():
    """S1 pin on general conductances: Z_t from the GPU = rows / columns of pinv(L_t) of the tier's Laplacian,
    assembled here from the generator's planes (brute force, numpy)."""
    from paper_2607_05818_b200 import Pdn
    torch_cuda()
    net = P.make_random(77, d=2, n=21, p=6, m=3, nl=4, drop=0.05, aniso=2.5)
    n = net.n
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-12)
    for t in range(2):
        Lt = np.zeros((n * n, n * n))
        for y in range(n):
            for x in range(n):
                i = y * n + x
                if x < n - 1 and net.gx[t][y, x] > 0:
                    g = net.gx[t][y, x]; Lt[i, i] += g; Lt[i + 1, i + 1] += g; Lt[i, i + 1] -= g; Lt[i + 1, i] -= g
                if y < n - 1 and net.gy[t][y, x] > 0:
                    g = net.gy[t][y, x]; Lt[i, i] += g; Lt[i + n, i + n] += g; Lt[i, i + n] -= g; Lt[i + n, i] -= g
        Lp = np.linalg.pinv(Lt, hermitian=True)
        term = net.bumps if t == 0 else net.loads
        ports = [int(s[0]) * n + int(s[1]) for s in net.tsv_site[0]] + [int(s[0]) * n + int(s[1]) for s in term]
        Z = pdn.port_matrix(t)
        ntsv = len(net.tsv_site[0])
        want = Lp[np.ix_(ports, ports)]
        ok = ~np.isnan(Z)
        assert ok[:ntsv, :].all() and ok[:, :ntsv].all() and np.diag(ok).all()
        assert np.allclose(Z[ok], want[ok], rtol=0, atol=1e-9 * np.abs(want).max())
    pdn.close()


@pytest.mark.parametrize("seed,d,n,p,kw", [
    (41, 2, 37, 9, {}),
    (42, 3, 70, 12, dict(drop=0.03, aniso=2.0)),
    (43, 4, 24, 6, {}),
])
def test_tsv_replanning_matches_a_fresh_context_and_the_oracle(seed, d, n, p, kw):
    """pdn_update_tsvs (NEXT-2): remove, add, move TSVs and change resistances; the updated context must give
    what a context created on the new network gives, and both must match the oracle of the new network."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import Pdn
    torch = torch_cuda()
    net = P.make_random(seed, d=d, n=n, p=p, m=5, nl=6, **kw)
    rng = np.random.default_rng(seed)
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10)

    def reff(obj):
        out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
        obj.reff(out)
        return out.cpu().numpy().reshape(net.m, net.nl)

    before = reff(pdn)
    for step in range(3):
        for i in range(d - 1):
            s, r = net.tsv_site[i].copy(), net.tsv_r[i].copy()
            if step == 0:      # drop two sites, add three new ones in the middle of the list, rescale one resistance
                keep = np.ones(len(s), bool); keep[rng.choice(len(s), 2, replace=False)] = False
                s, r = s[keep], r[keep]
                new = [x for x in P._distinct_sites(rng, n, 8).tolist() if x not in s.tolist()][:3]
                s = np.vstack([s[:2], np.array(new, dtype=np.int32), s[2:]]); r = np.concatenate([r[:2], rng.uniform(0.02, 0.2, 3), r[2:]])
                r[0] *= 3.0
            elif step == 1:    # permute the list and change every resistance: no new solves
                perm = rng.permutation(len(s)); s, r = s[perm], r[perm] * rng.uniform(0.5, 2.0, len(s))
            else:              # interface 0 only: replace everything but one site
                if i == 0:
                    new = [x for x in P._distinct_sites(rng, n, 10).tolist() if x not in s.tolist()][:4]
                    s = np.vstack([s[:1], np.array(new, dtype=np.int32)]); r = np.concatenate([r[:1], rng.uniform(0.02, 0.2, 4)])
            net.tsv_site[i], net.tsv_r[i] = np.ascontiguousarray(s, dtype=np.int32), r
        pdn.update_tsvs(net.tsv_site, net.tsv_r)
        st = pdn.stats()
        if step == 1:
            assert st["update_solves"] == 0
        got = reff(pdn)
        fresh, _ = gpu_all_pairs(net, rtol=1e-10)
        assert np.allclose(got, fresh, rtol=1e-8, atol=0)
        check(got, Oracle(net).reff_all())
    assert not np.allclose(got, before, rtol=1e-3)
    # a bad list is refused and leaves the context usable
    from paper_2607_05818_b200 import PdnError
    with pytest.raises(PdnError):
        pdn.update_tsvs([s[:0] for s in net.tsv_site], [r[:0] for r in net.tsv_r])
    assert np.allclose(reff(pdn), got, rtol=1e-12, atol=0)
    pdn.close()


def test_tsv_replanning_on_uniform_and_tiny_tiers():
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import Pdn
    torch = torch_cuda()
    for n in (4, 30):                      # n = 4: the mesh is its own coarsest level; n = 30: Eq. (3) fast path
        rng = np.random.default_rng(n)
        net = P.make_uniform(3, n, 0.7, 1.9, rt=0.05, tsv_sites=[P._distinct_sites(rng, n, 3) for _ in range(2)],
                             bumps=P._distinct_sites(rng, n, 3), loads=P._distinct_sites(rng, n, 2))
        pdn = Pdn.from_network(net, device="cuda:0")
        net.tsv_site[1] = np.vstack([net.tsv_site[1][1:], [[n - 1, 0]]]).astype(np.int32)
        if [n - 1, 0] in net.tsv_site[1][:-1].tolist():
            net.tsv_site[1] = net.tsv_site[1][:-1]
        net.tsv_r[1] = np.full(len(net.tsv_site[1]), 0.11)
        pdn.update_tsvs(net.tsv_site, net.tsv_r)
        out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
        pdn.reff(out)
        check(out.cpu().numpy().reshape(net.m, net.nl), Oracle(net).reff_all())
        pdn.close()


@pytest.mark.parametrize("seed,d,n,p,kw", [
    (61, 2, 33, 5, {}),
    (62, 4, 48, 7, dict(drop=0.04, aniso=0.4)),
    (63, 3, 4, 2, {}),                        # single-level mesh: direct path
    (64, 3, 40, 6, dict(uniform=True)),       # uniform tiers: Eq. (3) table
])
def test_arbitrary_tier_endpoints_against_the_oracle(seed, d, n, p, kw):
    """NEXT-3: R_eff between probes on ANY tiers (same tier, adjacent tiers, top-to-bottom, a probe on a TSV site,
    a bump, a load, a duplicate) against the oracle's per-pair solves of the whole 3D system; the bump x load block
    of the probe result equals pdn_reff; still right after TSV re-planning (the kept factor is replaced)."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import Pdn
    torch = torch_cuda()
    kw = dict(kw)
    if kw.pop("uniform", False):
        rng = np.random.default_rng(seed)
        net = P.make_uniform(d, n, 0.9, 1.4, rt=0.1, tsv_sites=[P._distinct_sites(rng, n, p) for _ in range(d - 1)],
                             bumps=P._distinct_sites(rng, n, 3), loads=P._distinct_sites(rng, n, 4))
    else:
        net = P.make_random(seed, d=d, n=n, p=p, m=3, nl=4, **kw)
    rng = np.random.default_rng(seed + 1000)
    nodes = [(int(rng.integers(d)), int(rng.integers(n)), int(rng.integers(n))) for _ in range(9)]
    nodes += [(0, *map(int, net.tsv_site[0][1])), (1, *map(int, net.tsv_site[0][1]))]      # both ends of one TSV
    nodes += [(0, *map(int, net.bumps[0])), (d - 1, *map(int, net.loads[2])), nodes[0]]    # a bump, a load, a duplicate
    nodes = np.array(nodes, dtype=np.int32)
    k = len(nodes)
    gid = nodes[:, 0].astype(np.int64) * n * n + nodes[:, 1] * n + nodes[:, 2]
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10)

    def check(o):
        out = torch.empty(k * k, dtype=torch.float64, device="cuda:0")
        pdn.reff_nodes(nodes, out)
        got = out.cpu().numpy().reshape(k, k)
        want = np.array([[o.reff_nodes(int(a), int(b)) for b in gid] for a in gid])
        assert np.all(np.diag(got) == 0.0)
        nz = want > 0
        rel = np.abs(got[nz] - want[nz]) / want[nz]
        assert rel.max() <= MAX_REL and rel.mean() <= MEAN_REL, (rel.max(), rel.mean())
        assert np.abs(got[~nz]).max() <= 1e-9 * want.max()       # duplicates: cancellation of equal terms
        full = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
        pdn.reff(full)
        assert abs(got[k - 3, k - 2] / full.cpu().numpy().reshape(net.m, net.nl)[0, 2] - 1.0) <= 1e-8
        # pdn_reff_from: one source against all the others (one row of the same matrix, by diagonal solves +
        # reciprocity), for a source on the top tier, on a middle / bottom tier and on a TSV site
        for s_ in (0, 3, 9):
            row = torch.empty(k, dtype=torch.float64, device="cuda:0")
            pdn.reff_from(nodes[s_], nodes, row)
            r_ = row.cpu().numpy()
            nzr = want[s_] > 0
            relr = np.abs(r_[nzr] - want[s_][nzr]) / want[s_][nzr]
            assert relr.max() <= MAX_REL and relr.mean() <= MEAN_REL, (s_, relr.max(), relr.mean())
            assert np.abs(r_[~nzr]).max() <= 1e-8 * want.max()

    check(Oracle(net))
    if n > 4:
        rng = np.random.default_rng(seed + 7)
        new = [x for x in P._distinct_sites(rng, n, 6).tolist() if x not in net.tsv_site[0].tolist()][:2]
        net.tsv_site[0] = np.vstack([net.tsv_site[0][:-1], np.array(new, dtype=np.int32)]).astype(np.int32)
        net.tsv_r[0] = np.concatenate([net.tsv_r[0][:-1], [0.07, 0.09]])
        pdn.update_tsvs(net.tsv_site, net.tsv_r)
        check(Oracle(net))
    with pytest.raises(Exception):
        pdn.reff_nodes(np.array([[d, 0, 0]], dtype=np.int32), torch.empty(1, dtype=torch.float64, device="cuda:0"))
    pdn.close()


@pytest.mark.parametrize("n", [1500, 2047])
@pytest.mark.parametrize("fast_path", [True, False])
def test_large_ragged_meshes_match_wu_closed_form(n, fast_path):
    """Sizes beyond BASELINE's and not powers of two (ragged tiles on every level, odd coarse meshes), ports in
    three corners: the intra-die R_jk from the GPU port matrix against Eq. (3), for the numerical path
    and for the spectral table."""
    from closed_forms import wu_mesh_reff
    from paper_2607_05818_b200 import PDN_NO_UNIFORM_FAST_PATH, Pdn
    torch_cuda()
    rng = np.random.default_rng(n)
    sites = [P._distinct_sites(rng, n, 6)]
    sites[0][0], sites[0][1], sites[0][2] = (0, 0), (n - 1, n - 1), (n - 1, 0)
    net = P.make_uniform(2, n, 0.8, 1.7, rt=0.1, tsv_sites=sites, bumps=np.array([[3, 3]]), loads=np.array([[5, 5]]))
    if fast_path:      # enough ports for the table to pay on a mesh this size (with 6 the library solves instead)
        extra = [s for s in P._distinct_sites(rng, n, 300).tolist() if s not in sites[0].tolist()]
        sites[0] = np.vstack([sites[0], np.array(extra, dtype=np.int32)])
        net = P.make_uniform(2, n, 0.8, 1.7, rt=0.1, tsv_sites=sites, bumps=np.array([[3, 3]]), loads=np.array([[5, 5]]))
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10, flags=0 if fast_path else PDN_NO_UNIFORM_FAST_PATH)
    Z = pdn.port_matrix(0)
    assert pdn.stats()["n_uniform_tiers"] == (2 if fast_path else 0)
    pdn.close()
    for j in range(6):
        for k in range(j + 1, 6):
            (y1, x1), (y2, x2) = sites[0][j], sites[0][k]
            want = wu_mesh_reff(n, n, 0.8, 1.7, x1, y1, x2, y2)
            assert abs((Z[j, j] + Z[k, k] - 2 * Z[j, k]) / want - 1.0) <= 1e-9


@pytest.mark.parametrize("aniso", [40.0, 1.0 / 40.0])
def test_strongly_anisotropic_tiers_converge_and_match_the_oracle(aniso):
    """Tiers whose x- and y-segments differ 40-fold (either way): the smoother widens its interval and deepens its
    polynomial by itself (pdn_api.cu: reduce_tier), the solves stay far from max_iter and the result is the oracle's."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import Pdn
    torch = torch_cuda()
    net = P.make_random(81, d=3, n=150, p=9, m=4, nl=5, aniso=aniso)
    pdn = Pdn.from_network(net, device="cuda:0")
    out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
    pdn.reff(out)
    assert pdn.stats()["pcg_iters_max"] <= 30
    pdn.close()
    check(out.cpu().numpy().reshape(net.m, net.nl), Oracle(net).reff_all())


def test_reff_map_over_a_whole_tier_against_the_oracle():
    """NEXT-3 / Fig. 6(d): the R_eff map from a bump to EVERY node of the bottom tier (stride 1) and to a
    sub-grid of a middle tier, against per-node solves of the oracle."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import Pdn
    torch_cuda()
    d, n = 3, 20
    net = P.make_random(71, d=d, n=n, p=6, m=2, nl=3, drop=0.03)
    o = Oracle(net)
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10)
    src = (0, int(net.bumps[1][0]), int(net.bumps[1][1]))
    a = src[1] * n + src[2]
    for tier, stride in ((d - 1, 1), (1, 3)):
        got = pdn.reff_map(src, tier, stride)
        ys = np.arange(0, n, stride)
        want = np.array([[o.reff_nodes(a, tier * n * n + int(y) * n + int(x)) for x in ys] for y in ys])
        assert got.shape == want.shape
        rel = np.abs(got - want) / want
        assert rel.max() <= MAX_REL and rel.mean() <= MEAN_REL, (rel.max(), rel.mean())
    pdn.close()


@pytest.mark.parametrize("seed,d,n,p,kw", [
    (51, 2, 33, 5, {}),
    (52, 3, 64, 8, dict(drop=0.04, aniso=0.4)),
    (53, 2, 4, 2, {}),                        # single-level mesh: direct path
])
def test_same_side_pairs_and_eq4_voltages_against_the_oracle(seed, d, n, p, kw):
    """NEXT-3: bump-bump / load-load effective resistances and the load voltages of Eq. (4),
    against the oracle (per-pair solves for R, a KCL solve for the voltages); the bump x load result of a
    PDN_TERMINAL_PAIRS context equals the default one; TSV re-planning keeps working on it."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import PDN_TERMINAL_PAIRS, Pdn
    torch = torch_cuda()
    net = P.make_random(seed, d=d, n=n, p=p, m=4, nl=7, **kw)
    o = Oracle(net)
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10, flags=PDN_TERMINAL_PAIRS)
    for side, nt in ((0, net.m), (1, net.nl)):
        out = torch.empty(nt * nt, dtype=torch.float64, device="cuda:0")
        pdn.reff_same_side(side, out)
        got, want = out.cpu().numpy().reshape(nt, nt), o.reff_same_side(side)
        off = ~np.eye(nt, dtype=bool)
        assert np.all(np.diag(got) == 0.0)
        assert np.allclose(got, got.T, rtol=1e-8, atol=0)
        rel = np.abs(got[off] - want[off]) / want[off]
        assert rel.max() <= MAX_REL and rel.mean() <= MEAN_REL
    cur = torch.tensor(np.random.default_rng(seed).uniform(0.0, 1.5, net.nl), dtype=torch.float64, device="cuda:0")
    v = torch.empty(net.nl, dtype=torch.float64, device="cuda:0")
    for b in range(net.m):
        pdn.load_voltages(b, cur, 0.8, v)
        want = o.load_voltages(b, cur.cpu().numpy(), 0.8)
        assert np.allclose(v.cpu().numpy(), want, rtol=0, atol=1e-8 * np.abs(0.8 - want).max())
    full = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
    pdn.reff(full)
    ref, _ = gpu_all_pairs(net, rtol=1e-10)
    assert np.allclose(full.cpu().numpy().reshape(net.m, net.nl), ref, rtol=1e-8, atol=0)
    Z = pdn.port_matrix(0)
    assert not np.isnan(Z).any()              # terminal-terminal entries exist now
    if n > 4:                                 # re-plan on a context that keeps the terminal rows
        rng = np.random.default_rng(seed)
        new = [x for x in P._distinct_sites(rng, n, 6).tolist() if x not in net.tsv_site[0].tolist()][:2]
        net.tsv_site[0] = np.vstack([net.tsv_site[0][1:], np.array(new, dtype=np.int32)]).astype(np.int32)
        net.tsv_r[0] = np.concatenate([net.tsv_r[0][1:], [0.07, 0.09]])
        pdn.update_tsvs(net.tsv_site, net.tsv_r)
        o2 = Oracle(net)
        out = torch.empty(net.nl * net.nl, dtype=torch.float64, device="cuda:0")
        pdn.reff_same_side(1, out)
        got, want = out.cpu().numpy().reshape(net.nl, net.nl), o2.reff_same_side(1)
        off = ~np.eye(net.nl, dtype=bool)
        assert (np.abs(got[off] - want[off]) / want[off]).max() <= MAX_REL
        pdn.reff(full)
        check(full.cpu().numpy().reshape(net.m, net.nl), o2.reff_all())
    pdn.close()
    plain = Pdn.from_network(net, device="cuda:0")
    from paper_2607_05818_b200 import PdnError
    with pytest.raises(PdnError):
        plain.reff_same_side(1, torch.empty(net.nl * net.nl, dtype=torch.float64, device="cuda:0"))
    plain.close()


@pytest.mark.parametrize("fast_path", [True, False])
def test_recombination_pins_series_law_and_separable_product_graph(fast_path):
    """S2-S3 pins that do not go through the oracle:
    (i) one TSV per interface => R = sum_t R^t(entry, exit) + sum Rt with every R^t from Eq. (3);
    (ii) identical uniform tiers with a TSV at EVERY node are the product graph P_n x P_n x P_d, whose two-point
    resistance has a closed DCT form (tests/closed_forms.py)."""
    from closed_forms import product_graph_reff, wu_mesh_reff
    from paper_2607_05818_b200 import PDN_NO_UNIFORM_FAST_PATH
    flags = 0 if fast_path else PDN_NO_UNIFORM_FAST_PATH
    # (i) series law, 3 tiers of 17 x 17, anisotropic
    n, rx, ry, rt = 17, 0.9, 2.3, 0.31
    sites = [np.array([[3, 12]]), np.array([[15, 1]])]
    bumps, loads = np.array([[0, 0], [8, 9]]), np.array([[16, 16], [2, 5], [15, 1]])
    net = P.make_uniform(3, n, rx, ry, rt=rt, tsv_sites=sites, bumps=bumps, loads=loads)
    got, _ = gpu_all_pairs(net, rtol=1e-11, flags=flags)

    def R2d(a, b):
        return 0.0 if tuple(a) == tuple(b) else wu_mesh_reff(n, n, rx, ry, a[1], a[0], b[1], b[0])
    for i, b in enumerate(bumps):
        for j, l in enumerate(loads):
            want = R2d(b, sites[0][0]) + rt + R2d(sites[0][0], sites[1][0]) + rt + R2d(sites[1][0], l)
            assert got[i, j] == pytest.approx(want, rel=1e-8)
    # (ii) product graph, 3 tiers of 6 x 6, TSV at every node
    n, d, rx, ry, rt = 6, 3, 1.2, 0.7, 0.45
    every = np.array([[y, x] for y in range(n) for x in range(n)])
    bumps, loads = np.array([[0, 0], [2, 3]]), np.array([[5, 5], [2, 3], [0, 4]])
    net = P.make_uniform(d, n, rx, ry, rt=rt, tsv_sites=[every] * (d - 1), bumps=bumps, loads=loads)
    got, _ = gpu_all_pairs(net, rtol=1e-11, flags=flags)
    for i, b in enumerate(bumps):
        for j, l in enumerate(loads):
            want = product_graph_reff(n, n, d, rx, ry, rt, (b[1], b[0], 0), (l[1], l[0], d - 1))
            assert got[i, j] == pytest.approx(want, rel=1e-8)
    # (iii) the same product graph, endpoints on ANY tier (pdn_reff_nodes): middle-middle, top-middle, same column
    torch = torch_cuda()
    from paper_2607_05818_b200 import Pdn
    nodes = np.array([[1, 2, 3], [1, 5, 0], [0, 2, 3], [2, 2, 3], [0, 0, 0], [2, 5, 5], [1, 0, 4]], dtype=np.int32)
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-11, flags=flags)
    out = torch.empty(len(nodes) ** 2, dtype=torch.float64, device="cuda:0")
    got = pdn.reff_nodes(nodes, out).cpu().numpy().reshape(len(nodes), len(nodes))
    pdn.close()
    for i, (ta, ya, xa) in enumerate(nodes):
        for j, (tb, yb, xb) in enumerate(nodes):
            if i != j:
                assert got[i, j] == pytest.approx(product_graph_reff(n, n, d, rx, ry, rt, (xa, ya, ta), (xb, yb, tb)), rel=1e-8)


def test_bump_on_tsv_site_and_shared_sites_between_interfaces():
    from oracle.reff_oracle import Oracle
    sites = [np.array([[2, 2], [5, 1]]), np.array([[2, 2], [0, 6]])]     # (2,2) used by both interfaces
    net = P.make_random(31, d=3, n=9, p=2, m=2, nl=2)
    net.tsv_site = [s.astype(np.int32) for s in sites]
    net.bumps = np.array([[2, 2], [8, 8]], dtype=np.int32)              # bump 0 sits on a TSV site
    net.loads = np.array([[0, 6], [4, 4]], dtype=np.int32)              # load 0 sits on a TSV site
    got, _ = gpu_all_pairs(net, rtol=1e-10)
    check(got, Oracle(net).reff_all())


@pytest.mark.parametrize("world,flags_name", [(2, None), (3, "PDN_TERMINAL_PAIRS")])
def test_sharded_port_solves_emulated_on_one_gpu(world, flags_name):
    """NEXT-4: `world` open contexts in one process play the ranks of a sharded run: each solves its slice of
    every tier's sources, the rows are exchanged (here: device copies between the contexts' buffers -- what a
    broadcast per rank does across GPUs), pdn_finish runs S2-S3 everywhere; every rank then equals the
    unsharded result and the oracle."""
    from oracle.reff_oracle import Oracle
    import paper_2607_05818_b200 as pkg
    from paper_2607_05818_b200 import Pdn, PdnError
    torch = torch_cuda()
    flags = getattr(pkg, flags_name) if flags_name else 0
    net = P.make_random(71, d=3, n=47, p=7, m=5, nl=6, drop=0.03)
    net.gx[1], net.gy[1] = P._planes(net.n, np.full((net.n, net.n), 0.8), np.full((net.n, net.n), 1.3))  # a uniform tier
    ref, _ = gpu_all_pairs(net, rtol=1e-10, flags=flags)
    ranks = [Pdn.from_network(net, device="cuda:0", rtol=1e-10, flags=flags, shard_rank=r, shard_world=world)
             for r in range(world)]
    out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
    with pytest.raises(PdnError):
        ranks[0].reff(out)                      # still open
    for src in range(world):                    # "broadcast" of rank src's pieces to everybody else
        pieces = [r.shard_pieces(src) for r in ranks]
        for k, (_, mine) in enumerate(pieces[src]):
            for dst in range(world):
                if dst != src:
                    assert pieces[dst][k][1].numel() == mine.numel()
                    pieces[dst][k][1].copy_(mine)
    for r in ranks:
        r.finish()
        r.reff(out)
        got = out.cpu().numpy().reshape(net.m, net.nl)
        assert np.allclose(got, ref, rtol=1e-9, atol=0)
        check(got, Oracle(net).reff_all())
        if flags:
            ll = torch.empty(net.nl * net.nl, dtype=torch.float64, device="cuda:0")
            r.reff_same_side(1, ll)
            want = Oracle(net).reff_same_side(1)
            off = ~np.eye(net.nl, dtype=bool)
            assert (np.abs(ll.cpu().numpy().reshape(net.nl, net.nl)[off] - want[off]) / want[off]).max() <= MAX_REL
        nodes = np.array([[1, 3, 40], [0, 20, 20], [2, 46, 0]], dtype=np.int32)     # probes on a finished sharded context
        rn = torch.empty(9, dtype=torch.float64, device="cuda:0")
        r.reff_nodes(nodes, rn)
        o = Oracle(net)
        gid = nodes[:, 0].astype(np.int64) * net.n ** 2 + nodes[:, 1] * net.n + nodes[:, 2]
        for a_ in range(3):
            for b_ in range(a_ + 1, 3):
                assert abs(rn[3 * a_ + b_].item() / o.reff_nodes(int(gid[a_]), int(gid[b_])) - 1.0) <= MAX_REL
        r.close()


@pytest.mark.parametrize("block,rtol", [(0, 1e-10), (1, 1e-10), (2, 1e-10), (3, None), (4, None)],
                         ids=["b0", "b1", "b2", "b3_default_rtol", "b4_default_rtol"])
def test_randomised_stacks_through_every_entry_point(block, rtol):
    """Seeded fuzz, 12 stacks per block: random d, n (1-level meshes, one node more / less than a tile, odd sizes),
    port counts, anisotropy (up to 12), removed segments, a uniform tier now and then, random flags, batch sizes and
    smoother depths, device or host planes -- pdn_reff, pdn_reff_nodes on random probes, then a TSV re-plan followed by
    pdn_reff (and the load-load pairs when the context keeps them), all against the oracle."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import PDN_NO_UNIFORM_FAST_PATH, PDN_TERMINAL_PAIRS, Pdn
    torch = torch_cuda()

    # rtol 1e-10: every single entry within 1e-8.  Default stopping rule (no rtol argument): the north_star bar
    # itself, max <= 1e-6 and mean <= 1e-8 per result array, on stacks far from BASELINE's distributions
    # (anisotropy 12, 10 % of the segments removed, smoother depth 2).
    def rel_err(got, want):
        nz = want > 0
        assert np.abs(got[~nz]).max(initial=0.0) <= 1e-9 * max(want.max(), 1.0)
        rel = np.abs(got[nz] / want[nz] - 1.0)
        if rtol is None:
            assert rel.mean() <= MEAN_REL if rel.size else True
            return rel.max(initial=0.0) * (1e-8 / MAX_REL)      # so that "<= 1e-8" below reads "max <= 1e-6"
        return rel.max(initial=0.0)

    for it in range(12):
        seed = 7000 + 100 * block + it
        rng = np.random.default_rng(seed)
        d, n = int(rng.integers(2, 6)), int(rng.choice([2, 3, 4, 5, 7, 9, 16, 17, 31, 33, 56, 57, 65, 90, 113]))
        p = int(rng.integers(1, min(n * n, 12) + 1))
        m, nl = int(rng.integers(1, min(n * n, 6) + 1)), int(rng.integers(1, min(n * n, 7) + 1))
        aniso = float(rng.choice([1.0, 1.0, 0.3, 3.0, 12.0]))
        drop = float(rng.choice([0.0, 0.0, 0.03, 0.1])) if n >= 5 else 0.0
        net = P.make_random(seed, d=d, n=n, p=p, m=m, nl=nl, aniso=aniso, drop=drop)
        if rng.random() < 0.25:
            t = int(rng.integers(d))
            net.gx[t], net.gy[t] = P._planes(n, np.full((n, n), 0.7), np.full((n, n), 1.9))
        flags = (PDN_TERMINAL_PAIRS if rng.random() < 0.4 else 0) | (PDN_NO_UNIFORM_FAST_PATH if rng.random() < 0.3 else 0)
        kw = dict(flags=flags, rhs_batch=int(rng.choice([0, 0, 1, 3, 7])), nu=int(rng.choice([0, 0, 2, 3, 5, 6])))
        if rtol is not None:
            kw["rtol"] = rtol
        what = f"seed {seed}: d={d} n={n} p={p} m={m} nl={nl} aniso={aniso} drop={drop} {kw}"
        pdn = Pdn.from_network(net, device="cuda:0" if rng.random() < 0.7 else None, **kw)
        o = Oracle(net)
        out = torch.empty(m * nl, dtype=torch.float64, device="cuda:0")
        pdn.reff(out)
        assert rel_err(out.cpu().numpy().reshape(m, nl), o.reff_all()) <= 1e-8, what
        k = int(rng.integers(1, 8))
        nodes = np.stack([rng.integers(0, d, k), rng.integers(0, n, k), rng.integers(0, n, k)], axis=1).astype(np.int32)
        rn = torch.empty(k * k, dtype=torch.float64, device="cuda:0")
        pdn.reff_nodes(nodes, rn)
        gid = nodes[:, 0].astype(np.int64) * n * n + nodes[:, 1] * n + nodes[:, 2]
        want = np.array([[o.reff_nodes(int(a), int(b)) for b in gid] for a in gid])
        assert rel_err(rn.cpu().numpy().reshape(k, k), want) <= 1e-8, what
        row = torch.empty(k, dtype=torch.float64, device="cuda:0")     # pdn_reff_from: the first probe against all of them
        pdn.reff_from(nodes[0], nodes, row)
        if rtol is None:
            assert rel_err(row.cpu().numpy(), want[0]) <= 1e-8, what
        else:   # the probes' diagonals come from loosely converged (second-order) solves whatever rtol is
            nz0 = want[0] > 0
            assert np.abs(row.cpu().numpy()[nz0] / want[0][nz0] - 1.0).max(initial=0.0) <= 1e-7, what
        if n * n > p + 1:
            new = [x for x in P._distinct_sites(np.random.default_rng(seed + 5), n, min(n * n, p + 3)).tolist()
                   if x not in net.tsv_site[0].tolist()][:1]
            keep = slice(1, None) if p > 1 else slice(None)
            net.tsv_site[0] = np.vstack([net.tsv_site[0][keep], np.array(new, dtype=np.int32).reshape(-1, 2)]).astype(np.int32)
            net.tsv_r[0] = np.concatenate([net.tsv_r[0][keep], [0.11] * len(new)])
            pdn.update_tsvs(net.tsv_site, net.tsv_r)
            o = Oracle(net)
            pdn.reff(out)
            assert rel_err(out.cpu().numpy().reshape(m, nl), o.reff_all()) <= 1e-8, what
            if flags & PDN_TERMINAL_PAIRS:
                ll = torch.empty(nl * nl, dtype=torch.float64, device="cuda:0")
                pdn.reff_same_side(1, ll)
                assert rel_err(ll.cpu().numpy().reshape(nl, nl), o.reff_same_side(1)) <= 1e-8, what
        pdn.close()


@pytest.mark.parametrize("n,kw", [(4, {}), (37, dict(drop=0.05, aniso=2.0)), (130, {}), (64, dict(uniform=True))])
def test_single_tier_is_the_2d_case(n, kw):
    """Degenerate stack: ONE tier, no TSVs -- R_eff between bumps and loads of the same mesh (Eq. 2 on a 2-D PDN), against
    the oracle and, on the uniform mesh, against Eq. (3) PAPER.md:49 directly; a bump that is also a load gives 0."""
    from closed_forms import wu_mesh_reff
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import Pdn, PdnError
    torch = torch_cuda()
    kw = dict(kw)
    if kw.pop("uniform", False):
        rng = np.random.default_rng(n)
        net = P.make_uniform(1, n, 0.6, 1.1, tsv_sites=[], bumps=P._distinct_sites(rng, n, 40), loads=P._distinct_sites(rng, n, 45))
    else:
        net = P.make_random(91, d=1, n=n, p=1, m=3, nl=5, **kw)
    net.loads[1] = net.bumps[0]                      # the same node on both lists
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10)
    out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
    pdn.reff(out)
    got = out.cpu().numpy().reshape(net.m, net.nl)
    want = Oracle(net).reff_all()
    assert abs(got[0, 1]) <= 1e-12 * want.max()
    nz = want > 0
    rel = np.abs(got[nz] / want[nz] - 1.0)
    assert rel.max() <= MAX_REL and rel.mean() <= MEAN_REL
    if net.name.startswith("uniform") or "uniform" in net.name:
        assert pdn.stats()["n_uniform_tiers"] == 1
    if n == 64:
        for i in range(0, net.m, 7):
            for j in range(2, net.nl, 9):
                (y1, x1), (y2, x2) = net.bumps[i], net.loads[j]
                assert got[i, j] == pytest.approx(wu_mesh_reff(n, n, 0.6, 1.1, x1, y1, x2, y2), rel=1e-9)
    bi = torch.tensor([2, 0], dtype=torch.int32, device="cuda:0")
    li = torch.tensor([4, 3], dtype=torch.int32, device="cuda:0")
    o2 = torch.empty(2, dtype=torch.float64, device="cuda:0")
    pdn.reff(o2, bi, li)
    assert np.allclose(o2.cpu().numpy(), got[[2, 0], [4, 3]], rtol=1e-12, atol=0)
    with pytest.raises(PdnError):
        pdn.reff_nodes(np.array([[0, 0, 0], [0, 1, 1]], dtype=np.int32), torch.empty(4, dtype=torch.float64, device="cuda:0"))
    pdn.close()


def test_two_host_threads_with_their_own_contexts():
    """The library is thread-compatible: contexts created and used concurrently from two host threads (shared
    device-memory pool, per-thread pinned scratch) give the same results as one after the other."""
    import threading
    nets = [P.make_random(61 + k, d=2 + k, n=40 + 9 * k, p=6, m=3, nl=4) for k in range(2)]
    ref = [gpu_all_pairs(net, rtol=1e-10)[0] for net in nets]
    got, err = [None, None], []

    def work(k):
        try:
            for _ in range(4):
                got[k] = gpu_all_pairs(nets[k], rtol=1e-10)[0]
        except Exception as e:      # noqa: BLE001
            err.append(e)
    th = [threading.Thread(target=work, args=(k,)) for k in range(2)]
    [t.start() for t in th]
    [t.join() for t in th]
    assert not err, err
    for k in range(2):
        assert np.allclose(got[k], ref[k], rtol=1e-9, atol=0)


def test_out_of_range_pair_index_yields_nan():
    torch = torch_cuda()
    from paper_2607_05818_b200 import Pdn
    net = P.make_config(1, seed=0)
    pdn = Pdn.from_network(net, device="cuda:0")
    bi = torch.tensor([0, 4, -1], dtype=torch.int32, device="cuda:0")
    li = torch.tensor([0, 0, 3], dtype=torch.int32, device="cuda:0")
    out = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    pdn.reff(out, bi, li)
    o = out.cpu().numpy()
    assert np.isfinite(o[0]) and np.isnan(o[1]) and np.isnan(o[2])
    pdn.close()


def test_error_statuses():
    torch_cuda()
    from paper_2607_05818_b200 import Pdn, PdnError
    net = P.make_config(1, seed=0)

    def expect(status, mutate):
        bad = P.make_config(1, seed=0)
        mutate(bad)
        with pytest.raises(PdnError) as e:
            Pdn.from_network(bad, device="cuda:0")
        assert e.value.status == status

    expect(1, lambda b: b.tsv_site.__setitem__(0, np.vstack([b.tsv_site[0][:-1], b.tsv_site[0][:1]])))  # duplicate
    expect(1, lambda b: b.tsv_r.__setitem__(0, -b.tsv_r[0]))                                            # r <= 0
    expect(1, lambda b: setattr(b, "bumps", np.array([[32, 0]], dtype=np.int32)))                       # out of range
    expect(1, lambda b: b.gx[0].__setitem__((3, 3), -1.0))                                              # negative g
    expect(1, lambda b: b.gy[1].__setitem__((3, 3), np.nan))

    def cut(b):   # split tier 1 in two halves
        b.gx[1][:, 15] = 0.0
    expect(2, cut)
    # isolated node
    def isolate(b):
        b.gx[0][4, 4] = b.gx[0][4, 3] = b.gy[0][4, 4] = b.gy[0][3, 4] = 0.0
    expect(2, isolate)
    # iteration cap reached
    with pytest.raises(PdnError) as e:
        Pdn.from_network(net, device="cuda:0", max_iter=1)
    assert e.value.status == 3
    # wrong n_pairs for the cross product
    import torch
    pdn = Pdn.from_network(net, device="cuda:0")
    five = torch.empty(5, dtype=torch.float64, device="cuda:0")
    with pytest.raises(ValueError):
        pdn.reff(five)                                     # refused by the binding ...
    assert pdn._lib.pdn_reff(pdn._h, 5, None, None, five.data_ptr()) == 1   # ... and by the library itself (PDN_E_ARG)
    pdn.close()


def test_binding_refuses_buffers_the_library_would_misread():
    """The C side reads raw doubles / int32s: wrong dtypes, sizes or sides are refused before the call."""
    torch = torch_cuda()
    from paper_2607_05818_b200 import Pdn
    net = P.make_config(1, seed=0)
    with pytest.raises(TypeError):
        Pdn(net.n, [g.astype(np.float32) for g in net.gx], net.gy, net.tsv_site, net.tsv_r, net.bumps, net.loads)
    pdn = Pdn.from_network(net, device="cuda:0")
    npairs = net.m * net.nl
    with pytest.raises(TypeError):
        pdn.reff(torch.empty(npairs, dtype=torch.float32, device="cuda:0"))
    out3 = torch.empty(3, dtype=torch.float64, device="cuda:0")
    with pytest.raises(TypeError):                         # torch's default integer dtype is int64
        pdn.reff(out3, torch.tensor([0, 1, 2], device="cuda:0"), torch.tensor([0, 1, 2], device="cuda:0"))
    i32 = torch.tensor([0, 1], dtype=torch.int32, device="cuda:0")
    with pytest.raises(ValueError):                        # one index per pair
        pdn.reff(out3, i32, i32)
    with pytest.raises(ValueError):                        # a host buffer on the device entry point
        pdn.reff(np.empty(npairs))
    with pytest.raises(ValueError):
        pdn.reff_host(torch.empty(npairs, dtype=torch.float64, device="cuda:0"))
    with pytest.raises(ValueError):
        pdn.reff_nodes(np.array([[0, 0, 0], [1, 1, 1]], dtype=np.int32), torch.empty(3, dtype=torch.float64, device="cuda:0"))
    m = pdn.reff_map((0, 0, 0), 1, stride=16)              # allocates on the context's device
    assert m.shape == (2, 2) and np.isfinite(m).all()
    pdn.close()


def test_initial_guess_is_rejected_where_it_does_not_help():
    """The closed-form guess comes from the tier's MEAN mesh.  A tier made of two halves whose conductances differ
    2.5-fold has a coefficient of variation of 0.43 -- the guess is tried -- but near most sources the mean mesh is off
    by a factor of 1.4-1.75, so the guess does not halve the residual there: those right-hand sides must fall back to
    x0 = 0 on the device (k_guess_check) and every result must still match the oracle; with the guess switched off the
    result is the same to solver tolerance."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import PDN_NO_INITIAL_GUESS
    n = 200
    net = P.make_random(55, d=2, n=n, p=80, m=40, nl=40, r_lo=0.9, r_hi=1.1)   # >= n/2 right-hand sides per tier: a table is built
    for t in range(2):
        net.gx[t][:, : n // 2] *= 2.5
        net.gy[t][:, : n // 2] *= 2.5
    got, st = gpu_all_pairs(net)
    assert st["n_guess_tiers"] == 2 and 0 < st["n_guess_rejected"]
    check(got, Oracle(net).reff_all())
    ref, st0 = gpu_all_pairs(net, flags=PDN_NO_INITIAL_GUESS)
    assert st0["n_guess_tiers"] == 0 and st0["n_guess_rejected"] == 0
    assert np.allclose(got, ref, rtol=1e-7, atol=0)
    print(f"guess rejected for {st['n_guess_rejected']} of {2 * (80 + 40)} right-hand sides; "
          f"rhs-iterations {st['rhs_iterations']} (x0 = 0 everywhere: {st0['rhs_iterations']})")


def test_more_than_65535_terminals():
    """m + n_loads > 65535: the kernels that used to put that dimension in gridDim.y (limit 65535) now walk it; a
    sample of the 1.04e9 pairs through the pair list against the oracle, and the terminal diagonals from 66 000
    bump / load solves on a 256^2 mesh (which start from the closed-form guess)."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import Pdn
    torch = torch_cuda()
    m, nl = 40000, 26000
    net = P.make_random(97, d=2, n=256, p=8, m=m, nl=nl)
    assert m + nl > 65535 and len({tuple(b) for b in net.bumps.tolist()}) == m
    pdn = Pdn.from_network(net, device="cuda:0")
    rng = np.random.default_rng(3)
    bi = np.concatenate([[0, m - 1], rng.integers(0, m, 22)]).astype(np.int32)
    li = np.concatenate([[nl - 1, 0], rng.integers(0, nl, 22)]).astype(np.int32)
    out = torch.empty(bi.size, dtype=torch.float64, device="cuda:0")
    pdn.reff(out, torch.from_numpy(bi).cuda(), torch.from_numpy(li).cuda())
    st = pdn.stats()
    pdn.close()
    o = Oracle(net)
    want = np.array([o.reff(int(b), int(l)) for b, l in zip(bi, li)])
    check(out.cpu().numpy(), want)
    assert st["n_guess_tiers"] == 2


def test_permuting_the_bump_and_load_lists_permutes_the_output():
    """S4 pin: R depends on the pair, not on where it sits in the create-time lists."""
    net = P.make_random(11, d=3, n=40, p=7, m=6, nl=9, drop=0.02)
    ref, _ = gpu_all_pairs(net, rtol=1e-11)
    rng = np.random.default_rng(5)
    pb, pl = rng.permutation(net.m), rng.permutation(net.nl)
    net.bumps, net.loads = np.ascontiguousarray(net.bumps[pb]), np.ascontiguousarray(net.loads[pl])
    got, _ = gpu_all_pairs(net, rtol=1e-11)
    assert np.allclose(got, ref[np.ix_(pb, pl)], rtol=1e-9, atol=0)


def test_pair_kernel_equals_per_pair_solves_of_c_from_the_port_matrices():
    """S4 pin (Eq. (18)-(22) PAPER.md:179-204): the bilinear split R(i,j) = u_i + w_j - 2 b_i^T x_j
    of the pair kernel against ONE naive solve per pair of the coupled system C x = b, C = [K B; B^T 0] built here
    in numpy from the tier port matrices the library returns (pdn_get_port_matrix), R = Z_0[s,s] + Z_{d-1}[l,l] - b^T x
    (reading G9).  Checks S2 (assembly), S3 (factor + substitution) and S4 without the oracle."""
    torch_cuda()
    from paper_2607_05818_b200 import Pdn
    d, n, p, m, nl = 4, 14, 5, 3, 4
    net = P.make_random(19, d=d, n=n, p=p, m=m, nl=nl, drop=0.03, aniso=1.7)
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-12)
    Z = [pdn.port_matrix(t) for t in range(d)]
    import torch
    out = torch.empty(m * nl, dtype=torch.float64, device="cuda:0")
    got = pdn.reff(out).cpu().numpy().reshape(m, nl)
    pdn.close()
    pc = [len(s) for s in net.tsv_site]
    off = np.concatenate([[0], np.cumsum(pc)])
    Pt = int(off[-1])
    K = np.zeros((Pt, Pt))
    B = np.zeros((Pt, d - 1))
    for i in range(d - 1):
        lo_prev = pc[i - 1] if i > 0 else 0               # ports of tier i: [lo_{i-1}] ++ [up_i] ++ terminals
        up = slice(lo_prev, lo_prev + pc[i])
        lo = slice(0, pc[i])                                # ports of tier i+1 start with lo_i
        blk = slice(off[i], off[i + 1])
        K[blk, blk] = Z[i][up, up] + Z[i + 1][lo, lo] + np.diag(net.tsv_r[i])
        if i + 1 < d - 1:
            nxt = slice(off[i + 1], off[i + 2])
            cpl = -Z[i + 1][lo, pc[i]:pc[i] + pc[i + 1]]    # -Z_{i+1}[lo_i, up_{i+1}]
            K[blk, nxt], K[nxt, blk] = cpl, cpl.T
        B[blk, i] = 1.0
    Cm = np.block([[K, B], [B.T, np.zeros((d - 1, d - 1))]])
    nt0, ntd = pc[0], (pc[-1] if d > 1 else 0)              # TSV ports of tier 0 / of tier d-1 (its lo ends)
    for i in range(m):
        for j in range(nl):
            b = np.zeros(Pt + d - 1)
            b[off[0]:off[1]] += Z[0][:nt0, nt0 + i]                       # Z_0[up_0, bump i]
            b[off[d - 2]:off[d - 1]] += Z[d - 1][:ntd, ntd + j]           # Z_{d-1}[lo_{d-2}, load j]
            b[Pt:] = 1.0
            x = np.linalg.solve(Cm, b)
            want = Z[0][nt0 + i, nt0 + i] + Z[d - 1][ntd + j, ntd + j] - b @ x
            assert got[i, j] == pytest.approx(want, rel=1e-9)


def test_failed_replanning_leaves_the_context_as_it_was():
    """pdn_update_tsvs is staged: tier 0's new port matrix is a pure remap (its interface only loses a site) and
    succeeds, then the added sites of tier 1 fail (iteration cap of 1, set through pdn_set_solver_opts).  The context
    must still answer for the OLD plan, bit for bit (reff, every port matrix), pdn_reff_nodes must still work, and the
    same update must go through once the cap is restored."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import Pdn, PdnError
    torch = torch_cuda()
    d, n = 4, 41
    net = P.make_random(23, d=d, n=n, p=6, m=4, nl=5, drop=0.02)
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10)
    out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
    before = pdn.reff(out).cpu().numpy().copy()
    z_before = [pdn.port_matrix(t) for t in range(d)]
    rng = np.random.default_rng(3)
    new_sites = [s.copy() for s in net.tsv_site]
    new_r = [r.copy() for r in net.tsv_r]
    new_sites[0], new_r[0] = new_sites[0][1:].copy(), new_r[0][1:].copy()   # interface 0 only LOSES a site: tier 0 needs no solve
    for i in range(1, d - 1):                               # the others get a new site: tiers 1 .. d-1 need solves
        cand = [x for x in P._distinct_sites(rng, n, 8).tolist() if x not in new_sites[i].tolist()][0]
        new_sites[i] = np.vstack([new_sites[i][1:], [cand]]).astype(np.int32)
        new_r[i] = np.concatenate([new_r[i][1:], [0.09]])
    pdn.set_solver_opts(max_iter=1)
    with pytest.raises(PdnError) as e:
        pdn.update_tsvs(new_sites, new_r)
    assert e.value.status == 3                              # PDN_E_NOCONV
    assert np.array_equal(pdn.reff(out).cpu().numpy(), before)
    for t in range(d):
        zt = pdn.port_matrix(t)
        assert zt.shape == z_before[t].shape and np.array_equal(np.nan_to_num(zt), np.nan_to_num(z_before[t]))
    pdn.set_solver_opts(max_iter=200)
    nodes = np.array([[0, 1, 2], [d - 1, 30, 7]], dtype=np.int32)
    rn = pdn.reff_nodes(nodes, torch.empty(4, dtype=torch.float64, device="cuda:0")).cpu().numpy()
    o_old = Oracle(net)
    assert abs(rn[1] / o_old.reff_nodes(1 * n + 2, (d - 1) * n * n + 30 * n + 7) - 1.0) <= MAX_REL
    pdn.update_tsvs(new_sites, new_r)                       # the same list now goes through
    net.tsv_site, net.tsv_r = new_sites, new_r
    check(pdn.reff(out).cpu().numpy().reshape(net.m, net.nl), Oracle(net).reff_all())
    pdn.close()


_SHARD_WORKER = r"""
import os, sys
import numpy as np
import torch, torch.distributed as dist
sys.path.insert(0, os.getcwd())
import pdn_inputs as P
from oracle.reff_oracle import Oracle
from paper_2607_05818_b200 import Pdn, PDN_TERMINAL_PAIRS
dist.init_process_group("gloo")                       # NCCL refuses two ranks on one device; gloo moves CUDA tensors
rank, world = dist.get_rank(), dist.get_world_size()
torch.cuda.set_device(0)
net = P.make_random(71, d=3, n=47, p=7, m=5, nl=6, drop=0.03)       # the same network on every rank
net.gx[1], net.gy[1] = P._planes(net.n, np.full((net.n, net.n), 0.8), np.full((net.n, net.n), 1.3))  # a uniform tier
flags = PDN_TERMINAL_PAIRS if os.environ.get("SHARD_TERMINAL_PAIRS") == "1" else 0
pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10, flags=flags, shard_rank=rank, shard_world=world)
pdn.exchange_and_finish(dist, world)                  # the product path, unchanged: broadcasts of library memory
out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
got = pdn.reff(out).cpu().numpy().reshape(net.m, net.nl)
want = Oracle(net).reff_all()
rel = np.abs(got - want) / want
assert rel.max() <= 1e-6 and rel.mean() <= 1e-8, (rel.max(), rel.mean())
ref = Pdn.from_network(net, device="cuda:0", rtol=1e-10, flags=flags)   # unsharded, same process
full = ref.reff(torch.empty_like(out)).cpu().numpy().reshape(net.m, net.nl)
assert np.allclose(got, full, rtol=1e-9, atol=0)
every = [torch.zeros_like(out) for _ in range(world)]                   # every rank holds the same result
dist.all_gather(every, out)
assert all(torch.equal(e, every[0]) for e in every)
pdn.close(); ref.close()
dist.destroy_process_group()
print("shard-ok", rank, f"{rel.max():.2e}")
"""


@pytest.mark.parametrize("terminal_pairs", [False, True])
def test_sharded_exchange_runs_for_real_between_two_processes_on_one_gpu(tmp_path, terminal_pairs):
    """NEXT-4: `Pdn.exchange_and_finish` -- pdn_shard_slice / pdn_shard_buffers views of library
    memory under torch.distributed.broadcast -- executed unchanged by two ranks (torchrun, one process per rank, both on
    cuda:0, backend gloo since NCCL will not place two ranks on one device); every rank must equal the oracle and the
    unsharded context, and all ranks must hold bit-identical results."""
    import subprocess
    import sys
    torch_cuda()
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    w = tmp_path / "shard_worker.py"
    w.write_text(_SHARD_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", SHARD_TERMINAL_PAIRS="1" if terminal_pairs else "0")
    r = subprocess.run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2",
                        "--master-addr", "127.0.0.1", "--master-port", "29547" if terminal_pairs else "29546", str(w)],
                       cwd=root, env=env, capture_output=True, text=True, timeout=600)
    assert r.returncode == 0, (r.stdout[-2000:], r.stderr[-4000:])
    assert r.stdout.count("shard-ok") == 2
