#!/usr/bin/env python
"""Small driver for compute-sanitizer ("race detection / sanitizers"): one pass of the hot
path on configs[0] (what smoke() runs) and on one ragged three-level stack whose sizes make every hand-written
kernel class appear -- k_pq3, k_down3<fused / plain>, k_up3<dot / plain>, k_tail, the DMMA GEMM (p >= 96), the
blocked Cholesky, k_pair_full, k_pair_list -- plus one TSV re-plan and one pdn_reff_nodes call.  Run as

    compute-sanitizer --tool memcheck|racecheck|synccheck|initcheck python tests/sanitizer_case.py

(one tool per gpurun call); results are checked against the oracle so that a run that "passes" the tool by
computing nothing fails here.  profiles/r2_sanitizer.md records the runs."""
import os
import sys

import numpy as np
import torch

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

import pdn_inputs as P  # noqa: E402
from oracle.reff_oracle import Oracle  # noqa: E402
from paper_2607_05818_b200 import Pdn  # noqa: E402


def run(net, name, replan):
    pdn = Pdn.from_network(net, device="cuda:0")
    out = torch.empty(net.m * net.nl, dtype=torch.float64, device="cuda:0")
    got = pdn.reff(out).cpu().numpy().reshape(net.m, net.nl)
    o = Oracle(net)
    rel = np.abs(got - o.reff_all()) / o.reff_all()
    assert rel.max() <= 1e-6 and rel.mean() <= 1e-8, (name, rel.max(), rel.mean())
    bi = torch.tensor([0, net.m - 1], dtype=torch.int32, device="cuda:0")
    li = torch.tensor([net.nl - 1, 0], dtype=torch.int32, device="cuda:0")
    two = pdn.reff(torch.empty(2, dtype=torch.float64, device="cuda:0"), bi, li).cpu().numpy()
    assert np.allclose(two, [got[0, -1], got[-1, 0]], rtol=1e-12, atol=0)
    st = pdn.stats()
    if replan:
        nodes = np.array([[0, 3, 5], [net.d - 1, net.n - 1, 0], [1, 10, 10]], dtype=np.int32)
        rn = pdn.reff_nodes(nodes, torch.empty(9, dtype=torch.float64, device="cuda:0")).cpu().numpy().reshape(3, 3)
        gid = nodes[:, 0].astype(np.int64) * net.n ** 2 + nodes[:, 1] * net.n + nodes[:, 2]
        assert abs(rn[0, 1] / o.reff_nodes(int(gid[0]), int(gid[1])) - 1.0) <= 1e-6
        rng = np.random.default_rng(1)
        cand = [x for x in P._distinct_sites(rng, net.n, 8).tolist() if x not in net.tsv_site[0].tolist()][0]
        net.tsv_site[0] = np.vstack([net.tsv_site[0][1:], [cand]]).astype(np.int32)
        pdn.update_tsvs(net.tsv_site, net.tsv_r)
        got = pdn.reff(out).cpu().numpy().reshape(net.m, net.nl)
        want = Oracle(net).reff_all()
        assert (np.abs(got - want) / want).max() <= 1e-6
    pdn.close()
    print(f"{name}: max rel err {rel.max():.2e}, {st['kernel_launches']} launches, {st['pcg_iters_max']} PCG iterations")


if __name__ == "__main__":
    run(P.make_config(1, seed=0), "configs[0]", replan=False)
    run(P.make_random(5, d=3, n=70, p=100, m=40, nl=60, drop=0.02, aniso=2.0), "ragged 3 x 70^2, 100 TSV/interface", replan=True)
    print("sanitizer case done")
