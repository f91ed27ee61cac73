"""pdn_load_voltages_static (include/pdn.h): Eq. (4), with the scratch in the library's static
__device__ array instead of the device pool -- for callers that cannot call cudaMalloc.

Collected last on purpose (the file name sorts after every other test file): the suite runs with `pytest -x`, and a
failure here must not hide the parity tests.  The test does not depend on anything the other tests leave behind: it
passes alone in a fresh process and after the whole suite.
"""
import numpy as np
import pytest

import pdn_inputs as P

pytestmark = pytest.mark.gpu


def torch_cuda():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("CUDA device required for -m gpu tests (no CPU fallback exists)")
    return torch


def test_static_scratch_entry_point_matches_the_pooled_path_on_two_calls_in_a_row():
    """Two calls in a row with different bumps and currents (the second finds the first one's R_b / R_LL in the
    shared array and must not be affected by them), each against pdn_load_voltages on the same context within the
    tolerance of the Eq. (4) parity test (tests/test_gpu_parity.py: 1e-8 of the largest drop), and against the
    oracle's KCL solve.  Once warm, the free device memory does not move across further calls."""
    from oracle.reff_oracle import Oracle
    from paper_2607_05818_b200 import PDN_TERMINAL_PAIRS, Pdn
    torch = torch_cuda()
    net = P.make_random(71, d=3, n=48, p=6, m=5, nl=70, drop=0.03, aniso=0.3)   # 70 loads: 2 x 2 tiles of k_pair_same, ragged
    o = Oracle(net)
    pdn = Pdn.from_network(net, device="cuda:0", rtol=1e-10, flags=PDN_TERMINAL_PAIRS)
    rng = np.random.default_rng(71)
    cases = [(0, rng.uniform(0.0, 1.5, net.nl), 0.8), (3, rng.uniform(0.0, 0.4, net.nl), 1.1)]
    v_pool = torch.empty(net.nl, dtype=torch.float64, device="cuda:0")
    v_stat = torch.empty(net.nl, dtype=torch.float64, device="cuda:0")
    want_pool = []
    for b, cur, vb in cases:                       # the existing path first (it may allocate)
        pdn.load_voltages(b, torch.tensor(cur, dtype=torch.float64, device="cuda:0"), vb, v_pool)
        want_pool.append(v_pool.cpu().numpy().copy())
    cur_dev = [torch.tensor(cur, dtype=torch.float64, device="cuda:0") for _, cur, _ in cases]
    launches0 = pdn.stats()["kernel_launches"]
    got = []
    for (b, _, vb), cd in zip(cases, cur_dev):     # two calls in a row, nothing of the library in between
        v_stat.fill_(float("nan"))
        pdn.load_voltages_static(b, cd, vb, v_stat)
        got.append(v_stat.cpu().numpy().copy())
    assert pdn.stats()["kernel_launches"] == launches0 + 6
    # No allocation: with every kernel of the process loaded by now (the CUDA runtime loads a kernel's code on its
    # first launch, which takes device memory once) the free memory does not move across two more calls, and the
    # repeat reproduces the bits.
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for (b, _, vb), cd, g in zip(cases, cur_dev, got):
        pdn.load_voltages_static(b, cd, vb, v_stat)
        assert torch.cuda.mem_get_info()[0] == free0
        assert np.array_equal(v_stat.cpu().numpy(), g)
    for (b, cur, vb), g, w in zip(cases, got, want_pool):
        assert np.all(np.isfinite(g))
        drop = np.abs(vb - w).max()
        assert np.allclose(g, w, rtol=0, atol=1e-8 * drop), np.abs(g - w).max() / drop
        oracle = o.load_voltages(b, cur, vb)
        assert np.allclose(g, oracle, rtol=0, atol=1e-8 * np.abs(vb - oracle).max())
    assert not np.allclose(got[0], got[1])         # the two calls really had different answers
    pdn.close()


def test_static_scratch_entry_point_rejects_more_loads_than_the_array_holds():
    from paper_2607_05818_b200 import PDN_STATIC_MAX_LOADS, PDN_TERMINAL_PAIRS, Pdn, PdnError
    torch = torch_cuda()
    nl = PDN_STATIC_MAX_LOADS + 1
    net = P.make_random(72, d=2, n=40, p=4, m=2, nl=nl)
    pdn = Pdn.from_network(net, device="cuda:0", flags=PDN_TERMINAL_PAIRS)
    cur = torch.ones(nl, dtype=torch.float64, device="cuda:0")
    v = torch.full((nl,), -7.0, dtype=torch.float64, device="cuda:0")
    with pytest.raises(PdnError) as e:
        pdn.load_voltages_static(0, cur, 0.8, v)
    assert e.value.status == 1 and "PDN_STATIC_MAX_LOADS" in str(e.value)
    assert bool((v == -7.0).all())                 # nothing was launched
    pdn.load_voltages(0, cur, 0.8, v)              # the pooled path takes the same context
    assert bool(torch.isfinite(v).all())
    pdn.close()
