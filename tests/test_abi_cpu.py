"""CPU-side checks of the boundary: libpdn.so builds (nvcc cross-compiles sm_100a without a GPU),
loads, and exports every symbol include/pdn.h declares.  No compute call is made here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    src = open(os.path.join(ROOT, "include", "pdn.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(pdn_[a-z_]+)\s*\(", src)))


def test_header_declares_the_north_star_calls():
    names = declared_functions()
    for must in ("pdn_create", "pdn_reff", "pdn_destroy"):
        assert must in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    import __graft_entry__ as g
    g.build()
    import paper_2607_05818_b200 as pkg
    lib = pkg.load_library()
    for name in declared_functions():
        assert hasattr(lib, name), f"{name} declared in pdn.h but not exported"
    assert set(pkg.EXPORTS) == set(declared_functions())


def test_struct_sizes_match_the_header_layout():
    from paper_2607_05818_b200 import binding as b
    assert ctypes.sizeof(b.PdnTier) == 24 and ctypes.sizeof(b.PdnTsv) == 24 and ctypes.sizeof(b.PdnSite) == 8
    assert ctypes.sizeof(b.PdnOpts) == 48
    assert ctypes.sizeof(b.PdnStats) == 16 + 16 + 8 + 8 + 8 + 4 * 8 + 8 + 24 + 3 * 64 + 8


def test_compute_calls_fail_loudly_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("this check is for the CPU-only container")
    import pdn_inputs as P
    from paper_2607_05818_b200 import Pdn, PdnError
    with pytest.raises(PdnError) as e:
        Pdn.from_network(P.make_config(1))
    assert e.value.status in (4, 5)      # PDN_E_CUDA / PDN_E_NOMEM: never a silent CPU result


def test_pure_status_helpers():
    import paper_2607_05818_b200 as pkg
    lib = pkg.load_library()
    assert lib.pdn_strerror(0) == b"ok" and b"connected" in lib.pdn_strerror(2)
    lib.pdn_destroy(None)                # NULL-safe


def test_argument_validation_runs_on_the_host_before_any_device_work():
    """pdn_create rejects malformed inputs with PDN_E_ARG on the host (no device needed): TSVs on a single tier, a TSV
    outside the mesh or on an interface that does not exist, a non-positive resistance, a duplicate site inside
    one interface, an interface without TSVs, a terminal outside the mesh."""
    import numpy as np
    import pdn_inputs as P
    from paper_2607_05818_b200 import Pdn, PdnError

    def status_of(mutate):
        net = P.make_config(1)
        mutate(net)
        with pytest.raises(PdnError) as e:
            Pdn(net.n, net.gx, net.gy, net.tsv_site, net.tsv_r, net.bumps, net.loads)
        return e.value.status

    def one_tier_with_tsvs(net):                 # a single tier is a 2-D PDN: it has no interface for a TSV
        net.gx, net.gy = net.gx[:1], net.gy[:1]
    assert status_of(one_tier_with_tsvs) == 1
    assert status_of(lambda n: n.tsv_site[0].__setitem__(0, [32, 0])) == 1
    assert status_of(lambda n: n.tsv_r[0].__setitem__(3, 0.0)) == 1
    assert status_of(lambda n: n.tsv_r[0].__setitem__(3, float("inf"))) == 1
    assert status_of(lambda n: n.tsv_site[0].__setitem__(1, n.tsv_site[0][0])) == 1
    assert status_of(lambda n: (n.tsv_site.__setitem__(0, n.tsv_site[0][:0]), n.tsv_r.__setitem__(0, n.tsv_r[0][:0]))) == 1
    assert status_of(lambda n: setattr(n, "loads", np.array([[0, -1]], dtype=np.int32))) == 1
