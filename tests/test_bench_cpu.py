"""CPU-side checks of bench.py: the reference (oracle) arm, alone and under a 2-rank torchrun launch, and the
max-over-ranks timing reduction the CUDA arm uses, over gloo (world_size 2)."""
import json
import os
import subprocess
import sys

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def run(cmd, **kw):
    return subprocess.run(cmd, cwd=ROOT, capture_output=True, text=True, timeout=300, **kw)


def test_reference_arm_prints_one_contract_line():
    r = run([sys.executable, "bench.py", "--impl", "reference", "--config", "1", "--steps", "2", "--warmup", "1",
             "--cpu-budget", "1"])
    assert r.returncode == 0, r.stderr
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1
    d = json.loads(lines[0])
    assert d["impl"] == "reference" and d["unit"] == "pairs/s" and d["value"] > 0 and d["higher_is_better"] is True
    assert d["cpu_baseline"]["kind"] == "oracle" and d["cpu_baseline"]["cores"] == 1
    assert d["e2e"] == {"value": d["value"], "unit": "pairs/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}
    assert d["vs_baseline"] is None and d["dtype"] == "f64" and "workload" in d["config"]


def test_reference_arm_under_torchrun_only_rank0_works():
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
             "127.0.0.1", "--master-port", "29541", "bench.py", "--gpus", "2", "--impl", "reference", "--config", "1",
             "--steps", "1", "--warmup", "0", "--cpu-budget", "1"], env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
    assert len(lines) == 1 and json.loads(lines[0])["n_gpus"] == 2


_WORKER = r"""
import os, sys, torch, torch.distributed as dist
sys.path.insert(0, os.getcwd())
import bench
dist.init_process_group("gloo")
rank = dist.get_rank()
ms = bench.max_over_ranks(10.0 + 5.0 * rank, None, dist)          # the reduction run_cuda uses (device=None: CPU)
assert ms == 15.0, ms
import pdn_inputs as P
a, b = P.make_config(1, seed=rank), P.make_config(1, seed=rank)     # one independent, reproducible network per rank
assert (a.gx[0] == b.gx[0]).all()
other = P.make_config(1, seed=1 - rank)
assert not (a.gx[0] == other.gx[0]).all()
dist.destroy_process_group()
print("ok", rank)
"""


def test_max_over_ranks_and_per_rank_networks_gloo_world2(tmp_path):
    w = tmp_path / "worker.py"
    w.write_text(_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
             "127.0.0.1", "--master-port", "29542", str(w)], env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    assert r.stdout.count("ok") == 2


_SHARD_WORKER = r"""
import os, sys, torch, torch.distributed as dist
sys.path.insert(0, os.getcwd())
from paper_2607_05818_b200 import shard_bounds
dist.init_process_group("gloo")
rank, world = dist.get_rank(), dist.get_world_size()
# the exchange Pdn.exchange_and_finish does, on CPU tensors: rank r owns rows shard_bounds(k, world)[r] of a k x q
# matrix; after one broadcast per rank every rank holds the whole matrix
k, q = 11, 5
full = torch.arange(k * q, dtype=torch.float64).reshape(k, q)
mine = torch.full((k, q), float("nan"), dtype=torch.float64)
lo, hi = shard_bounds(k, world)[rank]
mine[lo:hi] = full[lo:hi]
for r, (a, b) in enumerate(shard_bounds(k, world)):
    piece = mine[a:b].reshape(-1)          # contiguous view, as the row slices of the port matrix are
    dist.broadcast(piece, src=r)
assert torch.equal(mine, full)
assert shard_bounds(10, 4) == [(0, 2), (2, 5), (5, 7), (7, 10)] and shard_bounds(3, 2) == [(0, 1), (1, 3)]
dist.destroy_process_group()
print("ok", rank)
"""


def test_shard_bounds_and_row_exchange_gloo_world2(tmp_path):
    w = tmp_path / "shard_worker.py"
    w.write_text(_SHARD_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1")
    r = run([sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr",
             "127.0.0.1", "--master-port", "29543", str(w)], env=env)
    assert r.returncode == 0, r.stderr[-2000:]
    assert r.stdout.count("ok") == 2
