#!/usr/bin/env python
"""Benchmark of the bump x load effective-resistance path (BASELINE.json metric: pairs/sec, FP64).

One "step" = one pass of the whole hot path over one synthetic workload: pdn_create (S0 tier import,
S1 batched port reduction, S2 assembly, S3 factor + substitution) + pdn_reff for the full bump x load
cross product (S4) + pdn_destroy.  `value` times it with the conductance planes already resident in
HBM and the result left on the device; `e2e` times the same through the host-buffer entry points
(planes in pinned host memory, result copied back to the host) -- copies inside the timed region.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1..5] [--impl reference]

Default workload: configs[4] (8 tiers x 1024^2, 4,194,304 pairs) -- BASELINE.json's `metric` names no config,
so the headline is the largest single-GPU one.  Its oracle sample costs one sparse LU of the whole 3D system
(~4-5 min on one core, ~19 GB) plus a few pairs; `--config 4` (configs[3], LU ~1 min) and the others are
measured the same way and recorded under profiles/.

N > 1 (torchrun): every rank runs its own independent network of the same workload (seed = rank): the
path has no cross-problem exchange, so this is weak scaling without a collective (multi-GPU).
"""
import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import pdn_inputs as P  # noqa: E402

METRIC = "bump-load R_eff pairs/sec (FP64)"
UNIT = "pairs/s"


def workload_name(cfg):
    c = P.CONFIGS[cfg]
    return (f"configs[{cfg - 1}]: {c['d']} tiers x {c['n']}^2 mesh, {c['p']} TSV/interface, "
            f"{c['m']}x{c['nl']} pairs")


# ----------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "500", "-i", str(gpu_index)], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        if self.p is None:
            return out
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush()
        rows = [l.split(", ") for l in open(self.f.name).read().strip().splitlines() if l.count(",") >= 8]
        os.unlink(self.f.name)
        if not rows:
            return out
        sm = [float(r[1]) for r in rows if r[1].replace(".", "").isdigit()]
        out["sm_mhz"] = float(np.median(sm)) if sm else None
        out["sm_max_mhz"] = float(rows[0][2]) if rows[0][2].replace(".", "").isdigit() else None
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        out["reasons"] = [n for k, n in enumerate(names) if any(r[5 + k].strip() == "Active" for r in rows)]
        out["samples"] = len(rows)
        return out


# ----------------------------------------------------------------------------------------- oracle arm
class OracleTimer:
    """The oracle as it stands, timed on the host: the whole 3D system is factored ONCE (SuperLU is serial:
    1 core), then seeded pairs of the workload's 4096-pair sample are solved one at a time."""

    def __init__(self, cfg):
        from oracle.reff_oracle import Oracle
        self.cfg = cfg
        net = P.make_config(cfg, seed=0)
        t0 = time.perf_counter()
        self.o = Oracle(net)
        self.t_factor = time.perf_counter() - t0
        self.bi, self.li = P.sample_pairs(net, 4096, seed=0, cfg=cfg)
        self.pos = 0

    def sample(self, budget_s, max_pairs=4096):
        """Solves pairs for about `budget_s` seconds; returns (pairs, seconds)."""
        done = 0
        t1 = time.perf_counter()
        while done < max_pairs:
            k = self.pos % self.bi.size
            self.o.reff(int(self.bi[k]), int(self.li[k]))
            self.pos += 1
            done += 1
            if time.perf_counter() - t1 > budget_s:
                break
        return done, time.perf_counter() - t1

    def describe(self, pairs, secs):
        return (f"sparse LU of the whole 3D system once ({self.t_factor:.1f} s, not counted in value) + {pairs} seeded "
                f"pairs of the workload solved one at a time in {secs:.1f} s")


def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cfg = a.config
    ot = OracleTimer(cfg)
    per = max(2.0, a.cpu_budget / max(a.steps, 1))
    for _ in range(a.warmup):
        ot.sample(min(per, 2.0), max_pairs=2)
    pairs = secs = 0
    for _ in range(a.steps):
        n, t = ot.sample(per)
        pairs += n
        secs += t
    value = pairs / secs
    desc = ot.describe(pairs, secs)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": a.gpus, "steps": a.steps,
            "warmup": a.warmup, "ms_per_step": 1e3 * secs / max(a.steps, 1), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "cfg": cfg, "factor_s": round(ot.t_factor, 2),
                       "pairs_per_step": pairs / max(a.steps, 1)},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


# ----------------------------------------------------------------------------------------- CUDA arm
def max_over_ranks(ms, device, dist):
    """Step time of the job = the slowest rank's device time (all-reduce MAX; gloo on CPU in the tests)."""
    import torch
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def run_cuda(a):
    import torch
    import torch.distributed as dist
    from paper_2607_05818_b200 import PDN_TIME_KERNELS, Pdn

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    cfg = a.config
    sharded = a.shard and world > 1
    net = P.make_config(cfg, seed=0 if sharded else rank)   # one independent network per rank, or one for all
    if a.uniform:   # NEXT-1 variant: every tier gets its median segment conductances (same sites): Eq. (3) fast path
        for t in range(net.d):
            n_ = net.n
            net.gx[t][:, : n_ - 1] = np.median(net.gx[t][:, : n_ - 1][net.gx[t][:, : n_ - 1] > 0])
            net.gy[t][: n_ - 1, :] = np.median(net.gy[t][: n_ - 1, :][net.gy[t][: n_ - 1, :] > 0])
    npairs = net.m * net.nl
    gx_d = [torch.from_numpy(g).to(dev) for g in net.gx]
    gy_d = [torch.from_numpy(g).to(dev) for g in net.gy]
    gx_h = [torch.from_numpy(g).pin_memory() for g in net.gx]
    gy_h = [torch.from_numpy(g).pin_memory() for g in net.gy]
    out_d = torch.empty(npairs, dtype=torch.float64, device=dev)
    out_h = torch.empty(npairs, dtype=torch.float64).pin_memory()
    args = (net.n,), (net.tsv_site, net.tsv_r, net.bumps, net.loads)

    # PDN_NO_UNIFORM_FAST_PATH, PDN_PRECOND_F32, PDN_NO_INITIAL_GUESS
    base_flags = (8 if a.no_fast_path else 0) | (32 if a.precond_f32 else 0) | (64 if a.no_guess else 0)

    shard_kw = dict(shard_rank=rank, shard_world=world) if sharded else {}

    def step_device(flags=0):
        pdn = Pdn(net.n, gx_d, gy_d, *args[1], flags=flags | base_flags, rtol=a.rtol, nu=a.nu, rhs_batch=a.rhs_batch,
                  **shard_kw)
        if sharded:
            pdn.exchange_and_finish(dist, world)
        pdn.reff(out_d)
        st = pdn.stats()
        pdn.close()
        return st

    def step_host():
        pdn = Pdn(net.n, gx_h, gy_h, *args[1], flags=base_flags, rtol=a.rtol, nu=a.nu, rhs_batch=a.rhs_batch, **shard_kw)
        if sharded:
            pdn.exchange_and_finish(dist, world)
        pdn.reff_host(out_h)
        pdn.close()

    def timed(fn, steps):
        barrier()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        res = [fn() for _ in range(steps)]
        e1.record()
        barrier()
        return max_over_ranks(e0.elapsed_time(e1), dev, dist if world > 1 else None), res

    sampler = ClockSampler(local) if rank == 0 else None   # started before the warm-up: its spawn is not timed
    for _ in range(a.warmup):
        step_device()
    ms, stats = timed(lambda: step_device(), a.steps)
    clocks = sampler.stop() if sampler else None
    jobs = 1 if sharded else world               # networks solved per step by the whole job
    value = jobs * npairs * a.steps / (ms * 1e-3)

    if a.only_device:   # used under ncu: no extra legs, no JSON contract
        if rank == 0:
            print(json.dumps({"only_device": True, "value": value, "ms_per_step": ms / a.steps}))
        return
    # per-kernel-class device time (CUDA events on the launching stream around every launch)
    ms_prof, pstats = timed(lambda: step_device(PDN_TIME_KERNELS), a.steps)
    # end to end through the host-buffer entry points
    step_host()
    ms_e2e, _ = timed(step_host, a.steps)
    e2e_value = jobs * npairs * a.steps / (ms_e2e * 1e-3)
    h2d = sum(g.numel() * 8 for g in gx_h) * 2
    d2h = npairs * 8

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    peaks = {}
    pk_path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(pk_path):
        peaks = json.load(open(pk_path))
    peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json, sustained copy)" if "hbm_gbs" in peaks else "fallback 6650 GB/s"
    st = pstats[-1]
    cls_ms = {k: sum(s["class_ms"][k] for s in pstats) for k in st["class_ms"]}
    cls_by = {k: sum(s["class_bytes"][k] for s in pstats) for k in st["class_bytes"]}
    cls_n = {k: sum(s["class_launches"][k] for s in pstats) for k in st["class_launches"]}
    stencil_classes = ["pq", "down0", "up0", "down_coarse", "up_coarse"]
    dom = max(stencil_classes, key=lambda k: cls_ms[k])
    ach = cls_by[dom] / (cls_ms[dom] * 1e-3) / 1e9 if cls_ms[dom] > 0 else 0.0
    tot_ms = sum(cls_ms[k] for k in stencil_classes)
    tot_by = sum(cls_by[k] for k in stencil_classes)
    phase = tot_by / (tot_ms * 1e-3) / 1e9 if tot_ms > 0 else 0.0
    # DRAM traffic of the dominant kernel from the committed ncu capture (profiles/ncu_traffic.csv: bytes per
    # right-hand side of one launch on a mesh of the same size), scaled to this run's average right-hand sides per
    # launch -- NOT measured in this run (a run under ncu is never a bench value): `traffic_source` says so
    traffic = None
    tr_path = os.path.join(ROOT, "profiles", "ncu_traffic.csv")
    if os.path.exists(tr_path) and cls_n[dom] > 0:
        import csv
        for row in csv.DictReader(open(tr_path)):
            if int(row["n"]) == net.n and row["class"] == dom:
                per_rhs_alg = float(row["algorithmic_bytes_per_launch"]) / float(row["rhs_in_launch"])
                rhs_per_launch = (cls_by[dom] / cls_n[dom]) / per_rhs_alg
                traffic = float(row["dram_bytes_per_rhs"]) * rhs_per_launch

    last = stats[-1]
    # parity of what the timed steps produced, against the oracle's stored values (tests/golden, written by
    # tests/golden/make_golden.py from oracle/ only): max / mean relative error over the golden pairs
    parity = None
    gpath = os.path.join(ROOT, "tests", "golden", f"cfg{cfg}_reff.txt")
    if os.path.exists(gpath) and not a.uniform:
        g = np.loadtxt(gpath, comments="#")
        got = out_d.cpu().numpy().reshape(net.m, net.nl)[g[:, 0].astype(int), g[:, 1].astype(int)]
        rel = np.abs(got - g[:, 2]) / g[:, 2]
        parity = {"max_rel": float(rel.max()), "mean_rel": float(rel.mean()), "pairs_checked": int(rel.size),
                  "tolerance": {"max_rel": 1e-6, "mean_rel": 1e-8}, "expected": f"tests/golden/cfg{cfg}_reff.txt (oracle)"}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": a.steps, "warmup": a.warmup,
        "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "strong" if sharded else "weak",
        "vs_baseline": None,
        "dtype": "f64 (multigrid sweeps in f32 registers: --precond-f32)" if a.precond_f32 else "f64", "data": "synthetic",
        "config": {"workload": workload_name(cfg) + (" -- UNIFORM variant (median conductances)" if a.uniform else ""),
                   "cfg": cfg, "pairs_per_step_per_gpu": npairs, "uniform_tiers": last["n_uniform_tiers"],
                   "l2": "working set of every stencil launch exceeds the 126 MB L2 (no flush needed)"
                         if cfg >= 3 else "working set fits L2: latency-bound case, HBM fraction not meaningful",
                   "rtol": a.rtol or 1e-8, "nu": a.nu or 4, "preconditioner_sweeps": "f32" if a.precond_f32 else "f64",
                   "pcg_iters_max": last["pcg_iters_max"], "rhs_iterations": last["rhs_iterations"],
                   "initial_guess_tiers": last["n_guess_tiers"],
                   "ms_stencil": last["ms_stencil"], "ms_dense": last["ms_dense"], "ms_upload": last["ms_upload"]},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "ms_per_step": ms_e2e / a.steps},
        "gpu_launches": int(sum(s["kernel_launches"] for s in stats)),
        "parity": parity,
        "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": dom, "achieved": ach, "peak": peak, "unit": "GB/s",
                     "frac": ach / peak, "traffic": traffic,
                     "traffic_source": "ncu capture (profiles/ncu_traffic.csv), scaled by right-hand sides per launch; "
                                       "not measured in this run" if traffic is not None else None,
                     "peak_source": peak_src,
                     "launches": int(cls_n[dom]), "avg_launch_ms": cls_ms[dom] / max(cls_n[dom], 1),
                     "alg_bytes_per_launch": cls_by[dom] / max(cls_n[dom], 1),
                     "timing": "CUDA events around every launch on the launching stream, in a repeat of the same "
                               f"{a.steps} steps right after the timed region (so that `value` carries no event overhead)",
                     "ms_per_step_in_that_pass": ms_prof / a.steps,
                     "stencil_phase": {"achieved": phase, "frac": phase / peak, "ms": tot_ms,
                                       "share_of_step": tot_ms / ms_prof if ms_prof else None},
                     "classes": {k: {"ms": cls_ms[k], "GBps": (cls_by[k] / (cls_ms[k] * 1e-3) / 1e9) if cls_ms[k] > 0 else 0.0,
                                     "launches": int(cls_n[k])} for k in cls_ms}},
    }
    if a.replan > 0:   # NEXT-2: move K TSVs per interface, time the update against a full re-creation
        rng = np.random.default_rng([cfg, a.replan])
        sites = [s_.copy() for s_ in net.tsv_site]
        for i in range(net.d - 1):
            taken = {tuple(x) for x in sites[i].tolist()}
            k = 0
            while k < min(a.replan, len(sites[i])):
                cand = (int(rng.integers(0, net.n)), int(rng.integers(0, net.n)))
                if cand not in taken:
                    taken.add(cand)
                    sites[i][k] = cand
                    k += 1
        pdn = Pdn(net.n, gx_d, gy_d, *args[1], flags=base_flags, rtol=a.rtol, nu=a.nu, rhs_batch=a.rhs_batch)
        cur = [net.tsv_site, sites]
        times = []
        for rep in range(a.warmup + a.steps):      # alternate between the two plans
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            pdn.update_tsvs(cur[(rep + 1) % 2], net.tsv_r)
            pdn.reff(out_d)
            torch.cuda.synchronize()
            if rep >= a.warmup:
                times.append(time.perf_counter() - t0)
        stu = pdn.stats()
        pdn.close()
        line["replan"] = {"tsvs_moved_per_interface": a.replan, "ms_per_update": 1e3 * float(np.mean(times)),
                          "port_solves_per_update": int(stu["update_solves"]), "ms_solves": stu["ms_update_stencil"],
                          "ms_refactor": stu["ms_update_dense"], "ms_full_step": ms / a.steps,
                          "pairs_per_s": npairs / float(np.mean(times))}
    if a.emulate_shards > 1:   # NEXT-4: per-rank compute of a sharded run, measured on this one GPU
        emu = {}
        w_ = 2
        while w_ <= a.emulate_shards:
            ts = []
            for rep in range(a.warmup + a.steps):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                pdn = Pdn(net.n, gx_d, gy_d, *args[1], flags=base_flags, rtol=a.rtol, nu=a.nu, rhs_batch=a.rhs_batch,
                          shard_rank=rep % w_, shard_world=w_)
                torch.cuda.synchronize()
                t1 = time.perf_counter()
                pieces = sum(v.numel() * 8 for _, v in pdn.shard_pieces(rep % w_))
                pdn.close()           # (pdn_finish needs every rank's rows: S2-S3 time is the unsharded run's ms_dense)
                if rep >= a.warmup:
                    ts.append((t1 - t0, pieces))
            emu[str(w_)] = {"ms_rank_solves": 1e3 * float(np.mean([t[0] for t in ts])),
                            "ms_s2_s3_replicated": last["ms_dense"],
                            "bytes_rank_broadcasts": int(np.mean([t[1] for t in ts]))}
            w_ *= 2
        line["shard_emulation"] = {"ms_full_step_1gpu": ms / a.steps, "per_world": emu}
    if a.eq4:   # NEXT-3: same-side pairs and Eq. (4) voltages
        nl = net.nl
        rll = torch.empty(nl * nl, dtype=torch.float64, device=dev)
        cur = torch.rand(nl, dtype=torch.float64, device=dev)
        vout = torch.empty(nl, dtype=torch.float64, device=dev)

        def ev_ms(fn, reps):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            e0.record()
            for _ in range(reps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / reps

        t_create = []
        pdn = None
        for rep in range(a.warmup + a.steps):
            if pdn is not None:
                pdn.close()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            pdn = Pdn(net.n, gx_d, gy_d, *args[1], flags=base_flags | 16, rtol=a.rtol, nu=a.nu, rhs_batch=a.rhs_batch)
            torch.cuda.synchronize()
            if rep >= a.warmup:
                t_create.append(time.perf_counter() - t0)
        ms_ll = ev_ms(lambda: pdn.reff_same_side(1, rll), 5)
        ms_v = ev_ms(lambda: pdn.load_voltages(0, cur, 1.0, vout), 5)
        pdn.close()
        line["eq4"] = {"ms_create_with_terminal_pairs": 1e3 * float(np.mean(t_create)), "ms_create_default": ms / a.steps,
                       "load_load_pairs": nl * nl, "ms_load_load": ms_ll, "load_load_pairs_per_s": nl * nl / (ms_ll * 1e-3),
                       "ms_voltages_one_bump": ms_v}
    if a.nodes > 0:   # NEXT-3: arbitrary-tier endpoints (pdn_reff_nodes) and an R_eff map (Fig. 6(d))
        rng = np.random.default_rng(12345)
        k = a.nodes
        nodes = np.stack([rng.integers(0, net.d, k), rng.integers(0, net.n, k), rng.integers(0, net.n, k)], axis=1).astype(np.int32)
        out_n = torch.empty(k * k, dtype=torch.float64, device=dev)
        pdn = Pdn(net.n, gx_d, gy_d, *args[1], flags=base_flags, rtol=a.rtol, nu=a.nu, rhs_batch=a.rhs_batch)
        tn, tm = [], []
        stride = a.map_stride if a.map_stride > 0 else max(1, net.n // 32)
        for rep in range(a.warmup + a.steps):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            pdn.reff_nodes(nodes, out_n)
            torch.cuda.synchronize()
            t1 = time.perf_counter()
            rmap = pdn.reff_map((0, int(net.bumps[0][0]), int(net.bumps[0][1])), net.d - 1, stride)
            t2 = time.perf_counter()
            if rep >= a.warmup:
                tn.append(t1 - t0)
                tm.append(t2 - t1)
        pdn.close()
        line["nodes"] = {"probes": k, "pairs": k * k, "ms_reff_nodes": 1e3 * float(np.mean(tn)),
                         "pairs_per_s": k * k / float(np.mean(tn)), "map_points": int(rmap.size),
                         "ms_reff_map": 1e3 * float(np.mean(tm)), "ms_create": ms / a.steps}
        if a.nodes_check > 0:   # a few pairs against the oracle (factors the whole 3D system on the host: minutes)
            from oracle.reff_oracle import Oracle
            o = Oracle(net)
            got = out_n.cpu().numpy().reshape(k, k)
            gid = nodes[:, 0].astype(np.int64) * net.n * net.n + nodes[:, 1] * net.n + nodes[:, 2]
            pa, pb = rng.integers(0, k, a.nodes_check), rng.integers(0, k, a.nodes_check)
            rel = [abs(got[i, j] / o.reff_nodes(int(gid[i]), int(gid[j])) - 1.0) for i, j in zip(pa, pb) if gid[i] != gid[j]]
            line["nodes"]["parity"] = {"pairs_checked": len(rel), "max_rel_err": float(np.max(rel)), "mean_rel_err": float(np.mean(rel))}
    if not a.no_cpu_baseline:
        ot = OracleTimer(cfg)
        n, t = ot.sample(a.cpu_budget)
        line["cpu_baseline"] = {"value": n / t, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": ot.describe(n, t)}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--rtol", type=float, default=0.0)
    ap.add_argument("--nu", type=int, default=0)
    ap.add_argument("--rhs-batch", type=int, default=0)
    ap.add_argument("--cpu-budget", type=float, default=15.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--uniform", action="store_true", help="uniform-tier variant of the workload (Eq. 3 fast path)")
    ap.add_argument("--no-fast-path", action="store_true", help="solve uniform tiers numerically too")
    ap.add_argument("--no-guess", action="store_true",
                    help="PDN_NO_INITIAL_GUESS: start every port solve from x0 = 0 instead of the closed form of the mean mesh")
    ap.add_argument("--precond-f32", action="store_true",
                    help="opt-in PDN_PRECOND_F32: multigrid sweeps in FP32 registers (CG, residuals, results stay FP64)")
    ap.add_argument("--replan", type=int, default=0, metavar="K",
                    help="also time pdn_update_tsvs after moving K TSVs of every interface to new sites (NEXT-2)")
    ap.add_argument("--eq4", action="store_true",
                    help="also time the NEXT-3 leg: context with PDN_TERMINAL_PAIRS, load-load R_eff, Eq. (4) voltages")
    ap.add_argument("--nodes", type=int, default=0, metavar="K",
                    help="also time pdn_reff_nodes on K random probes over all tiers and an R_eff map of the bottom tier (NEXT-3)")
    ap.add_argument("--map-stride", type=int, default=0, metavar="S",
                    help="with --nodes: stride of the R_eff map of the bottom tier (default n/32; 1 = every node: pdn_reff_from)")
    ap.add_argument("--nodes-check", type=int, default=0, metavar="J", help="with --nodes: check J of the pairs against the oracle")
    ap.add_argument("--shard", action="store_true",
                    help="N > 1: ONE network, its port solves sharded over the ranks (NEXT-4, strong scaling) instead "
                         "of one independent network per rank")
    ap.add_argument("--emulate-shards", type=int, default=0, metavar="W",
                    help="1 GPU: also time what ONE rank of a W-rank sharded run computes (its slice of the port solves + "
                         "S2-S3), for W = 2, 4, ... <= W; the row exchange is not included (NEXT-4 estimate)")
    ap.add_argument("--only-device", action="store_true", help="run only the device-resident steps (for ncu)")
    a = ap.parse_args()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_cuda(a)


if __name__ == "__main__":
    main()
