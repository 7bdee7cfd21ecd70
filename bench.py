#!/usr/bin/env python
"""bench.py — headline benchmark of the B200 Barnes-Hut force path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: one
``tree_leapfrog(dt)`` = kick + drift, bbox, PH keys, radix sort, permute, octree, groups, moments,
opening radii, fused walk+force, un-permute, kick.  The workload is
BASELINE.json ``configs[1]`` (Plummer sphere, N = 1,048,576, eps = 0.005, theta = 0.4) unless
``--config`` says otherwise (0-based index into ``configs``).  Prints ONE JSON line.

metric  : tree-force interactions per second = (p-p + p-c interactions) / step time
value   : whole-job, inputs resident in HBM, timed with CUDA events on the library's stream,
          L2 flushed between steps (inputs at N = 1M are smaller than the 126 MB L2)
e2e     : the same metric through the C ABI with HOST buffers (tree_build_host + tree_force_host:
          H2D of pos+mass and D2H of acc+pot inside the timed region)
roofline: the fused walk+force kernel against the FP32 FMA peak (bound "alu")
N > 1   : the path is partitioned by independent problems: every rank runs its own replica of the
          workload (seed + rank), no data-path collective; scaling "weak".
          ``--sharded``: ONE problem over the N GPUs instead (every rank builds the same tree,
          walks a cost-balanced range of groups and peer-stores its results into all ranks); scaling "strong".
``--impl reference`` times the CPU oracle (oracle/) on the host cores on a bounded sample.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "tree-force interactions/s and effective FP32 Tflops (fraction of peak)"
UNIT = "interactions/s"
# FP32 peak: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x 1.965 GHz (B200_PROFILING.md: 148 SMs,
# clocks.max.sm 1965 MHz); MEASURED_PEAKS.json holds no FP32 number.  DESIGN.md "Roofline".
FP32_LANES_PER_SM = 128


def _peak_tflops(sm_count: int, sm_mhz: float) -> float:
    return sm_count * FP32_LANES_PER_SM * 2 * sm_mhz * 1e6 / 1e12


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.lines = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for nm, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def _ncu_traffic(workload: str):
    """DRAM bytes per launch of the walk kernel from the committed ncu --set full capture (or None)."""
    import csv
    path = os.path.join(ROOT, "profiles", "walk_dram_traffic.csv")
    try:
        with open(path) as fh:
            for row in csv.DictReader(fh):
                if row["workload"] == workload:
                    return int(row["dram_bytes_read"]) + int(row["dram_bytes_write"]), row["source"]
    except (OSError, KeyError, ValueError):
        pass
    return None, None


def _cpu_oracle_sample(cfg, pos, mass, budget_s: float = 15.0):
    """Time the oracle's tree force (as it stands) on a bounded sample of groups of this workload."""
    import numpy as np
    import oracle

    t0 = time.perf_counter()
    ot = oracle.Tree(pos, mass)
    t_build = time.perf_counter() - t0
    ng = ot.n_groups
    # calibrate on a few groups, then size the sample for ~budget_s
    probe = max(1, ng // 64)
    t0 = time.perf_counter()
    ot.force(cfg["theta"], cfg["eps"], g0=0, stride=max(1, ng // probe))
    t_probe = time.perf_counter() - t0
    per_group = t_probe / max(1, len(range(0, ng, max(1, ng // probe))))
    want = int(min(ng, max(probe, budget_s / max(per_group, 1e-9))))
    stride = max(1, ng // want)
    t0 = time.perf_counter()
    _, _, npp, npc = ot.force(cfg["theta"], cfg["eps"], g0=0, stride=stride)
    dt = time.perf_counter() - t0
    gsel = np.arange(0, ng, stride)
    gs = np.minimum(64, ot.n - 64 * gsel)
    inter = int(((npp[gsel].astype(np.int64) + npc[gsel].astype(np.int64)) * gs).sum())
    flops = int(((23 * npp[gsel].astype(np.int64) + 65 * npc[gsel].astype(np.int64)) * gs).sum())
    return dict(value=inter / dt, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                sample=f"oracle tree force (FP64 accumulate) on every {stride}th group "
                       f"({len(gsel)} of {ng} groups, {dt:.1f} s) of the same workload; "
                       f"oracle tree build of all N took {t_build:.1f} s",
                tflops_effective=flops / dt / 1e12, seconds=dt, build_seconds=t_build)


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from nbody_inputs import config
    cfg, pos, vel, mass = config(args.config, with_vel=False)
    pos, mass = pos.numpy(), mass.numpy()
    per_step_budget = max(2.0, min(15.0, 120.0 / max(1, args.steps + args.warmup)))
    vals = []
    last = None
    for i in range(args.warmup + args.steps):
        r = _cpu_oracle_sample(cfg, pos, mass, budget_s=per_step_budget)
        if i >= args.warmup:
            vals.append(r)
        last = r
    v = sum(x["value"] for x in vals) / len(vals)
    ms = 1e3 * sum(x["seconds"] + x["build_seconds"] for x in vals) / len(vals)
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": cfg["name"], "n": cfg["n"], "theta": cfg["theta"], "eps": cfg["eps"],
                   "note": "each step = oracle tree build + oracle tree force on a bounded sample of groups"},
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def run_ours(args):
    import torch
    import torch.distributed as dist

    from nbody_inputs import config
    from paper_1412_0659_b200 import Tree, effective_flops
    from paper_1412_0659_b200.replicas import replica_seed, reduce_max_sum, whole_job_rate

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    from nbody_inputs import CONFIGS
    cfg = dict(CONFIGS[args.config])
    if args.n:
        cfg["n"] = args.n
    sharded = bool(args.sharded)
    if not sharded:
        cfg["seed"] = replica_seed(cfg["seed"], rank)  # every rank its own replica of the workload
    from nbody_inputs import plummer, milky_way
    gen = plummer if cfg["model"] == "plummer" else milky_way
    gen_dev = dev if cfg["n"] > (1 << 22) else "cpu"
    pos, vel, mass = gen(cfg["n"], cfg["seed"], device=gen_dev)
    n = cfg["n"]
    dt = cfg.get("dt", 1e-3)
    h_pos, h_mass = pos.cpu().pin_memory(), mass.cpu().pin_memory()
    d_pos, d_vel, d_mass = pos.to(dev), vel.to(dev), mass.to(dev)
    h_acc = torch.empty((n, 3)).pin_memory(); h_pot = torch.empty(n).pin_memory()

    stream = torch.cuda.current_stream(dev)
    t = Tree(device=local, stream=stream.cuda_stream)
    if sharded:  # one problem over all ranks: same particles everywhere, the force pass is cut
        from paper_1412_0659_b200.sharded import ShardedTree
        drv = ShardedTree(t, device=dev)
        try:
            drv.connect(n)
        except RuntimeError as e:  # no peer access between these GPUs: every rank falls back to its own replica
            sys.stderr.write(f"[bench] --sharded unavailable ({e}); running replicas\n")
            sharded = False
            drv = t
    else:
        drv = t
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident steps: tree_leapfrog
    drv.build(d_pos, d_mass); drv.set_velocity(d_vel); drv.force(cfg["theta"], cfg["eps"])
    ke0, pe0 = t.energy()  # synchronised velocities: E(0) of the KDK run (T12)
    for _ in range(args.warmup):
        drv.leapfrog(dt)
    barrier()
    sampler = ClockSampler(local)
    sampler.start()
    l0 = t.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    phase_ms = {}
    pp_tot = pc_tot = 0
    wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.fill_(k & 0xff)  # L2 flush, outside the event pair
        ev[k][0].record(stream)
        drv.leapfrog(dt)
        ev[k][1].record(stream)
        ms, pp, pc = t.stats()  # synchronises; reads the library's own per-phase CUDA events (this rank's share)
        for key, v in ms.items():
            phase_ms[key] = phase_ms.get(key, 0.0) + v
        pp_tot += pp; pc_tot += pc
    barrier()
    wall = time.perf_counter() - wall0
    launches = t.launch_count() - l0
    ke1, pe1 = t.energy()
    energy = {"steps": args.warmup + args.steps, "dt": dt, "e0": ke0 + pe0, "e1": ke1 + pe1,
              "rel_drift": abs((ke1 + pe1) - (ke0 + pe0)) / abs(ke0 + pe0)}
    clocks = sampler.stop()
    step_ms = sum(a.elapsed_time(b) for a, b in ev)
    mx, sm = reduce_max_sum([step_ms, float(pp_tot), float(pc_tot), phase_ms["walk"]], dev)
    step_ms_max, walk_ms_max = mx[0], mx[3]
    pp_all, pc_all = sm[1], sm[2]
    value = (pp_all + pc_all) / (step_ms_max * 1e-3)

    # ---- end to end through the C ABI with host buffers (build + force, copies timed)
    if sharded:
        # the sharded pass has no *_host call: the same copies through torch, then build + sharded force
        d_acc = torch.empty((n, 3), device=dev); d_pot = torch.empty(n, device=dev)

        class _HostCalls:
            def build_host(self, hp, hm):
                d_pos.copy_(hp, non_blocking=True); d_mass.copy_(hm, non_blocking=True)
                drv.build(d_pos, d_mass)

            def force_host(self, theta, eps, ha, hp):
                drv.force(theta, eps, d_acc, d_pot)
                ha.copy_(d_acc, non_blocking=True); hp.copy_(d_pot, non_blocking=True)
                torch.cuda.synchronize(dev)

            def stats(self):
                return t.stats()

            def close(self):
                pass
        t2 = _HostCalls()
    else:
        t2 = Tree(device=local, stream=stream.cuda_stream)
    # The caller of the *_host calls owns the integration: between two steps the host positions drift by dt * v (outside
    # the timed region), so that every step builds a tree over new positions, as a host-side integrator would ask for.
    h_vel = vel.cpu()

    def host_drift():
        h_pos.add_(h_vel, alpha=dt)

    for _ in range(min(args.warmup, 3)):
        t2.build_host(h_pos, h_mass); t2.force_host(cfg["theta"], cfg["eps"], h_acc, h_pot)
        host_drift()
    barrier()
    e2e_s = 0.0
    e_pp = e_pc = 0
    e_phase = {}
    for k in range(args.steps):
        if k:
            host_drift()
        flush.fill_(k & 0xff)
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        t2.build_host(h_pos, h_mass)
        t2.force_host(cfg["theta"], cfg["eps"], h_acc, h_pot)  # returns after the D2H copies
        e2e_s += time.perf_counter() - t0
        ems, pp, pc = t2.stats()
        for key, v in ems.items():
            e_phase[key] = e_phase.get(key, 0.0) + v / args.steps
        e_pp += pp; e_pc += pc
    e2e_val = whole_job_rate(e2e_s, float(e_pp + e_pc), dev)  # each rank counts the interactions it evaluated
    t2.close()

    if rank == 0:
        props = torch.cuda.get_device_properties(dev)
        peak = _peak_tflops(props.multi_processor_count, 1965.0)
        flops = effective_flops(pp_tot, pc_tot)
        ach = flops / (phase_ms["walk"] * 1e-3) / 1e12
        traffic, traffic_src = _ncu_traffic(cfg["name"])
        peak_meas = t.fp32_peak()  # register-only FFMA kernel, run now on this GPU
        roof = {"bound": "alu", "kernel": "walk_force_kernel", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                "frac": ach / peak, "peak_measured": peak_meas, "frac_of_measured": ach / peak_meas if peak_meas else None,
                "traffic": traffic, "traffic_unit": "bytes of DRAM read+write per launch",
                "traffic_source": traffic_src,
                "peak_source": f"derived: {props.multi_processor_count} SMs x 128 FP32 lanes x 2 x 1.965 GHz "
                               "(MEASURED_PEAKS.json has no FP32 figure)",
                "flops_convention": "23 per p-p, 65 per p-c (PAPER.md L190-192)",
                "kernel_ms_avg": phase_ms["walk"] / args.steps,
                "kernel_share_of_step": phase_ms["walk"] / step_ms,
                "interactions_per_s_kernel": (pp_tot + pc_tot) / (phase_ms["walk"] * 1e-3)}
        cpu = None
        if world == 1 and not args.no_cpu:
            cpu = _cpu_oracle_sample(cfg, pos.cpu().numpy(), mass.cpu().numpy(), budget_s=15.0)
            if "steps" in cfg:  # config 5: energy drift of the oracle on its 262,144-particle version
                import oracle
                op, ov, om = gen(262144, 1006)
                t0 = time.perf_counter()
                *_, en = oracle.leapfrog(op.numpy(), ov.numpy(), om.numpy(), dt, args.warmup + args.steps,
                                         cfg["theta"], cfg["eps"])
                energy["oracle_262144"] = {"steps": args.warmup + args.steps, "seconds": time.perf_counter() - t0,
                                           "rel_drift": abs(en[-1].sum() - en[0].sum()) / abs(en[0].sum())}
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms_max / args.steps, "higher_is_better": True,
            "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": cfg["name"], ("n_total" if sharded else "n_per_gpu"): n, "model": cfg["model"], "theta": cfg["theta"],
                       "eps": cfg["eps"], "dt": dt, "leaf_size": 16, "group_size": 64,
                       "step": "tree_leapfrog = kick/drift + keys + sort + build + moments + walk+force + kick",
                       "l2": "flushed between steps (256 MB write)", "parallelism": (f"sharded force pass x{world} (replicated tree, peer stores)" if sharded
                                       else f"replicas x{world}")},
            "effective_tflops_step": effective_flops(pp_all, pc_all) / (step_ms_max * 1e-3) / 1e12,
            "pp_per_particle": (pp_all if sharded else pp_tot) / args.steps / n,
            "pc_per_particle": (pc_all if sharded else pc_tot) / args.steps / n,
            "phase_ms": {k: v / args.steps for k, v in phase_ms.items()},
            "roofline": roof,
            "energy": energy,
            "cpu_baseline": cpu,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 16 * n,
                    "ms_per_step": 1e3 * e2e_s / args.steps, "phase_ms": e_phase,
                    "call": "tree_build_host + tree_force_host (pinned host buffers; host positions drift by dt * v between steps)"},
            "gpu_launches": launches, "clocks": clocks, "wall_s_timed_region": wall,
        }
        print(json.dumps(line))
    drv.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=1, help="0-based index into BASELINE.json configs")
    ap.add_argument("--n", type=int, default=0, help="override N (debugging only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--sharded", action="store_true",
                    help="N > 1: one problem over all GPUs (sharded force pass, strong scaling) instead of replicas")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
