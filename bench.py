#!/usr/bin/env python
"""bench.py — headline benchmark of the B200 Barnes-Hut force path (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: one
``tree_leapfrog(dt)`` = kick + drift, bbox, PH keys, radix sort, octree, groups, moments, opening
radii, fused walk+force, kick.  The workload is the largest
single-GPU configuration of BASELINE.json, ``configs[3]`` (Milky-Way-shaped model, N = 134,217,728,
eps = 0.005, theta = 0.4; BASELINE.json's metric names no configuration), unless ``--config`` says
otherwise (0-based index into ``configs``).  Prints ONE JSON line.

metric   : tree-force interactions per second = (p-p + p-c interactions) / step time
value    : whole-job, inputs resident in HBM, timed with CUDA events on the library's stream; L2 is
           flushed between steps (and the inputs of the headline workload are far larger than L2)
e2e      : the same metric through the C ABI with HOST buffers (tree_build_host + tree_force_host:
           H2D of pos+mass and D2H of acc+pot inside the timed region)
roofline : the fused walk+force kernel against the FP32 FMA peak (bound "alu")
accuracy : median relative force error of the tree force against direct summation (tree_direct,
           FP64 on the device) on a 65,536-particle subsample (BASELINE.json configs 2 and 4 ask for it)
configs  : one summary per other BASELINE.json configuration, measured in the same process (N = 1 only;
           ``--no-configs`` skips them); configs[4] runs its 16 leapfrog steps and reports the energy
           drift beside the CPU oracle's on the 262,144-particle version of the same model
N > 1    : ONE problem over the N GPUs (sharded force pass, peer stores fused into the
           walk kernel), "scaling": "strong".  ``--replicas``: N independent replicas instead, "weak".
``--impl reference`` times the CPU oracle (oracle/) on the host cores on a bounded sample.
``--table NAME`` prints one of the measurement tables kept under profiles/ (bench_tables.py).
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
HEADLINE_CONFIG = 3  # mw_134m: the largest single-GPU configuration of BASELINE.json
# FP32 peak: 148 SMs x 128 FP32 lanes x 2 flop (FMA) x 1.965 GHz (B200_PROFILING.md: 148 SMs,
# clocks.max.sm 1965 MHz); MEASURED_PEAKS.json holds no FP32 number.  DESIGN.md "Roofline".
FP32_LANES_PER_SM = 128
SM_MHZ = 1965.0
# What the evaluators execute per interaction (bh_force.cu pp_one / pc_one): FP32 instructions and flops
# (an FMA = 2, add / mul / rsqrt = 1).  The paper's CONVENTION is 23 / 65.
INSTR_PP, INSTR_PC = 13, 32
XFLOP_PP, XFLOP_PC = 20, 54


def _peak_tflops(sm_count: int, sm_mhz: float = SM_MHZ) -> float:
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


# `ncu --set full` captures of the fused kernel kept under profiles/ as `--page raw --csv` exports (one launch each; the
# .md beside each names the command).  roofline.traffic is read from them, never from a hand-copied number.
NCU_RAW = {"mw_134m": "profiles/r2_walk134m_ncu_raw.csv", "plummer_1m": "profiles/r2_walk1m_ncu_raw.csv"}


def _ncu_traffic(workload: str):
    """DRAM bytes (read + written) of one launch of the walk kernel from the committed ncu export (or None)."""
    import csv
    rel = NCU_RAW.get(workload)
    if not rel:
        return None, None
    try:
        with open(os.path.join(ROOT, rel), newline="") as fh:
            rows = list(csv.reader(fh))
        hdr, units, vals = rows[0], rows[1], rows[2]
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
        tot = 0.0
        for name in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            i = hdr.index(name)
            tot += float(vals[i].replace(",", "")) * scale[units[i]]
        return int(tot), f"{rel} (ncu --set full, one launch: dram__bytes_read.sum + dram__bytes_write.sum)"
    except (OSError, KeyError, ValueError, IndexError):
        return None, None


def _config_dict(cfg, world: int, sharded: bool) -> dict:
    """The `config` object of the JSON line; both arms (ours / reference) print the same one."""
    n = cfg["n"]
    par = (f"sharded force pass x{world} (replicated tree, peer stores)" if sharded else f"replicas x{world}")
    return {"workload": cfg["name"], ("n_total" if sharded else "n_per_gpu"): n, "model": cfg["model"],
            "theta": cfg["theta"], "eps": cfg["eps"], "dt": cfg.get("dt", 1e-3), "leaf_size": 16, "group_size": 64,
            "step": "tree_leapfrog = kick/drift + keys + sort + build + moments + walk+force + kick",
            "l2": "flushed between steps (256 MB write); inputs larger than L2 from config 2 up",
            "parallelism": par}


# ---- the CPU oracle, timed as it stands (cpu_baseline leg and --impl reference) -------------------------------------
class OracleSampler:
    """Builds the oracle's tree of one workload ONCE; every call of ``sample`` times its tree force on a bounded,
    strided sample of groups."""

    def __init__(self, cfg, pos, mass):
        import oracle
        self.oracle = oracle
        self.cfg = cfg
        t0 = time.perf_counter()
        self.ot = oracle.Tree(pos, mass)
        self.build_seconds = time.perf_counter() - t0
        self.per_group = None
        import numpy as np
        # result arrays allocated once: at N = 134 M zeroing 4.3 GB per call would otherwise be timed as force work
        self.out = (np.zeros((self.ot.n, 3), np.float64), np.zeros(self.ot.n, np.float64))

    def sample(self, budget_s: float, g0: int = 0):
        import numpy as np
        ot, cfg = self.ot, self.cfg
        ng = ot.n_groups
        if self.per_group is None:  # calibrate on a few groups, then size the sample for ~budget_s
            probe = max(1, min(ng, 256))
            ps = max(1, ng // probe)
            t0 = time.perf_counter()
            ot.force(cfg["theta"], cfg["eps"], g0=ps // 2, stride=ps, out=self.out)
            self.per_group = (time.perf_counter() - t0) / len(range(ps // 2, ng, ps))
        want = int(min(ng, max(16, budget_s / max(self.per_group, 1e-9))))
        stride = max(1, ng // want)
        for attempt in range(2):
            g0 = g0 % stride
            t0 = time.perf_counter()
            _, _, npp, npc = ot.force(cfg["theta"], cfg["eps"], g0=g0, stride=stride, out=self.out)
            dt = time.perf_counter() - t0
            if attempt == 0 and dt < 0.5 * budget_s and stride > 1:  # the probe's groups were dearer than the average
                self.per_group = dt / len(range(g0, ng, stride))
                stride = max(1, int(stride * dt / budget_s))
                continue
            break
        gsel = np.arange(g0, ng, stride)
        gs = np.minimum(64, ot.n - 64 * gsel)
        inter = int(((npp[gsel].astype(np.int64) + npc[gsel].astype(np.int64)) * gs).sum())
        flops = int(((23 * npp[gsel].astype(np.int64) + 65 * npc[gsel].astype(np.int64)) * gs).sum())
        label = "full pass" if stride == 1 else f"extrapolated from every {stride}th group"
        return dict(value=inter / dt, unit=UNIT, cores=self.oracle.num_threads(), kind="oracle",
                    sample=f"oracle tree force (FP64 accumulate, as it stands) on {len(gsel)} of {ng} groups "
                           f"({label}, {dt:.1f} s) of the same workload; oracle tree build of all N took "
                           f"{self.build_seconds:.1f} s (once, not in the rate)",
                    tflops_effective=flops / dt / 1e12, seconds=dt, build_seconds=self.build_seconds)


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on the host cores (rank 0 only).  The oracle's tree of the
    workload is built once; every step times its tree force on a bounded sample of groups (another offset each step)."""
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if rank != 0:
        return 0
    import torch
    from nbody_inputs import CONFIGS, milky_way, plummer
    cfg = dict(CONFIGS[args.config])
    if args.n:
        cfg["n"] = args.n
    gen = plummer if cfg["model"] == "plummer" else milky_way
    gen_dev = "cuda" if (torch.cuda.is_available() and cfg["n"] > (1 << 22)) else "cpu"  # generation only
    pos, _, mass = gen(cfg["n"], cfg["seed"], device=gen_dev, with_vel=False)
    pos, mass = pos.cpu().numpy(), mass.cpu().numpy()
    smp = OracleSampler(cfg, pos, mass)
    total = max(1, args.steps + args.warmup)
    per_step_budget = max(1.0, min(15.0, 100.0 / total))
    vals, last = [], None
    for i in range(total):
        r = smp.sample(per_step_budget, g0=i)
        if i >= args.warmup:
            vals.append(r)
        last = r
    v = sum(x["value"] for x in vals) / len(vals)
    ms = 1e3 * sum(x["seconds"] for x in vals) / len(vals)
    sharded = world > 1 and not args.replicas
    line = {
        "impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(cfg, world, sharded),
        "note": "each step = the oracle's tree force on a bounded sample of groups of the workload (tree built once)",
        "cpu_baseline": {"value": v, "unit": UNIT, "cores": last["cores"], "kind": "oracle", "sample": last["sample"]},
        "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ---- our arm ------------------------------------------------------------------------------------------------------
def _roofline(pp, pc, walk_ms_sum, steps, step_ms_sum, sm_count, peak_meas, workload):
    """Roofline of the fused walk+force kernel (bound: FP32 ALUs).  `achieved` follows the contract of SURVEY.md
    §8(d): ALGORITHMIC flops = the paper's 23 / 65 per interaction; the executed-flop and pipe-slot fractions of the
    same launch are reported beside it (what the hardware really issued)."""
    from paper_1412_0659_b200 import effective_flops
    peak = _peak_tflops(sm_count)
    t = walk_ms_sum * 1e-3
    ach = effective_flops(pp, pc) / t / 1e12
    ach_x = (XFLOP_PP * pp + XFLOP_PC * pc) / t / 1e12
    slots = (INSTR_PP * pp + INSTR_PC * pc) / t / (sm_count * FP32_LANES_PER_SM * SM_MHZ * 1e6)
    traffic, traffic_src = _ncu_traffic(workload)
    return {"bound": "alu", "kernel": "walk_force_kernel", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
            "frac": ach / peak,
            "frac_basis": "algorithmic flops, the paper's convention: 23 per p-p, 65 per p-c (PAPER.md L190-192)",
            "achieved_executed": ach_x, "frac_executed": ach_x / peak,
            "frac_executed_basis": f"flops the evaluators execute: {XFLOP_PP} per p-p, {XFLOP_PC} per p-c (FMA = 2)",
            "fma_pipe_slot_frac": slots,
            "fma_pipe_slot_basis": f"FP32 instruction slots of the evaluators ({INSTR_PP} per p-p, {INSTR_PC} per p-c) / "
                                   "(SMs x 128 lanes x clock): the share of FMA-pipe issue slots the interactions fill",
            "peak_measured": peak_meas, "frac_of_measured": ach / peak_meas if peak_meas else None,
            "traffic": traffic, "traffic_unit": "bytes of DRAM read+write per launch", "traffic_source": traffic_src,
            "peak_source": f"derived: {sm_count} SMs x 128 FP32 lanes x 2 x 1.965 GHz "
                           "(MEASURED_PEAKS.json has no FP32 figure)",
            "kernel_ms_avg": walk_ms_sum / steps, "kernel_share_of_step": walk_ms_sum / step_ms_sum,
            "interactions_per_s_kernel": (pp + pc) / t}


def _accuracy(t, n, eps, acc, nsub=65536):
    """Median relative force error of the tree force in `acc` against tree_direct on a seeded subsample."""
    import numpy as np
    import torch
    from nbody_inputs import subsample_indices
    dev = acc.device
    idx = subsample_indices(n, nsub, device=dev)
    ad = torch.empty((idx.numel(), 3), dtype=torch.float64, device=dev)
    pd = torch.empty(idx.numel(), dtype=torch.float64, device=dev)
    t.direct(idx, eps, ad, pd)
    err = ((acc[idx].double() - ad).norm(dim=1) / ad.norm(dim=1)).cpu().numpy()
    return {"vs": "tree_direct (FP64 direct summation on the device) on a seeded subsample", "n_sub": int(idx.numel()),
            "median_rel_force_err": float(np.median(err)), "p99_rel_force_err": float(np.percentile(err, 99)),
            "bound": 2e-3}


def _generate(cfg, dev):
    from nbody_inputs import milky_way, plummer
    gen = plummer if cfg["model"] == "plummer" else milky_way
    gen_dev = dev if cfg["n"] > (1 << 22) else "cpu"
    pos, vel, mass = gen(cfg["n"], cfg["seed"], device=gen_dev)
    return pos.to(dev), vel.to(dev), mass.to(dev)


def _config_summary(k, dev, stream, flush, sm_count, with_oracle):
    """One BASELINE.json configuration in short: device-resident steps only (the headline line carries e2e)."""
    import torch
    from nbody_inputs import CONFIGS, milky_way
    from paper_1412_0659_b200 import Tree, effective_flops
    cfg = dict(CONFIGS[k])
    n, dt = cfg["n"], cfg.get("dt", 1e-3)
    steps = cfg.get("steps", 10 if n <= (1 << 20) else 5)
    warm = 0 if "steps" in cfg else 3  # configs[4] IS its 16 steps: nothing runs before them
    pos, vel, mass = _generate(cfg, dev)
    t = Tree(device=dev.index, stream=stream.cuda_stream)
    acc = torch.empty((n, 3), device=dev); pot = torch.empty(n, device=dev)
    t.build(pos, mass); t.set_velocity(vel); t.force(cfg["theta"], cfg["eps"], acc, pot)
    accuracy = _accuracy(t, n, cfg["eps"], acc)
    ke0, pe0 = t.energy()
    for _ in range(warm):
        t.leapfrog(dt)
    torch.cuda.synchronize(dev)
    ph, pp_t, pc_t, step_ms = {}, 0, 0, 0.0
    for s in range(steps):
        flush.fill_(s & 0xff)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        t.leapfrog(dt)
        e1.record(stream)
        ms, pp, pc = t.stats()
        step_ms += e0.elapsed_time(e1)
        for key, v in ms.items():
            ph[key] = ph.get(key, 0.0) + v / steps
        pp_t += pp; pc_t += pc
    ke1, pe1 = t.energy()
    out = {"config": k + 1, "workload": cfg["name"], "n": n, "steps": steps, "warmup": warm, "dt": dt,
           "ms_per_step": step_ms / steps, "value": (pp_t + pc_t) / (step_ms * 1e-3), "unit": UNIT,
           "effective_tflops_step": effective_flops(pp_t, pc_t) / (step_ms * 1e-3) / 1e12,
           "roofline_frac": effective_flops(pp_t, pc_t) / (ph["walk"] * steps * 1e-3) / 1e12 / _peak_tflops(sm_count),
           "pp_per_particle": pp_t / steps / n, "pc_per_particle": pc_t / steps / n,
           "phase_ms": ph, "accuracy": accuracy,
           "energy": {"steps": warm + steps, "rel_drift": abs((ke1 + pe1) - (ke0 + pe0)) / abs(ke0 + pe0)}}
    t.close()
    del pos, vel, mass, acc, pot
    torch.cuda.empty_cache()
    if "steps" in cfg and with_oracle:  # configs[4]: the oracle's drift on its 262,144-particle version, same steps
        import oracle
        op, ov, om = milky_way(262144, 1006)
        t0 = time.perf_counter()
        *_, en = oracle.leapfrog(op.numpy(), ov.numpy(), om.numpy(), dt, steps, cfg["theta"], cfg["eps"])
        out["energy"]["oracle_262144"] = {"steps": steps, "seconds": time.perf_counter() - t0,
                                          "rel_drift": abs(en[-1].sum() - en[0].sum()) / abs(en[0].sum())}
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist

    from nbody_inputs import CONFIGS
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

    cfg = dict(CONFIGS[args.config])
    if args.n:
        cfg["n"] = args.n
    sharded = world > 1 and not args.replicas
    if not sharded:
        cfg["seed"] = replica_seed(cfg["seed"], rank)  # every rank its own replica of the workload
    pos, vel, mass = _generate(cfg, dev)
    n = cfg["n"]
    dt = cfg.get("dt", 1e-3)
    d_pos, d_vel, d_mass = pos, vel, mass
    h_pos, h_mass = pos.cpu().pin_memory(), mass.cpu().pin_memory()
    h_acc = torch.empty((n, 3)).pin_memory(); h_pot = torch.empty(n).pin_memory()

    stream = torch.cuda.current_stream(dev)
    t = Tree(device=local, stream=stream.cuda_stream)
    if sharded:  # one problem over all ranks: same particles everywhere, the force pass is cut
        from paper_1412_0659_b200.sharded import ShardedTree
        drv = ShardedTree(t, device=dev)
        drv.connect(n)  # raises if the GPUs are not peer-capable: no silent fall-back to replicas
    else:
        drv = t
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)  # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident steps: tree_leapfrog
    acc0 = torch.empty((n, 3), device=dev); pot0 = torch.empty(n, device=dev)
    drv.build(d_pos, d_mass); drv.set_velocity(d_vel); drv.force(cfg["theta"], cfg["eps"], acc0, pot0)
    accuracy = None if (args.no_accuracy or rank != 0) else _accuracy(t, n, cfg["eps"], acc0)
    del acc0, pot0
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

    # ---- beside the headline (not part of `value`): the same steps with the error-targeted acceptance criterion
    # (tree_set_mac_relative): time per step and error against direct summation on the same workload
    relative = None
    if world == 1 and not args.no_accuracy:
        alpha, floor, rsteps = 3e-4, 1.0, min(args.steps, 5)
        acc_r = torch.empty((n, 3), device=dev)
        t.set_mac_relative(alpha)                      # scaled by |a| of the last pass of the steps above
        t.force(floor, cfg["eps"], acc_r)
        acc_rel = _accuracy(t, n, cfg["eps"], acc_r, nsub=16384)
        del acc_r
        t.leapfrog(dt)
        rev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(rsteps)]
        rpp = rpc = 0
        rwalk = 0.0
        for k in range(rsteps):
            flush.fill_(k & 0xff)
            rev[k][0].record(stream)
            t.leapfrog(dt)
            rev[k][1].record(stream)
            ms, pp, pc = t.stats()
            rpp += pp; rpc += pc; rwalk += ms["walk"]
        rms = sum(a.elapsed_time(b) for a, b in rev)
        relative = {"criterion": f"tree_set_mac_relative(alpha={alpha:g}), geometric floor theta={floor:g}; |a| of the previous pass",
                    "steps": rsteps, "ms_per_step": rms / rsteps, "walk_ms": rwalk / rsteps,
                    "value": (rpp + rpc) / (rms * 1e-3), "unit": UNIT,
                    "pp_per_particle": rpp / rsteps / n, "pc_per_particle": rpc / rsteps / n,
                    "roofline_frac": effective_flops(rpp, rpc) / (rwalk * 1e-3) / 1e12 / _peak_tflops(torch.cuda.get_device_properties(dev).multi_processor_count),
                    "accuracy": acc_rel, "speedup_of_step_vs_headline": (step_ms / args.steps) / (rms / rsteps)}
        t.set_mac("geometric")
    mx, sm = reduce_max_sum([step_ms, float(pp_tot), float(pc_tot), phase_ms["walk"]], dev)
    step_ms_max = mx[0]
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
        smc = props.multi_processor_count
        peak_meas = t.fp32_peak()  # register-only FFMA kernel, run now on this GPU
        roof = _roofline(pp_tot, pc_tot, phase_ms["walk"], args.steps, step_ms, smc, peak_meas, cfg["name"])
        cpu = None
        others = None
        host_pos, host_mass = pos.cpu().numpy(), mass.cpu().numpy()
    drv.close()
    del pos, vel, mass, d_pos, d_vel, d_mass, h_acc, h_pot, h_pos, h_mass, h_vel
    torch.cuda.empty_cache()
    if rank == 0:
        if world == 1 and not args.no_cpu:
            cpu = OracleSampler(cfg, host_pos, host_mass).sample(15.0)
        del host_pos, host_mass
        if world == 1 and not args.no_configs:
            others = []
            for k in sorted(CONFIGS):
                if k != args.config:
                    others.append(_config_summary(k, dev, stream, flush, smc, with_oracle=not args.no_cpu))
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": step_ms_max / args.steps, "higher_is_better": True,
            "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": _config_dict(cfg, world, sharded),
            "effective_tflops_step": effective_flops(pp_all, pc_all) / (step_ms_max * 1e-3) / 1e12,
            "pp_per_particle": (pp_all if sharded else pp_tot) / args.steps / n,
            "pc_per_particle": (pc_all if sharded else pc_tot) / args.steps / n,
            "phase_ms": {k: v / args.steps for k, v in phase_ms.items()},
            "roofline": roof,
            "accuracy": accuracy,
            "relative_mac": relative,
            "energy": energy,
            "cpu_baseline": cpu,
            "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 16 * n,
                    "ms_per_step": 1e3 * e2e_s / args.steps, "phase_ms": e_phase,
                    "call": "tree_build_host + tree_force_host (pinned host buffers; host positions drift by dt * v between steps)"},
            "gpu_launches": launches, "clocks": clocks, "wall_s_timed_region": wall,
            "configs": others,
        }
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=HEADLINE_CONFIG, help="0-based index into BASELINE.json configs")
    ap.add_argument("--n", type=int, default=0, help="override N (debugging only)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg (and the oracle's drift run)")
    ap.add_argument("--no-configs", action="store_true", help="skip the summaries of the other BASELINE.json configs")
    ap.add_argument("--no-accuracy", action="store_true", help="skip the error against direct summation")
    ap.add_argument("--replicas", action="store_true",
                    help="N > 1: N independent replicas (weak scaling) instead of ONE problem over all GPUs")
    ap.add_argument("--sharded", action="store_true", help="(default for N > 1; kept for older command lines)")
    ap.add_argument("--table", default="", help="print a measurement table instead (bench_tables.py): kernels | "
                                                "shard-scaling | shard-weak | mac-sweep | sass-histogram | walk-eval-split")
    ap.add_argument("--from-ncu", default="", help="--table kernels: the ncu CSV to read")
    ap.add_argument("--from-sass", default="", help="--table sass-histogram: the cuobjdump -sass listing to read")
    ap.add_argument("--worlds", default="1,2,4,8", help="--table shard-scaling: world sizes")
    args = ap.parse_args()
    if args.table:
        import bench_tables
        return bench_tables.run(args)
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
