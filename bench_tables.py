"""Measurement tables kept under profiles/ (markdown on stdout), run through ``python bench.py --table NAME``.

  kernels        per-kernel launch time and DRAM traffic of the step's HBM-bound phases, from an ncu CSV
                 (``--from-ncu FILE``: a ``--metrics gpu__time_duration.sum,dram__bytes_read.sum,dram__bytes_write.sum``
                 pass), against the measured copy bandwidth of MEASURED_PEAKS.json and the algorithmic bytes of DESIGN.md §5
  shard-scaling  per-rank cost of the sharded force pass measured on ONE GPU with W contexts
  shard-weak     the same with N = 13 M particles x W (the paper's weak-scaling set-up, Table II): per-rank
                 phase times in the rows of Table II; ``--n`` overrides the particles per rank
  sass-histogram instruction classes of the whole kernel and of every innermost loop of a ``cuobjdump -sass`` listing
                 (``--from-sass FILE``)
  walk-eval-split the fused kernel against its walk alone and its evaluation alone (tree_measure_listeval); ``--worlds``
                 takes the list of configurations here (default 2,4)
  mac-sweep      error versus cost of the acceptance criteria: opening angle x criterion on a
                 BASELINE.json configuration, force error against tree_direct on a 16,384 subsample

Nothing here is on the product path; the tables only call the library through its binding.
"""
from __future__ import annotations

import csv
import json
import os
import re
from collections import defaultdict

ROOT = os.path.dirname(os.path.abspath(__file__))

# Algorithmic bytes per particle (or per cell, marked "c") of each HBM-bound kernel of the step pipeline, DESIGN.md §5.
# n_c = cells, N = particles.  (read + written)
ALGO_BYTES = {
    "kick_drift_bbox_kernel": ("N", 48 + 32),
    "bbox_kernel": ("N", 16 + 16),
    "keys_kernel": ("N", 16 + 8),
    "sort_hist8_kernel": ("N", 8),
    "sort_onesweep_kernel": ("N", 12 + 12),
    "permute_step_kernel": ("N", 8 + 4 + 36 + 36),
    "permute_build_kernel": ("N", 4 + 16 + 20),
    "tree_levels_kernel": ("N", 8 + 2),
    "tree_emit_kernel": ("N", 2 + 3),  # level / leaf words read + 13 B per cell written (c_level, c_first, c_count, c_fcall), 0.234 cells per particle
    "groups_kernel": ("N", 16),
    "kick_kernel": ("N", 32 + 16),
    "gather_out_kernel": ("N", 20 + 16),
    "inverse_order_kernel": ("N", 4 + 4),
}


def _peak_gbs() -> float:
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return float(json.load(fh)["hbm_gbs"])
    except Exception:
        return 6555.8  # the driver's figure for this pool (B200_PROFILING.md fallback if absent)


def table_kernels(path: str, n_particles: int, skip_walk: bool = True):
    """ncu CSV (long format: one row per launch and metric) -> per-kernel averages."""
    rows = []
    with open(path, newline="") as fh:
        lines = [ln for ln in fh if not ln.startswith("==")]
    rd = csv.DictReader(lines)
    per = defaultdict(lambda: defaultdict(dict))  # kernel -> launch id -> metric -> value
    for r in rd:
        name = re.sub(r"\(.*", "", r.get("Kernel Name", "")).strip()
        name = re.sub(r"^void\s+", "", name)
        name = re.sub(r"<.*", "", name).replace("bh::", "")
        try:
            v = float(r["Metric Value"].replace(",", ""))
        except (KeyError, ValueError):
            continue
        unit = r.get("Metric Unit", "")
        m = r["Metric Name"]
        if m == "gpu__time_duration.sum":
            v *= {"ns": 1e-3, "us": 1.0, "ms": 1e3, "s": 1e6}.get(unit, 1e-3)  # -> us
        else:
            v *= {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}.get(unit, 1.0)
        per[name][r["ID"]][m] = v
    peak = _peak_gbs()
    print(f"| kernel | launches | avg us | DRAM MB / launch | DRAM GB/s | % of {peak:.1f} | algorithmic MB | algorithmic GB/s | % | DRAM / algorithmic |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    tot = []
    for name, launches in per.items():
        if skip_walk and name.startswith("walk_force"):
            continue
        ts = [d.get("gpu__time_duration.sum", 0.0) for d in launches.values()]
        by = [d.get("dram__bytes_read.sum", 0.0) + d.get("dram__bytes_write.sum", 0.0) for d in launches.values()]
        us = sum(ts) / len(ts)
        mb = sum(by) / len(by) / 1e6
        tot.append((sum(ts), name, len(ts), us, mb))
    for _, name, cnt, us, mb in sorted(tot, reverse=True):
        gbs = mb / us * 1e3 if us else 0.0
        algo = ALGO_BYTES.get(name)
        if algo:
            amb = algo[1] * n_particles / 1e6
            agbs = amb / us * 1e3
            extra = f"{amb:.1f} | {agbs:.0f} | {100 * agbs / peak:.0f} | {mb / amb:.2f}"
        else:
            extra = "- | - | - | -"
        print(f"| {name} | {cnt} | {us:.1f} | {mb:.1f} | {gbs:.0f} | {100 * gbs / peak:.0f} | {extra} |")


def _measure_shards(cfg, world: int, steps: int):
    import torch
    from nbody_inputs import milky_way, plummer
    from paper_1412_0659_b200 import Tree
    from paper_1412_0659_b200.sharded import connect_local, force_local, leapfrog_local
    gen = plummer if cfg["model"] == "plummer" else milky_way
    n = cfg["n"]
    pos, vel, mass = gen(n, cfg["seed"], device="cuda" if n > (1 << 22) else "cpu")
    pos, vel, mass = pos.cuda(), vel.cuda(), mass.cuda()
    trees = [Tree(device=0) for _ in range(world)]
    for t in trees:
        t.reserve(n)
    if world > 1:
        connect_local(trees)
    for t in trees:
        t.build(pos, mass); t.set_velocity(vel)
    force_local(trees, cfg["theta"], cfg["eps"])
    leapfrog_local(trees, cfg.get("dt", 1e-3))  # warm-up; from here on the partition follows exact counts
    rows = []
    for _ in range(steps):
        leapfrog_local(trees, cfg.get("dt", 1e-3))
        torch.cuda.synchronize()
        per_rank = []
        for t in trees:
            ms, pp, pc = t.stats()
            g_lo, g_hi, _, _ = t.shard_range()
            # phases this rank runs before the barrier (walk included) + its kick after it; the kick is timed from the
            # barrier, which on one GPU includes the other contexts' kernels, so it is taken from the W = 1 run
            own = ms["total"] - ms["integrate"] - ms["unpermute"]
            per_rank.append(dict(total=own, walk=ms["walk"], sched=ms["sched"], rest=own - ms["walk"] - ms["sched"],
                                 groups=g_hi - g_lo, flops=23 * pp + 65 * pc, pp=pp, pc=pc, sort=ms["sort"],
                                 tree=ms["build"], moments=ms["moments"],
                                 other=own - ms["walk"] - ms["sort"] - ms["build"] - ms["moments"]))
        rows.append(per_rank)
    for t in trees:
        t.close()
    return [{k: sum(row[r][k] for row in rows) / len(rows) for k in rows[0][r]} for r in range(world)]


def table_shard_scaling(config: int, worlds, steps: int):
    """For every world size W, W contexts on cuda:0 share the passes of a few leapfrog steps.  Their kernels run one
    after the other, each with the whole GPU, as they would on W GPUs, so the library's per-phase CUDA-event times of
    each context are the times one rank of a W-GPU run spends; what one GPU cannot show is the cost of the peer stores
    over NVLink (16 bytes per particle and peer, spread over the walk kernel) and of the barrier."""
    import torch
    from nbody_inputs import CONFIGS
    from paper_1412_0659_b200 import Tree
    cfg = dict(CONFIGS[config])
    # the integrate phase (kick + drift + bbox, and the sharded kick) of a single context, measured alone
    t = Tree(device=0)
    from nbody_inputs import milky_way, plummer
    gen = plummer if cfg["model"] == "plummer" else milky_way
    pos, vel, mass = gen(cfg["n"], cfg["seed"], device="cuda" if cfg["n"] > (1 << 22) else "cpu")
    t.build(pos.cuda(), mass.cuda()); t.set_velocity(vel.cuda()); t.force(cfg["theta"], cfg["eps"])
    t.leapfrog(cfg.get("dt", 1e-3)); t.leapfrog(cfg.get("dt", 1e-3))
    integ = t.stats()[0]["integrate"] * 1.5  # + the sharded pass's own kick kernel (half the kick/drift pass's bytes)
    t.close()
    del pos, vel, mass
    torch.cuda.empty_cache()
    print(f"# sharded force pass, per-rank times on one GPU: {cfg['name']}, N = {cfg['n']:,}, theta {cfg['theta']}, "
          f"eps {cfg['eps']}, {steps} leapfrog steps averaged")
    print("| ranks | slowest rank: step ms | its walk ms | its build+rest ms | its task list ms | walk ms min..max over ranks "
          "| flop share max / fair | step(1) / step(W) |")
    print("|---|---|---|---|---|---|---|---|")
    base = None
    for w in worlds:
        avg = _measure_shards(cfg, w, steps)
        for r in avg:
            r["total"] += integ; r["rest"] += integ
        slow = max(avg, key=lambda r: r["total"])
        if base is None:
            base = slow["total"]
        tot_flops = sum(r["flops"] for r in avg)
        share = max(r["flops"] for r in avg) / (tot_flops / w)
        walks = [r["walk"] for r in avg]
        print(f"| {w} | {slow['total']:.3f} | {slow['walk']:.3f} | {slow['rest']:.3f} | {slow['sched']:.3f} | "
              f"{min(walks):.3f} .. {max(walks):.3f} | {share:.3f} | {base / slow['total']:.2f} |", flush=True)


def table_shard_weak(n_per_rank: int, worlds, steps: int):
    """Weak scaling in the paper's set-up (13 million particles per GPU, Milky-Way model, theta = 0.4),
    emulated on one GPU like table_shard_scaling: W contexts share the steps of ONE problem of N = n_per_rank x W
    particles; the rows are those of the paper's Table II (L240-258).  NVLink stores and barriers are not in it."""
    import torch
    from nbody_inputs import milky_way
    from paper_1412_0659_b200 import Tree
    theta, eps, dt = 0.4, 0.01, 5e-4
    print(f"# weak scaling, {n_per_rank:,} particles per rank (PAPER.md L200), Milky-Way-shaped model, theta {theta}, eps {eps}, "
          f"dt {dt}: per-rank times of the slowest rank on one GPU, {steps} leapfrog steps averaged")
    print("| ranks | N total | sorting ms | tree construction ms | tree properties ms | compute gravity (walk + force) ms | "
          "other (kick/drift, keys, gather, opening, task list) ms | total ms | p-p / particle | p-c / particle | "
          "GPU TFLOP/s per rank (walk) | application TFLOP/s per rank | step(1) / step(W) |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|---|")
    base = None
    for w in worlds:
        n = n_per_rank * w
        cfg = dict(name=f"mw_weak_{w}", model="milky_way", n=n, seed=1100 + w, theta=theta, eps=eps, dt=dt)
        t = Tree(device=0)  # the integrate phase of a single context at this N, measured alone (see table_shard_scaling)
        pos, vel, mass = milky_way(n, cfg["seed"], device="cuda")
        t.build(pos, mass); t.set_velocity(vel); t.force(theta, eps)
        t.leapfrog(dt); t.leapfrog(dt)
        integ = t.stats()[0]["integrate"] * 1.5
        t.close()
        del pos, vel, mass
        torch.cuda.empty_cache()
        avg = _measure_shards(cfg, w, steps)
        for r in avg:
            r["total"] += integ; r["other"] += integ
        slow = max(avg, key=lambda r: r["total"])
        if base is None:
            base = slow["total"]
        pp = sum(r["pp"] for r in avg) / n
        pc = sum(r["pc"] for r in avg) / n
        print(f"| {w} | {n:,} | {slow['sort']:.2f} | {slow['tree']:.2f} | {slow['moments']:.2f} | {slow['walk']:.2f} | "
              f"{slow['other']:.2f} | {slow['total']:.2f} | {pp:.0f} | {pc:.0f} | {slow['flops'] / slow['walk'] / 1e9:.1f} | "
              f"{slow['flops'] / slow['total'] / 1e9:.1f} | {base / slow['total']:.3f} |", flush=True)
        torch.cuda.empty_cache()


def table_mac_sweep(config: int):
    """Opening angle x acceptance criterion x grouping on one BASELINE.json configuration: interaction counts, walk
    time, force error against tree_direct (FP64 direct summation on the device) on a 16,384 subsample."""
    import numpy as np
    import torch
    from nbody_inputs import config as make_config, subsample_indices
    from paper_1412_0659_b200 import Tree
    cfg, pos, vel, mass = make_config(config, device="cuda", with_vel=False)
    n, eps = cfg["n"], cfg["eps"]
    idx = subsample_indices(n, 16384, device="cuda")
    ad = torch.empty((idx.numel(), 3), dtype=torch.float64, device="cuda")
    pd = torch.empty(idx.numel(), dtype=torch.float64, device="cuda")
    acc = torch.empty((n, 3), device="cuda"); pot = torch.empty(n, device="cuda")
    adn = None
    print(f"# {cfg['name']}, N = {n:,}, eps {eps}: acceptance criterion x theta (group 64, leaf 16 unless stated)")
    print("| criterion | group | leaf | theta | p-p / particle | p-c / particle | walk+sched ms | median err | 99% err | max err | eff. TFLOP/s |")
    print("|---|---|---|---|---|---|---|---|---|---|---|")
    from paper_1412_0659_b200.binding import MAC_KINDS
    for mac_name, mac in MAC_KINDS.items():
        for group, leaf in ((64, 16), (32, 16), (128, 16), (64, 8), (64, 32)):
            if mac != 0 and (group, leaf) != (64, 16):
                continue
            t = Tree(device=0, leaf_size=leaf, group_size=group)
            t.set_mac(mac)
            t.build(pos, mass)
            if adn is None:
                t.direct(idx, eps, ad, pd); torch.cuda.synchronize(); adn = ad.cpu().numpy()
            for theta in (0.3, 0.4, 0.5, 0.6, 0.75, 0.9):
                ws = []
                for _ in range(3):
                    t.force(theta, eps, acc, pot); ms, pp, pc = t.stats(); ws.append(ms["walk"] + ms["sched"])
                a = acc[idx].double().cpu().numpy()
                err = np.linalg.norm(a - adn, axis=1) / np.linalg.norm(adn, axis=1)
                print(f"| {mac_name} | {group} | {leaf} | {theta} | {pp / n:.0f} | {pc / n:.0f} | {min(ws):.2f} | "
                      f"{np.median(err):.2e} | {np.percentile(err, 99):.2e} | {err.max():.2e} | "
                      f"{(23 * pp + 65 * pc) / min(ws) / 1e9:.1f} |", flush=True)
            t.close()
    # the error-targeted criterion (tree_set_mac_relative): theta = 1 as the geometric floor, alpha swept; every pass is
    # scaled by |a| of the canonical theta = 0.4 pass (handed in, so that the rows differ in alpha only)
    t = Tree(device=0)
    t.build(pos, mass)
    t.force(0.4, eps, acc, pot)
    amag = acc.norm(dim=1).contiguous()
    for alpha in (1e-4, 2e-4, 3e-4, 6e-4, 1e-3, 3e-3):
        ws = []
        for _ in range(3):
            t.set_mac_relative(alpha, amag)
            t.force(1.0, eps, acc, pot); ms, pp, pc = t.stats(); ws.append(ms["walk"] + ms["sched"])
        a = acc[idx].double().cpu().numpy()
        err = np.linalg.norm(a - adn, axis=1) / np.linalg.norm(adn, axis=1)
        print(f"| relative alpha={alpha:g} | 64 | 16 | 1.0 (floor) | {pp / n:.0f} | {pc / n:.0f} | {min(ws):.2f} | "
              f"{np.median(err):.2e} | {np.percentile(err, 99):.2e} | {err.max():.2e} | "
              f"{(23 * pp + 65 * pc) / min(ws) / 1e9:.1f} |", flush=True)
    t.close()


def table_sass_histogram(path: str):
    """Instruction histogram of a `cuobjdump -sass -fun KERNEL libbhtree.so` listing: whole kernel and every innermost
    loop (a backward branch that encloses no other), in the classes the roofline of the fused kernel talks about."""
    import collections
    ins = []
    for ln in open(path).read().splitlines():
        m = re.match(r"\s+/\*([0-9a-f]{4,})\*/\s+(.*?);", ln)
        if m:
            txt = re.sub(r"^@!?U?P\d+\s+", "", m.group(2).strip())
            ins.append((int(m.group(1), 16), txt.split()[0].split(".")[0], txt))
    loops = []
    for a, op, txt in ins:
        if op == "BRA":
            m = re.search(r"0x([0-9a-f]+)", txt)
            if m and int(m.group(1), 16) < a:
                loops.append((int(m.group(1), 16), a))
    inner = [l for l in loops if not any(o != l and l[0] <= o[0] and o[1] <= l[1] for o in loops)]
    scalar = ("FFMA", "FMUL", "FADD", "FSEL", "FSETP", "FMNMX", "FMNMX3")

    def cls(op):
        return op if op in ("FFMA2", "FMUL2", "FADD2", "MUFU", "LDS") else ("FP32 scalar" if op in scalar else "other")

    cols = ["FFMA2", "FMUL2", "FADD2", "MUFU", "LDS", "FP32 scalar", "other"]
    print("| region | instructions | " + " | ".join(cols) + " | packed with a .reuse operand | most frequent other |")
    print("|---|---|" + "---|" * (len(cols) + 2))

    def row(name, body):
        h = collections.Counter(cls(i[1]) for i in body)
        oth = collections.Counter(i[1] for i in body if cls(i[1]) == "other").most_common(5)
        reuse = sum(".reuse" in i[2] for i in body if i[1] in ("FFMA2", "FMUL2", "FADD2"))
        print(f"| {name} | {len(body)} | " + " | ".join(str(h.get(c, 0)) for c in cols) + f" | {reuse} | "
              + ", ".join(f"{k} {v}" for k, v in oth) + " |")

    row("whole kernel", ins)
    for tgt, a in sorted(inner, key=lambda x: -(x[1] - x[0])):
        body = [i for i in ins if tgt <= i[0] <= a]
        if len(body) >= 40:
            row(f"loop 0x{tgt:x}..0x{a:x}", body)
    # straight-line blocks (no branch, no branch target inside) of 400 instructions or more that are not innermost loops
    # themselves: a fully unrolled tile evaluator has no loop of its own
    targets = set()
    for a, op, txt in ins:
        if op in ("BRA", "BSSY", "CALL", "JMP", "BRX"):
            m = re.search(r"0x([0-9a-f]+)", txt)
            if m:
                targets.add(int(m.group(1), 16))
    blocks, cur = [], []
    for i in ins:
        if i[0] in targets and cur:
            blocks.append(cur); cur = []
        cur.append(i)
        if i[1] in ("BRA", "EXIT", "RET", "BRX", "JMP", "CALL"):
            blocks.append(cur); cur = []
    if cur:
        blocks.append(cur)
    for b in sorted(blocks, key=lambda b: -len(b)):
        if len(b) >= 400 and not any(tgt <= b[0][0] and b[-1][0] <= a for tgt, a in inner):
            row(f"block 0x{b[0][0]:x}..0x{b[-1][0]:x}", b)


def table_walk_eval_split(configs):
    """tree_measure_listeval on BASELINE.json configurations: the fused walk+force kernel against the walk alone and the
    evaluation alone (two kernels, lists through global memory)."""
    import torch
    from nbody_inputs import config as make_config
    from paper_1412_0659_b200 import Tree
    print("| workload | N | fused walk+force ms | walk alone ms | evaluation alone ms | evaluation / fused | walk / fused | "
          "max rel deviation of a from the fused pass |")
    print("|---|---|---|---|---|---|---|---|")
    for k in configs:
        cfg, pos, vel, mass = make_config(k, device="cuda")
        t = Tree(device=0)
        t.build(pos, mass); t.set_velocity(vel); t.force(cfg["theta"], cfg["eps"])
        for _ in range(3):
            t.leapfrog(cfg.get("dt", 1e-3))
        fused = []
        for _ in range(3):  # a plain force pass on the current tree, scheduled by the previous pass's counts
            t.force(cfg["theta"], cfg["eps"]); fused.append(t.stats()[0]["walk"])
        w, e, dev = t.measure_listeval()
        f = min(fused)
        print(f"| {cfg['name']} | {cfg['n']:,} | {f:.3f} | {w:.3f} | {e:.3f} | {e / f:.4f} | {w / f:.4f} | {dev:.2e} |", flush=True)
        t.close()
        del pos, vel, mass
        torch.cuda.empty_cache()


def run(args) -> int:
    if args.table == "kernels":
        from nbody_inputs import CONFIGS
        table_kernels(args.from_ncu, args.n or CONFIGS[args.config]["n"])
    elif args.table == "shard-scaling":
        table_shard_scaling(args.config, [int(x) for x in args.worlds.split(",")], args.steps)
    elif args.table == "shard-weak":
        table_shard_weak(args.n or 13_000_000, [int(x) for x in args.worlds.split(",")], args.steps)
    elif args.table == "mac-sweep":
        table_mac_sweep(args.config)
    elif args.table == "walk-eval-split":
        table_walk_eval_split([int(x) for x in args.worlds.split(",")] if args.worlds != "1,2,4,8" else [2, 4])
    elif args.table == "sass-histogram":
        table_sass_histogram(args.from_sass)
    else:
        raise SystemExit(f"unknown table {args.table!r}")
    return 0
