"""Per-rank cost of the sharded force pass, measured on ONE GPU.

    python -m paper_1412_0659_b200.shard_scaling [CONFIG] [--worlds 1,2,4,8] [--steps 3]

For every world size W, W contexts on cuda:0 share the passes of a few leapfrog steps on BASELINE.json
config CONFIG (0-based; default 1).  Their kernels run one after the other, each with the whole GPU, as
they would on W GPUs, so the library's per-phase CUDA-event times of each context are the times one rank
of a W-GPU run spends; what one GPU cannot show is the cost of the peer stores over NVLink (16 bytes per
particle and peer, spread over the walk kernel) and of the barrier.  The un-permute phase is timed from the
end of the walk, which here includes the other contexts' kernels, so it is taken from the W = 1 run (the
work is the same).  Printed per W: the slowest rank's step, its parts, the cost imbalance of the
partition, and the step time of W = 1 divided by it.
"""
from __future__ import annotations

import argparse

import torch

from nbody_inputs import CONFIGS, milky_way, plummer

from .binding import Tree
from .sharded import connect_local, force_local, leapfrog_local


def measure(cfg, world: int, steps: int):
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
            own = ms["total"] - ms["unpermute"]
            per_rank.append(dict(total=own, walk=ms["walk"], sched=ms["sched"], unpermute=ms["unpermute"],
                                 rest=own - ms["walk"] - ms["sched"], groups=g_hi - g_lo,
                                 flops=23 * pp + 65 * pc))
        rows.append(per_rank)
    for t in trees:
        t.close()
    # average over steps, per rank
    avg = []
    for r in range(world):
        avg.append({k: sum(row[r][k] for row in rows) / len(rows) for k in rows[0][r]})
    return avg


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("config", nargs="?", type=int, default=1)
    ap.add_argument("--worlds", default="1,2,4,8")
    ap.add_argument("--steps", type=int, default=3)
    a = ap.parse_args()
    cfg = dict(CONFIGS[a.config])
    print(f"# sharded force pass, per-rank times on one GPU: {cfg['name']}, N = {cfg['n']:,}, theta {cfg['theta']}, "
          f"eps {cfg['eps']}, {a.steps} leapfrog steps averaged")
    print("| ranks | slowest rank: step ms | its walk ms | its build+rest ms | its task list ms | walk ms min..max over ranks "
          "| flop share max / fair | step(1) / step(W) |")
    print("|---|---|---|---|---|---|---|---|")
    base = None
    unperm = measure(cfg, 1, a.steps)[0]["unpermute"]
    for w in [int(x) for x in a.worlds.split(",")]:
        avg = measure(cfg, w, a.steps)
        for r in avg:
            r["total"] += unperm; r["rest"] += unperm
        slow = max(avg, key=lambda r: r["total"])
        if base is None:
            base = slow["total"]
        tot_flops = sum(r["flops"] for r in avg)
        share = max(r["flops"] for r in avg) / (tot_flops / w)
        walks = [r["walk"] for r in avg]
        print(f"| {w} | {slow['total']:.3f} | {slow['walk']:.3f} | {slow['rest']:.3f} | {slow['sched']:.3f} | "
              f"{min(walks):.3f} .. {max(walks):.3f} | {share:.3f} | {base / slow['total']:.2f} |")


if __name__ == "__main__":
    main()
