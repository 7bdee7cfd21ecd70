"""Error-versus-cost sweep: opening angle x group size x leaf size on a BASELINE
config; force error against tree_direct (FP64 direct summation on the device) on a 16,384 subsample.

    python -m paper_1412_0659_b200.sweep [config index, default 1]

Prints a markdown table.  PAPER.md fixes theta = 0.4 (L133) and notes cost ~ theta^-3 (L31)."""
import sys, os, json
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import numpy as np, torch
from paper_1412_0659_b200 import Tree
from nbody_inputs import config, subsample_indices
cfgi = int(sys.argv[1]) if len(sys.argv) > 1 else 1
cfg, pos, vel, mass = config(cfgi, device="cuda", with_vel=False)
n = cfg["n"]; eps = cfg["eps"]
idx = subsample_indices(n, 16384, device="cuda")
ad = torch.empty((idx.numel(), 3), dtype=torch.float64, device="cuda"); pd = torch.empty(idx.numel(), dtype=torch.float64, device="cuda")
acc = torch.empty((n, 3), device="cuda"); pot = torch.empty(n, device="cuda")
first = True
print("| group | leaf | theta | p-p / particle | p-c / particle | walk ms | build ms | median err | 99% err | eff. TFLOP/s |")
print("|---|---|---|---|---|---|---|---|---|---|")
for group in (32, 64, 128):
    for leaf in (8, 16, 32):
        if leaf != 16 and group != 64: continue
        t = Tree(device=0, leaf_size=leaf, group_size=group)
        t.build(pos, mass)
        if first:
            t.direct(idx, eps, ad, pd); torch.cuda.synchronize(); adn = ad.cpu().numpy(); first = False
        for theta in (0.3, 0.4, 0.5, 0.6, 0.75):
            ws = []
            for r in range(3):
                t.force(theta, eps, acc, pot); ms, pp, pc = t.stats(); ws.append(ms["walk"] + ms["sched"])
            a = acc[idx].double().cpu().numpy()
            err = np.linalg.norm(a - adn, axis=1) / np.linalg.norm(adn, axis=1)
            bms = ms["keys"] + ms["sort"] + ms["permute"] + ms["build"] + ms["moments"]
            print(f"| {group} | {leaf} | {theta} | {pp/n:.0f} | {pc/n:.0f} | {min(ws):.2f} | {bms:.2f} | {np.median(err):.2e} | {np.percentile(err,99):.2e} | {(23*pp+65*pc)/min(ws)/1e9:.1f} |", flush=True)
        t.close()
