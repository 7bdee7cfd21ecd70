"""Oracle-only experiment for SURVEY.md 8(f) NEXT-2: does a multipole acceptance criterion built on TIGHT cell
boxes (l = longest side of the bounding box of the cell's particles, delta = |c.o.m. - box centre|) shorten the
interaction lists at equal error, compared with the canonical geometric cell (S5, S6)?

    python -m oracle.mac_variants [N] [plummer|mw]

Uses only oracle/ (test infrastructure) and the seeded generators: the tight criterion is fed to the oracle's walker
through its stored delta (r_open = l_c / theta + delta', delta' = l_tight / theta + delta_tight - l_c / theta), forces are
compared with the oracle's direct summation on a seeded 4096-subsample.  Result (profiles/r1k_tight_boxes_oracle.md):
no gain, so the CUDA path keeps the geometric cell."""
import sys, os, time
sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import numpy as np
import oracle
from nbody_inputs import plummer, milky_way
n = int(sys.argv[1]) if len(sys.argv) > 1 else 65536
model = sys.argv[2] if len(sys.argv) > 2 else "plummer"
pos, _, mass = (plummer if model == "plummer" else milky_way)(n, 1002, with_vel=False)
pos, mass = pos.numpy(), mass.numpy()
eps = 0.01
rng = np.random.default_rng(1)
tg = np.sort(rng.choice(n, 4096, replace=False)).astype(np.int64)
ad, pd = oracle.direct(pos, mass, eps, tg)
ot = oracle.Tree(pos, mass)
cells = ot.cells(); mom0 = ot.moments().copy(); sp = ot.sorted_particles()
lo, hi, org, k = ot.grid()
first = cells[:, 1]; cnt = cells[:, 2]; lev = cells[:, 0]
# tight boxes from particle ranges: cells sorted BFS; use per-cell slicing via reduceat on (first) needs sorted starts -> do loop by level
bmin = np.empty((len(cells), 3), np.float32); bmax = np.empty((len(cells), 3), np.float32)
order = np.argsort(first, kind="stable")
for c in range(len(cells)):
    s = sp[first[c]:first[c] + cnt[c], :3]
    bmin[c] = s.min(0); bmax[c] = s.max(0)
lt = (bmax - bmin).max(1).astype(np.float32)
ctr = 0.5 * (bmax.astype(np.float64) + bmin)
dt_ = np.linalg.norm(mom0[:, 1:4].astype(np.float64) - ctr, axis=1).astype(np.float32)
lc = np.ldexp(1.0, (int(k) - lev)).astype(np.float32)
def run(theta, tight):
    m = mom0.copy()
    if tight:
        th = np.float32(theta)
        m[:, 10] = (lt / th + dt_) - lc / th
    ot.set_moments(m)
    a, p, npp, npc = ot.force(theta, eps)
    rel = np.linalg.norm(a[tg] - ad, axis=1) / np.linalg.norm(ad, axis=1)
    cost = 13.0 * npp.sum() + 37.0 * npc.sum()
    return npp.mean(), npc.mean(), cost / len(npp), np.median(rel), np.percentile(rel, 99)
print("mac theta pp pc cost med99")
for tight in (0, 1):
    for theta in ([0.3, 0.4, 0.5, 0.6, 0.75] if not tight else [0.2, 0.25, 0.3, 0.35, 0.4, 0.5, 0.6]):
        r = run(theta, tight)
        print("tight" if tight else "geom ", theta, "pp %.0f pc %.0f cost %.0f  med %.2e p99 %.2e" % r, flush=True)
