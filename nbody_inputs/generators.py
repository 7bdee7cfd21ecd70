"""Counter-based seeded samplers: Plummer sphere and a Milky-Way-shaped 3-component model.

Every random number is a pure function of (seed, particle index, draw number), so any
particle can be generated independently, on the CPU or on the GPU (``device=``), in any
chunking.  All sampling maths is FP64 and is rounded to FP32 once, at the end.

Workload shapes follow BASELINE.json's five configs (see ``CONFIGS``).  Component shapes of
the Milky-Way-like model follow PAPER.md L129 (NFW halo, exponential disk, Hernquist bulge);
its numbers (masses, scale lengths, truncations, particle fractions) are BASELINE.json's.
"""
from __future__ import annotations

import math
from typing import Dict, Tuple

import torch

_M64 = (1 << 64) - 1


def _s64(c: int) -> int:
    """Two's-complement view of an unsigned 64-bit constant as a Python int for torch.int64."""
    c &= _M64
    return c - (1 << 64) if c >= (1 << 63) else c


_C1 = _s64(0xBF58476D1CE4E5B9)
_C2 = _s64(0x94D049BB133111EB)
_GOLD = _s64(0x9E3779B97F4A7C15)


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical shift right on int64 tensors (torch's >> is arithmetic)."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    """splitmix64 finaliser (Steele, Lea & Flood 2014); int64 arithmetic wraps mod 2^64."""
    z = (z ^ _lsr(z, 30)) * _C1
    z = (z ^ _lsr(z, 27)) * _C2
    return z ^ _lsr(z, 31)


def uniform01(seed: int, idx: torch.Tensor, draw) -> torch.Tensor:
    """u(seed, idx, draw) in (0,1), FP64, with 32-bit resolution: (k + 0.5) / 2^32.

    ``idx`` is an int64 tensor of particle indices; ``draw`` an int or an int64 tensor.
    """
    if not torch.is_tensor(draw):
        draw = torch.full_like(idx, int(draw))
    s = torch.full_like(idx, _s64(seed * 0x9E3779B97F4A7C15 + 0x632BE59BD9B4E019))
    z = _mix(s + draw * _GOLD)
    z = _mix(z ^ (idx * _C2 + _C1))
    k = _lsr(z, 32)
    return (k.to(torch.float64) + 0.5) * (1.0 / 4294967296.0)


def _iso_direction(seed, idx, d0):
    """Isotropic unit vector from draws d0 (cos theta) and d0+1 (azimuth)."""
    ct = 2.0 * uniform01(seed, idx, d0) - 1.0
    ph = (2.0 * math.pi) * uniform01(seed, idx, d0 + 1)
    st = torch.sqrt(torch.clamp(1.0 - ct * ct, min=0.0))
    return st * torch.cos(ph), st * torch.sin(ph), ct


def plummer(n: int, seed: int, device="cpu", with_vel: bool = True):
    """Plummer sphere, G = M = a = 1, m = 1/N (BASELINE.json configs 1-2).

    Positions: X1 uniform on (0, 0.999] (mass-fraction cut, r <= 38.7), r = (X1^-2/3 - 1)^-1/2,
    isotropic direction.  Velocities: Aarseth-Henon-Wielen rejection, v_esc = sqrt2 (1+r^2)^-1/4,
    draw (X4, X5) until 0.1 X5 < X4^2 (1 - X4^2)^3.5, v = X4 v_esc, isotropic direction.
    Returns pos [n,3] f32, vel [n,3] f32 (or None), mass [n] f32.
    """
    idx = torch.arange(n, dtype=torch.int64, device=device)
    x1 = 0.999 * uniform01(seed, idx, 0)
    r = 1.0 / torch.sqrt(x1 ** (-2.0 / 3.0) - 1.0)
    dx, dy, dz = _iso_direction(seed, idx, 1)
    pos = torch.stack((r * dx, r * dy, r * dz), dim=1).to(torch.float32)
    mass = torch.full((n,), 1.0 / n, dtype=torch.float32, device=device)
    vel = None
    if with_vel:
        q = torch.zeros(n, dtype=torch.float64, device=device)
        todo = torch.ones(n, dtype=torch.bool, device=device)
        k = 0
        while bool(todo.any()):
            sel = todo.nonzero(as_tuple=True)[0]
            x4 = uniform01(seed, sel, 16 + 2 * k)
            x5 = uniform01(seed, sel, 17 + 2 * k)
            ok = 0.1 * x5 < x4 * x4 * (1.0 - x4 * x4) ** 3.5
            q[sel[ok]] = x4[ok]
            todo[sel[ok]] = False
            k += 1
            if k > 4096:
                raise RuntimeError("rejection sampler did not terminate")
        v = q * math.sqrt(2.0) * (1.0 + r * r) ** (-0.25)
        ux, uy, uz = _iso_direction(seed, idx, 3)
        vel = torch.stack((v * ux, v * uy, v * uz), dim=1).to(torch.float32)
    return pos, vel, mass


# ---- Milky-Way-shaped model (units: kpc, 1e10 Msun, G = 1) --------------------------------
MW = dict(
    disk_mass=5.0, disk_rd=2.5, disk_z0=0.3, disk_rmax=25.0,
    bulge_mass=1.0, bulge_a=0.7, bulge_rmax=10.0,
    halo_mass=80.0, halo_rs=10.0, halo_rmax=200.0,
)


def _disk_frac(x):  # enclosed-mass fraction of an exponential disk, x = R/Rd (un-normalised)
    return 1.0 - (1.0 + x) * torch.exp(-x)


def _nfw_m(x):  # NFW enclosed-mass shape, x = r/rs
    return torch.log1p(x) - x / (1.0 + x)


def _invert_monotone(f, target, lo, hi, iters=64):
    """Vectorised bisection for f(x) = target on [lo, hi]; f increasing."""
    a = torch.full_like(target, lo)
    b = torch.full_like(target, hi)
    for _ in range(iters):
        mid = 0.5 * (a + b)
        below = f(mid) < target
        a = torch.where(below, mid, a)
        b = torch.where(below, b, mid)
    return 0.5 * (a + b)


def mw_counts(n: int) -> Tuple[int, int, int]:
    """(n_disk, n_bulge, n_halo): floor(N/6), floor(N/12), rest."""
    nb = n // 12
    nd = n // 6
    return nd, nb, n - nd - nb


def _mw_menc(r):
    """Spherically averaged analytic enclosed mass of the three components at radius r."""
    p = MW
    xd = torch.clamp(r, max=p["disk_rmax"]) / p["disk_rd"]
    md = p["disk_mass"] * _disk_frac(xd) / (1.0 - (1.0 + p["disk_rmax"] / p["disk_rd"]) * math.exp(-p["disk_rmax"] / p["disk_rd"]))
    rb = torch.clamp(r, max=p["bulge_rmax"])
    fb = (p["bulge_rmax"] / (p["bulge_rmax"] + p["bulge_a"])) ** 2
    mb = p["bulge_mass"] * (rb / (rb + p["bulge_a"])) ** 2 / fb
    xh = torch.clamp(r, max=p["halo_rmax"]) / p["halo_rs"]
    xm = p["halo_rmax"] / p["halo_rs"]
    mh = p["halo_mass"] * _nfw_m(xh) / (math.log1p(xm) - xm / (1.0 + xm))
    return md + mb + mh


def milky_way(n: int, seed: int, device="cpu", with_vel: bool = True):
    """3-component Milky-Way-shaped model (BASELINE.json configs 3-5).

    Slots are ordered disk, bulge, halo in the returned arrays (not sorted in space).
    Equal particle masses inside each component: 5/n_disk, 1/n_bulge, 80/n_halo.
    Velocities are NOT an equilibrium model (BASELINE.json is silent):
    disk = circular speed tangential in the plane; bulge/halo = isotropic Gaussian with
    1-D sigma = v_c/sqrt2, speed clipped at 2 v_c.
    """
    p = MW
    nd, nb, nh = mw_counts(n)
    idx = torch.arange(n, dtype=torch.int64, device=device)
    i_d, i_b, i_h = idx[:nd], idx[nd:nd + nb], idx[nd + nb:]
    pos = torch.empty((n, 3), dtype=torch.float64, device=device)
    mass = torch.empty(n, dtype=torch.float32, device=device)

    # disk: R from the truncated exponential-disk mass fraction, z ~ sech^2(z/z0)
    xmax = p["disk_rmax"] / p["disk_rd"]
    fmax = 1.0 - (1.0 + xmax) * math.exp(-xmax)
    R = p["disk_rd"] * _invert_monotone(_disk_frac, uniform01(seed, i_d, 0) * fmax, 0.0, xmax)
    az = (2.0 * math.pi) * uniform01(seed, i_d, 1)
    uz = torch.clamp(2.0 * uniform01(seed, i_d, 2) - 1.0, -math.tanh(10.0), math.tanh(10.0))
    pos[:nd, 0] = R * torch.cos(az)
    pos[:nd, 1] = R * torch.sin(az)
    pos[:nd, 2] = p["disk_z0"] * torch.atanh(uz)
    mass[:nd] = p["disk_mass"] / max(nd, 1)

    # bulge: Hernquist, M(r)/M = r^2/(r+a)^2 truncated at rmax
    ub = uniform01(seed, i_b, 0) * (p["bulge_rmax"] / (p["bulge_rmax"] + p["bulge_a"])) ** 2
    sq = torch.sqrt(ub)
    rb = p["bulge_a"] * sq / (1.0 - sq)
    dx, dy, dz = _iso_direction(seed, i_b, 1)
    pos[nd:nd + nb, 0] = rb * dx
    pos[nd:nd + nb, 1] = rb * dy
    pos[nd:nd + nb, 2] = rb * dz
    mass[nd:nd + nb] = p["bulge_mass"] / max(nb, 1)

    # halo: NFW truncated at rmax
    xm = p["halo_rmax"] / p["halo_rs"]
    mmax = math.log1p(xm) - xm / (1.0 + xm)
    rh = p["halo_rs"] * _invert_monotone(_nfw_m, uniform01(seed, i_h, 0) * mmax, 0.0, xm)
    dx, dy, dz = _iso_direction(seed, i_h, 1)
    pos[nd + nb:, 0] = rh * dx
    pos[nd + nb:, 1] = rh * dy
    pos[nd + nb:, 2] = rh * dz
    mass[nd + nb:] = p["halo_mass"] / max(nh, 1)

    vel = None
    if with_vel:
        vel = torch.empty((n, 3), dtype=torch.float64, device=device)
        r = torch.sqrt((pos * pos).sum(dim=1))
        vc = torch.sqrt(_mw_menc(r) / torch.clamp(r, min=1e-12))
        # disk: tangential circular speed at the cylindrical radius
        Rc = torch.sqrt(pos[:nd, 0] ** 2 + pos[:nd, 1] ** 2)
        vcd = torch.sqrt(_mw_menc(Rc) / torch.clamp(Rc, min=1e-12))
        vel[:nd, 0] = -vcd * torch.sin(az)
        vel[:nd, 1] = vcd * torch.cos(az)
        vel[:nd, 2] = 0.0
        # bulge + halo: isotropic Gaussian (Box-Muller), clipped at 2 v_c
        sph = idx[nd:]
        g = []
        for c in range(3):
            u1 = uniform01(seed, sph, 8 + 2 * c)
            u2 = uniform01(seed, sph, 9 + 2 * c)
            g.append(torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2))
        g = torch.stack(g, dim=1) * (vc[nd:] / math.sqrt(2.0)).unsqueeze(1)
        sp = torch.sqrt((g * g).sum(dim=1))
        lim = 2.0 * vc[nd:]
        g = g * torch.clamp(lim / torch.clamp(sp, min=1e-30), max=1.0).unsqueeze(1)
        vel[nd:] = g
        vel = vel.to(torch.float32)
    return pos.to(torch.float32), vel, mass


def milky_way_clumpy(n: int, seed: int, n_clumps: int = 64, clump_fraction: float = 0.2,
                     clump_scale: float = 0.02, device="cpu"):
    """Milky-Way-shaped model whose disk carries compact over-densities.

    The paper reports ~10 % more work once the disk has formed bars / spiral arms;
    its evolved snapshots are not available, so structure is emulated: the first
    ``clump_fraction`` of the disk particles are moved into ``n_clumps`` Plummer clumps of scale
    radius ``clump_scale`` (kpc) centred on the positions of disk particles drawn by hash.  Masses
    are unchanged.  Exercises deep trees, leaves at the last level and the load balance of the walk.
    Returns (pos, mass); no velocities.
    """
    pos, _, mass = milky_way(n, seed, device=device, with_vel=False)
    pos = pos.to(torch.float64)
    nd, nb, nh = mw_counts(n)
    nc = int(nd * clump_fraction)
    if nc == 0 or n_clumps <= 0:
        return pos.to(torch.float32), mass
    idx = torch.arange(nc, dtype=torch.int64, device=device)
    which = torch.clamp((uniform01(seed + 101, idx, 0) * n_clumps).to(torch.int64), max=n_clumps - 1)
    host = nc + torch.clamp((uniform01(seed + 101, torch.arange(n_clumps, dtype=torch.int64, device=device), 1)
                             * (nd - nc)).to(torch.int64), max=max(nd - nc - 1, 0))
    centre = pos[host]                                    # clump centres sit on unmoved disk particles
    x1 = torch.clamp(uniform01(seed + 101, idx, 2), max=0.99)
    r = clump_scale / torch.sqrt(x1 ** (-2.0 / 3.0) - 1.0)
    dx, dy, dz = _iso_direction(seed + 101, idx, 3)
    pos[:nc, 0] = centre[which, 0] + r * dx
    pos[:nc, 1] = centre[which, 1] + r * dy
    pos[:nc, 2] = centre[which, 2] + r * dz
    return pos.to(torch.float32), mass


def subsample_indices(n: int, k: int, seed: int = 2001, device="cpu") -> torch.Tensor:
    """k distinct particle indices out of n, seeded, sorted ascending (subsample for error stats).

    Selection = the k smallest values of the per-particle hash (ties are impossible to matter:
    a stable sort breaks them by index).
    """
    k = min(k, n)
    idx = torch.arange(n, dtype=torch.int64, device=device)
    u = uniform01(seed, idx, 0)
    sel = torch.argsort(u, stable=True)[:k]
    return torch.sort(sel).values


# BASELINE.json configs, 0-based as in its list; seeds from SURVEY.md §8(d).
CONFIGS: Dict[int, dict] = {
    0: dict(name="plummer_16k", model="plummer", n=16384, seed=1001, eps=0.01, theta=0.4),
    1: dict(name="plummer_1m", model="plummer", n=1048576, seed=1002, eps=0.005, theta=0.4),
    2: dict(name="mw_8m", model="milky_way", n=8388608, seed=1003, eps=0.01, theta=0.4),
    3: dict(name="mw_134m", model="milky_way", n=134217728, seed=1004, eps=0.005, theta=0.4),
    4: dict(name="mw_33m_leapfrog", model="milky_way", n=33554432, seed=1005, eps=0.01, theta=0.4,
            dt=0.0005, steps=16),
}


def config(k: int, device="cpu", n_override: int | None = None, with_vel: bool = True):
    """Generate BASELINE.json config k (0-based). Returns (cfg dict, pos, vel, mass)."""
    cfg = dict(CONFIGS[k])
    if n_override is not None:
        cfg["n"] = int(n_override)
    fn = plummer if cfg["model"] == "plummer" else milky_way
    pos, vel, mass = fn(cfg["n"], cfg["seed"], device=device, with_vel=with_vel)
    return cfg, pos, vel, mass
