"""Seeded synthetic particle models (the five BASELINE.json configs).

This module is the ONLY code shared by the CUDA path's tests/bench and the CPU oracle's tests.
It holds none of the method's arithmetic (no keys, no tree, no forces): it only draws positions
and masses.  The paper's own initial conditions came from the MAGI generator, which
is not available; these seed-driven spheres and the composite disk model stand in for them
(recipe: DESIGN.md "Input recipe").

All models: G = 1, total mass 1, equal masses 1/N, float64 maths -> float32 (x, y, z, m) rows.
Radii are drawn by inverse CDF of the TRUNCATED profile, directions isotropic.
"""
from __future__ import annotations

import numpy as np

__all__ = [
    "plummer", "hernquist", "nfw", "m31_like", "make_config", "CONFIGS", "random_active_subset", "isotropic_velocities", "LIVE_CONFIGS", "make_live_config", "m31_velocities",
]


def _rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(int(seed)))


def _isotropic(rng: np.random.Generator, r: np.ndarray) -> np.ndarray:
    n = r.shape[0]
    cth = rng.uniform(-1.0, 1.0, n)
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    sth = np.sqrt(np.maximum(0.0, 1.0 - cth * cth))
    return np.stack([r * sth * np.cos(phi), r * sth * np.sin(phi), r * cth], axis=1)


def _open_uniform(rng: np.random.Generator, n: int, hi: float) -> np.ndarray:
    """u in (0, hi): strictly inside so that inverse CDFs stay finite."""
    u = rng.uniform(0.0, 1.0, n)
    u = np.clip(u, 1e-15, 1.0 - 1e-15)
    return u * hi


def _r_plummer(rng, n, a=1.0, rmax=20.0):
    x = rmax / a
    m_r = x ** 3 / (1.0 + x * x) ** 1.5
    u = _open_uniform(rng, n, m_r)
    return a / np.sqrt(u ** (-2.0 / 3.0) - 1.0)


def _r_hernquist(rng, n, a=1.0, rmax=100.0):
    x = rmax / a
    m_r = (x / (1.0 + x)) ** 2
    s = np.sqrt(_open_uniform(rng, n, m_r))
    return a * s / (1.0 - s)


def _nfw_mu(x):
    return np.log1p(x) - x / (1.0 + x)


def _r_nfw(rng, n, rs=1.0, rmax=10.0):
    xmax = rmax / rs
    target = _open_uniform(rng, n, float(_nfw_mu(xmax)))
    lo = np.zeros(n)
    hi = np.full(n, xmax)
    # bisection in float64: mu is monotone on [0, xmax]; 60 halvings reach double precision
    for _ in range(60):
        mid = 0.5 * (lo + hi)
        below = _nfw_mu(mid) < target
        lo = np.where(below, mid, lo)
        hi = np.where(below, hi, mid)
    return rs * 0.5 * (lo + hi)


def _disk(rng, n, rd=1.0, zd=0.1, rmax=10.0):
    """Exponential surface density (R ~ Gamma(2, rd), truncated at rmax by rejection), sech^2 in z."""
    out_r = np.empty(n)
    filled = 0
    while filled < n:
        m = n - filled
        u1 = np.clip(rng.uniform(0.0, 1.0, m), 1e-300, 1.0)
        u2 = np.clip(rng.uniform(0.0, 1.0, m), 1e-300, 1.0)
        r = -rd * np.log(u1 * u2)
        r = r[r <= rmax]
        out_r[filled:filled + r.shape[0]] = r
        filled += r.shape[0]
    phi = rng.uniform(0.0, 2.0 * np.pi, n)
    u = np.clip(rng.uniform(0.0, 1.0, n), 1e-15, 1.0 - 1e-15)
    z = zd * np.arctanh(2.0 * u - 1.0)
    return np.stack([out_r * np.cos(phi), out_r * np.sin(phi), z], axis=1)


def _finish(rng: np.random.Generator, xyz64: np.ndarray) -> np.ndarray:
    """Cast to fp32, give every particle mass 1/N, and re-draw exact duplicate positions
    (shifted by a few fp32 ulps) so that no two particles coincide."""
    n = xyz64.shape[0]
    out = np.empty((n, 4), dtype=np.float32)
    out[:, :3] = xyz64.astype(np.float32)
    out[:, 3] = np.float32(1.0 / n)
    for _ in range(8):
        bits = out[:, :3].view(np.uint32).astype(np.uint64)
        h = (bits[:, 0] * np.uint64(0x9E3779B97F4A7C15)) ^ (bits[:, 1] * np.uint64(0xC2B2AE3D27D4EB4F)) \
            ^ (bits[:, 2] * np.uint64(0x165667B19E3779F9))
        order = np.argsort(h, kind="stable")
        hs = h[order]
        cand = np.nonzero(hs[1:] == hs[:-1])[0]
        if cand.size == 0:
            break
        a, b = order[cand], order[cand + 1]
        same = np.all(out[a, :3] == out[b, :3], axis=1)
        dup = b[same]
        if dup.size == 0:
            break
        jitter = rng.integers(1, 64, size=(dup.size, 3)).astype(np.float32)
        out[dup, :3] = out[dup, :3] + jitter * np.spacing(np.abs(out[dup, :3]) + np.float32(1e-30))
    return out


def plummer(n: int, seed: int = 1, a: float = 1.0, rmax: float = 20.0) -> np.ndarray:
    rng = _rng(seed)
    return _finish(rng, _isotropic(rng, _r_plummer(rng, n, a, rmax)))


def hernquist(n: int, seed: int = 1, a: float = 1.0, rmax: float = 100.0) -> np.ndarray:
    rng = _rng(seed)
    return _finish(rng, _isotropic(rng, _r_hernquist(rng, n, a, rmax)))


def nfw(n: int, seed: int = 1, rs: float = 1.0, rmax: float = 10.0) -> np.ndarray:
    rng = _rng(seed)
    return _finish(rng, _isotropic(rng, _r_nfw(rng, n, rs, rmax)))


def m31_like(n: int, seed: int = 1, components: bool = False):
    """NFW halo 81 % + Hernquist bulge 8 % + exponential disk 11 % by mass (BASELINE.json configs[3]);
    equal-mass particles, so the split is by count.  Scale radii in units of R_d = 1:
    halo r_s = 1.413 (cut at 10 r_s), bulge a = 0.113 (cut at 100 a), disk R_d = 1, z_d = 0.1."""
    rng = _rng(seed)
    n_bulge = int(round(0.08 * n))
    n_disk = int(round(0.11 * n))
    n_halo = n - n_bulge - n_disk
    halo = _isotropic(rng, _r_nfw(rng, n_halo, 1.413, 14.13))
    bulge = _isotropic(rng, _r_hernquist(rng, n_bulge, 0.113, 11.3))
    disk = _disk(rng, n_disk, 1.0, 0.1, 10.0)
    xyz = np.concatenate([halo, bulge, disk], axis=0)
    perm = rng.permutation(n)
    xyz = xyz[perm]
    pos_m = _finish(rng, xyz)
    if not components:
        return pos_m
    comp = np.concatenate([np.zeros(n_halo, np.uint8), np.ones(n_bulge, np.uint8), np.full(n_disk, 2, np.uint8)])[perm]
    return pos_m, comp      # component of every particle: 0 halo, 1 bulge, 2 disk (for m31_velocities)


def m31_velocities(pos_m: np.ndarray, comp: np.ndarray, seed: int = 2) -> np.ndarray:
    """Velocities (vx, vy, vz, 0) float32 for a live run of m31_like: a STAND-IN for the paper's M31 initial conditions (which come from a
    distribution-function code), good enough for orbits, level migration and tree ageing, not an equilibrium model.
    Everything is taken from the particles themselves under a spherical average (G = 1): M(<r) by sorting the radii, rho(r) from counts in
    256 logarithmic shells.  Halo and bulge particles: isotropic Gaussian with the spherical Jeans dispersion of the total profile,
    sigma^2(r) = (1/rho) int_r^inf rho M / s^2 ds.  Disk particles: the circular speed sqrt(M(<r)/r) about the z axis plus an isotropic
    Gaussian of 15 % of it (in place of the epicyclic dispersions)."""
    n = pos_m.shape[0]
    xyz = pos_m[:, :3].astype(np.float64)
    r = np.maximum(np.linalg.norm(xyz, axis=1), 1e-9)
    order = np.argsort(r, kind="stable")
    m_enc = np.empty(n)
    m_enc[order] = np.cumsum(pos_m[order, 3].astype(np.float64))
    edges = np.geomspace(max(r.min(), 1e-6), r.max() * (1 + 1e-9), 257)
    mass_in, _ = np.histogram(r, bins=edges, weights=pos_m[:, 3].astype(np.float64))
    mid = np.sqrt(edges[1:] * edges[:-1])
    rho = mass_in / (4.0 / 3.0 * np.pi * (edges[1:] ** 3 - edges[:-1] ** 3))
    m_mid = np.interp(mid, r[order], m_enc[order])
    f = rho * m_mid / mid ** 2
    seg = 0.5 * (f[1:] + f[:-1]) * np.diff(mid)
    tail = np.concatenate([np.cumsum(seg[::-1])[::-1], [0.0]])
    full = mass_in > 0                                                    # empty shells (far inside, far outside) take their neighbours' value
    sig = np.sqrt(np.interp(r, mid[full], tail[full] / rho[full]))
    rng = _rng(seed)
    vel = np.zeros((n, 4), np.float32)
    v = rng.normal(size=(n, 3)) * sig[:, None]
    disk = comp == 2
    vc = np.sqrt(m_enc[disk] / r[disk])
    R = np.maximum(np.hypot(xyz[disk, 0], xyz[disk, 1]), 1e-9)
    v[disk] = rng.normal(size=(int(disk.sum()), 3)) * (0.15 * vc)[:, None]
    v[disk, 0] += -vc * xyz[disk, 1] / R
    v[disk, 1] += vc * xyz[disk, 0] / R
    vel[:, :3] = v.astype(np.float32)
    return vel


def isotropic_velocities(pos_m: np.ndarray, model: str, seed: int = 2) -> np.ndarray:
    """Velocities (vx, vy, vz, 0) float32 for the live block-stepping runs: isotropic Gaussian with the local radial dispersion of the
    spherical Jeans equation, sigma^2(r) = (1/rho) int_r^rmax rho(s) M(<s) / s^2 ds (G = 1, total mass 1 inside the cut), integrated
    numerically on a logarithmic grid for the truncated profile.  A near-equilibrium start, not an exact distribution function:
    enough for the orbits, level migration and tree ageing of a time-to-solution measurement.  model: plummer | hernquist | nfw."""
    r = np.linalg.norm(pos_m[:, :3].astype(np.float64), axis=1)
    if model == "plummer":
        rmax, rho, mass = 20.0, (lambda x: (1.0 + x * x) ** -2.5), (lambda x: x ** 3 / (1.0 + x * x) ** 1.5)
    elif model == "hernquist":
        rmax, rho, mass = 100.0, (lambda x: 1.0 / (x * (1.0 + x) ** 3)), (lambda x: (x / (1.0 + x)) ** 2)
    elif model == "nfw":
        rmax, rho, mass = 10.0, (lambda x: 1.0 / (x * (1.0 + x) ** 2)), _nfw_mu
    else:
        raise ValueError(f"no velocity recipe for {model}")
    grid = np.geomspace(1e-6, rmax, 4096)
    f = rho(grid) * (mass(grid) / mass(rmax)) / grid ** 2
    seg = 0.5 * (f[1:] + f[:-1]) * np.diff(grid)
    tail = np.concatenate([np.cumsum(seg[::-1])[::-1], [0.0]])           # int_r^rmax
    sigma2 = tail / rho(grid)
    sig = np.sqrt(np.interp(np.clip(r, grid[0], rmax), grid, sigma2))
    rng = _rng(seed)
    vel = np.zeros((pos_m.shape[0], 4), np.float32)
    vel[:, :3] = (rng.normal(size=(pos_m.shape[0], 3)) * sig[:, None]).astype(np.float32)
    return vel


def random_active_subset(n: int, fraction: float, seed: int = 7) -> np.ndarray:
    """Ascending uint32 indices of a random subset (BASELINE.json configs[4], fixed seed)."""
    rng = _rng(seed)
    k = max(1, int(round(fraction * n)))
    if k >= n:
        return np.arange(n, dtype=np.uint32)
    idx = rng.choice(n, size=k, replace=False)
    idx.sort()
    return idx.astype(np.uint32)


# name -> (generator, N, eps, delta_acc, description) : BASELINE.json "configs" in order
CONFIGS = {
    # r_crit: critical separation for splitting wide i-groups.  The paper tunes it at run time from
    # timings (Brent's method); here it is a fixed number per workload, picked from a coarse sweep of the all-active walk time on
    # a B200 ("r_crit": NFW 0.125 ... 2, Hernquist 0.25 ... 64).  group_size: G of reading R3; a problem too
    # small to give every resident warp a group takes G = 8 (S = 4 lanes per i-particle).
    "plummer_2p13": dict(model=plummer, n=1 << 13, eps=1.0 / 64, delta_acc=2.0 ** -7, block=False, r_crit=1.0, group_size=8),
    "hernquist_2p20": dict(model=hernquist, n=1 << 20, eps=2.0 ** -7, delta_acc=2.0 ** -9, block=False, r_crit=16.0, group_size=32),
    "nfw_2p24_block": dict(model=nfw, n=1 << 24, eps=2.0 ** -8, delta_acc=2.0 ** -9, block=True, r_crit=0.5, group_size=32),
    "m31_2p24_block": dict(model=m31_like, n=1 << 24, eps=2.0 ** -8, delta_acc=2.0 ** -9, block=True, r_crit=0.5, group_size=32),
    "nfw_2p22_sweep": dict(model=nfw, n=1 << 22, eps=2.0 ** -8, delta_acc=2.0 ** -9, block=False, r_crit=0.5, group_size=32),
}


# Live block-stepping runs (moving particles): the same spheres with isotropic_velocities(); not BASELINE.json configs
# (those carry no velocities) but the workloads of the time-to-solution measurement SURVEY.md 8f row 1 asks for.
LIVE_CONFIGS = {
    "plummer_2p20_live": dict(model="plummer", n=1 << 20, eps=2.0 ** -7, delta_acc=2.0 ** -9, r_crit=1.0, group_size=32),
    "nfw_2p22_live": dict(model="nfw", n=1 << 22, eps=2.0 ** -8, delta_acc=2.0 ** -9, r_crit=0.5, group_size=32),
    "nfw_2p24_live": dict(model="nfw", n=1 << 24, eps=2.0 ** -8, delta_acc=2.0 ** -9, r_crit=0.5, group_size=32),
    # the paper's headline model under live stepping; velocities are m31_velocities' stand-in
    "m31_2p24_live": dict(model="m31_like", n=1 << 24, eps=2.0 ** -8, delta_acc=2.0 ** -9, r_crit=0.5, group_size=32),
}


def make_live_config(name: str, seed: int = 1, n: int | None = None) -> tuple[np.ndarray, np.ndarray, dict]:
    """Returns (pos_m float32 [N,4], vel float32 [N,4], parameters) of a live block-stepping workload."""
    cfg = dict(LIVE_CONFIGS[name])
    if n is not None:
        cfg["n"] = int(n)
    if cfg["model"] == "m31_like":
        pos, comp = m31_like(cfg["n"], seed, components=True)
        vel = m31_velocities(pos, comp, seed + 1000)
    else:
        pos = globals()[cfg["model"]](cfg["n"], seed)
        vel = isotropic_velocities(pos, cfg["model"], seed + 1000)
    cfg["name"] = name
    cfg["seed"] = seed
    return pos, vel, cfg


def make_config(name: str, seed: int = 1, n: int | None = None) -> tuple[np.ndarray, dict]:
    """Returns (pos_m float32 [N,4], parameters).  `n` overrides N (smaller parity-test sizes)."""
    cfg = dict(CONFIGS[name])
    if n is not None:
        cfg["n"] = int(n)
    pos = cfg["model"](cfg["n"], seed)
    cfg["name"] = name
    cfg["seed"] = seed
    return pos, cfg
