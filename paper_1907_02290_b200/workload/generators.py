"""Seeded synthetic particle distributions for the five BASELINE.json configs.

Harness code: these generators feed both the CUDA path and the CPU oracle and contain none of
the method's arithmetic.  The paper measures a
generated cold uniform sphere and names galaxy / cosmology / planetary runs only
as motivation; BASELINE.json's configs are the stand-ins.  All distributions
are textbook ones; numbers are drawn from numpy's PCG64 `default_rng(seed)` in the order written
here, generated in fp64 and rounded once to fp32 by the caller (`make_config`).  G = 1.
"""
from __future__ import annotations

import dataclasses

import numpy as np


@dataclasses.dataclass(frozen=True)
class Config:
    name: str
    n: int
    seed: int
    eps: float
    theta: float
    n_leaf: int
    n_grp: int
    kind: str              # "plummer" | "disk_halo" | "clumpy_box"
    n_reuse: int = 0       # extra evaluations that reuse the lists (config 5)
    dt: float = 0.0
    groups_per_dispatch: int = 0  # 0 = all groups in one dispatch
    eta: float = 1.2       # short-range configs: h = eta (m / rho)^(1/3)
    gamma: float = 5.0 / 3.0
    skin: float = 0.0      # neighbour lists reach 2 (1 + skin) h, so that they stay complete over the reuse steps


# BASELINE.json "configs", in order (config k is CONFIGS[k-1]).
CONFIGS = (
    Config("plummer_4k", 4096, 1, 1.0 / 64, 0.5, 8, 64, "plummer"),
    Config("plummer_1m", 1 << 20, 2, 1.0 / 256, 0.5, 16, 256, "plummer", groups_per_dispatch=256),
    Config("disk_halo_4m", 1 << 22, 3, 0.005, 0.4, 16, 512, "disk_halo"),
    Config("clumpy_box_8m", 1 << 23, 4, 1e-4, 0.5, 16, 256, "clumpy_box"),
    Config("plummer_4m_reuse", 1 << 22, 5, 1.0 / 512, 0.5, 16, 256, "plummer", n_reuse=8, dt=1.0 / 1024),
)


# Short-range (SPH) stand-ins for SURVEY.md section 8(f) NEXT-4: the paper names SPH runs and
# measures none, so these are this build's own workloads: a gas Plummer sphere with adaptive smoothing lengths.
SPH_CONFIGS = (
    Config("sph_plummer_32k", 1 << 15, 6, 0.0, 0.0, 16, 64, "sph_plummer"),
    Config("sph_plummer_1m", 1 << 20, 7, 0.0, 0.0, 16, 64, "sph_plummer", n_reuse=4, dt=1.0 / 4096, skin=0.1),
    Config("sph_plummer_4m", 1 << 22, 8, 0.0, 0.0, 16, 128, "sph_plummer", n_reuse=4, dt=1.0 / 4096, skin=0.1),
)


def _isotropic(rng: np.random.Generator, n: int) -> np.ndarray:
    ct = rng.uniform(-1.0, 1.0, n)
    ph = rng.uniform(0.0, 2.0 * np.pi, n)
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    return np.stack([st * np.cos(ph), st * np.sin(ph), ct], axis=1)


def plummer(n: int, seed: int, a: float = 1.0, mtot: float = 1.0, rcut: float = 22.8):
    """Plummer sphere by Aarseth-Henon-Wielen sampling, G = 1, equal masses mtot/n, r < rcut*a.

    Radii by inverting M(r): r = a (X^(-2/3) - 1)^(-1/2); speeds by von Neumann rejection on
    g(q) = q^2 (1 - q^2)^(7/2); shifted to zero centre of mass and zero momentum.
    Returns (pos[n,3], vel[n,3], mass[n]) in fp64.
    """
    rng = np.random.default_rng(seed)
    r = np.empty(n)
    filled = 0
    while filled < n:
        x = rng.uniform(0.0, 1.0, n - filled)
        x = x[x > 0.0]
        rr = a / np.sqrt(x ** (-2.0 / 3.0) - 1.0)
        rr = rr[rr < rcut * a]
        r[filled:filled + rr.size] = rr
        filled += rr.size
    pos = r[:, None] * _isotropic(rng, n)
    q = np.empty(n)
    filled = 0
    while filled < n:
        m = n - filled
        qq = rng.uniform(0.0, 1.0, m)
        yy = rng.uniform(0.0, 0.1, m)
        ok = yy < qq * qq * (1.0 - qq * qq) ** 3.5
        k = int(ok.sum())
        q[filled:filled + k] = qq[ok]
        filled += k
    speed = q * np.sqrt(2.0) * (1.0 + (r / a) ** 2) ** (-0.25) * np.sqrt(mtot / a)
    vel = speed[:, None] * _isotropic(rng, n)
    mass = np.full(n, mtot / n)
    pos -= pos.mean(axis=0)
    vel -= vel.mean(axis=0)
    return pos, vel, mass


def planetary_ring(n: int, seed: int, m_ring: float = 1e-6, r_in: float = 0.95, r_out: float = 1.05, h: float = 1e-4):
    """The paper's third shape ("planetary ring"; list reuse pays most here, the particles barely
    change neighbours): one central body of mass 1 at the origin (particle 0) and n - 1 equal light particles of total
    mass m_ring in a thin annulus r_in <= r < r_out (uniform in area), Gaussian thickness h x r, on circular Keplerian
    orbits (G = 1).  Not one of BASELINE.json's configs: reported beside them.  Returns (pos[n,3], vel[n,3], mass[n]) in fp64."""
    rng = np.random.default_rng(seed)
    k = n - 1
    r = np.sqrt(rng.uniform(r_in * r_in, r_out * r_out, k))
    phi = rng.uniform(0.0, 2.0 * np.pi, k)
    pos = np.zeros((n, 3))
    vel = np.zeros((n, 3))
    pos[1:, 0], pos[1:, 1], pos[1:, 2] = r * np.cos(phi), r * np.sin(phi), h * r * rng.normal(size=k)
    v = 1.0 / np.sqrt(r)
    vel[1:, 0], vel[1:, 1] = -v * np.sin(phi), v * np.cos(phi)
    mass = np.full(n, m_ring / k)
    mass[0] = 1.0
    return pos, vel, mass


def disk_halo(n: int, seed: int):
    """90% exponential disk (R_d = 1, sech^2 vertical profile, h = 0.1, total mass 0.1) plus
    10% Hernquist halo (a = 3, total mass 0.9, truncated at r = 100).  Positions only."""
    rng = np.random.default_rng(seed)
    nd = int(round(0.9 * n))
    nh = n - nd
    rr = rng.gamma(2.0, 1.0, nd)                       # surface density ~ exp(-R/R_d)
    ph = rng.uniform(0.0, 2.0 * np.pi, nd)
    u = rng.uniform(0.0, 1.0, nd)
    u = np.clip(u, 1e-12, 1.0 - 1e-12)
    z = 0.1 * np.arctanh(2.0 * u - 1.0)                 # rho(z) ~ sech^2(z/h)
    disk = np.stack([rr * np.cos(ph), rr * np.sin(ph), z], axis=1)
    a, rmax = 3.0, 100.0
    xmax = (rmax / (rmax + a)) ** 2                     # Hernquist M(<r)/M = (r/(r+a))^2
    x = rng.uniform(0.0, xmax, nh)
    s = np.sqrt(x)
    rh = a * s / (1.0 - s)
    halo = rh[:, None] * _isotropic(rng, nh)
    pos = np.concatenate([disk, halo], axis=0)
    mass = np.concatenate([np.full(nd, 0.1 / nd), np.full(nh, 0.9 / nh)])
    return pos, None, mass


def clumpy_box(n: int, seed: int, n_clump: int = 512):
    """30% uniform background in [0,1)^3 plus 70% in `n_clump` Plummer clumps: centres uniform,
    clump masses log-uniform over 2 decades, scale radii log-uniform in [0.002, 0.02], particle
    counts multinomial in clump mass, each clump cut at 10 scale radii.  Equal masses 1/n, open
    boundaries (no wrap)."""
    rng = np.random.default_rng(seed)
    nb = int(round(0.3 * n))
    nc = n - nb
    bg = rng.uniform(0.0, 1.0, (nb, 3))
    centres = rng.uniform(0.0, 1.0, (n_clump, 3))
    cm = 10.0 ** rng.uniform(0.0, 2.0, n_clump)
    radii = 10.0 ** rng.uniform(np.log10(0.002), np.log10(0.02), n_clump)
    counts = rng.multinomial(nc, cm / cm.sum())
    owner = np.repeat(np.arange(n_clump), counts)
    xmax = (10.0 ** 2 / (1.0 + 10.0 ** 2)) ** 1.5       # Plummer M(<10a)/M
    x = rng.uniform(0.0, xmax, nc)
    x = np.maximum(x, 1e-300)
    r = radii[owner] / np.sqrt(x ** (-2.0 / 3.0) - 1.0)
    cl = centres[owner] + r[:, None] * _isotropic(rng, nc)
    pos = np.concatenate([bg, cl], axis=0)
    mass = np.full(n, 1.0 / n)
    return pos, None, mass


def make_sph_fields(cfg: Config, posm: np.ndarray) -> np.ndarray:
    """[N,4] float32 (h, u, 0, 0) in the order of posm for a short-range config.  Smoothing length from the ANALYTIC
    Plummer density rho(r) = 3/(4 pi) (1 + r^2)^(-5/2) (M = a = 1): h = min(eta (m / rho)^(1/3), 1), which gives
    about (32/3) pi eta^3 = 58 neighbours inside 2h; specific internal energy u = 0.1 (1 + r^2)^(-1/2) (a hot core)."""
    r2 = np.sum(posm[:, :3].astype(np.float64) ** 2, axis=1)
    rho = 3.0 / (4.0 * np.pi) * (1.0 + r2) ** -2.5
    out = np.zeros((posm.shape[0], 4), np.float32)
    out[:, 0] = np.minimum(cfg.eta * np.cbrt(posm[:, 3].astype(np.float64) / rho), 1.0)
    out[:, 1] = 0.1 / np.sqrt(1.0 + r2)
    return out


def make_particles(cfg: Config, n: int | None = None):
    """Returns (posm float32 [n,4], vel float64 [n,3] or None) for a config; `n` overrides the
    particle count (same recipe, smaller problem) for tests."""
    n = cfg.n if n is None else int(n)
    if cfg.kind in ("plummer", "sph_plummer"):
        pos, vel, mass = plummer(n, cfg.seed)
    elif cfg.kind == "disk_halo":
        pos, vel, mass = disk_halo(n, cfg.seed)
    elif cfg.kind == "clumpy_box":
        pos, vel, mass = clumpy_box(n, cfg.seed)
    else:
        raise ValueError(cfg.kind)
    posm = np.empty((n, 4), dtype=np.float32)
    posm[:, :3] = pos
    posm[:, 3] = mass
    return posm, vel
