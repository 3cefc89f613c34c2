"""Seeded synthetic inputs shaped like the paper's workloads (configs C1-C5 of BASELINE.json).

This module holds NO lattice-Boltzmann arithmetic: it only builds density, velocity and
solid-mask fields.  It is the one module that both the CUDA path's callers (tests, bench.py)
and the oracle's callers use, so that both sides see bit-identical fp32 inputs.

The paper's own initial fields and device geometry are not published (PAPER.md:207-227,
Fig. 4; Fig. 7); these recipes stand in for them (DESIGN.md
"Input recipe").  Generator: numpy Generator(PCG64(200512764 + config index)); fields are
evaluated in fp64 and rounded once to fp32.

Layout: scalar fields [nz, ny, nx] (x fastest), u [3, nz, ny, nx], mask uint8 (1 = solid).
"""
from __future__ import annotations

import dataclasses

import numpy as np

SEED0 = 200512764


@dataclasses.dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    tau_r: float
    tau_b: float
    A: float
    beta: float
    A_nc: float
    rho_r: np.ndarray
    rho_b: np.ndarray | None          # None = single component
    u: np.ndarray
    solid: np.ndarray | None = None   # uint8, 1 = solid
    g: tuple = (0.0, 0.0, 0.0)
    phi_c: float = 0.9
    steps: int = 100                  # steps the config asks for
    info: dict = dataclasses.field(default_factory=dict)

    @property
    def shape(self):
        return (self.nz, self.ny, self.nx)

    @property
    def sites(self):
        return self.nx * self.ny * self.nz

    @property
    def fluid_sites(self):
        return self.sites if self.solid is None else int((self.solid == 0).sum())    # wall groups are 2, 3, 4: count, do not sum

    @property
    def params(self):
        return (self.tau_r, self.tau_b, self.A, self.beta, self.A_nc)


def _rng(index):
    return np.random.Generator(np.random.PCG64(SEED0 + index))


def _paint_droplets(phi, centres, radii, periodic=(True, True, True), reach=18.0):
    """phi <- max(phi, tanh((R_j - r_j)/2)) for every droplet, touching only a local box.

    Beyond R + reach the profile equals -1 to fp32 rounding (tanh(-9) = -1 + 3e-8)."""
    nz, ny, nx = phi.shape
    dims = (nx, ny, nz)
    for (cx, cy, cz), R in zip(centres, radii):
        idx, dist = [], []
        for a, c in enumerate((cx, cy, cz)):
            lo = int(np.floor(c - R - reach))
            hi = int(np.ceil(c + R + reach)) + 1
            n = dims[a]
            if hi - lo >= n:
                lo, hi = 0, n
                j = np.arange(lo, hi)
                d = np.abs(j - c)
                if periodic[a]:
                    d = np.minimum(d, n - d)
                idx.append(j)
                dist.append(d)
                continue
            j = np.arange(lo, hi)
            d = np.abs(j - c)
            if periodic[a]:
                j = j % n
            else:
                keep = (j >= 0) & (j < n)
                j, d = j[keep], d[keep]
            idx.append(j)
            dist.append(d)
        r = np.sqrt(dist[2][:, None, None] ** 2 + dist[1][None, :, None] ** 2 + dist[0][None, None, :] ** 2)
        val = np.tanh((R - r) / 2.0).astype(np.float32)
        sel = np.ix_(idx[2], idx[1], idx[0])
        phi[sel] = np.maximum(phi[sel], val)
    return phi


def _from_phi(phi):
    """rho_r = (1 + phi)/2, rho_b = (1 - phi)/2 evaluated in fp64, rounded once."""
    p = phi.astype(np.float64)
    return ((1.0 + p) / 2.0).astype(np.float32), ((1.0 - p) / 2.0).astype(np.float32)


def c1_droplet(n=32, R=8.0):
    """C1: one red droplet of radius 8 centred in a 32^3 periodic blue box (Laplace test)."""
    c = (n - 1) / 2.0
    phi = np.full((n, n, n), -1.0, np.float32)
    _paint_droplets(phi, [(c, c, c)], [R], reach=float(n))
    rr, rb = _from_phi(phi)
    return Workload("C1-droplet", n, n, n, 1.0, 1.0, 0.01, 0.7, 0.0, rr, rb,
                    np.zeros((3, n, n, n), np.float32), steps=100, info=dict(R=R))


def c2_taylor_green(n=256, tau=0.6, U0=0.02, steps=1000):
    """C2: single-component Taylor-Green vortex, arguments 2 pi x/n (G19)."""
    a = 2.0 * np.pi * np.arange(n) / n
    sx, cx = np.sin(a)[None, None, :], np.cos(a)[None, None, :]
    sy, cy = np.sin(a)[None, :, None], np.cos(a)[None, :, None]
    cz = np.cos(a)[:, None, None]
    u = np.zeros((3, n, n, n), np.float32)
    u[0] = (U0 * sx * cy * cz).astype(np.float32)
    u[1] = (-U0 * cx * sy * cz).astype(np.float32)
    return Workload("C2-taylor-green", n, n, n, tau, tau, 0.0, 0.0, 0.0,
                    np.ones((n, n, n), np.float32), None, u, steps=steps, info=dict(U0=U0))


def c3_spinodal(n=256, steps=5000, index=2):
    """C3: bicontinuous spinodal mixture, one draw xi per site so that rho = 1 exactly (G14)."""
    xi = _rng(index).uniform(-1.0, 1.0, size=(n, n, n))
    rr = (0.5 + 0.05 * xi).astype(np.float32)
    rb = (0.5 - 0.05 * xi).astype(np.float32)
    return Workload("C3-spinodal", n, n, n, 1.0, 1.0, 0.01, 0.7, 0.0, rr, rb,
                    np.zeros((3, n, n, n), np.float32), steps=steps)


def _fcc_centres(dims, d, R, rng, wall_axes):
    """FCC lattice of nearest-neighbour distance d: points (i, j, k) d/sqrt 2 with i+j+k even.
    Along periodic axes the spacing is stretched so that an even number of half-cells fits;
    along walled axes the lattice is centred between the planes R + 2 (+ the half-link wall
    offset) away from the walls, so no kept centre is closer than R + 2 to a wall.  Each
    centre is then jittered by U(-0.5, 0.5)^3."""
    half = d / np.sqrt(2.0)
    axes = []
    for ax in range(3):
        n = dims[ax]
        if ax in wall_axes:
            lo, hi = 0.5 + R + 2 + 0.5, n - 1.5 - R - 2 - 0.5      # room for the jitter
            m = int(np.floor((hi - lo) / half))
            axes.append(lo + ((hi - lo) - m * half) / 2.0 + half * np.arange(m + 1))
        else:
            m = max(2, 2 * int(round(n / half / 2.0)))
            axes.append((n / m) * np.arange(m))
    I, J, K = np.meshgrid(*(np.arange(len(a)) for a in axes), indexing="ij")
    keep = (I + J + K) % 2 == 0
    out = np.stack([axes[0][I[keep]], axes[1][J[keep]], axes[2][K[keep]]], axis=1)
    return out + rng.uniform(-0.5, 0.5, size=out.shape)


def c4_channel(nx=512, ny=128, nz=128, R=10.0, target=0.60, steps=10000, index=3):
    """C4: microfluidic-crystal channel, bounce-back walls at y and z faces, periodic in x,
    body force g_x = 1e-6, jittered FCC lattice of red droplets, near-contact force on.
    d is bisected (lower bound 2R + 1) towards a dispersed fraction `target`; the achieved
    fraction is reported in info."""
    z, y = np.arange(nz)[:, None, None], np.arange(ny)[None, :, None]
    solid = np.broadcast_to((y == 0) | (y == ny - 1) | (z == 0) | (z == nz - 1), (nz, ny, nx)).astype(np.uint8)
    fluid = solid == 0

    def build(d):
        centres = _fcc_centres((nx, ny, nz), d, R, _rng(index), wall_axes=(1, 2))
        phi = np.full((nz, ny, nx), -1.0, np.float32)
        _paint_droplets(phi, centres, [R] * len(centres), periodic=(True, False, False))
        frac = float(((1.0 + phi[fluid].astype(np.float64)) / 2.0).mean())
        return phi, frac, len(centres)

    lo, hi = 2 * R + 1.0, 4 * R
    d = lo
    phi, frac, nd = build(d)
    if frac > target + 0.01:                      # otherwise the densest allowed lattice is it
        for _ in range(10):
            d = 0.5 * (lo + hi)
            phi, frac, nd = build(d)
            if abs(frac - target) <= 0.01:
                break
            if frac < target:
                hi = d
            else:
                lo = d
    rr, rb = _from_phi(phi)
    rr[~fluid] = 0
    rb[~fluid] = 0
    return Workload("C4-channel", nx, ny, nz, 1.0, 1.0, 0.01, 0.7, 0.02, rr, rb,
                    np.zeros((3, nz, ny, nx), np.float32), solid=solid, g=(1e-6, 0.0, 0.0),
                    steps=steps, info=dict(d=d, droplets=nd, dispersed_fraction=frac, R=R))


def c5_emulsion(n=640, ndrops=3000, rmin=8.0, rmax=14.0, gap=3.0, steps=1000, index=4):
    """C5: dense emulsion, seeded random sequential addition of non-overlapping red droplets
    with radii U[rmin, rmax] (minimum-image centre distance >= R_i + R_j + gap)."""
    rng = _rng(index)
    centres = np.zeros((0, 3))
    radii = np.zeros(0)
    tries = 0
    while len(radii) < ndrops and tries < 200 * ndrops:
        tries += 1
        c = rng.uniform(0.0, n, size=3)
        R = rng.uniform(rmin, rmax)
        if len(radii):
            dlt = np.abs(centres - c)
            dlt = np.minimum(dlt, n - dlt)
            if (np.sqrt((dlt ** 2).sum(1)) < radii + R + gap).any():
                continue
        centres = np.vstack([centres, c])
        radii = np.append(radii, R)
    phi = np.full((n, n, n), -1.0, np.float32)
    _paint_droplets(phi, centres, radii)
    rr, rb = _from_phi(phi)
    frac = float(rr.mean(dtype=np.float64))
    return Workload("C5-emulsion", n, n, n, 1.0, 1.0, 0.01, 0.7, 0.02, rr, rb,
                    np.zeros((3, n, n, n), np.float32), steps=steps,
                    info=dict(droplets=int(len(radii)), red_fraction=frac))


def focuser(nx=96, ny=48, nz=1, wd=10, wc=12, t=4, li=24, wo=10, lo=8, u_d=0.01, u_c=0.01,
            tau=1.0, A=0.01, beta=0.7, A_nc=0.0, walls_z=False, steps=2000):
    """Flow-focusing device (Fig. 4): a dispersed (red) inlet of width wd between
    two continuous (blue) inlets of width wc, all on the x = 0 plane and kept apart by dividers of
    thickness t and length li, an orifice of width wo and length lo behind the junction, and an
    outlet chamber that ends in a pressure outlet on the x = nx-1 plane.  alpha = u_d / (2 u_c) as
    in the paper.  The device dimensions are NOT in the paper: these are stand-ins.

    Mask values: 1 wall at rest, 2 dispersed inlet, 3 continuous inlets, 4 outlet; what the groups
    are is in info["wall_groups"] and set on an Oracle or an LB by configure_walls()."""
    solid = np.zeros((nz, ny, nx), np.uint8)
    solid[:, 0, :] = 1
    solid[:, -1, :] = 1
    if walls_z:
        solid[0] = 1
        solid[-1] = 1
    y0d = (ny - wd) // 2
    y1d = y0d + wd
    solid[:, y0d - t:y0d, :li] = 1
    solid[:, y1d:y1d + t, :li] = 1
    # the continuous inlets reach from the dividers wc sites outwards, the rest of the face is wall
    lo_c, hi_c = max(1, y0d - t - wc), min(ny - 1, y1d + t + wc)
    solid[:, 1:lo_c, :li] = 1
    solid[:, hi_c:ny - 1, :li] = 1
    xo = li + max(wd, wc)
    y0o = (ny - wo) // 2
    solid[:, 1:y0o, xo:xo + lo] = 1
    solid[:, y0o + wo:ny - 1, xo:xo + lo] = 1
    face = solid[:, :, 0] == 0
    yy = np.broadcast_to(np.arange(ny)[None, :], (nz, ny))
    solid[:, :, 0] = np.where(face, np.where((yy >= y0d) & (yy < y1d), 2, 3), solid[:, :, 0])
    solid[:, :, -1] = np.where(solid[:, :, -1] == 0, 4, solid[:, :, -1])
    # red fills the dispersed channel up to the junction, blue everything else
    x = np.arange(nx, dtype=np.float64)[None, None, :]
    y = np.arange(ny, dtype=np.float64)[None, :, None]
    phi = np.tanh((li - 2.0 - x) / 2.0) * np.ones((nz, 1, 1))
    phi = np.where((y >= y0d) & (y < y1d), phi, -1.0)
    rr, rb = _from_phi(phi.astype(np.float32))
    walls = {2: dict(kind="inlet", u=(u_d, 0.0, 0.0), rho=(1.0, 0.0)),
             3: dict(kind="inlet", u=(u_c, 0.0, 0.0), rho=(0.0, 1.0)),
             4: dict(kind="outlet", u=(0.0, 0.0, 0.0), rho=(0.5, 0.5))}
    return Workload("focuser", nx, ny, nz, tau, tau, A, beta, A_nc, rr, rb,
                    np.zeros((3, nz, ny, nx), np.float32), solid=solid, steps=steps,
                    info=dict(alpha=u_d / (2.0 * u_c), wall_groups=walls, li=li, xo=xo, wd=wd, wc=wc))


def bijel(n=256, fraction=0.01, R=5.5, density=1.0, steps=2000, index=5):
    """Colloids in a phase-separating mixture (the paper's section 6 and Fig. 6-7, PAPER.md:286-351:
    "rigid colloids (of radius R = 5.5 lu) in a bicontinuous fluid"; the phi = 1 % rows of Fig. 6 are a
    1024^3 box with 15 407 colloids): the C3 spinodal mixture plus N = 3 fraction / (4 pi) (n / R)^3
     neutrally wetting spheres placed by seeded random sequential addition (gap >= 3
    lattice units, minimum image), at rest, neutrally buoyant by default; pair repulsion and
    lubrication on.  Positions only: no LB arithmetic here."""
    w = c3_spinodal(n, steps=steps, index=index)
    rng = _rng(index + 100)
    N = max(1, int(round(3.0 * fraction / (4.0 * np.pi) * (n / R) ** 3)))
    centres = np.zeros((0, 3))
    tries = 0
    while len(centres) < N and tries < 500 * N:
        tries += 1
        c = rng.uniform(0.0, n, size=3)
        if len(centres):
            d = np.abs(centres - c)
            d = np.minimum(d, n - d)
            if (np.sqrt((d ** 2).sum(1)) < 2 * R + 3.0).any():
                continue
        centres = np.vstack([centres, c])
    m = density * 4.0 / 3.0 * np.pi * R ** 3
    state = np.zeros((len(centres), 15))
    state[:, 0:3] = centres
    state[:, 9] = 1.0
    state[:, 13] = R
    state[:, 14] = m
    w.name = "bijel"
    w.info.update(particles=state, particle_options=dict(mobile=True, K=0.02, h_c=2.0, lubrication=True),
                  colloids=int(len(centres)), colloid_volume_fraction=float(len(centres) * 4.0 / 3.0 * np.pi * R ** 3 / n ** 3))
    return w


def configure_walls(obj, w):
    """Apply what a workload carries besides its fields to an oracle or an LB (same method names on
    both): info["wall_groups"] (velocities, open boundaries) and info["particles"] (rigid colloids)."""
    for group, d in sorted(w.info.get("wall_groups", {}).items()):
        obj.set_wall_velocity(group, *d["u"])
        obj.set_wall_type(group, d["kind"], *d["rho"])
    if "particles" in w.info:
        obj.set_particles(w.info["particles"])
        obj.set_particle_options(**w.info["particle_options"])


def get(name):
    """Workloads by name: full configs c1..c5 and the parity minis."""
    table = {
        "c1": c1_droplet,
        "c2": c2_taylor_green,
        "c3": c3_spinodal,
        "c4": c4_channel,
        "c5": c5_emulsion,
        "c2-mini": lambda: c2_taylor_green(64, steps=100),
        "c3-mini": lambda: c3_spinodal(64, steps=100),
        "c4-mini": lambda: c4_channel(128, 32, 32, R=6.0, steps=100),
        "c5-mini": lambda: c5_emulsion(96, 8, steps=100),
        "bijel": bijel,
        "bijel-mini": lambda: bijel(48, fraction=0.02, R=4.5, density=2.0, steps=100),
        "focuser": focuser,
        "focuser-3d": lambda: focuser(256, 96, 48, wd=20, wc=24, t=6, li=48, wo=20, lo=16, walls_z=True,
                                      A_nc=0.02, steps=20000),
        "focuser-large": lambda: focuser(1024, 256, 128, wd=56, wc=64, t=16, li=128, wo=40, lo=48, walls_z=True,
                                         A_nc=0.02, steps=20000),
        # dripping regime (Ca = rho nu u_c / sigma = 0.125 with sigma = 4 A tau / 9): droplets pinch off behind the orifice
        "focuser-drip": lambda: focuser(256, 96, 48, wd=20, wc=24, t=6, li=48, wo=14, lo=16, u_d=0.006, u_c=0.02,
                                        A=0.06, A_nc=0.02, walls_z=True, steps=36000),
    }
    return table[name]()
