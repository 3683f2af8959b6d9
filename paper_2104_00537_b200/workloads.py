"""Seeded synthetic SPH workloads (input generators only).

This module serves BOTH the CUDA library (through ``sph.py``) and the CPU oracle
(through ``oracle/``) with identical inputs.  It holds none of the method's
per-step arithmetic: no kernel function, no neighbour search, no cell/offset
conversion, no interaction or update formula.  The one physical recipe it holds is
the hydrostatic initial density rho(z) = rho0 (1 + rho0 |g| depth / B)^(1/gamma) of
the column and flume inputs (reading A18), which is input data, not a step of the
path.  It imports neither the binding nor the oracle.

Every case is a stand-in for the paper's SPHERIC Test-2 dam break
(section 5.3), whose case definition and data are not available here;
the shapes follow BASELINE.json ``configs`` and SURVEY.md section 8(d).

Recipe (stated again in DESIGN.md):
  * lattice sites at (i + 1/2) * dp; boundary = 2 extra lattice layers outside
    the floor and the side walls (open top), not jittered;
  * fluid sites jittered per axis with U(-j, j) * dp drawn from a counter-based
    hash of (seed, particle index, axis), so generation is order independent;
  * everything generated on the host in float64; velocities and densities are
    rounded to float32 (the state precision of the configs).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

FLUID = 0
BOUND_FIXED = 1
BOUND_MOVING0 = 2  # first moving-boundary group id

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _splitmix64(x: np.ndarray) -> np.ndarray:
    """Counter-based hash (SplitMix64 finaliser) on uint64 arrays."""
    with np.errstate(over="ignore"):
        x = (x + np.uint64(0x9E3779B97F4A7C15)) & _M64
        z = x
        z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
        z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, index: np.ndarray, stream: int) -> np.ndarray:
    """U[0,1) doubles from (seed, index, stream); order independent."""
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        ctr = (idx * np.uint64(16) + np.uint64(stream)) & _M64
        ctr = ctr ^ _splitmix64(np.full(1, seed, dtype=np.uint64))[0]
    h = _splitmix64(ctr)
    return (h >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal01(seed: int, index: np.ndarray, stream: int) -> np.ndarray:
    """N(0,1) doubles via Box-Muller on two hashed uniforms (streams s, s+8)."""
    u1 = uniform01(seed, index, stream)
    u2 = uniform01(seed, index, stream + 8)
    u1 = np.maximum(u1, 1e-300)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * math.pi * u2)


@dataclass
class Case:
    """One workload: particle arrays + the parameters both sides receive."""

    name: str
    pos: np.ndarray   # (n, 3) float64; 2-D cases use the (x, z) plane, y = 0
    vel: np.ndarray   # (n, 3) float32
    rho: np.ndarray   # (n,)   float32
    ptype: np.ndarray  # (n,)  uint8: 0 fluid, 1 fixed boundary, >= 2 moving group
    params: dict      # keys mirror sph_params (include/sph.h)
    nsteps: int = 0
    motions: list = field(default_factory=list)  # dicts: group, axis, stroke, period, phase
    notes: str = ""
    normals: np.ndarray | None = None  # (n, 3) float64, boundary particles: vector to the boundary interface (mDBC)
    box: tuple | None = None           # ((x0, y0, z0), (x1, y1, z1)): the tank's fluid-side interface planes

    @property
    def n(self) -> int:
        return int(self.pos.shape[0])

    @property
    def n_fluid(self) -> int:
        return int((self.ptype == FLUID).sum())

    @property
    def n_bound(self) -> int:
        return self.n - self.n_fluid


def _params(dim, dp, hcoef, c0, g, domain_min, domain_max, periodic=(0, 0, 0),
            cell_div=1, cell_size=0.0, alpha=0.01, delta=0.1, cfl=0.2):
    h = hcoef * math.sqrt(dim) * dp
    return dict(dim=dim, dp=dp, h=h, rho0=1000.0, c0=c0, gamma=7.0, alpha=alpha,
                delta=delta, g=tuple(g), cfl=cfl,
                domain_min=tuple(domain_min), domain_max=tuple(domain_max),
                periodic=tuple(periodic), eta2_coef=0.001, ddt_over_boundary=0,
                rho_bound_floor=0, cell_div=cell_div, cell_size=cell_size)


def _lattice(n_sites, lo=(0, 0, 0)):
    """Integer site indices of a box, x fastest. Returns (m,3) int64."""
    nx, ny, nz = n_sites
    i = np.arange(lo[0], lo[0] + nx, dtype=np.int64)
    j = np.arange(lo[1], lo[1] + ny, dtype=np.int64)
    k = np.arange(lo[2], lo[2] + nz, dtype=np.int64)
    kk, jj, ii = np.meshgrid(k, j, i, indexing="ij")
    return np.stack([ii.ravel(), jj.ravel(), kk.ravel()], axis=1)


def dam_break(name, dim, dp, tank_sites, fluid_sites, jitter, seed, c0_height,
              cell_div=1, shuffle=False, nsteps=0, layers=2, top_factor=2.0, obstacle=None):
    """Dam break in a tank with `layers` DBC layers (floor + side walls, open top).

    dim=3: tank_sites=(nx,ny,nz), fluid block at the corner (0,0,0).
    dim=2: plane (x,z): tank_sites=(nx,1,nz), fluid_sites=(fx,1,fz); y = 0.
    obstacle = ((i0, j0, k0), (ni, nj, nk)): a box of fixed boundary particles standing on lattice sites inside
    the tank (an obstacle in the path of the wave, the shape of the paper's performance case).
    """
    nx, ny, nz = tank_sites
    L = layers
    if dim == 3:
        outer = _lattice((nx + 2 * L, ny + 2 * L, nz + L), lo=(-L, -L, -L))
        inside = ((outer[:, 0] >= 0) & (outer[:, 0] < nx) & (outer[:, 1] >= 0)
                  & (outer[:, 1] < ny) & (outer[:, 2] >= 0))
    else:
        outer = _lattice((nx + 2 * L, 1, nz + L), lo=(-L, 0, -L))
        inside = (outer[:, 0] >= 0) & (outer[:, 0] < nx) & (outer[:, 2] >= 0)
    bsites = outer[~inside]
    fsites = _lattice(fluid_sites)
    if obstacle is not None:
        (i0, j0, k0), (ni, nj, nk) = obstacle
        osites = _lattice((ni, nj if dim == 3 else 1, nk), lo=(i0, j0 if dim == 3 else 0, k0))
        bsites = np.concatenate([bsites, osites], axis=0)
        in_obs = ((fsites[:, 0] >= i0) & (fsites[:, 0] < i0 + ni) & (fsites[:, 2] >= k0) & (fsites[:, 2] < k0 + nk))
        if dim == 3:
            in_obs &= (fsites[:, 1] >= j0) & (fsites[:, 1] < j0 + nj)
        fsites = fsites[~in_obs]
    nb, nf = len(bsites), len(fsites)

    bpos = (bsites.astype(np.float64) + 0.5) * dp
    fpos = (fsites.astype(np.float64) + 0.5) * dp
    fidx = np.arange(nf)
    for ax in range(3):
        if dim == 2 and ax == 1:
            continue
        fpos[:, ax] += (2.0 * uniform01(seed, fidx, ax) - 1.0) * jitter * dp
    if dim == 2:
        bpos[:, 1] = 0.0
        fpos[:, 1] = 0.0

    pos = np.concatenate([bpos, fpos], axis=0)
    ptype = np.concatenate([np.full(nb, BOUND_FIXED, np.uint8), np.full(nf, FLUID, np.uint8)])
    n = nb + nf
    vel = np.zeros((n, 3), np.float32)
    rho = np.full(n, 1000.0, np.float32)
    if shuffle:
        perm = np.argsort(_splitmix64(np.arange(n, dtype=np.uint64) ^ np.uint64(seed * 7919 + 13)),
                          kind="stable")
        pos, vel, rho, ptype = pos[perm], vel[perm], rho[perm], ptype[perm]

    g = (0.0, 0.0, -9.81)
    c0 = 10.0 * math.sqrt(9.81 * c0_height)
    m = 4.0 * dp
    dmin = (-m, -m if dim == 3 else 0.0, -m)
    dmax = (nx * dp + m, (ny * dp + m) if dim == 3 else 0.0, top_factor * nz * dp)
    p = _params(dim, dp, 1.2, c0, g, dmin, dmax, cell_div=cell_div)
    lo, hi = (0.0, 0.0, 0.0), (nx * dp, ny * dp, nz * dp)
    normals = box_normals(pos, ptype, lo, hi, dim=dim)
    if obstacle is not None:
        (i0, j0, k0), (ni, nj, nk) = obstacle
        normals += obstacle_normals(pos, ptype, (i0 * dp, j0 * dp, k0 * dp),
                                    ((i0 + ni) * dp, (j0 + nj) * dp, (k0 + nk) * dp), lo, hi, dim=dim)
    return Case(name, np.ascontiguousarray(pos), vel, rho, ptype, p, nsteps=nsteps,
                notes=f"dam break dim={dim} dp={dp} tank={tank_sites} fluid={fluid_sites} "
                      f"jitter={jitter} seed={seed}",
                normals=normals, box=(lo, hi))


def box_normals(pos, ptype, lo, hi, dim=3, open_top=True):
    """mDBC input ("a ghost node is projected into the fluid across a boundary interface"): for every
    boundary particle, the vector from the particle to the nearest point of the box interface [lo, hi] (the planes
    half a spacing inside the innermost boundary layer; the top is open).  Pure geometry; fluid rows are 0."""
    pos = np.asarray(pos, np.float64)
    nrm = np.zeros_like(pos)
    for ax in range(3):
        if dim == 2 and ax == 1:
            continue
        x = pos[:, ax]
        below = x < lo[ax]
        above = x > hi[ax]
        nrm[below, ax] = lo[ax] - x[below]
        if not (ax == 2 and open_top):
            nrm[above, ax] = hi[ax] - x[above]
    nrm[np.asarray(ptype) == FLUID] = 0.0
    return nrm


def obstacle_normals(pos, ptype, o_lo, o_hi, lo, hi, dim=3):
    """mDBC input for a solid box obstacle [o_lo, o_hi] standing inside the tank [lo, hi]: for every boundary particle
    inside the obstacle, the vector to the nearest obstacle face that is wetted, i.e. not lying on a tank plane (the
    faces are the interface: half a spacing outside the outermost particle layer).  A tie between faces goes to the
    lower axis, then to the lower side.  Pure geometry; all other rows are 0, so the result adds to box_normals."""
    pos = np.asarray(pos, np.float64)
    nrm = np.zeros_like(pos)
    axes = [ax for ax in range(3) if not (dim == 2 and ax == 1)]
    inside = np.asarray(ptype) != FLUID
    for ax in axes:
        inside &= (pos[:, ax] > o_lo[ax]) & (pos[:, ax] < o_hi[ax])
    rows = np.flatnonzero(inside)
    best = np.full(rows.size, np.inf)
    for ax in axes:
        for face, wetted in ((o_lo[ax], o_lo[ax] > lo[ax]), (o_hi[ax], o_hi[ax] < hi[ax])):
            if not wetted:
                continue
            d = face - pos[rows, ax]
            closer = np.abs(d) < best
            best[closer] = np.abs(d[closer])
            nrm[rows[closer]] = 0.0
            nrm[rows[closer], ax] = d[closer]
    return nrm


def periodic_cloud(name, n_side, dp, jitter, seed, cell_div=1, c0=None, dim=3,
                   vel_sigma=0.05, rho_sigma=0.001):
    """Fully periodic box of n_side^dim jittered lattice sites, no boundaries (config 3)."""
    if c0 is None:
        c0 = 10.0 * math.sqrt(9.81 * 0.3)
    L = n_side * dp
    hcoef = 1.2
    h = hcoef * math.sqrt(dim) * dp
    support_cell = 2.0 * h / cell_div
    ncell = int(math.floor(L / support_cell))
    cs = L / ncell
    sites = _lattice((n_side, n_side if dim == 3 else 1, n_side))
    n = len(sites)
    idx = np.arange(n)
    pos = (sites.astype(np.float64) + 0.5) * dp
    for ax in range(3):
        if dim == 2 and ax == 1:
            pos[:, 1] = 0.0
            continue
        pos[:, ax] += (2.0 * uniform01(seed, idx, ax) - 1.0) * jitter * dp
        pos[:, ax] = np.mod(pos[:, ax], L)
        pos[:, ax] = np.where(pos[:, ax] >= L, 0.0, pos[:, ax])
    vel = np.zeros((n, 3), np.float64)
    for ax in range(3):
        if dim == 2 and ax == 1:
            continue
        vel[:, ax] = normal01(seed, idx, 3 + ax) * vel_sigma * c0
    rho = 1000.0 * (1.0 + rho_sigma * normal01(seed, idx, 6))
    per = (1, 1 if dim == 3 else 0, 1)
    dmax = (L, L if dim == 3 else 0.0, L)
    p = _params(dim, dp, hcoef, c0, (0.0, 0.0, 0.0), (0.0, 0.0, 0.0), dmax, periodic=per,
                cell_div=cell_div, cell_size=cs)
    return Case(name, np.ascontiguousarray(pos), vel.astype(np.float32), rho.astype(np.float32),
                np.zeros(n, np.uint8), p,
                notes=f"periodic cloud n_side={n_side} dim={dim} dp={dp} jitter={jitter} seed={seed}")


def random_cloud(name, n, box, dp, seed, dim=3, periodic=(0, 0, 0), frac_bound=0.2,
                 cell_div=1, vel_sigma=0.05, rho_sigma=0.01):
    """Uniform random points in a box with a mix of fluid and boundary types.

    Test-only input: irregular spacing, borderline pairs and random types exercise the
    neighbour search far harder than a lattice does.
    """
    c0 = 10.0 * math.sqrt(9.81 * 0.3)
    hcoef = 1.2
    h = hcoef * math.sqrt(dim) * dp
    idx = np.arange(n)
    pos = np.zeros((n, 3), np.float64)
    dmin = [0.0, 0.0, 0.0]
    dmax = [0.0, 0.0, 0.0]
    cs = 0.0
    support_cell = 2.0 * h / cell_div
    for ax in range(3):
        if dim == 2 and ax == 1:
            continue
        pos[:, ax] = uniform01(seed, idx, ax) * box[ax]
        dmax[ax] = box[ax]
    if any(periodic):
        # one cell size for all axes; every periodic length must be a multiple of it
        Lp = [box[ax] for ax in range(3) if periodic[ax]]
        assert all(abs(l - Lp[0]) < 1e-12 for l in Lp), "periodic axes must share a length"
        ncell = int(math.floor(Lp[0] / support_cell))
        cs = Lp[0] / ncell
    else:
        for ax in range(3):
            if dim == 2 and ax == 1:
                continue
            dmin[ax] = -0.5 * h
            dmax[ax] = box[ax] + 0.5 * h
    vel = np.zeros((n, 3), np.float64)
    for ax in range(3):
        if dim == 2 and ax == 1:
            continue
        vel[:, ax] = normal01(seed, idx, 3 + ax) * vel_sigma * c0
    rho = 1000.0 * (1.0 + rho_sigma * normal01(seed, idx, 6))
    ptype = (uniform01(seed, idx, 7) < frac_bound).astype(np.uint8)  # 1 = fixed boundary
    vel[ptype != 0] = 0.0
    p = _params(dim, dp, hcoef, c0, (0.0, 0.0, -9.81), dmin, dmax, periodic=periodic,
                cell_div=cell_div, cell_size=cs)
    return Case(name, pos, vel.astype(np.float32), rho.astype(np.float32), ptype, p,
                notes=f"random cloud n={n} box={box} dim={dim} seed={seed}")


def hydrostatic_column(name, dp, tank_sites, depth_sites, seed=77, cell_div=1, dim=3):
    """Resting water column in a DBC tank with hydrostatic initial density.

    rho(z) = rho0 * (1 + rho0*|g|*(H - z)/B)^(1/gamma), B = c0^2 rho0 / gamma.  This is an
    input recipe (initial condition), not part of the method's per-step arithmetic.
    """
    nx, ny, nz = tank_sites
    fs = (nx, ny, depth_sites)
    case = dam_break(name, dim, dp, tank_sites, fs, 0.0, seed, depth_sites * dp,
                     cell_div=cell_div)
    p = case.params
    B = p["c0"] ** 2 * p["rho0"] / p["gamma"]
    H = depth_sites * dp
    z = case.pos[:, 2]
    depth = np.clip(H - z, 0.0, None)
    rho = p["rho0"] * (1.0 + p["rho0"] * 9.81 * depth / B) ** (1.0 / p["gamma"])
    case.rho = rho.astype(np.float32)
    case.notes += " hydrostatic rho"
    return case


def wave_flume(name, dp, length, width, height, depth, seed, cell_div=1, stroke=0.1,
               period=2.0, beach_slope=1.0 / 20.0, nsteps=0):
    """3-D wave flume (config 4): DBC bed and walls, piston of moving boundary particles at
    x = 0 (group 2), 1:beach_slope beach of boundary particles at the far end, still water of
    `depth` with hydrostatic initial density (A18)."""
    L = 2
    nx = int(round(length / dp))
    ny = int(round(width / dp))
    nz = int(round(height / dp))
    nd = int(round(depth / dp))
    outer = _lattice((nx + 2 * L, ny + 2 * L, nz + L), lo=(-L, -L, -L))
    x = (outer[:, 0] + 0.5) * dp
    z = (outer[:, 2] + 0.5) * dp
    # beach: rises `depth` over the last depth/beach_slope metres
    x_toe = length - depth / beach_slope
    zb = np.where(x > x_toe, (x - x_toe) * beach_slope, 0.0)
    inside = ((outer[:, 0] >= 0) & (outer[:, 0] < nx) & (outer[:, 1] >= 0)
              & (outer[:, 1] < ny) & (outer[:, 2] >= 0))
    in_beach = inside & (z < zb)
    beach_skin = in_beach & (z >= zb - (L + 0.5) * dp)
    is_wall = ~inside
    is_piston = is_wall & (outer[:, 0] < 0)
    is_fluid = inside & ~in_beach & (outer[:, 2] < nd)
    keep_b = is_wall | beach_skin
    # walls buried under the beach are not needed
    bsites = outer[keep_b]
    btype = np.where(is_piston[keep_b], BOUND_MOVING0, BOUND_FIXED).astype(np.uint8)
    fsites = outer[is_fluid]
    nb, nf = len(bsites), len(fsites)
    bpos = (bsites.astype(np.float64) + 0.5) * dp
    fpos = (fsites.astype(np.float64) + 0.5) * dp
    fidx = np.arange(nf)
    for ax in range(3):
        fpos[:, ax] += (2.0 * uniform01(seed, fidx, ax) - 1.0) * 0.01 * dp
    pos = np.concatenate([bpos, fpos], axis=0)
    ptype = np.concatenate([btype, np.zeros(nf, np.uint8)])
    n = nb + nf
    c0 = 10.0 * math.sqrt(9.81 * depth)
    m = 4.0 * dp
    p = _params(3, dp, 1.2, c0, (0.0, 0.0, -9.81), (-m - stroke, -m, -m),
                (length + m, width + m, 1.5 * height), cell_div=cell_div)
    B = c0 ** 2 * p["rho0"] / p["gamma"]
    dpt = np.clip(depth - pos[:, 2], 0.0, None)
    rho = p["rho0"] * (1.0 + p["rho0"] * 9.81 * dpt / B) ** (1.0 / p["gamma"])
    return Case(name, np.ascontiguousarray(pos), np.zeros((n, 3), np.float32),
                rho.astype(np.float32), ptype, p, nsteps=nsteps,
                motions=[dict(group=BOUND_MOVING0, axis=0, stroke=stroke, period=period,
                              phase=0.0)],
                notes=f"wave flume dp={dp} {length}x{width}x{height} depth={depth}")


# ----------------------------------------------------------------------------------------
# BASELINE.json configs (SURVEY.md section 8(d) sizes)
# ----------------------------------------------------------------------------------------

def config(i: int, cell_div: int = 1, scale: float = 1.0) -> Case:
    """BASELINE.json configs[i]; `scale` < 1 shrinks the site counts (tests only)."""
    seed = 1234 + i
    if i == 0:
        return dam_break("cfg0_tiny_dambreak3d", 3, 0.02, (50, 25, 25), (15, 25, 15), 0.01,
                         seed, 0.3, cell_div=cell_div, nsteps=100)
    if i == 1:
        # ~1 M fluid particles needs dp = 0.0014142; 4.0 x 2.0 tank, 1.0 x 2.0 column
        dp = 0.0014142 / scale
        nx, nz = int(round(4.0 / dp)), int(round(2.0 / dp))
        fx = int(round(1.0 / dp))
        return dam_break("cfg1_dambreak2d_1M", 2, dp, (nx, 1, nz), (fx, 1, nz), 0.01, seed, 2.0,
                         cell_div=cell_div, nsteps=1000)
    if i == 2:
        dp = 0.0027 / scale
        t = (int(round(1.6 / dp)), int(round(0.67 / dp)), int(round(0.4 / dp)))
        f = (int(round(0.4 / dp)), int(round(0.67 / dp)), int(round(0.3 / dp)))
        return dam_break("cfg2_dambreak3d_4M", 3, dp, t, f, 0.01, seed, 0.3,
                         cell_div=cell_div, nsteps=1000)
    if i == 3:
        n_side = max(24, int(round(252 * scale)))
        return periodic_cloud("cfg3_periodic_cloud_16M", n_side, 0.002, 0.2, seed,
                              cell_div=cell_div)
    if i == 4:
        dp = 0.00684 / scale
        return wave_flume("cfg4_wave_flume_30M", dp, 20.0, 1.0, 1.5, 0.8, seed,
                          cell_div=cell_div, nsteps=2000)
    if i == 5:
        # not a BASELINE.json config: config 2 with a box obstacle on the floor in the path of the wave (SURVEY.md
        # 8(f) rank 4, "Test-2-shaped workload"; the dimensions are ours, the paper's case definition is not available)
        dp = 0.0027 / scale
        t = (int(round(1.6 / dp)), int(round(0.67 / dp)), int(round(0.4 / dp)))
        f = (int(round(0.4 / dp)), int(round(0.67 / dp)), int(round(0.3 / dp)))
        obs = ((int(round(0.9 / dp)), int(round(0.235 / dp)), 0),
               (max(4, int(round(0.12 / dp))), max(4, int(round(0.2 / dp))), max(4, int(round(0.12 / dp)))))
        return dam_break("cfg5_dambreak3d_obstacle", 3, dp, t, f, 0.01, seed, 0.3,
                         cell_div=cell_div, nsteps=1000, obstacle=obs)
    raise ValueError(i)
