"""Seeded synthetic scene generators (inputs only).

This module is the ONE piece shared by the CUDA path and the CPU oracle: it
produces the fp32 input arrays (particle positions, velocities, boundary
samples, rigid-body descriptors) and the parameter dictionary of a scene.  It
holds none of the method's arithmetic: no SPH kernel, no neighbour search, no
Akinci volumes, no solver.  (Rigid-body mass / inertia are analytic solid
formulas of the scene description, not part of the SPH method.)

Scene conventions follow SURVEY.md section 8(d):
  * z is up, gravity g = (0, 0, -9.81);
  * one global lattice of spacing s = 2r, lattice site i sits at (i + 1/2) s;
  * the tank interior is the box of sites [0, n_a) per axis (nominal size
    n_a * s); the walls are the two site layers outside every face (closed
    box, edges and corners included), each layer pushed outward by 0.1 s along
    every axis in which it lies outside (reading R25);
  * fluid blocks are boxes of sites with a given initial velocity;
  * obstacles / rigid bodies are sampled on their surface at spacing s;
  * RNG: numpy.random.default_rng(seed).

The paper's own scenes (1.23M-particle splash on dragon
meshes, nine rigid bodies in a box, mu = 13000 column) are artist assets that
are not available; these procedural scenes stand in for them with the paper's
r, h = 4r, rho0 = 1000 kg/m^3 and BASELINE.json's configs.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

WALL_LAYERS = 2
WALL_SHIFT = 0.1  # in units of s, reading R25


@dataclass
class Body:
    """One rigid body = one contiguous range of boundary samples."""

    first_particle: int
    n_particles: int
    dynamic: int = 0
    mass: float = 0.0
    inertia_body: Tuple[float, float, float] = (1.0, 1.0, 1.0)
    com: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    quat: Tuple[float, float, float, float] = (1.0, 0.0, 0.0, 0.0)  # w, x, y, z
    lin_vel: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    ang_vel: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    contact_radius: float = 0.0


@dataclass
class Scene:
    name: str
    fluid_pos: np.ndarray       # (N_f, 3) float32
    fluid_vel: np.ndarray       # (N_f, 3) float32
    boundary_pos: np.ndarray    # (N_b, 3) float32, world coordinates at t = 0
    boundary_body: np.ndarray   # (N_b,) int32, index into bodies
    bodies: List[Body]
    params: Dict[str, object]   # keys mirror SphParams in include/sph.h
    steps: int = 1
    fluid_height: float = 1.0   # H in the velocity tolerance floor sqrt(|g| H)

    @property
    def n_fluid(self) -> int:
        return int(self.fluid_pos.shape[0])

    @property
    def n_boundary(self) -> int:
        return int(self.boundary_pos.shape[0])


# --------------------------------------------------------------------------
# lattice helpers
# --------------------------------------------------------------------------

def _site_coords(lo: int, hi: int, s: float) -> np.ndarray:
    return (np.arange(lo, hi, dtype=np.float64) + 0.5) * s


def block_sites(lo: Sequence[int], n: Sequence[int], s: float) -> np.ndarray:
    """All lattice sites of the box [lo, lo + n) as float64 coordinates, x fastest."""
    xs = _site_coords(lo[0], lo[0] + n[0], s)
    ys = _site_coords(lo[1], lo[1] + n[1], s)
    zs = _site_coords(lo[2], lo[2] + n[2], s)
    z, y, x = np.meshgrid(zs, ys, xs, indexing="ij")
    return np.stack([x.ravel(), y.ravel(), z.ravel()], axis=1)


def tank_walls(n_sites: Sequence[int], s: float, layers: int = WALL_LAYERS,
               shift: float = WALL_SHIFT) -> np.ndarray:
    """Closed box shell: `layers` site layers outside every face of [0, n_a)."""
    L = layers
    idx = [np.arange(-L, n + L) for n in n_sites]
    k, j, i = np.meshgrid(idx[2], idx[1], idx[0], indexing="ij")
    ijk = np.stack([i.ravel(), j.ravel(), k.ravel()], axis=1)
    n = np.asarray(n_sites)
    outside = (ijk < 0) | (ijk >= n)
    ijk = ijk[outside.any(axis=1)]
    pos = (ijk.astype(np.float64) + 0.5) * s
    # push outward along every axis in which the site lies outside (R25)
    pos += np.where(ijk < 0, -shift * s, 0.0)
    pos += np.where(ijk >= n, shift * s, 0.0)
    return pos


def box_shell(center: Sequence[float], size: Sequence[float], s: float) -> np.ndarray:
    """Surface lattice of an axis-aligned box: n_a = round(size_a / s) + 1 points per edge."""
    n = [int(round(size[a] / s)) + 1 for a in range(3)]
    ax = [np.linspace(-0.5 * size[a], 0.5 * size[a], n[a]) for a in range(3)]
    k, j, i = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    i, j, k = i.ravel(), j.ravel(), k.ravel()
    surf = (i == 0) | (i == n[0] - 1) | (j == 0) | (j == n[1] - 1) | (k == 0) | (k == n[2] - 1)
    p = np.stack([ax[0][i[surf]], ax[1][j[surf]], ax[2][k[surf]]], axis=1)
    return p + np.asarray(center, dtype=np.float64)


def sphere_shell(center: Sequence[float], radius: float, s: float) -> np.ndarray:
    """Fibonacci points, N = round(4 pi R^2 / s^2)."""
    n = int(round(4.0 * np.pi * radius * radius / (s * s)))
    k = np.arange(n, dtype=np.float64) + 0.5
    z = 1.0 - 2.0 * k / n
    phi = k * np.pi * (3.0 - np.sqrt(5.0))
    rxy = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    p = radius * np.stack([rxy * np.cos(phi), rxy * np.sin(phi), z], axis=1)
    return p + np.asarray(center, dtype=np.float64)


def cylinder_shell(center: Sequence[float], radius: float, height: float, s: float) -> np.ndarray:
    """Vertical cylinder: lateral rings at spacing s plus two caps of concentric rings."""
    nz = int(round(height / s)) + 1
    zs = np.linspace(-0.5 * height, 0.5 * height, nz)
    nphi = max(8, int(round(2.0 * np.pi * radius / s)))
    phi = 2.0 * np.pi * np.arange(nphi) / nphi
    ring = np.stack([radius * np.cos(phi), radius * np.sin(phi)], axis=1)
    lateral = np.concatenate([np.concatenate([ring, np.full((nphi, 1), z)], axis=1) for z in zs])
    caps = []
    nr = int(np.floor((radius - 0.5 * s) / s))
    for zc in (zs[0], zs[-1]):
        pts = [np.array([[0.0, 0.0, zc]])]
        for ir in range(1, nr + 1):
            rr = ir * s
            m = max(6, int(round(2.0 * np.pi * rr / s)))
            ph = 2.0 * np.pi * np.arange(m) / m
            pts.append(np.stack([rr * np.cos(ph), rr * np.sin(ph), np.full(m, zc)], axis=1))
        caps.append(np.concatenate(pts))
    p = np.concatenate([lateral] + caps)
    return p + np.asarray(center, dtype=np.float64)


# --------------------------------------------------------------------------
# scene assembly
# --------------------------------------------------------------------------

def default_params(r: float, dt: float) -> Dict[str, object]:
    """Parameter dictionary mirroring SphParams (include/sph.h)."""
    return dict(
        particle_radius=float(r),
        support_radius=float(4.0 * r),        # h = 4r
        rest_density=1000.0,
        particle_mass=0.0,                    # 0 => rho0 (2r)^3, reading R3
        dt=float(dt),
        gravity=(0.0, 0.0, -9.81),
        domain_min=(0.0, 0.0, 0.0),
        domain_max=(1.0, 1.0, 1.0),
        tank_min=(0.0, 0.0, 0.0),
        tank_max=(1.0, 1.0, 1.0),
        viscosity_mode=0,
        kinematic_viscosity=0.0,
        cg_rel_tol=1e-5,
        cg_max_iter=500,
        eta_density=1e-3,
        min_iter_density=2,
        max_iter_density=100,
        eta_divergence=1e-2,
        min_iter_divergence=1,
        max_iter_divergence=100,
        enable_divergence_solve=1,
        force_iterations=0,
        wcsph_stiffness=50000.0,
        wcsph_exponent=7.0,
        cfl_factor=0.0,                       # 0 => fixed dt (all BASELINE configs); > 0: CFL-adaptive dt, reading R26
        dt_min=0.0,
    )


def _finish(name: str, r: float, dt: float, tank_sites: Optional[Sequence[int]],
            fluid: List[Tuple[np.ndarray, Sequence[float]]],
            extra_bodies: List[Tuple[np.ndarray, Body]],
            steps: int, fluid_height: float, **overrides) -> Scene:
    s = 2.0 * r
    h = 4.0 * r
    fpos = np.concatenate([p for p, _ in fluid]) if fluid else np.zeros((0, 3))
    fvel = np.concatenate([np.broadcast_to(np.asarray(v, dtype=np.float64), p.shape)
                           for p, v in fluid]) if fluid else np.zeros((0, 3))
    bpos_list, bbody_list, bodies = [], [], []
    first = 0
    if tank_sites is not None:
        w = tank_walls(tank_sites, s)
        bpos_list.append(w)
        bbody_list.append(np.zeros(len(w), dtype=np.int32))
        bodies.append(Body(first_particle=0, n_particles=len(w), dynamic=0))
        first = len(w)
    for pts, body in extra_bodies:
        body.first_particle = first
        body.n_particles = len(pts)
        bpos_list.append(pts)
        bbody_list.append(np.full(len(pts), len(bodies), dtype=np.int32))
        bodies.append(body)
        first += len(pts)
    bpos = np.concatenate(bpos_list) if bpos_list else np.zeros((0, 3))
    bbody = np.concatenate(bbody_list) if bbody_list else np.zeros((0,), dtype=np.int32)

    prm = default_params(r, dt)
    allp = np.concatenate([fpos, bpos]) if len(bpos) else fpos
    if tank_sites is not None:
        tmin = np.zeros(3)
        tmax = np.asarray(tank_sites, dtype=np.float64) * s
        prm["tank_min"] = tuple(float(v) for v in tmin)
        prm["tank_max"] = tuple(float(v) for v in tmax)
        lo = np.minimum(allp.min(axis=0), tmin) - h
        hi = np.maximum(allp.max(axis=0), tmax) + h
    else:
        lo = allp.min(axis=0) - 2.0 * h
        hi = allp.max(axis=0) + 2.0 * h
        prm["tank_min"] = tuple(float(v) for v in lo)
        prm["tank_max"] = tuple(float(v) for v in hi)
    prm["domain_min"] = tuple(float(np.float32(v)) for v in lo)
    prm["domain_max"] = tuple(float(np.float32(v)) for v in hi)
    prm.update(overrides)
    return Scene(
        name=name,
        fluid_pos=np.ascontiguousarray(fpos, dtype=np.float32),
        fluid_vel=np.ascontiguousarray(fvel, dtype=np.float32),
        boundary_pos=np.ascontiguousarray(bpos, dtype=np.float32),
        boundary_body=np.ascontiguousarray(bbody, dtype=np.int32),
        bodies=bodies, params=prm, steps=steps, fluid_height=float(fluid_height))


def dam_break(fluid_sites: Sequence[int], tank_sites: Sequence[int], r: float = 0.01,
              dt: float = 4e-4, steps: int = 100, name: str = "dam_break",
              fluid_lo: Sequence[int] = (0, 0, 0), v0: Sequence[float] = (0.0, 0.0, 0.0),
              **overrides) -> Scene:
    """Fluid block of `fluid_sites` sites at `fluid_lo` inside a closed tank."""
    s = 2.0 * r
    f = block_sites(fluid_lo, fluid_sites, s)
    return _finish(name, r, dt, tank_sites, [(f, v0)], [], steps,
                   fluid_height=(fluid_lo[2] + fluid_sites[2]) * s, **overrides)


def free_block(n_sites: Sequence[int], r: float = 0.01, dt: float = 4e-4, seed: int = 0,
               jitter: float = 0.0, vel_scale: float = 0.0, gravity=(0.0, 0.0, 0.0),
               name: str = "free_block", **overrides) -> Scene:
    """Fluid-only block with no boundary: optional seeded position jitter (in units of s)
    and seeded random velocities (uniform in [-vel_scale, vel_scale]^3)."""
    s = 2.0 * r
    rng = np.random.default_rng(seed)
    f = block_sites((0, 0, 0), n_sites, s)
    if jitter > 0.0:
        f = f + rng.uniform(-jitter * s, jitter * s, size=f.shape)
    sc = _finish(name, r, dt, None, [(f, (0.0, 0.0, 0.0))], [], 1,
                 fluid_height=n_sites[2] * s, gravity=tuple(gravity), **overrides)
    if vel_scale > 0.0:
        sc.fluid_vel = rng.uniform(-vel_scale, vel_scale, size=f.shape).astype(np.float32)
    return sc


def random_cloud(n: int, box: Sequence[float], r: float = 0.01, seed: int = 0,
                 n_boundary: int = 0, name: str = "random_cloud", **overrides) -> Scene:
    """Uniform random fluid (and optionally boundary) points in a box: neighbour-search stress input."""
    rng = np.random.default_rng(seed)
    box = np.asarray(box, dtype=np.float64)
    f = rng.uniform(0.0, 1.0, size=(n, 3)) * box
    extra = []
    if n_boundary > 0:
        b = rng.uniform(0.0, 1.0, size=(n_boundary, 3)) * box
        extra.append((b, Body(0, 0, dynamic=0)))
    sc = _finish(name, r, 4e-4, None, [(f, (0.0, 0.0, 0.0))], extra, 1,
                 fluid_height=float(box[2]), **overrides)
    sc.fluid_vel = rng.uniform(-1.0, 1.0, size=f.shape).astype(np.float32)
    return sc


def _solid_box_inertia(mass: float, size: Sequence[float]) -> Tuple[float, float, float]:
    a, b, c = size
    return (mass * (b * b + c * c) / 12.0, mass * (a * a + c * c) / 12.0,
            mass * (a * a + b * b) / 12.0)


def make_rigid_box(center, size, density, s, dynamic=1) -> Tuple[np.ndarray, Body]:
    pts = box_shell(center, size, s)
    mass = density * size[0] * size[1] * size[2]
    return pts, Body(0, 0, dynamic=dynamic, mass=mass, inertia_body=_solid_box_inertia(mass, size),
                     com=tuple(float(c) for c in center), contact_radius=0.5 * min(size))


def make_rigid_sphere(center, radius, density, s, dynamic=1) -> Tuple[np.ndarray, Body]:
    pts = sphere_shell(center, radius, s)
    mass = density * 4.0 / 3.0 * np.pi * radius ** 3
    I = 0.4 * mass * radius * radius
    return pts, Body(0, 0, dynamic=dynamic, mass=mass, inertia_body=(I, I, I),
                     com=tuple(float(c) for c in center), contact_radius=radius)


def rigid_coupling(scale: float = 1.0, seed: int = 0, r: float = 0.01, dt: float = 4e-4,
                   steps: int = 1000, name: str = "rigid_coupling", **overrides) -> Scene:
    """Config 2: fluid block dropped onto three dynamic bodies resting on the tank floor.

    scale = 1 gives BASELINE.json's config 2 (300,000 fluid particles, tank 100x50x150 sites
    (reading R24), cube 0.2 m, sphere R = 0.15 m, box 0.3x0.1x0.1 m, body densities
    U[500, 2000] from the seed).  Smaller scales shrink the tank and the fluid block (site
    counts * scale) but keep body sizes, for tests.
    """
    s = 2.0 * r
    rng = np.random.default_rng(seed)
    q = lambda n: max(1, int(round(n * scale)))
    tank = (max(q(100), 50), max(q(50), 30), max(q(150), 40))
    fl_n = (q(75), q(40), q(100))
    fl_lo = ((tank[0] - fl_n[0]) // 2, (tank[1] - fl_n[1]) // 2, 25)
    f = block_sites(fl_lo, fl_n, s)
    dens = rng.uniform(500.0, 2000.0, size=3)
    # seeded, non-overlapping (x, y) slots along x; y jittered
    Lx, Ly = tank[0] * s, tank[1] * s
    xs = np.array([0.2, 0.5, 0.8]) * Lx + rng.uniform(-0.02, 0.02, size=3)
    ys = 0.5 * Ly + rng.uniform(-0.05, 0.05, size=3)
    gap = 0.5 * s  # bodies rest half a spacing above the inner wall layer's influence
    cube = make_rigid_box((xs[0], ys[0], 0.1 + gap), (0.2, 0.2, 0.2), dens[0], s)
    sph = make_rigid_sphere((xs[1], ys[1], 0.15 + gap), 0.15, dens[1], s)
    box = make_rigid_box((xs[2], ys[2], 0.05 + gap), (0.3, 0.1, 0.1), dens[2], s)
    return _finish(name, r, dt, tank, [(f, (0.0, 0.0, 0.0))], [cube, sph, box], steps,
                   fluid_height=(fl_lo[2] + fl_n[2]) * s, **overrides)


def viscous_column(scale: float = 1.0, r: float = 0.01, dt: float = 1e-3, steps: int = 500,
                   nu: float = 10.0, name: str = "viscous_column", **overrides) -> Scene:
    """Config 3: column 50x50x80 sites falling from z = 0.2 m in a 100^3-site tank (R24);
    implicit viscosity (mode 2), nu = 10 m^2/s, CG 1e-5."""
    q = lambda n: max(1, int(round(n * scale)))
    tank = (max(q(100), 20), max(q(100), 20), max(q(100), 20))
    n = (q(50), q(50), q(80))
    lo = ((tank[0] - n[0]) // 2, (tank[1] - n[1]) // 2, min(10, tank[2] - n[2]))
    kw = dict(viscosity_mode=2, kinematic_viscosity=nu, cg_rel_tol=1e-5, cg_max_iter=500)
    kw.update(overrides)
    return dam_break(n, tank, r=r, dt=dt, steps=steps, name=name, fluid_lo=lo, **kw)


def splash(n_target: float = 1.23e6, seed: int = 0, r: float = 0.005, dt: float = 2e-4,
           steps: int = 200, name: str = "splash", **overrides) -> Scene:
    """Config 4 (and its scaling sweep): two fluid blocks colliding at +-2 m/s against four
    static obstacles (2 boxes, 2 cylinders) in a closed tank.

    n_target = 1.23e6 gives tank 400x200x200 sites (4x2x2 m at s = 0.01), blocks of
    100x75x82 sites = 615,000 particles each.  Other sizes scale every site count by
    (n_target / 1.23e6)^(1/3); the actual particle count is in the returned scene.
    """
    s = 2.0 * r
    rng = np.random.default_rng(seed)
    k = (n_target / 1.23e6) ** (1.0 / 3.0)
    q = lambda n: max(2, int(round(n * k)))
    tank = (q(400), q(200), q(200))
    bn = (q(100), q(75), q(82))
    xa = q(77)
    xb = tank[0] - xa - bn[0]
    y0 = (tank[1] - bn[1]) // 2
    fa = block_sites((xa, y0, 0), bn, s)
    fb = block_sites((xb, y0, 0), bn, s)
    Lx, Ly = tank[0] * s, tank[1] * s
    extra = []
    for kk in range(4):
        cx = rng.uniform(0.4875, 0.5125) * Lx
        cy = (0.125 + 0.25 * kk) * Ly + rng.uniform(-0.025, 0.025) * Ly
        hgt = 0.6 * k
        if kk % 2 == 0:
            sz = (0.3 * k, 0.3 * k, hgt)
            pts = box_shell((cx, cy, 0.5 * hgt + 0.5 * s), sz, s)
        else:
            pts = cylinder_shell((cx, cy, 0.5 * hgt + 0.5 * s), 0.15 * k, hgt, s)
        extra.append((pts, Body(0, 0, dynamic=0)))
    return _finish(name, r, dt, tank, [(fa, (2.0, 0.0, 0.0)), (fb, (-2.0, 0.0, 0.0))], extra,
                   steps, fluid_height=bn[2] * s, **overrides)


# --------------------------------------------------------------------------
# BASELINE.json configs
# --------------------------------------------------------------------------

def config(idx: int, seed: int = 0, **overrides) -> Scene:
    """The five BASELINE.json configs (synthetic stand-ins)."""
    if idx == 0:
        return dam_break((20, 20, 20), (25, 25, 25), r=0.01, dt=4e-4, steps=100,
                         name="config0_dam_break_8k", **overrides)
    if idx == 1:
        kw = dict(viscosity_mode=1, kinematic_viscosity=0.01)
        kw.update(overrides)
        return dam_break((50, 50, 50), (100, 50, 50), r=0.01, dt=4e-4, steps=500,
                         name="config1_dam_break_125k", **kw)
    if idx == 2:
        return rigid_coupling(1.0, seed=seed, name="config2_rigid_coupling_300k", **overrides)
    if idx == 3:
        return viscous_column(1.0, name="config3_viscous_column_200k", **overrides)
    if idx == 4:
        return splash(1.23e6, seed=seed, name="config4_splash_1p23M", **overrides)
    raise ValueError(f"unknown config {idx}")
