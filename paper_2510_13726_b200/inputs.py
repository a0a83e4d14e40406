"""Seeded synthetic inputs shared by the oracle tests, the GPU parity tests and bench.py.

This module holds NO arithmetic of the method (no collision, streaming, wall function,
porosity rule or force sum): it only makes input arrays -- initial density/velocity,
signed-distance fields of synthetic shapes, the rotor-frame reference grid -- and the
five workload recipes of BASELINE.json.  The arrays are cast
to fp32 once here so both sides start from identical values.  It imports neither the
CUDA binding nor the oracle; `apply_case` drives whichever lattice object it is handed
through the method names both expose.

The paper's real workload is the model rotor of its ref. [19]; that
geometry is not available, the rotor below is a synthetic stand-in with the same
proportions (R/c_tip = 3.91, three blades, hub).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

PERIODIC, MIRROR = 0, 1


def _grid(nx, ny, nz):
    z, y, x = np.meshgrid(np.arange(nz, dtype=np.float64), np.arange(ny, dtype=np.float64),
                          np.arange(nx, dtype=np.float64), indexing="ij")
    return x, y, z


def taylor_green(n: int, u0: float = 0.05):
    """3-D Taylor-Green vortex on n^3 (BASELINE.json config 1).  Returns rho[n^3], u[3,n^3] fp32."""
    x, y, z = _grid(n, n, n)
    k = 2.0 * np.pi / n
    u = np.stack([u0 * np.sin(k * x) * np.cos(k * y) * np.cos(k * z),
                  -u0 * np.cos(k * x) * np.sin(k * y) * np.cos(k * z),
                  np.zeros_like(x)])
    rho = 1.0 + 3.0 * (u0 ** 2 / 16.0) * (np.cos(2 * k * x) + np.cos(2 * k * y)) * (np.cos(2 * k * z) + 2.0)
    return rho.reshape(-1).astype(np.float32), u.reshape(3, -1).astype(np.float32)


def noisy_uniform(nx, ny, nz, mean, sigma, seed):
    """u = mean + N(0, sigma^2) per component, C order (z,y,x,component), rho = 1."""
    rng = np.random.default_rng(seed)
    noise = rng.standard_normal((nz, ny, nx, 3))
    u = np.asarray(mean, np.float64)[None, None, None, :] + sigma * noise
    u = np.moveaxis(u, 3, 0).reshape(3, -1)
    rho = np.ones(nx * ny * nz)
    return rho.astype(np.float32), u.astype(np.float32)


def sphere_phi(nx, ny, nz, centre, r):
    x, y, z = _grid(nx, ny, nz)
    phi = np.sqrt((x - centre[0]) ** 2 + (y - centre[1]) ** 2 + (z - centre[2]) ** 2) - r
    return phi.reshape(-1).astype(np.float32)


def tanh_transition(phi, eps):
    """A smooth transition function s for Def. 1: normalised tanh ramp,
    s(-eps/2)=0, s(0)=1/2, s(eps/2)=1.  Values outside the band are 0/1."""
    phi = np.asarray(phi, np.float64)
    s = 0.5 * (1.0 + np.tanh(4.0 * phi / eps) / np.tanh(2.0))
    return np.clip(s, 0.0, 1.0).astype(np.float32)


def wall_phi(nx, ny, nz, offset=1.25):
    """Plane wall: phi = y - offset (solid below)."""
    x, y, z = _grid(nx, ny, nz)
    return (y - offset).reshape(-1).astype(np.float32)


def rotor_reference_grid(R: float, spacing: float = 0.5, clip: float = 4.0, margin: float = 4.0):
    """Synthetic three-blade rotor + hub in the rotor frame (axis = +x), as a signed-distance
    grid at `spacing` cells (reference grid at double resolution).
    Returns sdf[gz,gy,gx] fp32, tag[gz,gy,gx] u8 (1..3 blades, 4 hub), origin[3] (position of
    node (0,0,0) relative to the rotor centre)."""
    c_tip = R / 3.913
    hx = 0.3 * R + margin
    hy = R + margin
    gx = int(round(2 * hx / spacing)) + 1
    gy = int(round(2 * hy / spacing)) + 1
    gz = gy
    origin = np.array([-hx, -hy, -hy])
    xs = origin[0] + spacing * np.arange(gx)
    ys = origin[1] + spacing * np.arange(gy)
    sdf = np.empty((gz, gy, gx), np.float32)
    tag = np.empty((gz, gy, gx), np.uint8)
    Y, X = np.meshgrid(ys, xs, indexing="ij")
    for kz in range(gz):
        zc = origin[2] + spacing * kz
        best = np.sqrt(X * X + Y * Y + zc * zc) - 0.1 * R  # hub sphere
        btag = np.full(best.shape, 4, np.uint8)
        for b in range(3):
            az = 2.0 * np.pi * b / 3.0
            s = Y * np.cos(az) + zc * np.sin(az)          # span coordinate
            ch = -Y * np.sin(az) + zc * np.cos(az)        # chordwise (tangential)
            t = np.clip((s - 0.1 * R) / (0.9 * R), 0.0, 1.0)
            c = c_tip * (1.5 - 0.5 * t)
            beta = np.deg2rad(4.0 + 31.0 * (1.0 - t) ** 2)
            p = np.cos(beta) * ch + np.sin(beta) * X
            q = -np.sin(beta) * ch + np.cos(beta) * X
            A = 0.5 * c
            B = 0.09 * c
            rho_e = np.sqrt((p / A) ** 2 + (q / B) ** 2)
            g = np.sqrt((p / A ** 2) ** 2 + (q / B ** 2) ** 2)
            with np.errstate(divide="ignore", invalid="ignore"):
                pe = np.where(g > 1e-12, (rho_e - 1.0) * rho_e / g, -B)
            pb = np.maximum(np.maximum(pe, 0.1 * R - s), s - R)
            m = pb < best
            best = np.where(m, pb, best)
            btag = np.where(m, np.uint8(b + 1), btag)
        sdf[kz] = np.clip(best, -clip, clip)
        tag[kz] = btag
    return sdf, tag, origin


@dataclass
class Case:
    """One workload recipe: everything needed to set up a lattice on either side."""
    name: str
    nx: int
    ny: int
    nz: int
    steps: int
    mode: tuple = (PERIODIC, PERIODIC, PERIODIC)
    params: dict = field(default_factory=dict)      # tau0, sigma, smagorinsky_cs, body_force, ...
    rho: Optional[np.ndarray] = None
    u: Optional[np.ndarray] = None
    with_neq: bool = False
    phi: Optional[np.ndarray] = None                 # static geometry
    tag: Optional[np.ndarray] = None
    d_override: Optional[np.ndarray] = None
    fringe: Optional[tuple] = None                   # (x0, x1, u_in)
    rotor: Optional[dict] = None                     # kwargs of set_rotor
    wall_model: bool = False
    wall_function: int = 0                           # 0 truncated Spalding (the paper's), 1 Musker
    wm_variant: tuple = (0, 0)                       # (slip, shear) readings of PAPER.md:314 / :324, DESIGN R22
    fsi_boxes: Optional[list] = None                 # region split: [(x0,x1,y0,y1,z0,z1), ...]

    @property
    def n(self):
        return self.nx * self.ny * self.nz


def apply_case(case: Case, lattice) -> None:
    """Drive `lattice` (oracle.Lattice or the CUDA binding's Lattice) into the case's initial state."""
    if case.phi is not None:
        lattice.set_static_geometry(case.phi, case.tag, case.d_override)
    if case.fringe is not None:
        lattice.set_fringe(*case.fringe)
    if case.rotor is not None:
        lattice.set_rotor(**case.rotor)
    lattice.enable_wall_model(case.wall_model)
    if case.wall_function:
        lattice.set_wall_function(case.wall_function)
    if tuple(case.wm_variant) != (0, 0):
        lattice.set_wall_model_variant(*case.wm_variant)
    if case.fsi_boxes is not None:
        lattice.set_fsi_region(case.fsi_boxes)
    lattice.init_equilibrium(case.rho, case.u, case.with_neq)


def with_region_split(case: Case, margin: int = 6) -> Case:
    """The same recipe with the paper's bulk / FSI region split: boxes around everything that
    is not plain fluid -- the inflow fringe slab, the volume the rotor sweeps, a static sphere, the wall
    layer -- each widened by `margin` cells; the rest of the lattice runs the bulk RRLBM-LES model."""
    import dataclasses
    nx, ny, nz = case.nx, case.ny, case.nz
    boxes = []
    if case.fringe is not None:
        boxes.append((max(0, case.fringe[0] - 1), min(nx, case.fringe[1] + 1), 0, ny, 0, nz))
    if case.rotor is not None:
        sdf = case.rotor["sdf"]
        gz, gy, gx = sdf.shape
        sp, org, ctr = case.rotor["spacing"], case.rotor["origin"], case.rotor["centre"]
        hx = max(abs(org[0]), abs(org[0] + (gx - 1) * sp))          # axis +x: axial half-extent of the grid
        hr = max(abs(org[1]), abs(org[1] + (gy - 1) * sp), abs(org[2]), abs(org[2] + (gz - 1) * sp))
        boxes.append((max(0, int(np.floor(ctr[0] - hx)) - margin), min(nx, int(np.ceil(ctr[0] + hx)) + margin + 1),
                      max(0, int(np.floor(ctr[1] - hr)) - margin), min(ny, int(np.ceil(ctr[1] + hr)) + margin + 1),
                      max(0, int(np.floor(ctr[2] - hr)) - margin), min(nz, int(np.ceil(ctr[2] + hr)) + margin + 1)))
    if case.phi is not None:
        near = np.flatnonzero(np.asarray(case.phi).reshape(-1) < 2.0)   # cells within 2 of the static surface
        if near.size:
            x, y, z = near % nx, (near // nx) % ny, near // (nx * ny)
            boxes.append((max(0, int(x.min()) - margin), min(nx, int(x.max()) + margin + 1),
                          max(0, int(y.min()) - margin), min(ny, int(y.max()) + margin + 1),
                          max(0, int(z.min()) - margin), min(nz, int(z.max()) + margin + 1)))
    return dataclasses.replace(case, name=case.name + "+split", fsi_boxes=boxes)


DEFAULTS = dict(sigma=0.995, smagorinsky_cs=0.1, kappa=0.41, E=9.8, newton_max_iter=10,
                newton_tol=1e-4, sampling_distance=2.0, eps_cells=2.0)


def case_tgv(n=32, steps=10) -> Case:
    """Config 1: 3-D Taylor-Green vortex, periodic, tau=0.55, U0=0.05, d=1, no wall model."""
    rho, u = taylor_green(n, 0.05)
    return Case("tgv", n, n, n, steps, params=dict(DEFAULTS, tau0=0.55), rho=rho, u=u, with_neq=True)


def case_sphere(nx=128, ny=64, nz=64, r=10.0, steps=200, seed=20002) -> Case:
    """Config 2: channel with a static sphere as smoothed porosity, fringe inflow u=0.05, noise 1e-3."""
    centre = (nx / 4.0, ny / 2.0 - 0.5, nz / 2.0 - 0.5)
    phi = sphere_phi(nx, ny, nz, centre, r)
    rho, u = noisy_uniform(nx, ny, nz, (0.05, 0.0, 0.0), 1e-3, seed)
    return Case("sphere", nx, ny, nz, steps, params=dict(DEFAULTS, tau0=0.52), rho=rho, u=u,
                phi=phi, tag=np.ones(nx * ny * nz, np.uint8), d_override=tanh_transition(phi, 2.0),
                fringe=(0, 4, (0.05, 0.0, 0.0)))


def case_channel(nx=256, ny=128, nz=128, steps=500, re_tau=1000.0, seed=30003) -> Case:
    """Config 3: turbulent half-channel, body force, porosity-0 wall + wall-model layer, y MIRROR on top."""
    u_tau = 0.0025
    H = ny - 1.75                       # wall (phi=0) at y=1.25, mirror plane at y=ny-0.5
    nu = u_tau * H / re_tau
    g = u_tau ** 2 / H
    phi = wall_phi(nx, ny, nz, 1.25)
    rho, u = noisy_uniform(nx, ny, nz, (0.05, 0.0, 0.0), 0.0025, seed)
    d0 = np.clip(np.asarray(phi, np.float64) / 2.0 + 0.5, 0.0, 1.0)   # start at rest inside the wall
    u = (u.astype(np.float64) * d0[None, :]).astype(np.float32)
    return Case("channel", nx, ny, nz, steps, mode=(PERIODIC, MIRROR, PERIODIC),
                params=dict(DEFAULTS, tau0=0.5 + 3.0 * nu, body_force=(g, 0.0, 0.0)), rho=rho, u=u,
                phi=phi, tag=np.ones(nx * ny * nz, np.uint8), wall_model=True)


_ROTOR_CACHE: dict = {}


def case_rotor(nx=512, ny=256, nz=256, R=80.0, steps=1000, u_in=0.04, tsr=6.0, omega=None) -> Case:
    """Configs 4/5: one synthetic 3-blade rotor, axis +x, fringe inflow, wall model on, per-blade forces."""
    if R not in _ROTOR_CACHE:
        _ROTOR_CACHE[R] = rotor_reference_grid(R)
    sdf, tag, origin = _ROTOR_CACHE[R]
    if omega is None:
        omega = tsr * u_in / R
    c_tip = R / 3.913
    nu = omega * R * c_tip / 38882.0
    centre = (nx / 4.0, ny / 2.0 - 0.5, nz / 2.0 - 0.5)
    n = nx * ny * nz
    rho = np.ones(n, np.float32)
    u = np.zeros((3, n), np.float32)
    u[0] = u_in
    rotor = dict(sdf=sdf, tag=tag, spacing=0.5, origin=tuple(origin), centre=centre,
                 axis=(1.0, 0.0, 0.0), omega=omega, theta0=0.0, n_tags=4)
    return Case("rotor", nx, ny, nz, steps, params=dict(DEFAULTS, tau0=0.5 + 3.0 * nu), rho=rho, u=u,
                fringe=(0, 4, (u_in, 0.0, 0.0)), rotor=rotor, wall_model=True)


def baseline_config(k: int) -> Case:
    """The five configs of BASELINE.json at full size (1-based)."""
    if k == 1:
        return case_tgv(32, 10)
    if k == 2:
        return case_sphere(128, 64, 64, 10.0, 200)
    if k == 3:
        return case_channel(256, 128, 128, 500)
    if k == 4:
        return case_rotor(512, 256, 256, 80.0, 1000, omega=0.003)
    if k == 5:
        return case_rotor(768, 384, 364, 120.0, 200, omega=0.002)
    raise ValueError(k)
