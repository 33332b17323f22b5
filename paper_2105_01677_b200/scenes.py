"""Seeded synthetic dam-break-shaped scenes (inputs only).

This module is the ONE piece shared by the CPU oracle (``oracle/``) and the
CUDA path (``paper_2105_01677_b200/csrc``).  It holds none of the method's
arithmetic: no kernel function, no n0/lambda, no cell keys.  It only lays
particles on a cubic lattice, tags them FLUID / WALL / DUMMY, and draws the
seeded jitter.  The recipe is stated in DESIGN.md ("Input recipe") and follows
SURVEY.md section 8(d):

* Tank: open-top rectangular box of ``tank = (nx, ny, nz)`` lattice sites,
  particle centres at ``(i + 1/2) * l0``.
* Walls: 3 layers on the floor and the four sides; the innermost layer is
  WALL (carries pressure), the outer two are DUMMY (Listing 2
  comments "fluid or boundary p." / "dummy p."; reading Q3 in DESIGN.md).
* Fluid: rectangular blocks of lattice sites (the paper's dam-break column,
  PAPER.md:318-341 section 5.2, is a block at rest in one corner of the tank).
* Jitter: ``numpy.random.Generator(PCG64(seed)).uniform(-j, j, (N_fluid, 3))``
  with ``j = 1e-3 * l0`` on fluid positions only (BASELINE.json configs).
* Order: one z-major sweep over all sites (z slowest, x fastest); optional
  seeded shuffle so that the sort in ``mps_bin`` has real work to do.

The paper's own scene files (PAPER.md:292 item 3, "previously built simulation
scenario") are not available; these scenes stand in for them.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Dict, List, Optional, Sequence, Tuple

import numpy as np

FLUID, WALL, DUMMY, GHOST = 0, 1, 2, 3

BASE_SEED = 2105016770  # config k uses BASE_SEED + k


@dataclass
class Scene:
    """Particle arrays (caller's original order) plus the physical parameters."""

    name: str
    x: np.ndarray
    y: np.ndarray
    z: np.ndarray
    u: np.ndarray
    v: np.ndarray
    w: np.ndarray
    type: np.ndarray   # int32: FLUID/WALL/DUMMY
    phase: np.ndarray  # int32: 0 or 1
    params: Dict[str, object] = field(default_factory=dict)
    route: int = 0     # 0 explicit (EoS), 1 PPE
    steps: int = 20

    @property
    def n(self) -> int:
        return int(self.x.shape[0])

    @property
    def n_fluid(self) -> int:
        return int(np.count_nonzero(self.type == FLUID))


def default_params(l0: float) -> Dict[str, object]:
    """Physical/numerical parameters common to every config (DESIGN.md readings).

    n0_n, n0_lap, lam = 0 mean "compute the lattice closed form yourself": the
    oracle and the CUDA library each do so with their own code.
    """
    return dict(
        dim=3,
        l0=float(l0),
        re_n=2.1 * l0,       # density / gradient radius (BASELINE.json config 1)
        re_lap=3.1 * l0,     # Laplacian radius
        dt=0.05 * l0,        # reading Q14: c0*dt/l0 = 0.5 (5e-4 s at l0 = 0.01)
        g=(0.0, 0.0, -9.81),
        n_phases=1,
        rho=(1000.0, 1000.0),
        nu=(1.0e-6, 1.0e-6),
        c0=10.0,             # reading Q14
        gamma=7.0,
        beta=0.97,
        compress=1.0e-7,     # PAPER.md:282 Listing 2
        ppe_relax=1.0,
        cg_rtol=1.0e-8,
        cg_maxit=2000,
        cs=0.0,              # Smagorinsky constant, 0 = off
        grad_variant=0,
        ppe_source=0,        # 0 Eq. 8; 1 higher-order source (Eq. 15); 2 + error-compensating parts (Eq. 17-18)
        ppe_laplacian=0,     # 0 Eq. 10 form; 1 higher-order Laplacian (Eq. 16)
        kernel=0,            # 0 w = re/r - 1 (Eq. 3); 1 w = (1 - r/re)^3 (Eq. 4)
        rebin_every=1,       # 1 exact sets at every sweep; K > 1 the paper's list reuse
        ppe_operator=1,      # CUDA path only: 0 matrix-free operator, 1 coefficients assembled once per solve
        cg_warm_start=0,     # 1: CG starts from the particle's previous pressure instead of 0
        key_mode=0,          # 0 linear x-fastest cell key, 1 Morton (3 x 10-bit interleave)
        row_skin=0.0,        # CUDA path only: Verlet skin of mps_step's rows in units of l0 (0: default, < 0: off)
        clamp_negative_p=1,
        rho_pair_mean=0,
        nu_pair_mean=1,
        cell_div=1,
        domain_min=(0.0, 0.0, 0.0),
        domain_max=(0.0, 0.0, 0.0),
        max_neighbours=300,
        n0_n=0.0,
        n0_lap=0.0,
        lam=0.0,
    )


def _lattice_scene(
    name: str,
    l0: float,
    tank: Tuple[int, int, int],
    blocks: Sequence[Tuple[Tuple[int, int, int], Tuple[int, int, int], int]],
    seed: int,
    jitter: float = 1.0e-3,
    shuffle: bool = False,
    wall_layers: int = 3,
    wall_phase_split_z: Optional[int] = None,
) -> Scene:
    """Build a tank scene.

    ``blocks``: list of ``(lo, hi, phase)`` half-open lattice-site boxes of fluid.
    ``wall_layers``: 0 gives an isolated fluid blob (used by the pins).
    ``wall_phase_split_z``: WALL/DUMMY sites with ``iz >= split`` get phase 1.
    """
    nx, ny, nz = tank
    L = wall_layers
    ix = np.arange(-L, nx + L, dtype=np.int64)
    iy = np.arange(-L, ny + L, dtype=np.int64)
    iz = np.arange(-L, nz, dtype=np.int64) if L > 0 else np.arange(0, nz, dtype=np.int64)
    Z, Y, X = np.meshgrid(iz, iy, ix, indexing="ij")  # z slowest, x fastest
    X = X.ravel()
    Y = Y.ravel()
    Z = Z.ravel()
    inside = (X >= 0) & (X < nx) & (Y >= 0) & (Y < ny) & (Z >= 0)
    in_wall_box = (X >= -1) & (X < nx + 1) & (Y >= -1) & (Y < ny + 1) & (Z >= -1)

    typ = np.full(X.shape, -1, dtype=np.int32)
    phase = np.zeros(X.shape, dtype=np.int32)
    for lo, hi, ph in blocks:
        m = (
            (X >= lo[0]) & (X < hi[0]) & (Y >= lo[1]) & (Y < hi[1])
            & (Z >= lo[2]) & (Z < hi[2])
        )
        typ[m] = FLUID
        phase[m] = ph
    if L > 0:
        typ[~inside & in_wall_box] = WALL
        typ[~inside & ~in_wall_box] = DUMMY
        if wall_phase_split_z is not None:
            phase[(~inside) & (Z >= wall_phase_split_z)] = 1
    keep = typ >= 0
    X, Y, Z, typ, phase = X[keep], Y[keep], Z[keep], typ[keep], phase[keep]

    x = (X.astype(np.float64) + 0.5) * l0
    y = (Y.astype(np.float64) + 0.5) * l0
    z = (Z.astype(np.float64) + 0.5) * l0
    fl = np.nonzero(typ == FLUID)[0]
    if jitter > 0.0 and fl.size:
        rng = np.random.Generator(np.random.PCG64(seed))
        d = rng.uniform(-jitter * l0, jitter * l0, size=(fl.size, 3))
        x[fl] += d[:, 0]
        y[fl] += d[:, 1]
        z[fl] += d[:, 2]
    n = x.shape[0]
    if shuffle:
        prm = np.random.Generator(np.random.PCG64(seed ^ 0x5EED)).permutation(n)
        x, y, z, typ, phase = x[prm], y[prm], z[prm], typ[prm], phase[prm]

    p = default_params(l0)
    p["domain_min"] = (-L * l0, -L * l0, -L * l0 if L > 0 else 0.0)
    p["domain_max"] = ((nx + L) * l0, (ny + L) * l0, nz * l0)
    zeros = np.zeros(n, dtype=np.float64)
    return Scene(
        name=name,
        x=np.ascontiguousarray(x), y=np.ascontiguousarray(y), z=np.ascontiguousarray(z),
        u=zeros.copy(), v=zeros.copy(), w=zeros.copy(),
        type=np.ascontiguousarray(typ), phase=np.ascontiguousarray(phase),
        params=p,
    )


def dam_break(
    l0: float,
    tank: Tuple[int, int, int],
    fluid: Tuple[int, int, int],
    seed: int,
    name: str = "dam_break",
    **kw,
) -> Scene:
    """Fluid block ``fluid`` (sites) at rest in the corner x=y=z=0 of ``tank``."""
    return _lattice_scene(name, l0, tank, [((0, 0, 0), tuple(fluid), 0)], seed, **kw)


def fluid_blob(l0: float, m: Tuple[int, int, int], seed: int = 0, jitter: float = 0.0) -> Scene:
    """Isolated m[0] x m[1] x m[2] block with no walls (pins T3, T4, T10)."""
    s = _lattice_scene("blob", l0, tuple(m), [((0, 0, 0), tuple(m), 0)], seed,
                       jitter=jitter, wall_layers=0)
    pad = 8.0 * l0
    s.params["domain_min"] = (-pad, -pad, -pad)
    s.params["domain_max"] = (m[0] * l0 + pad, m[1] * l0 + pad, m[2] * l0 + pad)
    return s


def dam_break_2d(l0: float, tank: Tuple[int, int], fluid: Tuple[int, int], seed: int,
                 name: str = "dam_break_2d", jitter: float = 1.0e-3, shuffle: bool = False) -> Scene:
    """Two-dimensional dam break in the x-y plane (gravity along -y, z = 0 for every particle):
    the shape of the paper's own timed scenes (section 5.2 and PAPER.md:397:
    column height = 2 x column length, floor = 4 x column length).  Walls as in 3D: 3 layers on
    the floor and both sides, innermost WALL, outer two DUMMY; open top."""
    nx, ny = tank
    L = 3
    ix = np.arange(-L, nx + L, dtype=np.int64)
    iy = np.arange(-L, ny, dtype=np.int64)
    Y, X = np.meshgrid(iy, ix, indexing="ij")  # y slowest, x fastest
    X = X.ravel()
    Y = Y.ravel()
    inside = (X >= 0) & (X < nx) & (Y >= 0)
    in_wall_box = (X >= -1) & (X < nx + 1) & (Y >= -1)
    typ = np.full(X.shape, -1, dtype=np.int32)
    typ[(X >= 0) & (X < fluid[0]) & (Y >= 0) & (Y < fluid[1])] = FLUID
    typ[~inside & in_wall_box] = WALL
    typ[~inside & ~in_wall_box] = DUMMY
    keep = typ >= 0
    X, Y, typ = X[keep], Y[keep], typ[keep]
    x = (X.astype(np.float64) + 0.5) * l0
    y = (Y.astype(np.float64) + 0.5) * l0
    fl = np.nonzero(typ == FLUID)[0]
    if jitter > 0.0 and fl.size:
        rng = np.random.Generator(np.random.PCG64(seed))
        d = rng.uniform(-jitter * l0, jitter * l0, size=(fl.size, 2))
        x[fl] += d[:, 0]
        y[fl] += d[:, 1]
    n = x.shape[0]
    if shuffle:
        prm = np.random.Generator(np.random.PCG64(seed ^ 0x5EED)).permutation(n)
        x, y, typ = x[prm], y[prm], typ[prm]
    p = default_params(l0)
    p.update(dim=2, g=(0.0, -9.81, 0.0))
    p["domain_min"] = (-L * l0, -L * l0, -0.5 * l0)
    p["domain_max"] = ((nx + L) * l0, ny * l0, 0.5 * l0)
    zeros = np.zeros(n, dtype=np.float64)
    return Scene(name=name, x=np.ascontiguousarray(x), y=np.ascontiguousarray(y), z=zeros.copy(),
                 u=zeros.copy(), v=zeros.copy(), w=zeros.copy(), type=np.ascontiguousarray(typ),
                 phase=np.zeros(n, dtype=np.int32), params=p)


def water_drop(radius_sites: int = 20, l0: float = 0.875 / 20, rate: float = 100.0) -> Scene:
    """The paper's water-drop test (section 5.1, Table 1): a 2D disc
    of fluid, no walls, no gravity, initial velocity field (-rate x, rate y), Eq. 4 kernel, r_e = 3 l0,
    dt = 1e-5 s.  Reading of the garbled geometry (Q17): Table 1 prints b(0) = 0.875 m and
    ab(0) = 0.766 m^2 = 0.875^2, so the disc radius is 0.875 m ("9 x 10^-2" in the text is a typo),
    and 1257 particles are exactly the sites of a square lattice with i^2 + j^2 <= 20^2, so
    l0 = 0.875 / 20 = 0.04375 m ("5 x 10^-2" rounded).  No jitter."""
    R = radius_sites
    ii, jj = np.meshgrid(np.arange(-R, R + 1), np.arange(-R, R + 1), indexing="ij")
    m = (ii * ii + jj * jj) <= R * R
    x = ii[m].astype(np.float64) * l0
    y = jj[m].astype(np.float64) * l0
    n = x.shape[0]
    p = default_params(l0)
    p.update(dim=2, g=(0.0, 0.0, 0.0), re_n=3.0 * l0, re_lap=3.0 * l0, kernel=1, dt=1.0e-5)
    span = 4.0 * R * l0
    p["domain_min"] = (-span, -span, -0.5 * l0)
    p["domain_max"] = (span, span, 0.5 * l0)
    zeros = np.zeros(n, dtype=np.float64)
    return Scene(name="water_drop", x=np.ascontiguousarray(x), y=np.ascontiguousarray(y), z=zeros.copy(),
                 u=-rate * x, v=rate * y, w=zeros.copy(), type=np.zeros(n, np.int32),
                 phase=np.zeros(n, np.int32), params=p)


SWEEP_M = (23, 40, 69, 89, 147)  # config 5: N = 66k / 250k / 1.0M / 2.0M / 7.9M


def make_scene(config: int, seed: Optional[int] = None, shuffle: bool = False,
               sweep_index: int = 0) -> Scene:
    """The five BASELINE.json configs (1-based, as SURVEY.md 8(d) numbers them)."""
    if seed is None:
        seed = BASE_SEED + config + (sweep_index if config == 5 else 0)
    if config == 1:
        s = dam_break(0.01, (40, 20, 30), (20, 20, 10), seed, "config1_dam4k_explicit",
                      shuffle=shuffle)
        s.params.update(dt=5.0e-4, grad_variant=0)
        s.route, s.steps = 0, 20
    elif config == 2:
        s = dam_break(0.005, (80, 40, 60), (40, 40, 20), seed, "config2_dam32k_ppe",
                      shuffle=shuffle)
        s.params.update(grad_variant=0)
        s.route, s.steps = 1, 20
    elif config == 3:
        # tank size is a DESIGN.md reading (BASELINE.json gives the fluid block only)
        s = dam_break(0.005, (200, 50, 100), (100, 50, 50), seed, "config3_dam250k",
                      shuffle=shuffle)
        s.params.update(grad_variant=2)
        s.route, s.steps = 1, 100
    elif config == 4:
        l0 = 0.004
        s = _lattice_scene(
            "config4_twophase500k", l0, (100, 50, 125),
            [((0, 0, 0), (100, 50, 50), 0), ((0, 0, 50), (100, 50, 100), 1)],
            seed, shuffle=shuffle, wall_phase_split_z=50)
        s.params.update(n_phases=2, rho=(1000.0, 800.0), nu=(1.0e-6, 5.0e-6),
                        cs=0.12, grad_variant=0, rho_pair_mean=0, nu_pair_mean=1)
        s.route, s.steps = 1, 50
    elif config == 5:
        m = SWEEP_M[sweep_index]
        s = dam_break(0.005, (4 * m, m, 2 * m), (2 * m, m, m), seed,
                      f"config5_sweep_m{m}", shuffle=shuffle)
        s.route, s.steps = 0, 50
    elif config == 6:
        # not a BASELINE.json config: the paper's own timed workload shape (2D dam break,
        # PAPER.md:397, "about 1 fps at about 200,000 particles"), context only
        c = (100, 316, 700)[sweep_index] if sweep_index < 3 else 316
        s = dam_break_2d(0.005, (4 * c, 3 * c), (c, 2 * c), seed, f"paper_shape_2d_dam_c{c}",
                         shuffle=shuffle)
        s.route, s.steps = 1, 50
    else:
        raise ValueError(f"unknown config {config}")
    return s


def small_tank(l0: float = 0.01, tank=(12, 8, 10), fluid=(6, 6, 6), seed: int = 7,
               shuffle: bool = False, jitter: float = 1.0e-3) -> Scene:
    """A few-thousand-particle tank for fast tests (6^3 fluid block: pin T9)."""
    return dam_break(l0, tank, fluid, seed, "small_tank", shuffle=shuffle, jitter=jitter)


def hydrostatic_tank(l0: float = 0.01, foot=(20, 20), depth: int = 10, height: int = 14,
                     seed: int = 11) -> Scene:
    """Fluid filling the whole footprint, at rest (pin T11, hydrostatic rho*g*h)."""
    s = dam_break(l0, (foot[0], foot[1], height), (foot[0], foot[1], depth), seed,
                  "hydrostatic", jitter=0.0)
    s.params.update(dt=5.0e-4)
    s.route = 1
    return s


def random_cloud(n: int, side: float, seed: int) -> Scene:
    """n uniform random points in a cube (pin T1; not a physical scene)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    xyz = rng.uniform(0.0, side, size=(n, 3))
    zeros = np.zeros(n)
    l0 = side / 31.0
    p = default_params(l0)
    p["domain_min"] = (0.0, 0.0, 0.0)
    p["domain_max"] = (side, side, side)
    return Scene("cloud", np.ascontiguousarray(xyz[:, 0]), np.ascontiguousarray(xyz[:, 1]),
                 np.ascontiguousarray(xyz[:, 2]), zeros.copy(), zeros.copy(), zeros.copy(),
                 np.zeros(n, np.int32), np.zeros(n, np.int32), p)
