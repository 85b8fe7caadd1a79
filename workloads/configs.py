"""The five BASELINE.json configurations as seeded synthetic inputs (numpy only).

Units: Hartree atomic units (hbar = m = 1, lengths in bohr).  Grid point (i, j, k)
sits at (i*dx, j*dx, k*dx) (corner origin).  Boundary flags follow
include/tdse.h: 0 = periodic, 1 = zero Dirichlet.

Nothing here evaluates the method: atom lists and scalar parameters only.
Geometry recipes are stated in DESIGN.md ("Input recipe") and SURVEY.md section 8(d).
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace
from typing import List, Optional, Sequence, Tuple

import numpy as np

PERIODIC = 0
DIRICHLET = 1

CONFIG_NAMES = {
    0: "cfg0_coulomb_well_64c_f64",
    1: "cfg1_fcc111_slab_128c_f64",
    2: "cfg2_thermal_slab_256x256x512_f32",
    3: "cfg3_thin_film_batch64_128c_f32",
    4: "cfg4_large_grid_stress",
}

# atom record = (x, y, z, Z, soft2, screen); screen <= 0 means "unscreened"
ATOM_FIELDS = 6


@dataclass
class Workload:
    name: str
    nx: int
    ny: int
    nz: int
    batch: int
    dtype: str                      # "f32" | "f64"
    dx: float
    dt: float
    mass: float
    hbar: float
    bc: Tuple[int, int, int]        # (bcx, bcy, bcz)
    absorb_lo: int
    absorb_hi: int
    strength: float
    power: int
    atoms: List[np.ndarray]         # one [natoms, 6] float64 array per batch entry
    vmin: float
    vmax: float
    rcut: float                     # <= 0: no cutoff
    packet: dict                    # x0,y0,z0,sigma,kx,ky,kz,amplitude (0 => normalised)
    k_det: int
    every: int
    steps: int
    seeds: List[Optional[int]] = field(default_factory=list)
    dy: Optional[float] = None      # None: cubic cells (dy = dz = dx); else the anisotropic mesh of PAPER.md:87, 142
    dz: Optional[float] = None

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def np_dtype(self):
        return np.float32 if self.dtype == "f32" else np.float64

    def with_(self, **kw) -> "Workload":
        return replace(self, **kw)


def _dt_rule(dx: float, vabs_max: float, hbar: float = 1.0, mass: float = 1.0) -> float:
    """BASELINE.json configs[0]: dt = 0.5*hbar / (6 hbar^2/(m dx^2) + max|V|)."""
    return 0.5 * hbar / (6.0 * hbar * hbar / (mass * dx * dx) + vabs_max)


def fcc111_slab(lx: float, ly: float, z_top: float, nlayers: int, a: float = 6.82,
                Z: float = 29.0, soft2: float = 0.1, screen: float = 0.5) -> np.ndarray:
    """fcc(111) slab: layers stacked toward +z from z_top, ABC stacking.

    In-plane vectors a1 = (d, 0), a2 = (d/2, d*sqrt(3)/2), d = a/sqrt(2); layer m is
    shifted by m*(a1+a2)/3 and sits at z_top + m*a/sqrt(3).  Lattice points with
    0 <= x < lx and 0 <= y < ly are kept (the box is not commensurate with the
    lattice; the seam is accepted).  Order: layer, a2 index, a1 index.
    """
    d = a / math.sqrt(2.0)
    a1 = np.array([d, 0.0])
    a2 = np.array([0.5 * d, 0.5 * d * math.sqrt(3.0)])
    dz = a / math.sqrt(3.0)
    rows = []
    jmax = int(math.ceil(ly / a2[1])) + 2
    imax = int(math.ceil(lx / d)) + 2
    for m in range(nlayers):
        shift = (m % 3) * (a1 + a2) / 3.0
        for j in range(-2, jmax + 1):
            for i in range(-jmax - 2, imax + 1):
                p = i * a1 + j * a2 + shift
                if 0.0 <= p[0] < lx and 0.0 <= p[1] < ly:
                    rows.append((p[0], p[1], z_top + m * dz, Z, soft2, screen))
    return np.asarray(rows, dtype=np.float64).reshape(-1, ATOM_FIELDS)


def molecule_template(bond: float = 2.6) -> Tuple[np.ndarray, np.ndarray]:
    """Rigid planar 20-atom 'ring plus chain' molecule in its own xy-plane.

    Ring of 6 at radius `bond` (Z = 6,6,7,6,6,7); an 8-atom zig-zag chain (+-30 deg
    about +x) leaving ring vertex 0 (Z = 6 x6, 8, 8); H (Z = 1) radially outside ring
    vertices 1..5 and one H continuing the chain.  Returns (xyz[20,3], Z[20]).
    """
    pos, zs = [], []
    ring_z = [6, 6, 7, 6, 6, 7]
    for v in range(6):
        ang = math.radians(60.0 * v)
        pos.append((bond * math.cos(ang), bond * math.sin(ang), 0.0))
        zs.append(ring_z[v])
    chain_z = [6, 6, 6, 6, 6, 6, 8, 8]
    p = np.array(pos[0])
    for n in range(8):
        ang = math.radians(30.0 if n % 2 == 0 else -30.0)
        p = p + bond * np.array([math.cos(ang), math.sin(ang), 0.0])
        pos.append(tuple(p))
        zs.append(chain_z[n])
    for v in range(1, 6):
        ang = math.radians(60.0 * v)
        pos.append((2.0 * bond * math.cos(ang), 2.0 * bond * math.sin(ang), 0.0))
        zs.append(1)
    ang = math.radians(30.0)          # chain atom index 8 would use +30 deg
    p = p + bond * np.array([math.cos(ang), math.sin(ang), 0.0])
    pos.append(tuple(p))
    zs.append(1)
    xyz = np.asarray(pos, dtype=np.float64)
    xyz -= xyz.mean(axis=0)           # pose rotates about the centroid
    return xyz, np.asarray(zs, dtype=np.float64)


def _film_atoms(rng: np.random.Generator, lx: float, ly: float, z_top: float,
                nmol: int, soft2: float, screen: float) -> np.ndarray:
    xyz, zs = molecule_template()
    rows = []
    for _ in range(nmol):
        cx = rng.uniform(0.0, lx)
        cy = rng.uniform(0.0, ly)
        az = rng.uniform(0.0, 2.0 * math.pi)
        tilt = math.radians(rng.uniform(0.0, 15.0))
        rx = np.array([[1, 0, 0],
                       [0, math.cos(tilt), -math.sin(tilt)],
                       [0, math.sin(tilt), math.cos(tilt)]])
        rz = np.array([[math.cos(az), -math.sin(az), 0],
                       [math.sin(az), math.cos(az), 0],
                       [0, 0, 1]])
        p = xyz @ (rz @ rx).T + np.array([cx, cy, z_top - 4.0])
        for q, z in zip(p, zs):
            rows.append((q[0], q[1], q[2], z, soft2, screen))
    return np.asarray(rows, dtype=np.float64).reshape(-1, ATOM_FIELDS)


def _thermal(atoms: np.ndarray, seed: int, sd: float = 0.1) -> np.ndarray:
    rng = np.random.default_rng(seed)
    out = atoms.copy()
    out[:, 0:3] += rng.normal(0.0, sd, size=(atoms.shape[0], 3))
    return out


CFG4_ZTOP_FRAC = 0.38     # as config 1


def make_config(idx: int, *, n: Optional[Sequence[int]] = None, batch: Optional[int] = None,
                steps: Optional[int] = None, dtype: Optional[str] = None) -> Workload:
    """Build configuration `idx` (0..4) of BASELINE.json.

    `n=(nx,ny,nz)`, `batch`, `steps`, `dtype` override the stated size for reduced
    parity cases: the recipe (spacing, physics, fractions of the box) is unchanged, so
    a smaller grid is a smaller box with the same structure.
    """
    hbar = mass = 1.0
    if idx == 0:
        nx, ny, nz = n or (64, 64, 64)
        dx = 0.2
        cx, cy, cz = ((nx - 1) / 2 * dx, (ny - 1) / 2 * dx, (nz - 1) / 2 * dx)
        atoms = np.array([[cx, cy, cz, 1.0, 0.5, 0.0]])
        return Workload(
            name=CONFIG_NAMES[0], nx=nx, ny=ny, nz=nz, batch=batch or 1, dtype=dtype or "f64",
            dx=dx, dt=_dt_rule(dx, 1.0 / math.sqrt(0.5)), mass=mass, hbar=hbar,
            bc=(DIRICHLET, DIRICHLET, DIRICHLET), absorb_lo=0, absorb_hi=0, strength=0.05, power=2,
            atoms=[atoms] * (batch or 1), vmin=-50.0, vmax=0.0, rcut=0.0,
            packet=dict(x0=cx, y0=cy, z0=cz - 3.0, sigma=1.5, kx=0.0, ky=0.0, kz=1.0, amplitude=0.0),
            k_det=min(10, nz - 1), every=10, steps=steps or 500, seeds=[None] * (batch or 1))

    if idx in (1, 2, 3):
        if idx == 1:
            nx, ny, nz = n or (128, 128, 128)
            dx, nlayers, ztop_frac, absorb, every, nsteps, dt_, nb = 0.15, 4, 0.38, 16, 10, 4000, "f64", 1
        elif idx == 2:
            nx, ny, nz = n or (256, 256, 512)
            dx, nlayers, ztop_frac, absorb, every, nsteps, dt_, nb = 0.1, 6, 0.5, 24, 20, 8000, "f32", 1
        else:
            nx, ny, nz = n or (128, 128, 128)
            dx, nlayers, ztop_frac, absorb, every, nsteps, dt_, nb = 0.15, 3, 0.55, 16, 10, 4000, "f32", 64
        nb = batch or nb
        lx, ly, lz = nx * dx, ny * dx, nz * dx
        z_top = ztop_frac * lz
        slab = fcc111_slab(lx, ly, z_top, nlayers)
        atoms, seeds = [], []
        for b in range(nb):
            if idx == 1:
                atoms.append(slab); seeds.append(None)
            elif idx == 2:
                atoms.append(_thermal(slab, 2 + b)); seeds.append(2 + b)
            else:
                rng = np.random.default_rng(3000 + b)
                film = _film_atoms(rng, lx, ly, z_top, 12, 0.1, 0.5)
                atoms.append(np.concatenate([slab, film], axis=0)); seeds.append(3000 + b)
        z0 = 0.2 * lz if idx != 2 else 0.25 * lz
        absorb = min(absorb, max(nz // 8, 0))
        return Workload(
            name=CONFIG_NAMES[idx], nx=nx, ny=ny, nz=nz, batch=nb, dtype=dtype or dt_,
            dx=dx, dt=_dt_rule(dx, 200.0), mass=mass, hbar=hbar,
            bc=(PERIODIC, PERIODIC, DIRICHLET), absorb_lo=absorb, absorb_hi=absorb, strength=0.05, power=2,
            atoms=atoms, vmin=-200.0, vmax=0.0, rcut=0.0,
            packet=dict(x0=lx / 2, y0=ly / 2, z0=z0, sigma=4.0, kx=0.0, ky=0.0, kz=3.0, amplitude=0.0),
            k_det=min(10, nz - 1), every=every, steps=steps or nsteps, seeds=seeds)

    if idx == 4:
        dt_ = dtype or "f32"
        nx, ny, nz = n or ((512, 512, 512) if dt_ == "f32" else (384, 384, 384))
        dx = 0.15
        nb = batch or 1
        lx, ly, lz = nx * dx, ny * dx, nz * dx
        # "config-1 slab physics, scaled" (reading 19): config 1's fractions of the box -- slab top at 0.38 Lz,
        # packet at 0.2 Lz, detector plane at 10/128 of the box height -- on the larger grid
        slab = fcc111_slab(lx, ly, CFG4_ZTOP_FRAC * lz, 4)
        atoms, seeds = [], []
        for b in range(nb):
            atoms.append(slab if b == 0 else _thermal(slab, 4000 + b))
            seeds.append(None if b == 0 else 4000 + b)
        absorb = min(16, max(nz // 8, 0))
        return Workload(
            name=CONFIG_NAMES[4] + ("_%dc_%s" % (nx, dt_)), nx=nx, ny=ny, nz=nz, batch=nb, dtype=dt_,
            dx=dx, dt=_dt_rule(dx, 200.0), mass=mass, hbar=hbar,
            bc=(PERIODIC, PERIODIC, DIRICHLET), absorb_lo=absorb, absorb_hi=absorb, strength=0.05, power=2,
            atoms=atoms, vmin=-200.0, vmax=0.0, rcut=16.0,
            packet=dict(x0=lx / 2, y0=ly / 2, z0=0.2 * lz, sigma=4.0, kx=0.0, ky=0.0, kz=3.0, amplitude=0.0),
            k_det=min(max(1, (10 * nz + 64) // 128), nz - 1), every=10, steps=steps or 2000, seeds=seeds)

    raise ValueError("config index must be 0..4")


def shard_for_rank(w: Workload, idx: int, rank: int, world: int) -> Workload:
    """Weak-scaling shard of configuration `idx` for one rank.

    Entries are independent, so sharding is a partition of entry seeds with no exchange step:
    rank r owns global entries [r*batch, (r+1)*batch).  For cfg 3 each global entry g has film seed
    3000 + g; for cfg 2 / cfg 4 the thermal seed is base + g; cfg 0 / cfg 1 have no per-entry
    randomness (replicas).  rank 0 of any world size reproduces make_config(idx) exactly.
    """
    if world < 1 or not (0 <= rank < world):
        raise ValueError("rank/world")
    if rank == 0:
        return w
    lx, ly, lz = w.nx * w.dx, w.ny * w.dx, w.nz * w.dx
    g0 = rank * w.batch
    if idx == 3:
        z_top = 0.55 * lz
        slab = fcc111_slab(lx, ly, z_top, 3)
        atoms, seeds = [], []
        for b in range(w.batch):
            seed = 3000 + g0 + b
            film = _film_atoms(np.random.default_rng(seed), lx, ly, z_top, 12, 0.1, 0.5)
            atoms.append(np.concatenate([slab, film], axis=0)); seeds.append(seed)
        return w.with_(atoms=atoms, seeds=seeds)
    if idx == 2:
        slab = fcc111_slab(lx, ly, 0.5 * lz, 6)
        seeds = [2 + g0 + b for b in range(w.batch)]
        return w.with_(atoms=[_thermal(slab, s) for s in seeds], seeds=seeds)
    if idx == 4:
        slab = fcc111_slab(lx, ly, CFG4_ZTOP_FRAC * lz, 4)
        seeds = [4000 + g0 + b for b in range(w.batch)]
        return w.with_(atoms=[_thermal(slab, s) for s in seeds], seeds=seeds)
    return w


def random_state(seed: int, shape: Sequence[int], dtype=np.float64) -> Tuple[np.ndarray, np.ndarray]:
    """Seeded smooth-free random (R, I_half) pair for raw-state parity cases."""
    rng = np.random.default_rng(seed)
    r = rng.standard_normal(size=tuple(shape)).astype(dtype)
    i = rng.standard_normal(size=tuple(shape)).astype(dtype)
    return r, i


def random_potential(seed: int, shape: Sequence[int], lo: float, hi: float, dtype=np.float64) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.uniform(lo, hi, size=tuple(shape)).astype(dtype)


# ------------------------------------------------------------------------------------------------
# The paper's own mesh (section 2.3), as inputs only: sizes, spacings, a synthetic unit-cell
# potential per configuration, packet and detector parameters.  Stands in for the DFT potentials, which are not available.
# ------------------------------------------------------------------------------------------------
BOHR_PER_ANGSTROM = 1.0 / 0.529177210903
HARTREE_PER_EV = 1.0 / 27.211386245988


@dataclass
class PaperMesh:
    name: str
    nx: int
    ny: int
    nz: int                         # 420 cell planes + 100 absorber planes appended below
    batch: int
    dtype: str
    dx: float
    dy: float
    dz: float
    dt: float                       # eq (11)
    bc: Tuple[int, int, int]        # periodic on all three axes
    absorb_lo: int                  # 100 planes at the bottom, none at the top
    absorb_hi: int
    strength: float
    power: int
    cells_mz_my_mx: Tuple[int, int, int]
    cell_edges: Tuple[float, float, float]
    cell_origin: Tuple[float, float, float]
    unit_cells: List[np.ndarray]    # one [mz][my][mx] float64 grid per configuration
    vmin: float
    vmax: float
    packet: dict
    k_det: int
    every: int                      # h = 20
    steps: int                      # 5000
    mass: float = 1.0
    hbar: float = 1.0

    @property
    def cells(self) -> int:
        return self.nx * self.ny * self.nz


def paper_mesh(batch: int = 8, steps: int = 5000, n: Optional[Sequence[int]] = None, seed: int = 5000,
               dtype: str = "f32") -> PaperMesh:
    """240 x 240 x (420 + 100) points on the 35.4 x 40.9 x 70.0 Angstrom domain: anisotropic spacings,
    a 16 x 16 x 420 unit cell repeated 15 x 15 times in x and y, a 100-plane absorber appended below the cell, periodic
    on all axes; packet above the surface at r_z = 42.0 A moving down with E = 60 eV, sigma = 1.8 A;
    detector plane at z_det = 37.6 A, a frame every h = 20 steps; 5000 steps (the data-set runs).
    `n` = (nx, ny, nz_cell) shrinks the mesh for tests (nx, ny multiples of 16; the absorber keeps nz_cell * 100 // 420 planes).
    The unit-cell potential is synthetic: four attractive atomic layers below 28.35 A with a lateral corrugation, plus a
    seeded smooth bump per configuration above the top layer (standing in for one C6-SAM orientation)."""
    nx, ny, nzc = n or (240, 240, 420)
    assert nx % 16 == 0 and ny % 16 == 0
    nabs = 100 * nzc // 420
    A = BOHR_PER_ANGSTROM
    dx, dy, dz = 35.4 * A / 240, 40.9 * A / 240, 70.0 * A / 420
    mx, my, mz = 16, 16, nzc
    ax, ay, az = mx * dx, my * dy, (mz - 1) * dz
    zs = np.arange(mz) * dz                                   # heights above the bottom of the cell
    scale = nzc / 420.0                                       # reduced meshes keep the proportions along z
    z_top = 28.35 * A * scale
    xs, ys = np.arange(mx) / mx, np.arange(my) / my
    corr = 1.0 + 0.3 * np.cos(2 * np.pi * xs)[None, None, :] * np.cos(2 * np.pi * ys)[None, :, None]
    base = np.zeros((mz, my, mx))
    for layer in range(4):
        zc = z_top - layer * 2.08 * A * scale
        base += -18.0 * np.exp(-0.5 * ((zs - zc) / (0.45 * A * scale)) ** 2)[:, None, None] * corr
    cells = []
    for b in range(batch):
        rng = np.random.default_rng(seed + b)
        cx, cy = rng.uniform(0, 1, 2)
        zc = z_top + rng.uniform(1.0, 6.0) * A * scale
        bump = (-6.0 * np.exp(-0.5 * ((zs - zc) / (1.2 * A * scale)) ** 2)[:, None, None]
                * (1.0 + 0.8 * np.cos(2 * np.pi * (xs - cx))[None, None, :] * np.cos(2 * np.pi * (ys - cy))[None, :, None]))
        cells.append(np.ascontiguousarray(base + bump))
    energy = 60.0 * HARTREE_PER_EV
    k = math.sqrt(2.0 * energy)                               # = 2 pi / lambda of eq (4), PAPER.md:56 (hbar = m = 1)
    lx, ly = nx * dx, ny * dy
    z0 = (nabs + 42.0 / 70.0 * (nzc - 1)) * dz
    k_det = nabs + int(round(37.6 / 70.0 * (nzc - 1)))
    return PaperMesh(
        name="paper_mesh_%dx%dx%d_%s" % (nx, ny, nzc + nabs, dtype), nx=nx, ny=ny, nz=nzc + nabs, batch=batch, dtype=dtype,
        dx=dx, dy=dy, dz=dz, dt=0.2 * min(dx, dy, dz) ** 2,
        bc=(PERIODIC, PERIODIC, PERIODIC), absorb_lo=nabs, absorb_hi=0, strength=0.05, power=2,
        cells_mz_my_mx=(mz, my, mx), cell_edges=(ax, ay, az), cell_origin=(0.0, 0.0, nabs * dz), unit_cells=cells,
        vmin=-50.0, vmax=0.0,
        packet=dict(x0=lx / 2, y0=ly / 2, z0=z0, sigma=1.8 * A * scale, kx=0.0, ky=0.0, kz=-k, amplitude=0.0),
        k_det=k_det, every=20, steps=steps)
