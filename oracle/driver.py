"""ctypes driver around oracle/tdse_oracle.c (TEST INFRASTRUCTURE -- see package docstring).

No arithmetic of the method happens here beyond the coefficient definitions of PAPER.md:87
(`coefficients`) and dtype rounding of inputs; every loop lives in the C file.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
import threading
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = [os.path.join(_HERE, "tdse_oracle.c"), os.path.join(_HERE, "tdse_oracle_step.inc")]
_SO = os.path.join(_HERE, "_build", "liboracle_tdse.so")
_LOCK = threading.Lock()

PERIODIC, DIRICHLET = 0, 1


_FLAGS = {
    # the build every parity test and pin runs: no FMA contraction, literal grouping of eqs (8)-(9)
    "parity": ["-O2", "-ffp-contract=off"],
    # the same source with the flags BASELINE.md section 3 names for the timed serial / OpenMP figures; timing only
    "timing": ["-O3", "-march=native"],
}
_LIBS = {}


def _so_path(variant: str) -> str:
    return _SO if variant == "parity" else _SO.replace(".so", "_%s.so" % variant)


def build(force: bool = False, variant: str = "parity") -> str:
    """Compile the oracle with gcc (parity: -O2 -ffp-contract=off -fopenmp). Returns the .so path."""
    so = _so_path(variant)
    os.makedirs(os.path.dirname(so), exist_ok=True)
    newest = max(os.path.getmtime(p) for p in _SRC)
    if force or not os.path.exists(so) or os.path.getmtime(so) < newest:
        tmp = so + ".tmp.%d" % os.getpid()
        cmd = ["gcc"] + _FLAGS[variant] + ["-fopenmp", "-std=c99", "-shared", "-fPIC", "-o", tmp, _SRC[0], "-lm"]
        subprocess.run(cmd, check=True, cwd=_HERE)
        os.replace(tmp, so)
    return so


def lib(variant: str = "parity"):
    with _LOCK:
        if variant not in _LIBS:
            L = C.CDLL(build(variant=variant))
            dp, fp, ip = C.POINTER(C.c_double), C.POINTER(C.c_float), C.POINTER(C.c_int)
            L.oracle_max_threads.restype = C.c_int
            L.oracle_set_threads.argtypes = [C.c_int]
            L.oracle_potential.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [C.c_int] * 3 + \
                [dp, C.c_int, C.c_double, C.c_double, C.c_double, dp]
            L.oracle_mask.argtypes = [C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, dp]
            L.oracle_wavepacket.argtypes = [C.c_int] * 3 + [C.c_double] * 11 + [dp, dp]
            L.oracle_stagger.argtypes = [C.c_int] * 6 + [C.c_double] * 4 + [dp, dp, dp, dp]
            for sfx, rp in (("f64", dp), ("f32", fp)):
                f = getattr(L, "oracle_step_" + sfx)
                f.restype = C.c_int
                f.argtypes = [C.c_int] * 6 + [C.c_double] * 4 + [rp, rp, rp, rp, C.c_int,
                              C.POINTER(C.c_longlong), C.c_int, C.c_int, C.c_double,
                              dp, dp, C.c_int, ip]
                g = getattr(L, "oracle_norm_" + sfx)
                g.restype = None
                g.argtypes = [C.c_int] * 6 + [C.c_double] * 5 + [rp, rp, rp, rp, dp, dp]
                h = getattr(L, "oracle_plane_density_" + sfx)
                h.restype = None
                h.argtypes = [C.c_int] * 3 + [rp, rp, dp]
            L.oracle_potential_cell.argtypes = [C.c_int] * 3 + [C.c_double] * 3 + [dp] + [C.c_int] * 3 + [C.c_double] * 8 + [dp]
            L.oracle_dissimilarity.restype = C.c_double
            L.oracle_dissimilarity.argtypes = [dp, dp, C.c_int, C.c_double, C.c_int, C.c_int]
            _LIBS[variant] = L
    return _LIBS[variant]


def max_threads(variant: str = "parity") -> int:
    return int(lib(variant).oracle_max_threads())


def set_threads(n: int, variant: str = "parity") -> None:
    lib(variant).oracle_set_threads(int(n))


def _p(a: np.ndarray, ct):
    return a.ctypes.data_as(C.POINTER(ct))


def coefficients(dx: float, dt: float, mass: float, hbar: float,
                 dy: Optional[float] = None, dz: Optional[float] = None) -> Tuple[float, float, float, float]:
    """c_x = hbar dt/(2 m dx^2) (same for y, z), c_v = dt/hbar."""
    dy = dx if dy is None else dy
    dz = dx if dz is None else dz
    return (hbar * dt / (2.0 * mass * dx * dx), hbar * dt / (2.0 * mass * dy * dy),
            hbar * dt / (2.0 * mass * dz * dz), dt / hbar)


def paper_time_step(dx: float, dy: float, dz: float, mass: float, hbar: float) -> float:
    """eq (11): dt = (m / 5 hbar) min(dx, dy, dz)^2."""
    return mass / (5.0 * hbar) * min(dx, dy, dz) ** 2


def paper_wavelength(energy: float, mass: float, hbar: float) -> float:
    """eq (4): lambda = sqrt(2 hbar^2 pi^2 / (m E))."""
    return float(np.sqrt(2.0 * hbar * hbar * np.pi ** 2 / (mass * energy)))


def potential(nx, ny, nz, dx, bc, atoms, vmin, vmax, rcut=0.0, dy=None, dz=None) -> np.ndarray:
    atoms = np.ascontiguousarray(np.asarray(atoms, dtype=np.float64).reshape(-1, 6))
    V = np.empty((nz, ny, nx), dtype=np.float64)
    dy = dx if dy is None else dy
    dz = dx if dz is None else dz
    lib().oracle_potential(nx, ny, nz, dx, dy, dz, bc[0], bc[1], bc[2], _p(atoms, C.c_double),
                           atoms.shape[0], vmin, vmax, rcut, _p(V, C.c_double))
    return V


def potential_cell(nx, ny, nz, dx, cell, a, origin, vmin, vmax, dy=None, dz=None) -> np.ndarray:
    """Unit-cell potential cell[mz][my][mx] of edge lengths a = (ax, ay, az), tiled in x, y and trilinearly
    interpolated onto the mesh."""
    cell = np.ascontiguousarray(cell, dtype=np.float64)
    mz, my, mx = cell.shape
    V = np.empty((nz, ny, nx), dtype=np.float64)
    dy = dx if dy is None else dy
    dz = dx if dz is None else dz
    lib().oracle_potential_cell(nx, ny, nz, dx, dy, dz, _p(cell, C.c_double), mx, my, mz, a[0], a[1], a[2],
                                origin[0], origin[1], origin[2], vmin, vmax, _p(V, C.c_double))
    return V


def mask(nz, w_lo, w_hi, strength=0.05, power=2) -> np.ndarray:
    M = np.empty(nz, dtype=np.float64)
    lib().oracle_mask(nz, w_lo, w_hi, strength, power, _p(M, C.c_double))
    return M


def wavepacket(nx, ny, nz, dx, x0, y0, z0, sigma, kx, ky, kz, amplitude=0.0, dy=None, dz=None):
    R0 = np.empty((nz, ny, nx), dtype=np.float64)
    J0 = np.empty((nz, ny, nx), dtype=np.float64)
    dy = dx if dy is None else dy
    dz = dx if dz is None else dz
    lib().oracle_wavepacket(nx, ny, nz, dx, dy, dz, x0, y0, z0, sigma, kx, ky, kz, amplitude,
                            _p(R0, C.c_double), _p(J0, C.c_double))
    return R0, J0


def stagger(bc, coef, V, R0, J0) -> np.ndarray:
    nz, ny, nx = R0.shape
    V = np.ascontiguousarray(V, dtype=np.float64)
    out = np.empty_like(R0)
    lib().oracle_stagger(nx, ny, nz, bc[0], bc[1], bc[2], coef[0], coef[1], coef[2], coef[3],
                         _p(V, C.c_double), _p(R0, C.c_double), _p(J0, C.c_double), _p(out, C.c_double))
    return out


def dissimilarity(frames_k, frames_j, dA: float, s0: int, s1: int) -> float:
    """eq (16), over the frames s0..s1 (inclusive) of two [nframes][ny][nx] trajectories."""
    a = np.ascontiguousarray(frames_k, dtype=np.float64)
    b = np.ascontiguousarray(frames_j, dtype=np.float64)
    assert a.shape == b.shape and 0 <= s0 <= s1 < a.shape[0]
    npix = int(np.prod(a.shape[1:]))
    return float(lib().oracle_dissimilarity(_p(a, C.c_double), _p(b, C.c_double), npix, float(dA), int(s0), int(s1)))


class OracleRun:
    """One batch entry of the hot path, step by step.

    dtype: arithmetic type of the recurrence ("f64" | "f32").
    round_to: if "f32" while dtype == "f64", every input (V, M, R0, I_half, coefficients) is
    rounded to float and promoted back, so that the run is the exact-arithmetic image of an
    fp32 run (used as the truth for fp32 parity).
    """

    def __init__(self, nx, ny, nz, dx, dt, mass=1.0, hbar=1.0, dtype="f64",
                 bc=(DIRICHLET, DIRICHLET, DIRICHLET), absorb_lo=0, absorb_hi=0,
                 strength=0.05, power=2, round_to: Optional[str] = None, dy=None, dz=None):
        assert dtype in ("f64", "f32")
        self.nx, self.ny, self.nz = int(nx), int(ny), int(nz)
        self.dx, self.dt, self.mass, self.hbar = float(dx), float(dt), float(mass), float(hbar)
        self.dy = self.dx if dy is None else float(dy)       # anisotropic mesh of the paper
        self.dz = self.dx if dz is None else float(dz)
        self.dtype = dtype
        self.np = np.float64 if dtype == "f64" else np.float32
        self.round_to = round_to if round_to else dtype
        self.bc = tuple(int(b) for b in bc)
        coef = coefficients(dx, dt, mass, hbar, self.dy, self.dz)
        self.coef = tuple(self._round_scalar(c) for c in coef)
        self.M = self._round(mask(self.nz, absorb_lo, absorb_hi, strength, power))
        self.V = None
        self.R = None
        self.I = None
        self.k_det, self.every = 0, 0
        self.D = np.zeros((self.ny, self.nx), dtype=np.float64)
        self.trace = []
        self.counter = C.c_longlong(0)
        self.keep_frames, self.include_t0 = False, True
        self.frames = []              # frame mode: rho at s = 0 (optional), h, 2h, ...
        self.step_variant = "parity"  # bench.py's timed legs may switch the recurrence to the "timing" build

    # -- rounding of inputs to the run's storage dtype --------------------------------
    def _round(self, a: np.ndarray) -> np.ndarray:
        a = np.asarray(a, dtype=np.float64)
        if self.round_to == "f32":
            a = a.astype(np.float32)
        return np.ascontiguousarray(a.astype(self.np))

    def _round_scalar(self, x: float) -> float:
        return float(np.float32(x)) if self.round_to == "f32" else float(x)

    # -- inputs ---------------------------------------------------------------------
    def set_potential_atoms(self, atoms, vmin, vmax, rcut=0.0):
        self.V64 = potential(self.nx, self.ny, self.nz, self.dx, self.bc, atoms, vmin, vmax, rcut, self.dy, self.dz)
        self.V = self._round(self.V64)
        return self

    def set_potential_cell(self, cell, a, origin, vmin, vmax):
        self.V64 = potential_cell(self.nx, self.ny, self.nz, self.dx, cell, a, origin, vmin, vmax, self.dy, self.dz)
        self.V = self._round(self.V64)
        return self

    def set_potential_grid(self, V):
        self.V64 = np.asarray(V, dtype=np.float64).reshape(self.nz, self.ny, self.nx)
        self.V = self._round(self.V64)
        return self

    def set_wavepacket(self, x0, y0, z0, sigma, kx, ky, kz, amplitude=0.0):
        assert self.V is not None, "potential first (the staggered start needs V)"
        R0, J0 = wavepacket(self.nx, self.ny, self.nz, self.dx, x0, y0, z0, sigma, kx, ky, kz, amplitude, self.dy, self.dz)
        Ih = stagger(self.bc, coefficients(self.dx, self.dt, self.mass, self.hbar, self.dy, self.dz),
                     self.V.astype(np.float64), R0, J0)
        self.R, self.I = self._round(R0), self._round(Ih)
        self.counter = C.c_longlong(0)
        return self

    def set_state(self, R, I_half):
        self.R = self._round(np.asarray(R).reshape(self.nz, self.ny, self.nx))
        self.I = self._round(np.asarray(I_half).reshape(self.nz, self.ny, self.nx))
        self.counter = C.c_longlong(0)
        return self

    def set_detector(self, k_plane, every):
        self.k_det, self.every = int(k_plane), int(every)
        self.D[:] = 0.0
        self.trace = []
        self.counter = C.c_longlong(0)
        return self

    def set_frames(self, keep: bool = True, include_t0: bool = True):
        """Frame mode: keep every sampled detector frame (the paper's trajectory rho = {rho(0), rho(h dt), ...})."""
        self.keep_frames, self.include_t0 = bool(keep), bool(include_t0)
        self.frames = []
        return self

    def plane_density(self) -> np.ndarray:
        ct = C.c_double if self.dtype == "f64" else C.c_float
        rho = np.empty((self.ny, self.nx), dtype=np.float64)
        getattr(lib(), "oracle_plane_density_" + self.dtype)(self.nx, self.ny, self.k_det, _p(self.R, ct), _p(self.I, ct),
                                                             _p(rho, C.c_double))
        return rho

    # -- the recurrence -------------------------------------------------------------
    def step(self, n: int):
        assert self.V is not None and self.R is not None
        if self.keep_frames and self.every > 0:
            # advance from one sampling step to the next so that a frame can be taken from the state in memory
            if self.counter.value == 0 and self.include_t0 and not self.frames:
                self.frames.append(self.plane_density())
            left = int(n)
            while left > 0:
                m = min(left, self.every - int(self.counter.value % self.every))
                self._advance(m)
                left -= m
                if self.counter.value % self.every == 0:
                    self.frames.append(self.plane_density())
            return self
        return self._advance(n)

    def _advance(self, n: int):
        ct = C.c_double if self.dtype == "f64" else C.c_float
        f = getattr(lib(self.step_variant), "oracle_step_" + self.dtype)
        cap = n // self.every + 2 if self.every > 0 else 1
        tr = np.zeros(cap, dtype=np.float64)
        ns = C.c_int(0)
        f(self.nx, self.ny, self.nz, *self.bc, *self.coef,
          _p(self.V, ct), _p(self.M, ct), _p(self.R, ct), _p(self.I, ct), int(n),
          C.byref(self.counter), self.k_det, self.every, self.dx * self.dy,
          _p(self.D, C.c_double), _p(tr, C.c_double), cap, C.byref(ns))
        self.trace.extend(tr[: ns.value].tolist())
        return self

    def norm(self) -> Tuple[float, float]:
        ct = C.c_double if self.dtype == "f64" else C.c_float
        g = getattr(lib(), "oracle_norm_" + self.dtype)
        qv, qp = C.c_double(0), C.c_double(0)
        g(self.nx, self.ny, self.nz, *self.bc, *self.coef, self.dx * self.dy * self.dz,
          _p(self.V, ct), _p(self.M, ct), _p(self.R, ct), _p(self.I, ct), C.byref(qv), C.byref(qp))
        return qv.value, qp.value

    @classmethod
    def from_workload(cls, w, entry: int = 0, dtype: Optional[str] = None,
                      round_to: Optional[str] = None) -> "OracleRun":
        """Set up batch entry `entry` of a workloads.Workload (inputs only; no stepping)."""
        o = cls(w.nx, w.ny, w.nz, w.dx, w.dt, w.mass, w.hbar, dtype or w.dtype, w.bc,
                w.absorb_lo, w.absorb_hi, w.strength, w.power, round_to=round_to,
                dy=getattr(w, "dy", None), dz=getattr(w, "dz", None))
        o.set_potential_atoms(w.atoms[entry], w.vmin, w.vmax, w.rcut)
        o.set_wavepacket(**w.packet)
        o.set_detector(w.k_det, w.every)
        return o
