"""Thin ctypes binding over libtdse.so (include/tdse.h).  Argument marshalling only.

Every step of the path runs in the library's CUDA kernels; PyTorch is used for device memory
(the workspace tensor) and the CUDA stream handle.  There is no CPU fallback: if libtdse.so has
not been built, or no CUDA device is present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Optional, Sequence, Tuple

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libtdse.so")

TDSE_F32, TDSE_F64 = 0, 1
TDSE_BC_PERIODIC, TDSE_BC_DIRICHLET = 0, 1
TDSE_OK, TDSE_EINVAL, TDSE_ENOMEM, TDSE_ECUDA, TDSE_ESTATE, TDSE_EUNSTABLE = 0, -1, -2, -3, -4, -5
TDSE_KERNEL_AUTO, TDSE_KERNEL_TWOPASS, TDSE_KERNEL_FUSED = 0, 1, 2

_ERRNAMES = {TDSE_EINVAL: "TDSE_EINVAL", TDSE_ENOMEM: "TDSE_ENOMEM", TDSE_ECUDA: "TDSE_ECUDA",
             TDSE_ESTATE: "TDSE_ESTATE", TDSE_EUNSTABLE: "TDSE_EUNSTABLE"}

# every symbol include/tdse.h declares (tests check that the library exports all of them)
SYMBOLS = [
    "tdse_create", "tdse_destroy", "tdse_workspace_bytes", "tdse_bind", "tdse_set_boundary",
    "tdse_set_potential", "tdse_set_potential_device", "tdse_set_potential_grid",
    "tdse_set_wavepacket", "tdse_set_state", "tdse_set_detector", "tdse_step",
    "tdse_detector_read", "tdse_detector_device", "tdse_read_psi", "tdse_read_potential",
    "tdse_norm", "tdse_set_option", "tdse_get_info", "tdse_last_error",
    "tdse_set_frames", "tdse_frames_read", "tdse_frames_device", "tdse_dissimilarity", "tdse_set_spacing", "tdse_set_potential_cell", "tdse_set_potential_batch", "tdse_set_frame_stream", "tdse_frames_sync",
    "tdse_dissimilarity_static",
]

TDSE_STATIC_SCRATCH_DOUBLES = 262144   # include/tdse.h: size of the fixed scratch array behind tdse_dissimilarity_static


class TdseError(RuntimeError):
    def __init__(self, code: int, where: str, text: str):
        super().__init__("%s failed with %s (%d): %s" % (where, _ERRNAMES.get(code, "?"), code, text))
        self.code = code


class Atom(C.Structure):
    _fields_ = [(n, C.c_double) for n in ("x", "y", "z", "Z", "soft2", "screen")]


_lib = None


def load():
    """dlopen libtdse.so and declare the prototypes.  Raises if the library has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise RuntimeError("libtdse.so is missing at %s: run `python -m paper_2401_07416_b200.build` "
                           "(or __graft_entry__.build()); there is no CPU fallback" % LIB_PATH)
    L = C.CDLL(LIB_PATH)
    vp, ip, dp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_double)
    L.tdse_create.argtypes = [C.POINTER(vp)] + [C.c_int] * 4 + [C.c_double] * 4 + [C.c_int]
    L.tdse_destroy.argtypes = [vp]
    L.tdse_workspace_bytes.argtypes = [C.c_int] * 6
    L.tdse_workspace_bytes.restype = C.c_size_t
    L.tdse_bind.argtypes = [vp, vp, C.c_size_t, vp]
    L.tdse_set_boundary.argtypes = [vp] + [C.c_int] * 5 + [C.c_double, C.c_int]
    L.tdse_set_potential.argtypes = [vp, C.c_int, C.POINTER(Atom), C.c_int] + [C.c_double] * 3
    L.tdse_set_potential_device.argtypes = [vp, C.c_int, vp, C.c_int] + [C.c_double] * 3
    L.tdse_set_potential_grid.argtypes = [vp, C.c_int, vp, C.c_int]
    L.tdse_set_potential_batch.argtypes = [vp, vp, ip, C.c_int] + [C.c_double] * 3
    L.tdse_set_wavepacket.argtypes = [vp, C.c_int] + [C.c_double] * 8
    L.tdse_set_state.argtypes = [vp, C.c_int, vp, vp, C.c_int]
    L.tdse_set_detector.argtypes = [vp, C.c_int, C.c_int, C.c_int]
    L.tdse_step.argtypes = [vp, C.c_int]
    L.tdse_detector_read.argtypes = [vp, C.c_int, dp, dp, C.c_int, ip]
    L.tdse_detector_device.argtypes = [vp, C.POINTER(vp), C.POINTER(vp), ip]
    L.tdse_set_spacing.argtypes = [vp, C.c_double, C.c_double]
    L.tdse_set_potential_cell.argtypes = [vp, C.c_int, vp, C.c_int] + [C.c_int] * 3 + [C.c_double] * 8
    L.tdse_set_frames.argtypes = [vp, C.c_int, C.c_int]
    L.tdse_frames_read.argtypes = [vp, C.c_int, C.c_int, C.c_int, dp, ip]
    L.tdse_frames_device.argtypes = [vp, C.POINTER(vp), ip, ip]
    L.tdse_set_frame_stream.argtypes = [vp, dp, C.c_int, C.c_int, C.c_int]
    L.tdse_frames_sync.argtypes = [vp, ip]
    L.tdse_dissimilarity.argtypes = [vp, C.c_int, C.c_int, dp]
    L.tdse_dissimilarity_static.argtypes = [vp] + [C.c_int] * 4 + [C.c_double, C.c_int, C.c_int, vp, vp]
    L.tdse_read_psi.argtypes = [vp, C.c_int, vp, vp]
    L.tdse_read_potential.argtypes = [vp, C.c_int, vp]
    L.tdse_norm.argtypes = [vp, C.c_int, dp, dp]
    L.tdse_set_option.argtypes = [vp, C.c_char_p, C.c_longlong]
    L.tdse_get_info.argtypes = [vp, C.c_char_p, C.POINTER(C.c_longlong)]
    L.tdse_last_error.argtypes = [vp]
    L.tdse_last_error.restype = C.c_char_p
    for name in SYMBOLS:
        f = getattr(L, name)
        if name not in ("tdse_workspace_bytes", "tdse_last_error"):
            f.restype = C.c_int
    _lib = L
    return L


def dissimilarity_static(frames, first_frame, last_frame, dA, out, stream=None):
    """tdse_dissimilarity_static: eq (16) for callers that may not allocate GPU memory (a job that gave all of HBM to the
    grids, a process whose device memory belongs to one pool, a loop that cannot take cudaMalloc's device-wide stall).

    frames: device tensor [batch][frames_per_entry][ny][nx], float64, contiguous; out: device tensor [batch][batch],
    float64, contiguous -- both on the current device, both the caller's.  Nothing is allocated here or in the library:
    the partial sums go to a fixed 2 MiB array inside libtdse.so that all calls on a GPU share (so calls that may
    overlap on the GPU must be ordered by the caller).  Asynchronous on `stream`; raises TdseError(TDSE_EINVAL) when
    batch*batch*frames exceeds TDSE_STATIC_SCRATCH_DOUBLES.  The first call on a GPU looks up the array's address and
    belongs in set-up code, ahead of any stream capture."""
    L = load()
    batch, per_entry, ny, nx = (int(v) for v in frames.shape)
    sptr = stream.cuda_stream if stream is not None else 0
    code = L.tdse_dissimilarity_static(frames.data_ptr(), batch, per_entry, ny, nx, float(dA), int(first_frame),
                                       int(last_frame), out.data_ptr(), sptr)
    if code != TDSE_OK:
        raise TdseError(code, "tdse_dissimilarity_static", (L.tdse_last_error(None) or b"").decode())
    return out


def atoms_array(atoms) -> "C.Array":
    a = np.ascontiguousarray(np.asarray(atoms, dtype=np.float64).reshape(-1, 6))
    arr = (Atom * max(a.shape[0], 1))()
    C.memmove(arr, a.ctypes.data, a.nbytes)
    return arr, a.shape[0]


class Tdse:
    """One libtdse context.  Method names mirror the C calls without the `tdse_` prefix."""

    def __init__(self, nx, ny, nz, batch=1, dx=1.0, dt=1.0, mass=1.0, hbar=1.0, dtype="f64",
                 pingpong: bool = True, stream=None, device="cuda:0"):
        import torch
        self._torch = torch
        self.L = load()
        self.nx, self.ny, self.nz, self.batch = int(nx), int(ny), int(nz), int(batch)
        self.dx = float(dx)
        self.dtype = dtype
        self.np_dtype = np.float32 if dtype == "f32" else np.float64
        self._h = C.c_void_p()
        self.device = torch.device(device)
        # tdse_create records the current device; every later call runs there whatever device is current then
        with torch.cuda.device(self.device):
            code = self.L.tdse_create(C.byref(self._h), self.nx, self.ny, self.nz, self.batch,
                                      float(dx), float(dt), float(mass), float(hbar),
                                      TDSE_F32 if dtype == "f32" else TDSE_F64)
        if code != TDSE_OK:
            raise TdseError(code, "tdse_create", (self.L.tdse_last_error(None) or b"").decode())
        nbytes = self.L.tdse_workspace_bytes(self.nx, self.ny, self.nz, self.batch,
                                             TDSE_F32 if dtype == "f32" else TDSE_F64, 1 if pingpong else 0)
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)   # torch owns the memory
        self.stream = stream
        sptr = stream.cuda_stream if stream is not None else 0
        self._check(self.L.tdse_bind(self._h, self.workspace.data_ptr(), nbytes, sptr), "tdse_bind")

    # -- plumbing ---------------------------------------------------------------------------
    def _check(self, code, where):
        if code != TDSE_OK:
            raise TdseError(code, where, (self.L.tdse_last_error(self._h) or b"").decode())

    def close(self):
        if getattr(self, "_h", None) is not None and self._h:
            self.L.tdse_destroy(self._h)     # synchronises both streams: the host frame buffer may go afterwards
            self._h = C.c_void_p()
            self._frames_host = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # -- the C calls -------------------------------------------------------------------------
    def set_boundary(self, bcx, bcy, bcz, absorb_lo=0, absorb_hi=0, strength=0.05, power=2):
        self._check(self.L.tdse_set_boundary(self._h, bcx, bcy, bcz, absorb_lo, absorb_hi, strength, power),
                    "tdse_set_boundary")

    def set_potential(self, b, atoms, vmin, vmax, rcut=0.0):
        arr, n = atoms_array(atoms)
        self._check(self.L.tdse_set_potential(self._h, b, arr, n, vmin, vmax, rcut), "tdse_set_potential")

    def set_potential_device(self, b, atoms_tensor, natoms, vmin, vmax, rcut=0.0):
        self._check(self.L.tdse_set_potential_device(self._h, b, atoms_tensor.data_ptr(), natoms, vmin, vmax, rcut),
                    "tdse_set_potential_device")

    def set_potential_batch(self, atoms, offsets, vmin, vmax, rcut=0.0):
        """atoms: concatenated [total][6] list (numpy array on the host, or a device tensor); offsets: batch + 1 ints."""
        off = np.ascontiguousarray(offsets, dtype=np.int32)
        assert off.size == self.batch + 1
        if hasattr(atoms, "data_ptr"):
            ptr, dev = atoms.data_ptr(), 1
        else:
            atoms = np.ascontiguousarray(np.asarray(atoms, dtype=np.float64).reshape(-1, 6))
            ptr, dev = atoms.ctypes.data, 0
        self._check(self.L.tdse_set_potential_batch(self._h, ptr, off.ctypes.data_as(C.POINTER(C.c_int)), dev, vmin, vmax, rcut),
                    "tdse_set_potential_batch")

    def set_potential_cell(self, b, cell, a, origin, vmin, vmax):
        if hasattr(cell, "data_ptr"):
            mz, my, mx = cell.shape
            ptr, dev = cell.data_ptr(), 1
        else:
            cell = np.ascontiguousarray(cell, dtype=np.float64)
            mz, my, mx = cell.shape
            ptr, dev = cell.ctypes.data, 0
        self._check(self.L.tdse_set_potential_cell(self._h, b, ptr, dev, mx, my, mz, float(a[0]), float(a[1]), float(a[2]),
                                                   float(origin[0]), float(origin[1]), float(origin[2]), vmin, vmax),
                    "tdse_set_potential_cell")

    def set_potential_grid(self, b, V):
        if hasattr(V, "data_ptr"):
            self._check(self.L.tdse_set_potential_grid(self._h, b, V.data_ptr(), 1), "tdse_set_potential_grid")
        else:
            V = np.ascontiguousarray(V, dtype=self.np_dtype)
            assert V.size == self.nx * self.ny * self.nz
            self._check(self.L.tdse_set_potential_grid(self._h, b, V.ctypes.data, 0), "tdse_set_potential_grid")

    def set_wavepacket(self, b, x0, y0, z0, sigma, kx, ky, kz, amplitude=0.0):
        self._check(self.L.tdse_set_wavepacket(self._h, b, x0, y0, z0, sigma, kx, ky, kz, amplitude),
                    "tdse_set_wavepacket")

    def set_state(self, b, R, I_half):
        if hasattr(R, "data_ptr"):
            self._check(self.L.tdse_set_state(self._h, b, R.data_ptr(), I_half.data_ptr(), 1), "tdse_set_state")
        else:
            R = np.ascontiguousarray(R, dtype=self.np_dtype)
            I_half = np.ascontiguousarray(I_half, dtype=self.np_dtype)
            assert R.size == I_half.size == self.nx * self.ny * self.nz
            self._check(self.L.tdse_set_state(self._h, b, R.ctypes.data, I_half.ctypes.data, 0), "tdse_set_state")

    def set_detector(self, k_plane, every, max_samples=0):
        self.max_samples = int(max_samples)
        self._check(self.L.tdse_set_detector(self._h, k_plane, every, max_samples), "tdse_set_detector")

    def step(self, n):
        self._check(self.L.tdse_step(self._h, int(n)), "tdse_step")

    def detector_read(self, b) -> Tuple[np.ndarray, np.ndarray]:
        img = np.empty((self.ny, self.nx), dtype=np.float64)
        cap = max(getattr(self, "max_samples", 0), 1)
        tr = np.zeros(cap, dtype=np.float64)
        ns = C.c_int(0)
        self._check(self.L.tdse_detector_read(self._h, b, img.ctypes.data_as(C.POINTER(C.c_double)),
                                              tr.ctypes.data_as(C.POINTER(C.c_double)), cap, C.byref(ns)),
                    "tdse_detector_read")
        return img, tr[: min(ns.value, getattr(self, "max_samples", 0))]

    def detector_device(self):
        img, tr, ms = C.c_void_p(), C.c_void_p(), C.c_int(0)
        self._check(self.L.tdse_detector_device(self._h, C.byref(img), C.byref(tr), C.byref(ms)), "tdse_detector_device")
        return img.value, tr.value, ms.value

    def set_spacing(self, dy, dz):
        self._check(self.L.tdse_set_spacing(self._h, float(dy), float(dz)), "tdse_set_spacing")

    def set_frames(self, max_frames, include_t0=True):
        self._check(self.L.tdse_set_frames(self._h, int(max_frames), 1 if include_t0 else 0), "tdse_set_frames")

    def frames_read(self, b, first=0, count=None) -> np.ndarray:
        if count is None:
            count = self.get_info("nframes") - first
        out = np.empty((count, self.ny, self.nx), dtype=np.float64)
        n = C.c_int(0)
        self._check(self.L.tdse_frames_read(self._h, b, int(first), int(count), out.ctypes.data_as(C.POINTER(C.c_double)),
                                            C.byref(n)), "tdse_frames_read")
        return out

    def set_frame_stream(self, capacity, ring_slots=4, include_t0=True, pinned=True):
        """Streamed frame mode: torch owns the (page-locked) host buffer [batch][capacity][ny][nx]; the library fills it."""
        torch = self._torch
        fresh = None
        if capacity > 0:
            buf = torch.empty((self.batch, int(capacity), self.ny, self.nx), dtype=torch.float64)
            fresh = buf.pin_memory() if pinned else buf
        ptr = C.cast(fresh.data_ptr(), C.POINTER(C.c_double)) if capacity > 0 else None
        # The previous host buffer stays referenced until the library call has returned: that call is what waits for
        # copies still in flight into it (tdse.h: the buffer must stay valid until then), and torch's pinned-memory
        # allocator, which knows nothing of the library's copy stream, could otherwise hand the block out again.
        self._check(self.L.tdse_set_frame_stream(self._h, ptr, int(capacity), int(ring_slots), 1 if include_t0 else 0),
                    "tdse_set_frame_stream")
        self._frames_host = fresh

    def frames_sync(self) -> np.ndarray:
        """Frames landed so far as a numpy view [batch][nframes][ny][nx] of the host buffer."""
        n = C.c_int(0)
        self._check(self.L.tdse_frames_sync(self._h, C.byref(n)), "tdse_frames_sync")
        return self._frames_host.numpy()[:, : n.value]

    def dissimilarity(self, first_frame, last_frame) -> np.ndarray:
        d = np.empty((self.batch, self.batch), dtype=np.float64)
        self._check(self.L.tdse_dissimilarity(self._h, int(first_frame), int(last_frame),
                                              d.ctypes.data_as(C.POINTER(C.c_double))), "tdse_dissimilarity")
        return d

    def read_psi(self, b) -> Tuple[np.ndarray, np.ndarray]:
        R = np.empty((self.nz, self.ny, self.nx), dtype=self.np_dtype)
        I = np.empty((self.nz, self.ny, self.nx), dtype=self.np_dtype)
        self._check(self.L.tdse_read_psi(self._h, b, R.ctypes.data, I.ctypes.data), "tdse_read_psi")
        return R, I

    def read_potential(self, b) -> np.ndarray:
        V = np.empty((self.nz, self.ny, self.nx), dtype=self.np_dtype)
        self._check(self.L.tdse_read_potential(self._h, b, V.ctypes.data), "tdse_read_potential")
        return V

    def norm(self, b) -> Tuple[float, float]:
        qv, qp = C.c_double(0), C.c_double(0)
        self._check(self.L.tdse_norm(self._h, b, C.byref(qv), C.byref(qp)), "tdse_norm")
        return qv.value, qp.value

    def set_option(self, key: str, value: int):
        self._check(self.L.tdse_set_option(self._h, key.encode(), int(value)), "tdse_set_option")

    def get_info(self, key: str) -> int:
        v = C.c_longlong(0)
        self._check(self.L.tdse_get_info(self._h, key.encode(), C.byref(v)), "tdse_get_info")
        return int(v.value)

    # -- convenience: one workloads.Workload -> configured context -----------------------------
    @classmethod
    def from_workload(cls, w, **kw) -> "Tdse":
        t = cls(w.nx, w.ny, w.nz, w.batch, w.dx, w.dt, w.mass, w.hbar, w.dtype, **kw)
        if getattr(w, "dy", None) or getattr(w, "dz", None):
            t.set_spacing(w.dy or w.dx, w.dz or w.dx)
        t.set_boundary(*w.bc, w.absorb_lo, w.absorb_hi, w.strength, w.power)
        if w.batch > 1:
            t.set_potential_batch(np.concatenate(w.atoms, axis=0), np.concatenate([[0], np.cumsum([a.shape[0] for a in w.atoms])]),
                                  w.vmin, w.vmax, w.rcut)
        else:
            t.set_potential(0, w.atoms[0], w.vmin, w.vmax, w.rcut)
        p = w.packet
        t.set_wavepacket(-1, p["x0"], p["y0"], p["z0"], p["sigma"], p["kx"], p["ky"], p["kz"], p["amplitude"])
        t.set_detector(w.k_det, w.every, max(1, w.steps // max(w.every, 1)))
        return t
