"""ctypes binding of the CPU oracle (oracle/bte_ref.cpp).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl
reference` legs may import this package.  It imports nothing from the CUDA
package and shares no code with it.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libbte_ref.so")
_SRC = [os.path.join(_HERE, "bte_ref.cpp"), os.path.join(_HERE, "bte_ref.h")]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc: -O2 -ffp-contract=off (no FMA contraction)."""
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fPIC", "-shared", "-pthread",
           "-o", _SO, _SRC[0]]
    subprocess.run(cmd, check=True, cwd=_HERE)
    return _SO


class _BC(C.Structure):
    _fields_ = [("type", C.c_int32), ("dT_wall", C.c_double)]


class _Problem(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("dim", C.c_int32),
        ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
        ("solid_mask", C.c_void_p),
        ("n_bands", C.c_int32),
        ("C", C.c_void_p), ("v", C.c_void_p), ("tau", C.c_void_p),
        ("n_dirs", C.c_int32),
        ("s", C.c_void_p), ("w", C.c_void_p),
        ("face_bc", _BC * 6),
        ("interface_bc", _BC),
        ("Q", C.c_void_p),
        ("diagnostics", C.c_int32),
        ("literal_one_over_pi", C.c_int32),
    ]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.bte_ref_create.argtypes = [C.POINTER(_Problem), C.POINTER(C.c_void_p)]
        L.bte_ref_create.restype = C.c_int
        L.bte_ref_destroy.argtypes = [C.c_void_p]
        L.bte_ref_destroy.restype = None
        L.bte_ref_set_threads.argtypes = [C.c_void_p, C.c_int32]
        L.bte_ref_set_threads.restype = None
        L.bte_ref_set_dir_order.argtypes = [C.c_void_p, C.c_void_p]
        L.bte_ref_iterate.argtypes = [C.c_void_p, C.c_int32]
        for name in ("bte_ref_get_temperature", "bte_ref_get_heat_flux", "bte_ref_set_temperature",
                     "bte_ref_get_intensity", "bte_ref_face_flux", "bte_ref_face_flux_band",
                     "bte_ref_boundary_power"):
            getattr(L, name).argtypes = [C.c_void_p, C.c_void_p]
            getattr(L, name).restype = C.c_int
        L.bte_ref_residual.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        L.bte_ref_updates_per_sweep.argtypes = [C.c_void_p]
        L.bte_ref_updates_per_sweep.restype = C.c_int64
        L.bte_ref_iterations_done.argtypes = [C.c_void_p]
        L.bte_ref_iterations_done.restype = C.c_int64
        L.bte_ref_pi_face.argtypes = [C.c_void_p, C.c_int32]
        L.bte_ref_pi_face.restype = C.c_double
        _lib = L
    return _lib


def _f64(a):
    return np.ascontiguousarray(a, dtype=np.float64)


class RefSolver:
    """Oracle handle built from a `workloads.Problem` (or any object with the same fields)."""

    def __init__(self, p, diagnostics: bool = False, literal_one_over_pi: bool = False, threads: int = 1):
        L = lib()
        self._keep = dict(
            C=_f64(p.C), v=_f64(p.v), tau=_f64(p.tau), s=_f64(p.s), w=_f64(p.w),
            mask=None if p.mask is None else np.ascontiguousarray(p.mask, dtype=np.uint8),
            Q=None if p.Q is None else _f64(p.Q))
        k = self._keep
        pr = _Problem()
        pr.nx, pr.ny, pr.nz, pr.dim = p.nx, p.ny, p.nz, p.dim
        pr.dx, pr.dy, pr.dz = p.dx, p.dy, p.dz
        pr.solid_mask = None if k["mask"] is None else k["mask"].ctypes.data
        pr.n_bands = len(k["C"])
        pr.C, pr.v, pr.tau = k["C"].ctypes.data, k["v"].ctypes.data, k["tau"].ctypes.data
        pr.n_dirs = len(k["w"])
        pr.s, pr.w = k["s"].ctypes.data, k["w"].ctypes.data
        for f in range(6):
            pr.face_bc[f].type, pr.face_bc[f].dT_wall = int(p.face_bc[f][0]), float(p.face_bc[f][1])
        pr.interface_bc.type, pr.interface_bc.dT_wall = int(p.interface_bc[0]), float(p.interface_bc[1])
        pr.Q = None if k["Q"] is None else k["Q"].ctypes.data
        pr.diagnostics = int(diagnostics)
        pr.literal_one_over_pi = int(literal_one_over_pi)
        h = C.c_void_p()
        rc = L.bte_ref_create(C.byref(pr), C.byref(h))
        self.h = None
        if rc != 0:
            raise ValueError(f"bte_ref_create failed with code {rc}")
        self.h = h
        self.shape = (p.nz, p.ny, p.nx)
        self.B, self.D = pr.n_bands, pr.n_dirs
        self.n_cells = p.nx * p.ny * p.nz
        if threads != 1:
            L.bte_ref_set_threads(self.h, threads)

    def __del__(self):
        if getattr(self, "h", None):
            lib().bte_ref_destroy(self.h)
            self.h = None

    def set_threads(self, n):
        lib().bte_ref_set_threads(self.h, int(n))

    def set_dir_order(self, perm):
        if perm is None:
            return lib().bte_ref_set_dir_order(self.h, None)
        a = np.ascontiguousarray(perm, dtype=np.int32)
        rc = lib().bte_ref_set_dir_order(self.h, a.ctypes.data)
        if rc:
            raise ValueError("bad permutation")

    def iterate(self, n):
        rc = lib().bte_ref_iterate(self.h, int(n))
        if rc:
            raise RuntimeError("bte_ref_iterate failed")

    def _get(self, fn, shape):
        out = np.empty(shape, dtype=np.float64)
        rc = getattr(lib(), fn)(self.h, out.ctypes.data)
        if rc:
            raise RuntimeError(f"{fn} failed ({rc})")
        return out

    def temperature(self):
        return self._get("bte_ref_get_temperature", self.shape)

    def heat_flux(self):
        return self._get("bte_ref_get_heat_flux", (3,) + self.shape)

    def set_temperature(self, dT):
        a = _f64(dT)
        assert a.size == self.n_cells
        lib().bte_ref_set_temperature(self.h, a.ctypes.data)

    def residual(self):
        a, b = C.c_double(), C.c_double()
        lib().bte_ref_residual(self.h, C.byref(a), C.byref(b))
        return a.value, b.value

    def intensity(self):
        return self._get("bte_ref_get_intensity", (self.B, self.D) + self.shape)

    def face_flux(self):
        return self._get("bte_ref_face_flux", (6,) + self.shape)

    def face_flux_band(self):
        return self._get("bte_ref_face_flux_band", (self.B, 6) + self.shape)

    def boundary_power(self):
        return self._get("bte_ref_boundary_power", (4,))

    def pi_face(self, f):
        return lib().bte_ref_pi_face(self.h, int(f))

    @property
    def updates_per_sweep(self):
        return lib().bte_ref_updates_per_sweep(self.h)

    @property
    def iterations_done(self):
        return lib().bte_ref_iterations_done(self.h)
