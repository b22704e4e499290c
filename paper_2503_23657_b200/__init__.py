"""paper_2503_23657_b200 -- thin Python binding of the B200 phonon-BTE sweep library.

Argument marshalling only: every step of the hot path runs in the CUDA kernels behind the
C-ABI of include/bte.h (csrc/bte_api.cu, csrc/bte_kernels.cuh).  PyTorch supplies device
memory and streams, nothing else.  There is no CPU fallback: if the shared library is missing
or no CUDA device is present, construction fails loudly.

Entry points mirror the C names: bte_workspace_bytes, bte_create, bte_iterate,
bte_get_temperature, bte_get_heat_flux, bte_set_temperature, bte_residual, bte_solve_host, ...
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_HERE, "csrc")
_SO = os.path.join(_HERE, "libbte_b200.so")
_SOURCES = [os.path.join(_CSRC, f) for f in ("bte_api.cu", "bte_kernels.cuh", "bte_sweep2.cuh", "bte_static.cuh", "bte_internal.h")] + \
           [os.path.join(os.path.dirname(_HERE), "include", "bte.h")]

NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-shared", "-Xcompiler", "-fPIC"]

STATUS = {0: "BTE_OK", 1: "BTE_ERR_INVALID_ARG", 2: "BTE_ERR_QUADRATURE", 3: "BTE_ERR_WORKSPACE",
          4: "BTE_ERR_CUDA", 5: "BTE_ERR_UNSUPPORTED", 6: "BTE_ERR_TOO_LARGE"}
BTE_FP64, BTE_FP32_STORE_FP64_ACC = 0, 1

EXPORTS = ["bte_workspace_bytes", "bte_create", "bte_iterate", "bte_get_temperature", "bte_get_heat_flux",
           "bte_set_temperature", "bte_residual", "bte_solve_host", "bte_set_sweep_timing",
           "bte_get_sweep_timing", "bte_updates_per_sweep",
           "bte_iterations_done", "bte_kernel_launches_per_iteration", "bte_kernel_path", "bte_plan_info", "bte_schedule_info", "bte_destroy",
           "bte_status_string", "bte_last_cuda_error", "bte_set_option", "bte_residual_static"]


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile the CUDA library in-tree for sm_100a (nvcc cross-compiles without a GPU)."""
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SOURCES):
        return _SO
    cmd = ["nvcc"] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", _SO, os.path.join(_CSRC, "bte_api.cu")]
    subprocess.run(cmd, check=True, cwd=_CSRC)
    return _SO


class BteError(RuntimeError):
    def __init__(self, code, where):
        self.code = code
        super().__init__(f"{where}: {STATUS.get(code, code)}")


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
        ("precision", C.c_int32),
    ]


_lib = None


def lib():
    """Load libbte_b200.so (must have been built; raises if it is missing)."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise FileNotFoundError(f"{_SO} is missing: run paper_2503_23657_b200.build() (no fallback path exists)")
        L = C.CDLL(_SO)
        vp, i32, i64, dp = C.c_void_p, C.c_int32, C.c_int64, C.POINTER(C.c_double)
        L.bte_workspace_bytes.argtypes = [C.POINTER(_Problem)]
        L.bte_workspace_bytes.restype = C.c_size_t
        L.bte_create.argtypes = [C.POINTER(_Problem), vp, C.c_size_t, vp, C.POINTER(vp)]
        L.bte_iterate.argtypes = [vp, i32, vp]
        L.bte_get_temperature.argtypes = [vp, vp, vp]
        L.bte_get_heat_flux.argtypes = [vp, vp, vp]
        L.bte_set_temperature.argtypes = [vp, vp, vp]
        L.bte_residual.argtypes = [vp, dp, dp]
        L.bte_solve_host.argtypes = [vp, vp, i32, i32, vp, vp, vp]
        L.bte_set_sweep_timing.argtypes = [vp, i32]
        L.bte_get_sweep_timing.argtypes = [vp, dp, C.POINTER(i64)]
        L.bte_updates_per_sweep.argtypes = [vp]
        L.bte_updates_per_sweep.restype = i64
        L.bte_iterations_done.argtypes = [vp]
        L.bte_iterations_done.restype = i64
        L.bte_kernel_launches_per_iteration.argtypes = [vp]
        L.bte_kernel_launches_per_iteration.restype = i32
        L.bte_plan_info.argtypes = [C.POINTER(_Problem), i32, C.POINTER(i64)]
        L.bte_kernel_path.argtypes = [vp]
        L.bte_kernel_path.restype = i32
        L.bte_schedule_info.argtypes = [vp, C.POINTER(i64)]
        L.bte_schedule_info.restype = None
        L.bte_destroy.argtypes = [vp]
        L.bte_destroy.restype = None
        L.bte_status_string.argtypes = [C.c_int]
        L.bte_status_string.restype = C.c_char_p
        L.bte_last_cuda_error.restype = i32
        L.bte_set_option.argtypes = [i32, i32]
        L.bte_residual_static.argtypes = [vp, vp, vp, vp, vp, i64, vp, vp]
        _lib = L
    return _lib


OPTIONS = {"force_generic": 0, "warps": 1, "publish_period": 2, "start_slack": 3, "schedule": 4}


def bte_set_option(name, value) -> None:
    """Process-wide test / tuning option (include/bte.h bte_set_option); 0 restores the default."""
    rc = lib().bte_set_option(OPTIONS[name], int(value))
    if rc:
        raise BteError(rc, "bte_set_option")


STATIC_MAX_CELLS = 1 << 24


def bte_residual_static(dT_new, dT_old, q_new, q_old, solid_mask, eps_out, stream=None) -> None:
    """Allocation-free Eq. 23 stopping test (include/bte.h bte_residual_static).  Every argument is a contiguous CUDA
    tensor the caller owns: dT_* float64 [n_cells], q_* float64 [3][n_cells], solid_mask uint8 [n_cells] or None,
    eps_out float64 [2] (receives eps_T, eps_q).  Asynchronous on `stream` (default: torch's current stream)."""
    import torch
    for t, dt in ((dT_new, torch.float64), (dT_old, torch.float64), (q_new, torch.float64), (q_old, torch.float64),
                  (eps_out, torch.float64)) + (() if solid_mask is None else ((solid_mask, torch.uint8),)):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dt):
            raise ValueError("bte_residual_static takes contiguous CUDA tensors (float64; uint8 mask)")
    n = dT_new.numel()
    if dT_old.numel() != n or q_new.numel() != 3 * n or q_old.numel() != 3 * n or eps_out.numel() < 2 or \
            (solid_mask is not None and solid_mask.numel() != n):
        raise ValueError("bte_residual_static: sizes do not match")
    s = torch.cuda.current_stream(dT_new.device) if stream is None else stream
    with torch.cuda.device(dT_new.device):
        rc = lib().bte_residual_static(dT_new.data_ptr(), dT_old.data_ptr(), q_new.data_ptr(), q_old.data_ptr(),
                                       None if solid_mask is None else solid_mask.data_ptr(), n, eps_out.data_ptr(),
                                       C.c_void_p(s.cuda_stream))
    if rc:
        raise BteError(rc, "bte_residual_static")


def _marshal(p, precision=None):
    """workloads.Problem-like object -> (bte_problem struct, keep-alive arrays)."""
    f64 = lambda a: np.ascontiguousarray(a, dtype=np.float64)
    keep = dict(C=f64(p.C), v=f64(p.v), tau=f64(p.tau), s=f64(p.s), w=f64(p.w),
                mask=None if p.mask is None else np.ascontiguousarray(p.mask, dtype=np.uint8),
                Q=None if p.Q is None else f64(p.Q))
    pr = _Problem()
    pr.nx, pr.ny, pr.nz, pr.dim = p.nx, p.ny, p.nz, p.dim
    pr.dx, pr.dy, pr.dz = p.dx, p.dy, p.dz
    pr.solid_mask = None if keep["mask"] is None else keep["mask"].ctypes.data
    pr.n_bands = len(keep["C"])
    pr.C, pr.v, pr.tau = keep["C"].ctypes.data, keep["v"].ctypes.data, keep["tau"].ctypes.data
    pr.n_dirs = len(keep["w"])
    pr.s, pr.w = keep["s"].ctypes.data, keep["w"].ctypes.data
    for f in range(6):
        pr.face_bc[f].type, pr.face_bc[f].dT_wall = int(p.face_bc[f][0]), float(p.face_bc[f][1])
    pr.interface_bc.type, pr.interface_bc.dT_wall = int(p.interface_bc[0]), float(p.interface_bc[1])
    pr.Q = None if keep["Q"] is None else keep["Q"].ctypes.data
    pr.precision = int(p.precision if precision is None else precision)
    return pr, keep


def bte_workspace_bytes(p, precision=None) -> int:
    pr, _keep = _marshal(p, precision)
    return int(lib().bte_workspace_bytes(C.byref(pr)))


def bte_plan_info(p, resident_ctas=148, precision=None):
    """Host-only plan summary (no GPU needed)."""
    pr, _keep = _marshal(p, precision)
    out = (C.c_int64 * 8)()
    rc = lib().bte_plan_info(C.byref(pr), int(resident_ctas), out)
    if rc:
        raise BteError(rc, "bte_plan_info")
    keys = ["kernel_path", "work_units", "order_ok", "steps_per_unit", "warps_per_cta", "band_groups", "masked",
            "workspace_bytes"]
    return dict(zip(keys, [int(x) for x in out]))


class Solver:
    """One bte_solver handle; the device workspace is a torch uint8 tensor owned here."""

    def __init__(self, p, precision=None, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2503_23657_b200 needs a CUDA device (there is no CPU fallback)")
        L = lib()
        self.torch = torch
        self.device = torch.device(device)
        pr, keep = _marshal(p, precision)
        need = int(L.bte_workspace_bytes(C.byref(pr)))
        if need == 0:
            # let bte_create report the precise status
            need = 256
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(need + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            self._ws_ptr = (base + 255) & ~255
            h = C.c_void_p()
            rc = L.bte_create(C.byref(pr), C.c_void_p(self._ws_ptr), C.c_size_t(need), self._stream(stream), C.byref(h))
        self.h = None
        if rc != 0:
            raise BteError(rc, "bte_create")
        self.h = h
        self.shape = (p.nz, p.ny, p.nx)
        self.n_cells = p.nx * p.ny * p.nz
        self.workspace_bytes = need

    def _stream(self, stream=None):
        s = self.torch.cuda.current_stream(self.device) if stream is None else stream
        return C.c_void_p(s.cuda_stream)

    def __del__(self):
        if getattr(self, "h", None):
            lib().bte_destroy(self.h)
            self.h = None

    def iterate(self, n, stream=None):
        rc = lib().bte_iterate(self.h, int(n), self._stream(stream))
        if rc:
            raise BteError(rc, "bte_iterate")

    def temperature(self, stream=None):
        out = self.torch.empty(self.shape, dtype=self.torch.float64, device=self.device)
        rc = lib().bte_get_temperature(self.h, C.c_void_p(out.data_ptr()), self._stream(stream))
        if rc:
            raise BteError(rc, "bte_get_temperature")
        return out

    def heat_flux(self, stream=None):
        out = self.torch.empty((3,) + self.shape, dtype=self.torch.float64, device=self.device)
        rc = lib().bte_get_heat_flux(self.h, C.c_void_p(out.data_ptr()), self._stream(stream))
        if rc:
            raise BteError(rc, "bte_get_heat_flux")
        return out

    def set_temperature(self, dT, stream=None):
        t = self.torch.as_tensor(np.ascontiguousarray(dT, dtype=np.float64)).to(self.device).contiguous()
        assert t.numel() == self.n_cells
        rc = lib().bte_set_temperature(self.h, C.c_void_p(t.data_ptr()), self._stream(stream))
        self.torch.cuda.current_stream(self.device).synchronize()
        if rc:
            raise BteError(rc, "bte_set_temperature")

    def residual(self):
        a, b = C.c_double(), C.c_double()
        rc = lib().bte_residual(self.h, C.byref(a), C.byref(b))
        if rc:
            raise BteError(rc, "bte_residual")
        return a.value, b.value

    def solve_host(self, Q_host, n, want_q=True, reset=True, out=None, stream=None):
        """End-to-end call with HOST buffers (numpy arrays or pinned torch CPU tensors).
        `out` = (dT, q) preallocated host buffers (q may be None) to avoid allocation in timed loops."""
        ptr = lambda a: C.c_void_p(a.ctypes.data if isinstance(a, np.ndarray) else a.data_ptr())
        if out is None:
            dT = np.empty(self.shape, dtype=np.float64)
            q = np.empty((3,) + self.shape, dtype=np.float64) if want_q else None
        else:
            dT, q = out
        rc = lib().bte_solve_host(self.h, None if Q_host is None else ptr(Q_host), int(n), int(bool(reset)),
                                  ptr(dT), None if q is None else ptr(q), self._stream(stream))
        if rc:
            raise BteError(rc, "bte_solve_host")
        return dT, q

    def set_sweep_timing(self, max_launches):
        rc = lib().bte_set_sweep_timing(self.h, int(max_launches))
        if rc:
            raise BteError(rc, "bte_set_sweep_timing")

    def sweep_timing(self):
        """(summed sweep-kernel device time [ms], launches covered) since the last call."""
        ms, n = C.c_double(), C.c_int64()
        rc = lib().bte_get_sweep_timing(self.h, C.byref(ms), C.byref(n))
        if rc:
            raise BteError(rc, "bte_get_sweep_timing")
        return ms.value, n.value

    @property
    def updates_per_sweep(self):
        return int(lib().bte_updates_per_sweep(self.h))

    @property
    def iterations_done(self):
        return int(lib().bte_iterations_done(self.h))

    @property
    def launches_per_iteration(self):
        return int(lib().bte_kernel_launches_per_iteration(self.h))

    @property
    def kernel_path(self):
        return int(lib().bte_kernel_path(self.h))

    def schedule_info(self):
        out = (C.c_int64 * 6)()
        lib().bte_schedule_info(self.h, out)
        keys = ["work_units", "ctas", "threads_per_cta", "wavefront_steps", "thread_slot_updates", "workspace_bytes"]
        return dict(zip(keys, [int(x) for x in out]))
