"""Bench-only CUDA objects (not part of the product library): the plain-ALU FMA peak microbenchmark that bench.py
runs before its timed region (roofline denominator, measured in the same run)."""
import ctypes as C
import os
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libfma_peak.so")
_SRC = os.path.join(_HERE, "fma_peak.cu")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared", "-Xcompiler", "-fPIC"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        subprocess.run(["nvcc"] + NVCC_FLAGS + ["-o", _SO, _SRC], check=True, cwd=_HERE)
    return _SO


def measure_fma_peak(dtype: str, device, reps: int = 5):
    """Achieved FMA/s of a register-only FFMA2 ('f32') or DFMA ('f64') chain on all SMs -> (TFLOP/s, SM count)."""
    import torch
    if not os.path.exists(_SO):
        raise FileNotFoundError(f"{_SO} is missing: run __graft_entry__.build()")
    L = C.CDLL(_SO)
    L.bte_measure_fma_peak.argtypes = [C.c_int, C.c_void_p, C.c_void_p, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_int)]
    with torch.cuda.device(device):
        scratch = torch.zeros(4 << 20, dtype=torch.uint8, device=device)
        v, sms = C.c_double(), C.c_int()
        rc = L.bte_measure_fma_peak(1 if dtype == "f32" else 0, C.c_void_p(scratch.data_ptr()),
                                    C.c_void_p(torch.cuda.current_stream(device).cuda_stream), reps, C.byref(v), C.byref(sms))
        if rc:
            raise RuntimeError("bte_measure_fma_peak failed")
    return 2.0 * v.value / 1e12, sms.value
