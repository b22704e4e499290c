"""bte_residual_static (include/bte.h): the allocation-free Eq. 23 stopping test whose scratch is a file-scope
__device__ array of the library, against the existing path (bte_iterate + bte_residual, scratch in the caller's
workspace).  Collected last on purpose (the suite runs with pytest -x).

The snapshots handed to the new entry point are bte_get_temperature / bte_get_heat_flux before and after one
iteration, so both paths see the same fp64 values and differ only in summation grouping: the tolerance is the
residual tolerance of tests/test_gpu_parity.py::check for the fp64 path, rtol 1e-6 (measured ~1e-15).
"""
import ctypes as C

import numpy as np
import pytest

import paper_2503_23657_b200 as bte
import workloads as W

RES_RTOL = 1e-6


def test_rejects_sizes_beyond_the_static_array():
    """No CUDA call is made before the size check: runs without a GPU.  The pointers are never dereferenced."""
    bte.build()
    L = bte.lib()
    fake = C.c_void_p(256)
    assert bte.STATIC_MAX_CELLS == 1 << 24
    rc = L.bte_residual_static(fake, fake, fake, fake, None, bte.STATIC_MAX_CELLS + 1, fake, None)
    assert bte.STATUS[rc] == "BTE_ERR_TOO_LARGE"
    assert b"BTE_STATIC_MAX_CELLS" in L.bte_status_string(rc)
    assert bte.STATUS[L.bte_residual_static(fake, fake, fake, fake, None, 0, fake, None)] == "BTE_ERR_INVALID_ARG"
    assert bte.STATUS[L.bte_residual_static(None, fake, fake, fake, None, 8, fake, None)] == "BTE_ERR_INVALID_ARG"
    assert bte.STATUS[L.bte_residual_static(fake, fake, fake, fake, None, 8, None, None)] == "BTE_ERR_INVALID_ARG"


CASES = [(3, (40, 36, 32), W.FP64),                  # voxel-masked, generic kernels: N_solid != N_cell
         (4, (45, 130, 36), W.FP32_STORE_FP64_ACC)]   # all solid (mask = NULL), fast path; 210 600 cells = 52 blocks


@pytest.mark.gpu
@pytest.mark.parametrize("k,grid,prec", CASES)
def test_residual_static_matches_bte_residual_twice_in_a_row(k, grid, prec):
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    bte.lib()
    p = W.config(k, grid=grid)
    g = bte.Solver(p, precision=prec)
    mask = None if p.mask is None else torch.as_tensor(np.ascontiguousarray(p.mask, dtype=np.uint8)).cuda().reshape(-1)
    eps = torch.full((2, 2), float("nan"), dtype=torch.float64, device="cuda")
    g.iterate(4)
    snaps = [(g.temperature(), g.heat_flux())]
    want = []
    for _ in range(2):
        g.iterate(1)
        snaps.append((g.temperature(), g.heat_flux()))
        want.append(g.residual())
    before = torch.cuda.memory_allocated()
    # two calls in a row on one stream, no synchronisation in between: the second reuses the array the first left
    for c in range(2):
        (T0, q0), (T1, q1) = snaps[c], snaps[c + 1]
        bte.bte_residual_static(T1, T0, q1, q0, mask, eps[c])
    assert torch.cuda.memory_allocated() == before
    got = eps.cpu().numpy()
    for c in range(2):
        for name, a, b in (("eps_T", got[c, 0], want[c][0]), ("eps_q", got[c, 1], want[c][1])):
            assert np.isfinite(a) and b > 0
            assert abs(a - b) <= RES_RTOL * b, f"call {c} {name}: static {a!r} vs bte_residual {b!r}"
    assert got[0, 0] != got[1, 0]                      # the two calls really had different inputs
    # same inputs again: bit-identical (fixed summation order; nothing of the earlier calls leaks in)
    again = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    bte.bte_residual_static(snaps[1][0], snaps[0][0], snaps[1][1], snaps[0][1], mask, again)
    assert again.cpu().numpy().tobytes() == got[0].tobytes()


@pytest.mark.gpu
def test_residual_static_degenerate_values():
    """0/0 -> 0 (identical all-zero snapshots), ragged single block, and a mask that removes the largest cell."""
    import torch
    n = 1000
    z, z3 = torch.zeros(n, dtype=torch.float64, device="cuda"), torch.zeros(3 * n, dtype=torch.float64, device="cuda")
    eps = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    bte.bte_residual_static(z, z, z3, z3, None, eps)
    assert eps.cpu().tolist() == [0.0, 0.0]
    rng = np.random.default_rng(3)
    T0, T1 = rng.normal(size=n), rng.normal(size=n)
    q0, q1 = rng.normal(size=(3, n)), rng.normal(size=(3, n))
    m = (rng.uniform(size=n) > 0.3).astype(np.uint8)
    T1[5], m[5] = 1e6, 0                               # a void cell must not enter the maximum
    s = m.astype(bool)
    qm0, qm1 = np.sqrt((q0 ** 2).sum(0))[s], np.sqrt((q1 ** 2).sum(0))[s]
    eT = np.sqrt(((T1 - T0)[s] ** 2).sum() / s.sum()) / np.abs(T1[s]).max()
    eq = np.sqrt(((qm1 - qm0) ** 2).sum() / s.sum()) / qm1.max()
    dev = lambda a: torch.as_tensor(np.ascontiguousarray(a)).cuda().reshape(-1)
    bte.bte_residual_static(dev(T1), dev(T0), dev(q1), dev(q0), dev(m), eps)
    a, b = eps.cpu().tolist()
    assert abs(a - eT) <= 1e-12 * eT and abs(b - eq) <= 1e-12 * eq
