"""CPU-only checks of the C-ABI boundary: the library builds, loads and exports every symbol
include/bte.h declares; host-side validation and workspace sizing work without a GPU."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import paper_2503_23657_b200 as bte
import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def L():
    bte.build()
    return bte.lib()


def test_exports_every_declared_symbol(L):
    hdr = open(os.path.join(ROOT, "include", "bte.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(bte_[a-z_]+)\s*\(", hdr))
    assert {"bte_create", "bte_iterate", "bte_get_temperature", "bte_get_heat_flux", "bte_residual"} <= names
    for n in names:
        assert hasattr(L, n), f"{n} declared in include/bte.h but not exported"
    assert names == set(bte.EXPORTS)


def test_status_strings(L):
    assert L.bte_status_string(0) == b"ok"
    assert b"workspace" in L.bte_status_string(3)


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
def test_workspace_bytes_for_all_configs(L, k):
    grid = None if k < 2 else {2: (64, 64, 64), 3: (128, 64, 64), 4: (256, 128, 128)}[k]
    p = W.config(k, grid=grid)
    n = bte.bte_workspace_bytes(p)
    assert n > 0 and n % 256 == 0
    assert n < 60e9                      # fits one B200 (180 GB) with room to spare
    if k == 2:
        assert bte.bte_workspace_bytes(p, precision=W.FP32_STORE_FP64_ACC) < n


def test_invalid_problems_are_rejected_on_the_host(L):
    p = W.config(2, grid=(8, 8, 8))
    assert bte.bte_workspace_bytes(p) > 0
    bad = W.config(2, grid=(8, 8, 8)); bad.tau = -bad.tau
    assert bte.bte_workspace_bytes(bad) == 0
    bad = W.config(2, grid=(8, 8, 8)); bad.face_bc[0] = (W.BC_PERIODIC, 0.0)
    assert bte.bte_workspace_bytes(bad) == 0
    bad = W.config(2, grid=(8, 8, 8)); bad.w = bad.w * 1.01
    assert bte.bte_workspace_bytes(bad) == 0
    bad = W.config(2, grid=(8, 8, 8)); bad.mask = np.zeros((8, 8, 8), np.uint8)
    assert bte.bte_workspace_bytes(bad) == 0
    bad = W.config(1, grid=(8, 8, 1)); bad.s = bad.s.copy(); bad.s[0] = [0.6, 0.0, 0.8]   # specular needs closure
    assert bte.bte_workspace_bytes(bad) == 0


def test_create_reports_workspace_and_argument_errors_without_touching_cuda(L):
    pr, keep = bte._marshal(W.config(0))
    h = C.c_void_p()
    assert L.bte_create(C.byref(pr), None, 0, None, C.byref(h)) == 3          # BTE_ERR_WORKSPACE
    assert L.bte_create(C.byref(pr), C.c_void_p(128), 1 << 30, None, C.byref(h)) == 3   # misaligned
    assert h.value is None
    pr.n_bands = 0
    assert L.bte_create(C.byref(pr), None, 0, None, C.byref(h)) == 1          # BTE_ERR_INVALID_ARG
    assert L.bte_iterate(None, 1, None) == 1
    assert L.bte_updates_per_sweep(None) == 0


def test_product_does_not_import_the_oracle():
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2503_23657_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(root, f)).read()
                assert "import oracle" not in txt and "bte_ref" not in txt, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".cpp", ".h")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2503_23657_b200" not in txt.replace("paper_2503_23657_b200/csrc", "") or f == "bte_ref.h"


def test_options_replace_environment_variables(L):
    """bte_set_option is the only test / tuning hook: the product never reads the environment."""
    for root, _, files in os.walk(os.path.join(ROOT, "paper_2503_23657_b200")):
        for f in files:
            if f.endswith((".cu", ".cuh", ".h")):
                assert "getenv" not in open(os.path.join(root, f)).read(), f
    p = W.config(4, grid=(40, 34, 20))
    assert bte.bte_plan_info(p)["kernel_path"] == 2
    try:
        bte.bte_set_option("force_generic", 1)
        assert bte.bte_plan_info(p)["kernel_path"] == 1
        bte.bte_set_option("force_generic", 0)
        bte.bte_set_option("warps", 4)
        assert bte.bte_plan_info(p)["warps_per_cta"] == 4
    finally:
        bte.bte_set_option("force_generic", 0)
        bte.bte_set_option("warps", 0)
    assert bte.bte_plan_info(p)["kernel_path"] == 2
    assert L.bte_set_option(99, 1) == 1 and L.bte_set_option(-1, 1) == 1     # BTE_ERR_INVALID_ARG


def test_specular_face_needs_a_vanishing_first_moment(L):
    """|sum w s| > 1e-9 * 4 pi with a SPECULAR face -> BTE_ERR_QUADRATURE (Eq. 7 conserves energy only
    for a table whose first moment vanishes).  The skewed table below keeps sum w = 4 pi and stays closed under the
    x and y mirror flips (weights equal within each mirror orbit) but has a net z moment."""
    p = W.config(4, grid=(8, 8, 8))                     # x, y faces specular
    w = p.w.copy()
    up = p.s[:, 2] > 0
    w[up] *= 1.0 + 1e-6
    w *= 4 * np.pi / w.sum()
    bad = W.config(4, grid=(8, 8, 8)); bad.w = w
    pr, keep = bte._marshal(bad)
    out = (C.c_int64 * 8)()
    assert L.bte_plan_info(C.byref(pr), 148, out) == 2  # BTE_ERR_QUADRATURE
    ok = W.config(2, grid=(8, 8, 8)); ok.w = w          # no specular face: the same table is accepted
    pr, keep = bte._marshal(ok)
    assert L.bte_plan_info(C.byref(pr), 148, out) == 0
