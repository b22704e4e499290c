"""Host logic of the CUDA library, checked without a GPU: which kernel path a problem takes, and that the ticket
order of the sweep schedule is topological for any number of resident CTAs (a wrong order would dead-lock the
spin-waiting persistent kernel)."""
import numpy as np
import pytest

import paper_2503_23657_b200 as bte
import workloads as W


@pytest.fixture(scope="module", autouse=True)
def _built():
    bte.build()


@pytest.mark.parametrize("k,grid,path", [(0, None, 1), (1, None, 2), (1, (45, 71, 1), 1), (2, (64, 64, 64), 2), (3, (128, 64, 64), 2),
                                         (4, (256, 128, 128), 2), (2, (19, 37, 21), 1), (4, (43, 34, 20), 2)])
def test_kernel_path_selection(k, grid, path):
    info = bte.bte_plan_info(W.config(k, grid=grid))
    assert info["kernel_path"] == path
    assert info["order_ok"] == 1
    assert info["masked"] == (1 if (k == 3 and path == 2) else 0)


@pytest.mark.parametrize("slots", [1, 7, 148, 296, 100000])
@pytest.mark.parametrize("prec", [W.FP64, W.FP32_STORE_FP64_ACC])
def test_ticket_order_is_topological_for_any_cta_count(slots, prec):
    for p in (W.config(4, grid=(40, 130, 52)), W.config(3, grid=(36, 68, 40)), W.config(2, grid=(12, 10, 8))):
        info = bte.bte_plan_info(p, resident_ctas=slots, precision=prec)
        assert info["kernel_path"] == 2 and info["order_ok"] == 1
        groups = 8 if prec == W.FP32_STORE_FP64_ACC else 15
        assert info["band_groups"] == groups
        tiles = -(-p.ny // 64) * -(-p.nz // (2 * info["warps_per_cta"]))
        assert info["work_units"] == 8 * groups * tiles
        assert info["steps_per_unit"] == p.nx + 31 + info["warps_per_cta"] - 1


def test_fast_path_needs_symmetric_16_direction_octants_and_few_bands():
    p = W.config(2, grid=(12, 10, 8))
    assert bte.bte_plan_info(p)["kernel_path"] == 2
    q = W.config(2, grid=(12, 10, 8)); q.s, q.w = W.quadrature_3d(4, 8)          # 4 directions per octant
    assert bte.bte_plan_info(q)["kernel_path"] == 1
    q = W.config(2, grid=(12, 10, 8)); q.C, q.v, q.tau = W.band_table(17)        # more than 16 bands
    assert bte.bte_plan_info(q)["kernel_path"] == 1
    q = W.config(2, grid=(12, 10, 8)); q.C, q.v, q.tau = W.band_table(3)         # rotate the table: no mirror symmetry
    th = 0.3
    R = np.array([[np.cos(th), -np.sin(th), 0], [np.sin(th), np.cos(th), 0], [0, 0, 1]])
    q.s = q.s @ R.T
    q.face_bc = [(W.BC_ISOTHERMAL, 0.0)] * 6
    assert bte.bte_plan_info(q)["kernel_path"] == 1
    with pytest.raises(bte.BteError):
        bad = W.config(2, grid=(12, 10, 8)); bad.tau = -bad.tau
        bte.bte_plan_info(bad)
