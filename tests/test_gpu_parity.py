"""GPU parity: the CUDA path (through the C-ABI of include/bte.h) against the fp64 CPU oracle,
element by element, on the same seeded inputs after the same iteration count.

Error norms are reading G12: err_T = max|dT_gpu - dT_ref| / max|dT_ref|,
err_q = max||q_gpu - q_ref||_2 / max||q_ref||_2.  Tolerances are north_star's:
1e-10 for fp64, 1e-4 for fp32-storage/fp64-accumulate (against the fp64 oracle).
"""
import os

import numpy as np
import pytest

import workloads as W

pytestmark = pytest.mark.gpu

TOL = {W.FP64: 1e-10, W.FP32_STORE_FP64_ACC: 1e-4}
NCPU = max(1, min(32, os.cpu_count() or 1))


@pytest.fixture(scope="module")
def bte():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2503_23657_b200 as m
    m.lib()          # fails loudly if the in-tree .so is missing
    return m


@pytest.fixture
def option(bte):
    """bte_set_option for the duration of one test (the library never reads the environment)."""
    used = []

    def set_(name, value):
        bte.bte_set_option(name, value)
        used.append(name)
    yield set_
    for name in used:
        bte.bte_set_option(name, 0)


def errors(dT, q, dT_ref, q_ref):
    eT = np.max(np.abs(dT - dT_ref)) / max(np.max(np.abs(dT_ref)), 1e-300)
    dq = np.sqrt(((q - q_ref) ** 2).sum(axis=0))
    qn = np.sqrt((q_ref ** 2).sum(axis=0))
    eq = np.max(dq) / max(np.max(qn), 1e-300)
    return eT, eq


def run_both(bte, p, n, precision=None, checkpoints=()):
    import oracle
    prec = p.precision if precision is None else precision
    ref = oracle.RefSolver(p, threads=NCPU)
    gpu = bte.Solver(p, precision=prec)
    done = 0
    out = []
    for stop in sorted(set(checkpoints) | {n}):
        ref.iterate(stop - done)
        gpu.iterate(stop - done)
        done = stop
        dT = gpu.temperature().cpu().numpy()
        q = gpu.heat_flux().cpu().numpy()
        eT, eq = errors(dT, q, ref.temperature(), ref.heat_flux())
        rT, rq = ref.residual()
        gT, gq = gpu.residual()
        out.append((stop, eT, eq, (rT, rq), (gT, gq)))
    return out, gpu, ref


def check(bte, p, n, precision=None, checkpoints=(), res_rtol=None):
    prec = p.precision if precision is None else precision
    tol = TOL[prec]
    out, gpu, ref = run_both(bte, p, n, prec, checkpoints)
    for stop, eT, eq, (rT, rq), (gT, gq) in out:
        assert eT <= tol, f"{p.name} n={stop}: err_T={eT:.3e} > {tol}"
        assert eq <= tol, f"{p.name} n={stop}: err_q={eq:.3e} > {tol}"
        # Eq. 23 residuals: same definition on both sides
        rt = res_rtol if res_rtol is not None else (1e-6 if prec == W.FP64 else 1e-4)
        if rT > 1e3 * tol and np.isfinite(rT):
            assert abs(gT - rT) <= rt * rT, f"{p.name} n={stop}: eps_T {gT} vs {rT}"
        if rq > 1e3 * tol and np.isfinite(rq):
            assert abs(gq - rq) <= rt * rq, f"{p.name} n={stop}: eps_q {gq} vs {rq}"
    assert gpu.iterations_done == n
    assert gpu.updates_per_sweep == p.updates_per_sweep == ref.updates_per_sweep
    return out


# ---------------------------------------------------------------- shrunken configs (T2)
SHRUNK = {0: (57, 1, 1), 1: (45, 70, 1), 2: (19, 37, 21), 3: (40, 36, 32), 4: (43, 34, 19)}
# even ny, nz: served by the fast path (tiles of 64 x 8/16 rows: ragged in y and z, two tiles in y for 4')
SHRUNK_FAST = {2: (21, 38, 22), 4: (45, 130, 36)}


@pytest.mark.parametrize("k", [0, 1, 2, 3, 4])
@pytest.mark.parametrize("prec", [W.FP64, W.FP32_STORE_FP64_ACC])
def test_shrunken_configs(bte, k, prec):
    """Every config at a size that spans several tiles with a ragged tail on every axis
    (generic path: tiles are 32 rows in y and 8/16 in z), checked at n = 1, 2, 10, 30."""
    p = W.config(k, grid=SHRUNK[k])
    check(bte, p, 30, precision=prec, checkpoints=(1, 2, 10))


@pytest.mark.parametrize("k", [2, 4])
@pytest.mark.parametrize("prec", [W.FP64, W.FP32_STORE_FP64_ACC])
def test_shrunken_configs_fast_path(bte, k, prec, option):
    """The 3-D unmasked configs on the fast sweep kernel, and the same problem forced onto the generic one."""
    p = W.config(k, grid=SHRUNK_FAST[k])
    assert bte.Solver(p, precision=prec).kernel_path == 2
    check(bte, p, 30, precision=prec, checkpoints=(1, 2, 10))
    option("force_generic", 1)
    assert bte.Solver(p, precision=prec).kernel_path == 1
    check(bte, p, 6, precision=prec, checkpoints=(1,))


@pytest.mark.parametrize("warps", [4, 8])
def test_fast_path_tile_heights(bte, warps, option):
    """Both CTA shapes of the fast path (tiles of 8 and 16 rows in z), several z tiles, periodic + specular faces."""
    option("warps", warps)
    p = W.config(4, grid=(37, 66, 52))
    p.face_bc = [(W.BC_PERIODIC, 0.0), (W.BC_PERIODIC, 0.0), (W.BC_SPECULAR, 0.0), (W.BC_DIFFUSE, 0.0),
                 (W.BC_ISOTHERMAL, 0.1), (W.BC_SPECULAR, 0.0)]
    assert bte.Solver(p).kernel_path == 2
    check(bte, p, 12, checkpoints=(1, 3))
    check(bte, p, 4, precision=W.FP64)


@pytest.mark.parametrize("seed", range(6))
def test_masked_grids_on_the_fast_path(bte, seed):
    """Voxel masks on the fast sweep kernel (even ny, nz, 16 directions per octant): random masks with isothermal or
    diffuse interfaces, periodic axes whose wrap may land on void cells, both precisions."""
    p = W.random_problem(seed, dim=3, shape=(14 + seed, 10 + 2 * seed, 8 + 2 * (seed % 3)), masked=True,
                         periodic_axis=(seed % 3 if seed % 2 else None),
                         interface_type=(W.BC_DIFFUSE if seed % 2 == 0 else W.BC_ISOTHERMAL), n_polar=8, n_azimuth=16)
    assert bte.Solver(p).kernel_path == 2
    check(bte, p, 12, precision=W.FP64, checkpoints=(1, 3))
    check(bte, p, 12, precision=W.FP32_STORE_FP64_ACC)


def test_finfet_mask_fast_vs_generic(bte, option):
    """Config 3 (fin + slab, diffuse interfaces, periodic x) at a size with several z tiles on both kernel paths."""
    p = W.config(3, grid=(36, 68, 40))
    assert bte.Solver(p).kernel_path == 2
    check(bte, p, 20, checkpoints=(1, 5))
    check(bte, p, 6, precision=W.FP64, checkpoints=(1,))
    option("force_generic", 1)
    assert bte.Solver(p).kernel_path == 1
    check(bte, p, 6, precision=W.FP64, checkpoints=(1,))


# ---------------------------------------------------------------- random problems: every BC mix
@pytest.mark.parametrize("seed", range(8))
@pytest.mark.parametrize("dim", [1, 2, 3])
def test_random_masked_problems(bte, seed, dim):
    p = W.random_problem(seed, dim=dim, shape=(13 + seed, 9 + 5 * (seed % 3), 6 + seed % 4),
                         masked=(seed % 2 == 0), periodic_axis=(seed % 3 if seed % 4 == 1 else None),
                         interface_type=(W.BC_DIFFUSE if seed % 3 else W.BC_ISOTHERMAL))
    check(bte, p, 12, precision=W.FP64, checkpoints=(1, 3))
    check(bte, p, 12, precision=W.FP32_STORE_FP64_ACC)


@pytest.mark.parametrize("bc", [W.BC_ISOTHERMAL, W.BC_DIFFUSE, W.BC_SPECULAR, W.BC_PERIODIC])
def test_each_bc_type_alone(bte, bc):
    """One BC type on all side faces, z- isothermal so a steady state exists."""
    for grid in ((33, 34, 9), (33, 34, 10)):          # generic path / fast path
        p = W.config(2, grid=grid)
        fb = [(bc, 0.25 if bc == W.BC_ISOTHERMAL else 0.0)] * 4 + [(W.BC_ISOTHERMAL, -0.3), (W.BC_DIFFUSE, 0.0)]
        p.face_bc = fb
        assert bte.Solver(p).kernel_path == (2 if grid[2] % 2 == 0 else 1)
        check(bte, p, 15, precision=W.FP64, checkpoints=(1, 2))


def test_periodic_wrap_onto_void_uses_interface_bc(bte):
    """Reading: a periodic wrap that lands on a void cell falls through to interface_bc."""
    p = W.config(3, grid=(12, 20, 16))
    p.mask = p.mask.copy()
    p.mask[:, :, 0] = 0          # x=0 plane void: wrap from x=nx-1 hits void
    p.mask[0, 0, 0] = 1
    p.Q = p.Q * p.mask
    check(bte, p, 10, precision=W.FP64, checkpoints=(1,))


# ---------------------------------------------------------------- edge cases
def test_single_cell_and_tiny_grids(bte):
    for shape, dim in [((1, 1, 1), 1), ((1, 1, 1), 3), ((2, 1, 1), 2), ((1, 3, 2), 3), ((3, 1, 1), 1)]:
        p = W.random_problem(3, dim=dim, shape=shape, masked=False)
        check(bte, p, 6, precision=W.FP64, checkpoints=(1,))


@pytest.mark.parametrize("grid", [(9, 8, 7), (10, 8, 8)])          # generic / fast path
def test_zero_iterations_and_zero_source(bte, grid):
    p = W.config(2, grid=grid)
    g = bte.Solver(p)
    g.iterate(0)
    assert g.iterations_done == 0
    assert float(g.temperature().abs().max()) == 0.0
    eT, eq = g.residual()
    assert np.isinf(eT) and np.isinf(eq)
    p.Q = None
    p.face_bc = [(W.BC_DIFFUSE, 0.0)] * 4 + [(W.BC_ISOTHERMAL, 0.0), (W.BC_DIFFUSE, 0.0)]
    g = bte.Solver(p)
    g.iterate(3)
    assert float(g.temperature().abs().max()) == 0.0
    assert g.residual() == (0.0, 0.0)          # 0/0 -> 0 (reading G11)


@pytest.mark.parametrize("grid", [(17, 9, 11), (18, 10, 12)])      # generic / fast path
def test_set_temperature_restart(bte, grid):
    import oracle
    p = W.config(2, grid=grid)
    rng = np.random.default_rng(7)
    dT0 = rng.uniform(-1, 1, size=(p.nz, p.ny, p.nx))
    ref = oracle.RefSolver(p); ref.set_temperature(dT0); ref.iterate(1)
    g = bte.Solver(p); g.set_temperature(dT0); g.iterate(1)
    eT, eq = errors(g.temperature().cpu().numpy(), g.heat_flux().cpu().numpy(), ref.temperature(), ref.heat_flux())
    assert eT <= 1e-10 and eq <= 1e-10


@pytest.mark.parametrize("k", [3, 4])                               # generic (masked) / fast path
def test_bitwise_deterministic(bte, k):
    p = W.config(k, grid=(24, 40, 24))
    a = bte.Solver(p); a.iterate(7)
    b = bte.Solver(p); b.iterate(3); b.iterate(4)
    assert (a.temperature() == b.temperature()).all()
    assert (a.heat_flux() == b.heat_flux()).all()


@pytest.mark.parametrize("grid", [(20, 12, 9), (20, 12, 10)])      # generic / fast path
def test_solve_host_matches_device_path(bte, grid):
    p = W.config(2, grid=grid)
    g = bte.Solver(p); g.iterate(5)
    h = bte.Solver(p)
    dT, q = h.solve_host(np.ascontiguousarray(p.Q), 5)
    assert (dT == g.temperature().cpu().numpy()).all()
    assert (q == g.heat_flux().cpu().numpy()).all()
    dT2, _ = h.solve_host(None, 5)      # state is reset on every call
    assert (dT2 == dT).all()


def test_non_default_stream(bte):
    import torch
    p = W.config(1, grid=(40, 33, 1))
    a = bte.Solver(p); a.iterate(4)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        b = bte.Solver(p); b.iterate(4); t = b.temperature()
    s.synchronize()
    assert (a.temperature() == t).all()


# ---------------------------------------------------------------- full sizes (T3)
def test_config0_full_matches_oracle_and_golden(bte):
    p = W.config(0)
    check(bte, p, p.n_iter, checkpoints=(1, 10, 35))
    gold = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "cfg0_kn1_film.txt"))
    g = bte.Solver(p); g.iterate(p.n_iter)
    dT = g.temperature().cpu().numpy().ravel()
    qx = g.heat_flux().cpu().numpy()[0].ravel()
    assert np.max(np.abs(dT - gold[:, 1])) <= 1e-10 * np.max(np.abs(gold[:, 1]))
    assert np.max(np.abs(qx - gold[:, 2])) <= 1e-10 * np.max(np.abs(gold[:, 2]))


@pytest.mark.slow
def test_config1_full(bte):
    """Full-size config 1 at n = 50 (parity at n = 50)."""
    p = W.config(1)
    check(bte, p, 50, checkpoints=(1, 10))


@pytest.mark.slow
@pytest.mark.parametrize("prec", [W.FP64, W.FP32_STORE_FP64_ACC])
def test_config2_full(bte, prec):
    """Full-size config 2 at n = 50 in both precisions."""
    p = W.config(2)
    check(bte, p, 50, precision=prec, checkpoints=(1, 10))


@pytest.mark.slow
def test_config3_full(bte):
    """Full-size config 3 (voxel mask, diffuse interfaces, periodic x) at n = 50."""
    p = W.config(3)
    check(bte, p, 50, checkpoints=(1, 10))


@pytest.mark.slow
def test_config4_full_sampled(bte):
    """Full-size config 4 in the launch configuration bench.py times: n = 5 iterations against the
    (multi-threaded, bit-identical) oracle on every cell; the converged state is checked by
    test_config4_full_converged_energy_balance and, like for like, by test_config4_replica_converged_state."""
    p = W.config(4)
    out = check(bte, p, 5, checkpoints=(1, 2))
    assert out[-1][1] <= 1e-4


@pytest.mark.slow
@pytest.mark.parametrize("prec", [W.FP64, W.FP32_STORE_FP64_ACC])
def test_config4_replica_converged_state(bte, prec):
    """Like-for-like converged-state check: the 64x32x32 replica of the large slab is run to
    eps_T <= 1e-8 on BOTH sides (same iteration count, checked every 50 iterations); rounding differences must not
    accumulate over the ~10^3 iterations, in either precision."""
    import oracle
    p = W.config(4, grid=(64, 32, 32))
    ref = oracle.RefSolver(p, threads=NCPU)
    gpu = bte.Solver(p, precision=prec)
    n = 0
    while n < 4000:
        ref.iterate(50); gpu.iterate(50); n += 50
        if ref.residual()[0] <= 1e-8:
            break
    rT, _ = ref.residual()
    gT, _ = gpu.residual()
    assert rT <= 1e-8, f"oracle did not converge in {n} iterations (eps_T = {rT})"
    assert gT <= (1.05e-8 if prec == W.FP64 else 1e-6)      # fp32: the residual floors at the fp32 rounding level
    eT, eq = errors(gpu.temperature().cpu().numpy(), gpu.heat_flux().cpu().numpy(), ref.temperature(), ref.heat_flux())
    assert eT <= TOL[prec] and eq <= TOL[prec], (n, eT, eq)


@pytest.mark.slow
def test_progress_epoch_wraps_without_hanging(bte):
    """The per-unit progress words carry the iteration number in their upper bits and are re-zeroed every 30000
    iterations; run a tiny fast-path problem across that boundary (it is long converged by then)."""
    p = W.config(2, grid=(8, 8, 8))
    g = bte.Solver(p)
    assert g.kernel_path == 2
    g.iterate(29990)
    a = g.temperature().clone()
    g.iterate(25)                      # crosses iteration 30000
    b = g.temperature()
    assert g.iterations_done == 30015
    assert bool(((a - b).abs() <= 1e-9 * a.abs().max()).all())
    import oracle
    ref = oracle.RefSolver(p); ref.iterate(3000)          # converged reference (fixed point)
    assert np.abs(b.cpu().numpy() - ref.temperature()).max() <= 1e-8 * np.abs(ref.temperature()).max()


@pytest.mark.parametrize("warps", [4, 8])
@pytest.mark.parametrize("prec", [W.FP64, W.FP32_STORE_FP64_ACC])
@pytest.mark.parametrize("k", [3, 4])
def test_repeated_runs_are_bitwise_identical(bte, k, prec, warps, option):
    """Race detector for the tile pipeline (inter-tile progress flags, staged faces, accumulator hand-over between band
    groups): several y and z tiles, every run of the same problem must give the same bits."""
    option("warps", warps)
    p = W.config(k, grid=(45, 130, 36) if k == 4 else (40, 68, 40))
    ref = None
    for _ in range(5):
        g = bte.Solver(p, precision=prec)
        assert g.kernel_path == 2
        g.iterate(4)
        t = g.temperature()
        if ref is None:
            ref = t.clone()
        assert bool((t == ref).all())


@pytest.mark.parametrize("grid", [(1, 2, 2), (2, 4, 2), (1, 130, 36), (3, 66, 20), (7, 2, 34)])
def test_fast_path_degenerate_extents(bte, grid):
    """Fast path with fewer cells along x than the lane skew / the publication period, single-row tiles, and several
    tiles in y and z at the same time (a unit finishes before its downstream tile may start)."""
    p = W.config(4, grid=grid)
    assert bte.Solver(p).kernel_path == 2
    check(bte, p, 6, precision=W.FP64, checkpoints=(1, 2))
    check(bte, p, 6, precision=W.FP32_STORE_FP64_ACC)
    q = W.config(3, grid=grid)           # the same extents with the fin mask, periodic x, diffuse interfaces
    if q.mask.sum() > 0:
        check(bte, q, 6, precision=W.FP64, checkpoints=(1,))


@pytest.mark.slow
def test_config4_full_converged_energy_balance(bte):
    """Full-size config 4 run to eps_T <= 1e-8 (the oracle cannot follow it there): the power leaving through the
    isothermal face must match the total source.  With cell-centred q (Eq. 4; the conservative flux is the face flux,
    reading G18) the match is first order in the cell size: 6 % on a 64x32x32 replica, 2 % at full resolution."""
    def balance(grid):
        p = W.config(4, grid=grid)
        g = bte.Solver(p)
        n = 0
        while n < 5000 and (n == 0 or g.residual()[0] > 1e-8):
            g.iterate(50)
            n += 50
        assert g.residual()[0] <= 1e-8
        qz0 = g.heat_flux()[2, 0].sum().item()                       # bottom layer, z- is the isothermal face
        return -qz0 * p.dx * p.dy / (p.Q.sum() * p.dx * p.dy * p.dz), float(g.temperature().min())
    coarse, _ = balance((64, 32, 32))
    fine, tmin = balance(None)
    assert abs(1 - fine) < 0.03 and abs(1 - fine) < abs(1 - coarse) < 0.09
    assert tmin >= 0.0                                               # heating only: no undershoot below the wall


# ---------------------------------------------------------------- generic path beyond one chunk / 16 bands
def test_generic_path_two_direction_chunks_per_octant(bte):
    """32 directions per octant (8 polar x 32 azimuth: two chunks of 16 on the generic path, hemispherical partial sums
    from 2 x 4 slots) on a masked grid with diffuse interfaces and a diffuse box face."""
    p = W.random_problem(11, dim=3, shape=(13, 11, 9), masked=True, interface_type=W.BC_DIFFUSE,
                         bc_types=(W.BC_ISOTHERMAL, W.BC_DIFFUSE), n_polar=8, n_azimuth=32)
    assert len(p.w) == 256
    g = bte.Solver(p)
    assert g.kernel_path == 1
    check(bte, p, 12, precision=W.FP64, checkpoints=(1, 3))
    check(bte, p, 12, precision=W.FP32_STORE_FP64_ACC)


def test_generic_path_seventeen_bands(bte):
    """More than 16 bands (the fast path's parameter table holds 16): generic path, masked grid, diffuse interface."""
    p = W.random_problem(12, dim=3, shape=(12, 10, 8), n_bands=17, masked=True, interface_type=W.BC_DIFFUSE,
                         n_polar=8, n_azimuth=16)
    assert len(p.C) == 17
    g = bte.Solver(p)
    assert g.kernel_path == 1
    check(bte, p, 12, precision=W.FP64, checkpoints=(1, 3))
    check(bte, p, 12, precision=W.FP32_STORE_FP64_ACC)


# ---------------------------------------------------------------- reading G15 where it is weakest
def test_fp32_moments_antisymmetric_fifteen_bands(bte):
    """G15 as built: on the fast path the moments of ONE octant are summed in fp32 over 16 directions and all bands
    (tau spans three decades, so the 1/tau weights of M0 span three decades too).  Attacked where it is weakest: an
    antisymmetric +-dT_w film problem (signed intensities that cancel in M0, dT crosses zero) with the 15-band table,
    far into the iteration; error norm G12 against the fp64 oracle, and against the fp64 GPU path."""
    p = W.config(4, grid=(48, 34, 20))
    p.Q = None
    p.face_bc = [(W.BC_ISOTHERMAL, 0.5), (W.BC_ISOTHERMAL, -0.5), (W.BC_SPECULAR, 0.0), (W.BC_SPECULAR, 0.0),
                 (W.BC_SPECULAR, 0.0), (W.BC_SPECULAR, 0.0)]
    assert bte.Solver(p).kernel_path == 2
    out = check(bte, p, 300, precision=W.FP32_STORE_FP64_ACC, checkpoints=(5, 50))
    assert out[-1][1] <= 2e-5 and out[-1][2] <= 2e-5          # measured ~1e-6: an order of magnitude of margin
    a = bte.Solver(p, precision=W.FP64); a.iterate(300)
    b = bte.Solver(p, precision=W.FP32_STORE_FP64_ACC); b.iterate(300)
    eT, eq = errors(b.temperature().cpu().numpy(), b.heat_flux().cpu().numpy(),
                    a.temperature().cpu().numpy(), a.heat_flux().cpu().numpy())
    assert eT <= 2e-5 and eq <= 2e-5
    # antisymmetry about the mid-plane survives in fp32 to the same level
    dT = b.temperature().cpu().numpy()
    assert np.abs(dT + dT[:, :, ::-1]).max() <= 2e-5 * np.abs(dT).max()


@pytest.mark.slow
def test_config4_full_fp32_vs_fp64_gpu(bte):
    """Full-size config 4: the fp32-storage path against the fp64 GPU path (itself checked against the oracle at n = 5)
    at n = 5 and far into the iteration (n = 200), reading G15, tolerance 1e-4."""
    p = W.config(4)
    a = bte.Solver(p, precision=W.FP64)
    b = bte.Solver(p, precision=W.FP32_STORE_FP64_ACC)
    for n in (5, 195):
        a.iterate(n); b.iterate(n)
        eT, eq = errors(b.temperature().cpu().numpy(), b.heat_flux().cpu().numpy(),
                        a.temperature().cpu().numpy(), a.heat_flux().cpu().numpy())
        assert eT <= 1e-4 and eq <= 1e-4, (a.iterations_done, eT, eq)


def test_set_temperature_masks_void_cells(bte):
    """bte_set_temperature with nonzero values on void cells: void cells read 0 on both kernel paths (bte.h)."""
    import oracle
    for grid in ((12, 10, 8), (11, 9, 7)):              # fast (masked) / generic
        p = W.config(3, grid=grid)
        rng = np.random.default_rng(3)
        dT0 = rng.uniform(0.5, 1.0, size=(p.nz, p.ny, p.nx))          # nonzero everywhere, void cells included
        g = bte.Solver(p, precision=W.FP64)
        g.set_temperature(dT0)
        t = g.temperature().cpu().numpy()
        assert not t[p.mask == 0].any() and (t[p.mask == 1] == dT0[p.mask == 1]).all()
        ref = oracle.RefSolver(p); ref.set_temperature(dT0 * p.mask); ref.iterate(2)
        g.iterate(2)
        eT, eq = errors(g.temperature().cpu().numpy(), g.heat_flux().cpu().numpy(), ref.temperature(), ref.heat_flux())
        assert eT <= 1e-10 and eq <= 1e-10


def test_g14_directions_in_a_coordinate_plane(bte):
    """Reading G14 on the CUDA path: a quadrature with directions that have s_x = 0 or s_y = 0 exactly (azimuth offset
    0; isothermal faces only, such a table is not reflection-closed per octant), against the oracle."""
    mu, wmu = np.polynomial.legendre.leggauss(4)
    s, w = [], []
    for m, wm in zip(mu, wmu):
        st = np.sqrt(1.0 - m * m)
        for k in range(8):
            cx, cy = np.cos(k * np.pi / 4), np.sin(k * np.pi / 4)
            cx = 0.0 if abs(cx) < 1e-12 else cx
            cy = 0.0 if abs(cy) < 1e-12 else cy
            s.append((st * cx, st * cy, m)); w.append(wm * np.pi / 4)
    p = W.config(2, grid=(9, 8, 7))
    p.s, p.w = np.array(s), np.array(w)
    p.face_bc = [(W.BC_ISOTHERMAL, 0.1 * f) for f in range(6)]
    check(bte, p, 10, precision=W.FP64, checkpoints=(1, 2))
    check(bte, p, 10, precision=W.FP32_STORE_FP64_ACC)
