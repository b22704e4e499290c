"""Pins for the CPU oracle, part 3: the stopping test (Eq. 23), reading G14 and specular interfaces.

  Eq. 23 (readings G11): eps_T = sqrt(sum_i (dT_i^{n+1} - dT_i^n)^2 / N_solid) / max_i |dT_i^{n+1}|,
      eps_q the same with |q_i| magnitudes.  Recomputed here in numpy from temperature() / heat_flux()
      snapshots taken at n and n+1 on a MASKED 3-D problem -- the formula is retyped from the paper, but the
      inputs come from two independent oracle calls, so a wrong normalisation (N_cell instead of N_solid),
      the maximum taken at iteration n, or a component-wise difference of q instead of |q| fails.
  G14: a direction with s_a = 0 on an active axis drops that axis (coefficient 0) and contributes nothing
      to H / Pi of faces normal to a.  Pinned by dense solve (P5 style) and by the hemispherical normaliser.
  Specular solid/void interfaces (Eq. 7): mirror symmetry -- a specular interface plane is
      equivalent to the mirror-extended solid without the interface.
"""
import numpy as np
import pytest

import oracle
import workloads as W


def masked_problem(seed=4, shape=(9, 8, 7), n_bands=3, interface=(W.BC_DIFFUSE, 0.0)):
    p = W.random_problem(seed, dim=3, shape=shape, n_bands=n_bands, masked=True,
                         bc_types=(W.BC_ISOTHERMAL, W.BC_DIFFUSE, W.BC_SPECULAR), interface_type=interface[0])
    return p


def eq23(dT0, dT1, q0, q1, solid):
    """Eq. 23 retyped from PAPER.md:299-304 with readings G11 (N = solid cells, max over solid cells at n+1)."""
    n_solid = int(solid.sum())
    dT0, dT1 = dT0[solid], dT1[solid]
    qm0 = np.sqrt((q0 ** 2).sum(0))[solid]
    qm1 = np.sqrt((q1 ** 2).sum(0))[solid]
    eT = np.sqrt(((dT1 - dT0) ** 2).sum() / n_solid) / np.abs(dT1).max()
    eq = np.sqrt(((qm1 - qm0) ** 2).sum() / n_solid) / qm1.max()
    return eT, eq


@pytest.mark.parametrize("n", [1, 2, 7, 30])
def test_residual_is_eq23_on_a_masked_grid(n):
    p = masked_problem()
    solid = p.mask.astype(bool)
    assert 0 < solid.sum() < solid.size            # N_solid != N_cell, so the normalisation is tested
    r = oracle.RefSolver(p)
    r.iterate(n)
    dT0, q0 = r.temperature(), r.heat_flux()
    r.iterate(1)
    dT1, q1 = r.temperature(), r.heat_flux()
    eT, eq = r.residual()
    eT_ref, eq_ref = eq23(dT0, dT1, q0, q1, solid)
    assert abs(eT - eT_ref) <= 1e-13 * eT_ref
    assert abs(eq - eq_ref) <= 1e-13 * eq_ref
    # the plausible misreadings give clearly different numbers on this problem (so the pin has teeth)
    n_cell = solid.size
    wrong_N = eT_ref * np.sqrt(solid.sum() / n_cell)
    wrong_max = np.sqrt(((dT1 - dT0)[solid] ** 2).sum() / solid.sum()) / np.abs(dT0[solid]).max()
    wrong_q = np.sqrt((((q1 - q0) ** 2).sum(0))[solid].sum() / solid.sum()) / np.sqrt((q1 ** 2).sum(0))[solid].max()
    assert abs(eT - wrong_N) > 1e-3 * eT_ref
    assert abs(eT - wrong_max) > 1e-6 * eT_ref
    assert abs(eq - wrong_q) > 1e-3 * eq_ref


def test_residual_first_iteration_counts_from_zero_state():
    """n = 0 -> 1: dT^0 = 0 and |q|^0 = 0, so eps_T = rms(dT^1)/max|dT^1| (a number of order 1, not 0)."""
    p = masked_problem(seed=6)
    solid = p.mask.astype(bool)
    r = oracle.RefSolver(p)
    r.iterate(1)
    dT1, q1 = r.temperature(), r.heat_flux()
    eT, eq = r.residual()
    eT_ref, eq_ref = eq23(np.zeros_like(dT1), dT1, np.zeros_like(q1), q1, solid)
    assert abs(eT - eT_ref) <= 1e-13 * eT_ref and abs(eq - eq_ref) <= 1e-13 * eq_ref
    assert 0.05 < eT <= 1.0


def test_residual_zero_over_zero():
    """G11: 0/0 -> 0.  All walls at dT_w = 0 and Q = 0: every iterate is exactly 0, so both norms are 0/0 and the
    oracle must report (0, 0), not nan.  (The x/0 -> +inf branch cannot be reached from the public interface:
    with C, tau > 0 the sweep operator is positive, so a nonzero dT^n never gives dT^{n+1} == 0 exactly.)"""
    C, v, tau = W.band_table(2)
    s, w = W.quadrature_3d(2, 4)
    bcs = [(W.BC_ISOTHERMAL, 0.0)] * 6
    p = W.Problem(name="zero", nx=4, ny=3, nz=2, dim=3, dx=1e-8, dy=1e-8, dz=1e-8, C=C, v=v, tau=tau, s=s, w=w,
                  face_bc=bcs, Q=None)
    r = oracle.RefSolver(p)
    r.iterate(3)
    assert r.residual() == (0.0, 0.0)
    assert not r.temperature().any() and not r.heat_flux().any()


# ---------------------------------------------------------------------------------------------- G14
def quadrature_with_in_plane_directions(n_polar=4, n_azimuth=8):
    """Azimuth offset 0: directions with phi = 0, pi/2, pi, 3pi/2 lie in coordinate planes (s_y = 0 or s_x = 0
    up to rounding -> forced to exact 0 here so the s_a = 0 branch is really taken)."""
    mu, wmu = np.polynomial.legendre.leggauss(n_polar)
    phi = np.arange(n_azimuth) * (2.0 * np.pi / n_azimuth)
    s, w = [], []
    for m, wm in zip(mu, wmu):
        st = np.sqrt(1.0 - m * m)
        for ph in phi:
            cx, cy = np.cos(ph), np.sin(ph)
            cx = 0.0 if abs(cx) < 1e-12 else cx
            cy = 0.0 if abs(cy) < 1e-12 else cy
            s.append((st * cx, st * cy, m))
            w.append(wm * 2.0 * np.pi / n_azimuth)
    return np.array(s), np.array(w)


def test_g14_direction_in_a_coordinate_plane_dense_solve():
    """One sweep with directions that have s_x = 0 or s_y = 0 equals the dense solve of Eq. 21
    in which the zero component simply contributes no face term -- whichever sign the oracle assigns."""
    rng = np.random.default_rng(11)
    nx, ny, nz = 5, 4, 3
    C, v, tau = W.band_table(2, seed=W.MASTER_SEED + 5)
    s, w = quadrature_with_in_plane_directions()
    assert (s[:, 0] == 0).any() and (s[:, 1] == 0).any()
    iso = [(W.BC_ISOTHERMAL, float(t)) for t in rng.uniform(-1, 1, 6)]
    d = (9e-9, 12e-9, 15e-9)
    p = W.Problem(name="g14", nx=nx, ny=ny, nz=nz, dim=3, dx=d[0], dy=d[1], dz=d[2], C=C, v=v, tau=tau, s=s, w=w,
                  face_bc=iso, Q=rng.uniform(0, 1e17, size=(nz, ny, nx)))
    r = oracle.RefSolver(p, diagnostics=True)
    dT0 = rng.uniform(-1, 1, size=(nz, ny, nx))
    r.set_temperature(dT0)
    r.iterate(1)
    e = r.intensity()                                   # [B, D, nz, ny, nx]
    N = nx * ny * nz
    n = (nx, ny, nz)
    idx = lambda i, j, k: i + nx * (j + ny * k)
    sumC = C.sum()
    for b in range(len(C)):
        for dd in range(len(w)):
            A = np.zeros((N, N))
            rhs = np.zeros(N)
            for k in range(nz):
                for j in range(ny):
                    for i in range(nx):
                        row = idx(i, j, k)
                        A[row, row] = 1.0 / tau[b]
                        rhs[row] = (C[b] * dT0[k, j, i] / (4 * np.pi)) / tau[b] + C[b] * p.Q[k, j, i] / sumC / (4 * np.pi)
                        cell = (i, j, k)
                        for a in range(3):
                            sa = s[dd, a]
                            if sa == 0.0:
                                continue                  # G14: the axis drops out
                            flux = v[b] * abs(sa) / d[a]  # (1/V) |v.n| S
                            A[row, row] += flux           # outflow through the downwind face (Eq. 21 diagonal)
                            up = list(cell)
                            up[a] -= 1 if sa > 0 else -1
                            if 0 <= up[a] < n[a]:
                                A[row, idx(*up)] -= flux  # inflow from the upwind neighbour (Eq. 21 off-diagonal, G5)
                            else:
                                f = 2 * a + (0 if sa > 0 else 1)
                                rhs[row] += flux * C[b] * iso[f][1] / (4 * np.pi)   # Eq. 5
            x = np.linalg.solve(A, rhs)
            assert np.abs(x - e[b, dd].ravel()).max() <= 1e-12 * np.abs(x).max()


def test_g14_in_plane_directions_do_not_enter_pi_of_that_face():
    """Pi_f = sum_{s.n<0} w |s.n| (reading G10): directions with s.n = 0 contribute nothing, whichever octant
    they were filed under.  Checked on the x faces and y faces against a numpy sum."""
    C, v, tau = W.band_table(1)
    s, w = quadrature_with_in_plane_directions()
    bcs = [(W.BC_ISOTHERMAL, 0.0)] + [(W.BC_DIFFUSE, 0.0)] * 5
    p = W.Problem(name="g14pi", nx=3, ny=3, nz=3, dim=3, dx=1e-8, dy=1e-8, dz=1e-8, C=C, v=v, tau=tau, s=s, w=w,
                  face_bc=bcs, Q=np.full((3, 3, 3), 1e16))
    r = oracle.RefSolver(p, diagnostics=True)
    for f in range(6):
        a, sign = f // 2, (-1.0 if f % 2 == 0 else 1.0)     # outward normal = sign * e_a
        sn = sign * s[:, a]
        assert abs(r.pi_face(f) - (w * np.abs(sn))[sn < 0].sum()) <= 1e-14
    # and the converged solution conserves energy with such a table (P4): isothermal power == int Q dV
    for _ in range(400):
        r.iterate(50)
        if r.residual()[0] < 1e-13:
            break
    pw = r.boundary_power()                             # net outflow by BC type [iso, diffuse, specular, periodic]
    total_Q = p.Q.sum() * p.dx * p.dy * p.dz
    assert abs(pw[W.BC_ISOTHERMAL] / total_Q - 1.0) < 1e-9
    assert abs(pw[W.BC_DIFFUSE]) < 1e-9 * total_Q


# ---------------------------------------------------------------------------------------------- specular interface
def test_specular_interface_equals_mirror_extension():
    """Eq. 7 at a solid/void interface: a solid slab 0 <= i < n whose x+ side is a specular solid/void interface
    plane behaves like the x-mirror-extended solid (2n cells, mirrored source, both outer x faces carrying the
    original x- boundary condition) restricted to the first half."""
    rng = np.random.default_rng(3)
    n, ny, nz = 4, 3, 3
    C, v, tau = W.band_table(2, seed=W.MASTER_SEED + 9)
    s, w = W.quadrature_3d(2, 4)
    Qh = rng.uniform(0, 1e17, size=(nz, ny, n))
    side = [(W.BC_DIFFUSE, 0.0), (W.BC_DIFFUSE, 0.0), (W.BC_ISOTHERMAL, 0.1), (W.BC_DIFFUSE, 0.0)]
    # (a) masked: box of 2n cells in x, right half void, interface specular; the x+ box face is never reached
    mask = np.zeros((nz, ny, 2 * n), dtype=np.uint8)
    mask[:, :, :n] = 1
    Qa = np.zeros((nz, ny, 2 * n))
    Qa[:, :, :n] = Qh
    pa = W.Problem(name="spec_if", nx=2 * n, ny=ny, nz=nz, dim=3, dx=8e-9, dy=9e-9, dz=1e-8, C=C, v=v, tau=tau, s=s, w=w,
                   face_bc=[(W.BC_ISOTHERMAL, 0.7), (W.BC_ISOTHERMAL, -5.0)] + side,
                   interface_bc=(W.BC_SPECULAR, 0.0), mask=mask, Q=Qa)
    # (b) all solid mirror extension
    Qb = np.concatenate([Qh, Qh[:, :, ::-1]], axis=2)
    pb = W.Problem(name="spec_mirror", nx=2 * n, ny=ny, nz=nz, dim=3, dx=8e-9, dy=9e-9, dz=1e-8, C=C, v=v, tau=tau,
                   s=s, w=w, face_bc=[(W.BC_ISOTHERMAL, 0.7), (W.BC_ISOTHERMAL, 0.7)] + side, Q=Qb)
    ra, rb = oracle.RefSolver(pa), oracle.RefSolver(pb)
    for r in (ra, rb):
        for _ in range(400):
            r.iterate(50)
            if r.residual()[0] < 1e-14:
                break
    Ta, Tb = ra.temperature(), rb.temperature()
    qa, qb = ra.heat_flux(), rb.heat_flux()
    sc = np.abs(Tb).max()
    assert np.abs(Ta[:, :, :n] - Tb[:, :, :n]).max() <= 1e-10 * sc
    assert np.abs(qa[:, :, :, :n] - qb[:, :, :, :n]).max() <= 1e-10 * np.abs(qb).max()
    assert not Ta[:, :, n:].any()                      # void cells read 0
