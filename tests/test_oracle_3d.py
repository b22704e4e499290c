"""Pins for the CPU oracle, part 2: multi-dimensional properties.

  P4  energy balance: power through isothermal faces = int Q dV; adiabatic faces carry no net
      flux per band; G10: the literal 1/pi of Eq. 6 leaks, the discrete Pi_f does not
  P5  (i) one sweep == dense LU solve of A e = b with A from Eq. 21 (reading G5)
      (ii) the converged iteration == dense solve of the coupled (band x dir x cell) system
  P6  linearity / shift invariance (reading G3)
  P7  mirror and axis-permutation symmetry
  P8  B identical bands with C/B == one band
  G9  result independent of the (band, direction) visiting order; thread count
"""
import numpy as np
import pytest

import oracle
import workloads as W

FOUR_PI = 4 * np.pi


def small(dim=3, shape=(5, 4, 3), bcs=None, n_bands=2, quad=(2, 4), mask=None, Q=None, seed=0,
          interface=(W.BC_DIFFUSE, 0.0)):
    rng = np.random.default_rng(seed)
    nx, ny, nz = shape
    C, v, tau = W.band_table(n_bands, seed=W.MASTER_SEED + seed)
    s, w = W.quadrature_3d(*quad)
    if bcs is None:
        bcs = [(W.BC_ISOTHERMAL, 0.3), (W.BC_DIFFUSE, 0.0), (W.BC_SPECULAR, 0.0),
               (W.BC_ISOTHERMAL, -0.2), (W.BC_DIFFUSE, 0.0), (W.BC_SPECULAR, 0.0)]
    if Q is None:
        Q = rng.uniform(0, 1e17, size=(nz, ny, nx))
    if mask is not None:
        Q = Q * mask
    return W.Problem(name="small", nx=nx, ny=ny, nz=nz, dim=dim, dx=11e-9, dy=13e-9, dz=17e-9,
                     C=C, v=v, tau=tau, s=s, w=w, face_bc=list(bcs), interface_bc=interface,
                     mask=mask, Q=Q)


def converge(r, tol=1e-13, chunk=50, cap=40000):
    n = 0
    while n < cap:
        r.iterate(chunk)
        n += chunk
        if r.residual()[0] < tol:
            break
    return n


# ---------------------------------------------------------------- P5 (i)
@pytest.mark.parametrize("shape,dim", [((8, 8, 8), 3), ((9, 7, 1), 2), ((12, 1, 1), 1)])
def test_one_sweep_is_dense_solve_of_eq21(shape, dim):
    rng = np.random.default_rng(5)
    nx, ny, nz = shape
    iso = [(W.BC_ISOTHERMAL, float(t)) for t in rng.uniform(-1, 1, 6)]
    mask = (rng.uniform(size=(nz, ny, nx)) > 0.15).astype(np.uint8)
    p = small(dim=dim, shape=shape, bcs=iso, mask=mask, interface=(W.BC_ISOTHERMAL, 0.4), seed=3)
    r = oracle.RefSolver(p, diagnostics=True)
    dT0 = rng.uniform(-1, 1, size=(nz, ny, nx)) * mask
    r.set_temperature(dT0)
    r.iterate(1)
    e = r.intensity()
    delta = [p.dx, p.dy, p.dz]
    n = [nx, ny, nz]
    N = nx * ny * nz
    solid = mask.ravel().astype(bool)
    idx = lambda i, j, k: i + nx * (j + ny * k)
    sumC = p.C.sum()
    for b in range(len(p.C)):
        for d in range(0, len(p.w), 3):
            A = np.zeros((N, N))
            rhs = np.zeros(N)
            for k in range(nz):
                for j in range(ny):
                    for i in range(nx):
                        c = idx(i, j, k)
                        if not solid[c]:
                            A[c, c] = 1.0
                            continue
                        A[c, c] = 1.0 / p.tau[b]
                        rhs[c] = (p.C[b] / FOUR_PI) * dT0.ravel()[c] / p.tau[b] + p.C[b] * p.Q.ravel()[c] / sumC / FOUR_PI
                        ijk = [i, j, k]
                        for a in range(dim):
                            vn = p.v[b] * abs(p.s[d, a]) / delta[a]   # |v.n| S_ij / V_i
                            A[c, c] += vn                              # outflow face: H(v.n) term of A_ii
                            u = list(ijk)
                            u[a] -= 1 if p.s[d, a] >= 0 else -1
                            if 0 <= u[a] < n[a] and solid[idx(*u)]:
                                A[c, idx(*u)] -= vn                    # inflow face: A_ij (with S_ij, G5)
                            else:
                                if 0 <= u[a] < n[a]:
                                    Tw = 0.4
                                else:
                                    Tw = iso[2 * a + (0 if p.s[d, a] >= 0 else 1)][1]
                                rhs[c] += vn * p.C[b] * Tw / FOUR_PI    # Eq. 5
            x = np.linalg.solve(A, rhs)
            ref = e[b, d].ravel()
            assert np.abs(x[solid] - ref[solid]).max() < 1e-12 * np.abs(x).max()


# ---------------------------------------------------------------- P5 (ii)
def coupled_dense_solution(p):
    """Fixed point of the whole iteration as ONE linear system over (band, dir, solid cell)."""
    nx, ny, nz = p.nx, p.ny, p.nz
    n = [nx, ny, nz]
    delta = [p.dx, p.dy, p.dz]
    B, D = len(p.C), len(p.w)
    N = nx * ny * nz
    solid = np.ones(N, bool) if p.mask is None else p.mask.ravel().astype(bool)
    Qf = np.zeros(N) if p.Q is None else p.Q.ravel()
    idx = lambda i, j, k: i + nx * (j + ny * k)
    col = lambda b, d, c: (b * D + d) * N + c
    M = np.zeros((B * D * N, B * D * N))
    rhs = np.zeros(B * D * N)
    sumC, sumCt = p.C.sum(), (p.C / p.tau).sum()
    refl = []
    for a in range(3):
        t = p.s.copy()
        t[:, a] *= -1
        refl.append([int(np.argmin(np.abs(p.s - t[d]).max(1))) for d in range(D)])
    for b in range(B):
        for d in range(D):
            for k in range(nz):
                for j in range(ny):
                    for i in range(nx):
                        c = idx(i, j, k)
                        r = col(b, d, c)
                        if not solid[c]:
                            M[r, r] = 1.0
                            continue
                        M[r, r] += 1.0
                        # e0 coupling: -(C_b/4pi) dT_c, dT_c = sum_b' sum_d' (w/tau_b') e / sum(C/tau)  (Eq. 16)
                        for b2 in range(B):
                            for d2 in range(D):
                                M[r, col(b2, d2, c)] -= (p.C[b] / FOUR_PI) * p.w[d2] / p.tau[b2] / sumCt
                        rhs[r] += (p.C[b] / FOUR_PI) * p.tau[b] * Qf[c] / sumC
                        ijk = [i, j, k]
                        for a in range(p.dim):
                            ca = p.v[b] * p.tau[b] * abs(p.s[d, a]) / delta[a]
                            M[r, r] += ca
                            sg = 1 if p.s[d, a] >= 0 else -1
                            u = list(ijk)
                            u[a] -= sg
                            side = 0 if sg > 0 else 1
                            bc = None
                            if 0 <= u[a] < n[a]:
                                if solid[idx(*u)]:
                                    M[r, col(b, d, idx(*u))] -= ca
                                    continue
                                bc = p.interface_bc
                            else:
                                bc = p.face_bc[2 * a + side]
                                if bc[0] == W.BC_PERIODIC:
                                    u[a] %= n[a]
                                    if solid[idx(*u)]:
                                        M[r, col(b, d, idx(*u))] -= ca
                                        continue
                                    bc = p.interface_bc
                            if bc[0] == W.BC_ISOTHERMAL:
                                rhs[r] += ca * p.C[b] * bc[1] / FOUR_PI
                            elif bc[0] == W.BC_SPECULAR:
                                M[r, col(b, refl[a][d], c)] -= ca
                            else:  # diffuse, discrete normalisation
                                nsign = -sg  # outward normal of the upwind face
                                sn = nsign * p.s[:, a]
                                Pi = (p.w * np.where(sn < 0, -sn, 0)).sum()
                                for d2 in range(D):
                                    if sn[d2] > 0:
                                        M[r, col(b, d2, c)] -= ca * p.w[d2] * sn[d2] / Pi
    x = np.linalg.solve(M, rhs).reshape(B, D, N)
    dT = np.einsum("bdc,d,b->c", x, p.w, 1 / p.tau) / sumCt
    q = np.einsum("bdc,d,da,b->ac", x, p.w, p.s, p.v)
    return x, dT * solid, q * solid


@pytest.mark.parametrize("case", ["mixed", "periodic_masked", "2d"])
def test_converged_iteration_is_coupled_dense_solve(case):
    rng = np.random.default_rng(11)
    if case == "mixed":
        p = small(shape=(4, 4, 4), quad=(2, 4))
    elif case == "periodic_masked":
        mask = np.ones((3, 4, 4), np.uint8)
        mask[2, 1:3, 0] = 0
        mask[0, 0, 3] = 0
        bcs = [(W.BC_PERIODIC, 0.0), (W.BC_PERIODIC, 0.0), (W.BC_DIFFUSE, 0.0), (W.BC_SPECULAR, 0.0),
               (W.BC_ISOTHERMAL, 0.1), (W.BC_DIFFUSE, 0.0)]
        p = small(shape=(4, 4, 3), bcs=bcs, mask=mask, quad=(2, 4))
    else:
        bcs = [(W.BC_SPECULAR, 0.0), (W.BC_DIFFUSE, 0.0), (W.BC_ISOTHERMAL, 0.2), (W.BC_SPECULAR, 0.0)] + \
              [(W.BC_SPECULAR, 0.0)] * 2
        p = small(dim=2, shape=(6, 5, 1), bcs=bcs, quad=(2, 4))
    # shrink the box so the iteration converges quickly (Kn ~ 1)
    p.dx = p.dy = p.dz = 40e-9
    x, dT, q = coupled_dense_solution(p)
    r = oracle.RefSolver(p, diagnostics=True)
    converge(r, tol=1e-15, cap=20000)
    T = r.temperature().ravel()
    assert np.abs(T - dT).max() < 1e-10 * np.abs(dT).max()
    assert np.abs(r.heat_flux().reshape(3, -1) - q).max() < 1e-10 * np.abs(q).max()
    e = r.intensity().reshape(x.shape)
    assert np.abs(e - x).max() < 1e-10 * np.abs(x).max()


# ---------------------------------------------------------------- P4, G10
def test_energy_balance_and_diffuse_normalisation():
    p = W.config(2, grid=(6, 6, 6))
    p.C, p.v, p.tau = p.C[2::4], p.v[2::4], p.tau[2::4]     # 4 of the 15 bands: same physics, 4x faster
    vol = p.dx * p.dy * p.dz
    total_Q = p.Q.sum() * vol
    r = oracle.RefSolver(p, diagnostics=True)
    converge(r, tol=1e-12, cap=30000)
    pw = r.boundary_power()
    assert abs(pw[W.BC_ISOTHERMAL] / total_Q - 1) < 1e-8
    assert abs(pw[W.BC_DIFFUSE]) < 1e-8 * total_Q
    # adiabatic faces carry zero net flux per band
    fb = r.face_flux_band()
    assert np.abs(fb[:, 1, :, :, -1]).max() < 1e-9 * np.abs(fb[:, 4]).max()   # x+ face, diffuse
    # cell-wise conservation of the face fluxes: sum_faces F A = Q V (every cell, G18)
    ff = r.face_flux()
    div = (ff[0] + ff[1]) * p.dy * p.dz + (ff[2] + ff[3]) * p.dx * p.dz + (ff[4] + ff[5]) * p.dx * p.dy
    assert np.abs(div - p.Q * vol).max() < 1e-9 * (p.Q * vol).max()
    # Eq. 6 taken literally (1/pi) leaks energy with this quadrature (reading G10)
    r2 = oracle.RefSolver(p, diagnostics=True, literal_one_over_pi=True)
    converge(r2, tol=1e-12, cap=30000)
    leak = r2.boundary_power()[W.BC_ISOTHERMAL] / total_Q
    assert abs(leak - 1) > 1e-2


def test_no_source_flux_is_divergence_free():
    bcs = [(W.BC_ISOTHERMAL, 1.0), (W.BC_ISOTHERMAL, -1.0), (W.BC_SPECULAR, 0.0), (W.BC_DIFFUSE, 0.0),
           (W.BC_DIFFUSE, 0.0), (W.BC_SPECULAR, 0.0)]
    p = small(shape=(6, 5, 4), bcs=bcs, Q=np.zeros((4, 5, 6)), quad=(4, 8))
    p.dx = p.dy = p.dz = 30e-9
    r = oracle.RefSolver(p, diagnostics=True)
    converge(r, tol=1e-14)
    ff = r.face_flux()
    div = (ff[0] + ff[1]) / p.dx + (ff[2] + ff[3]) / p.dy + (ff[4] + ff[5]) / p.dz
    assert np.abs(div).max() < 1e-10 * np.abs(ff).max() / p.dx
    pw = r.boundary_power()
    assert abs(pw.sum()) < 1e-10 * np.abs(ff).max() * p.dy * p.dz * 20


# ---------------------------------------------------------------- P6
def test_linearity_and_shift_invariance():
    p = small(shape=(5, 4, 3))
    n = 30

    def run(prob):
        r = oracle.RefSolver(prob)
        r.iterate(n)
        return r.temperature(), r.heat_flux()

    T1, q1 = run(p)
    p2 = small(shape=(5, 4, 3))
    p2.Q = 2.5 * p.Q
    p2.face_bc = [(t, 2.5 * x) for t, x in p.face_bc]
    T2, q2 = run(p2)
    assert np.abs(T2 - 2.5 * T1).max() < 1e-12 * np.abs(T2).max()
    assert np.abs(q2 - 2.5 * q1).max() < 1e-12 * np.abs(q2).max()
    # shift: at convergence, adding a constant to all isothermal walls shifts dT, leaves q
    p.dx = p.dy = p.dz = 30e-9
    p3 = small(shape=(5, 4, 3))
    p3.dx = p3.dy = p3.dz = 30e-9
    p3.face_bc = [(t, x + 7.0 if t == W.BC_ISOTHERMAL else x) for t, x in p.face_bc]
    ra, rb = oracle.RefSolver(p), oracle.RefSolver(p3)
    converge(ra, tol=1e-15)
    converge(rb, tol=1e-15)
    assert np.abs(rb.temperature() - ra.temperature() - 7.0).max() < 1e-11
    assert np.abs(rb.heat_flux() - ra.heat_flux()).max() < 1e-10 * np.abs(ra.heat_flux()).max()


# ---------------------------------------------------------------- P7
def transform(p, perm, flips):
    """Apply the signed axis permutation new_axis a = old axis perm[a] (flipped if flips[a])."""
    n_old = [p.nx, p.ny, p.nz]
    d_old = [p.dx, p.dy, p.dz]

    def tf(field):  # field [nz,ny,nx] -> transformed
        f = np.transpose(field, (2, 1, 0))            # [x,y,z]
        f = np.transpose(f, perm)
        for a in range(3):
            if flips[a]:
                f = np.flip(f, axis=a)
        return np.ascontiguousarray(np.transpose(f, (2, 1, 0)))

    s = p.s[:, perm].copy()
    for a in range(3):
        if flips[a]:
            s[:, a] *= -1
    fb = []
    for a in range(3):
        lo, hi = p.face_bc[2 * perm[a]], p.face_bc[2 * perm[a] + 1]
        fb += [hi, lo] if flips[a] else [lo, hi]
    return W.Problem(name="t", nx=n_old[perm[0]], ny=n_old[perm[1]], nz=n_old[perm[2]], dim=3,
                     dx=d_old[perm[0]], dy=d_old[perm[1]], dz=d_old[perm[2]], C=p.C, v=p.v, tau=p.tau,
                     s=s, w=p.w, face_bc=fb, interface_bc=p.interface_bc,
                     mask=None if p.mask is None else tf(p.mask), Q=tf(p.Q)), tf


@pytest.mark.parametrize("perm,flips", [((0, 1, 2), (1, 0, 0)), ((1, 0, 2), (0, 0, 0)),
                                        ((2, 0, 1), (0, 1, 1)), ((0, 2, 1), (1, 1, 1))])
def test_signed_axis_permutation_symmetry(perm, flips):
    rng = np.random.default_rng(2)
    mask = (rng.uniform(size=(4, 5, 6)) > 0.2).astype(np.uint8)
    p = small(shape=(6, 5, 4), mask=mask, quad=(4, 8))
    pt, tf = transform(p, perm, flips)
    ra, rb = oracle.RefSolver(p), oracle.RefSolver(pt)
    ra.iterate(12)
    rb.iterate(12)
    Ta, Tb = ra.temperature(), rb.temperature()
    assert np.abs(tf(Ta) - Tb).max() < 1e-13 * np.abs(Ta).max()
    qa, qb = ra.heat_flux(), rb.heat_flux()
    for a in range(3):
        exp = tf(qa[perm[a]]) * (-1 if flips[a] else 1)
        assert np.abs(exp - qb[a]).max() < 1e-13 * np.abs(qa).max()


def test_config3_mirror_symmetric_in_y():
    p = W.config(3, grid=(16, 16, 16))
    r = oracle.RefSolver(p)
    r.iterate(10)
    T = r.temperature()
    assert np.abs(T - T[:, ::-1, :]).max() < 1e-13 * np.abs(T).max()
    q = r.heat_flux()
    assert np.abs(q[1] + q[1][:, ::-1, :]).max() < 1e-12 * np.abs(q).max()


def test_config1_2d_has_no_qz():
    p = W.config(1, grid=(24, 24, 1))
    r = oracle.RefSolver(p)
    r.iterate(10)
    q = r.heat_flux()
    assert np.abs(q[2]).max() < 1e-13 * np.abs(q).max()      # G16


# ---------------------------------------------------------------- P8, G9
def test_gray_equivalence():
    p1 = small(shape=(5, 4, 3), n_bands=1)
    pB = small(shape=(5, 4, 3), n_bands=1)
    Bn = 4
    pB.C = np.repeat(p1.C / Bn, Bn)
    pB.v = np.repeat(p1.v, Bn)
    pB.tau = np.repeat(p1.tau, Bn)
    ra, rb = oracle.RefSolver(p1), oracle.RefSolver(pB)
    ra.iterate(15)
    rb.iterate(15)
    assert np.abs(ra.temperature() - rb.temperature()).max() < 1e-13 * np.abs(ra.temperature()).max()
    assert np.abs(ra.heat_flux() - rb.heat_flux()).max() < 1e-13 * np.abs(ra.heat_flux()).max()


def test_direction_order_and_threads_do_not_matter():
    rng = np.random.default_rng(9)
    mask = (rng.uniform(size=(4, 5, 6)) > 0.2).astype(np.uint8)
    p = small(shape=(6, 5, 4), mask=mask, quad=(4, 8), n_bands=3)
    ra, rb, rc = oracle.RefSolver(p), oracle.RefSolver(p), oracle.RefSolver(p, threads=3)
    rb.set_dir_order(rng.permutation(len(p.w)))
    for r in (ra, rb, rc):
        r.iterate(8)
    assert np.array_equal(ra.temperature(), rc.temperature())          # threads: bit-identical
    assert np.array_equal(ra.heat_flux(), rc.heat_flux())
    assert np.abs(ra.temperature() - rb.temperature()).max() < 1e-14 * np.abs(ra.temperature()).max()
    assert np.abs(ra.heat_flux() - rb.heat_flux()).max() < 1e-13 * np.abs(ra.heat_flux()).max()


def test_invalid_inputs_are_rejected():
    p = small()
    p.tau = -p.tau
    with pytest.raises(ValueError):
        oracle.RefSolver(p)
    p = small()
    p.face_bc[0] = (W.BC_PERIODIC, 0.0)      # unpaired periodic
    with pytest.raises(ValueError):
        oracle.RefSolver(p)
    p = small()
    p.s = p.s.copy()
    p.s[0] = [0.6, 0.0, 0.8]                 # breaks closure under reflection; specular requested
    with pytest.raises(ValueError):
        oracle.RefSolver(p)
