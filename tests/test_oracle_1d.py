"""Pins for the CPU oracle, part 1: quadrature sums and the 1-D gray film.

These check oracle/ against what the paper and the mathematics fix (never
against itself and never against the CUDA path):
  P1  quadrature integrates 1 -> 4pi, s -> 0, s s^T -> 4pi/3 I        (Eq. 14)
  P2a ballistic limit: uniform mid temperature, wall jumps           ("slip")
  P2b diffusive limit: linear bulk profile, closed-form k_eff        (derivation in DESIGN.md)
  P2c Kn = 1: radiative-equilibrium integral equation (own Nystrom)  (ref [59])
  P3  steady face flux constant in x
  golden: tests/golden/cfg0_kn1_film.txt (written by tests/golden/make_golden.py from oracle/ only)
"""
import os

import numpy as np
import pytest
from scipy.special import expn

import oracle
import workloads as W

FOUR_PI = 4 * np.pi


def film(nx, L, C=1.6e6, v=6400.0, tau=15.6e-12, n_mu=16, dTh=0.5, dTc=-0.5):
    s, w = W.quadrature_1d(n_mu)
    return W.Problem(name="film", nx=nx, ny=1, nz=1, dim=1, dx=L / nx, dy=1.0, dz=1.0,
                     C=np.array([C]), v=np.array([v]), tau=np.array([tau]), s=s, w=w,
                     face_bc=[(W.BC_ISOTHERMAL, dTh), (W.BC_ISOTHERMAL, dTc)] + [(W.BC_SPECULAR, 0.0)] * 4)


# ---------------------------------------------------------------- P1
@pytest.mark.parametrize("table", ["3d", "1d", "gl_theta"])
def test_quadrature_sums(table):
    if table == "3d":
        s, w = W.quadrature_3d()
    elif table == "1d":
        s, w = W.quadrature_1d()
    else:
        s, w = W.quadrature_gl_theta_octant()
    assert abs(w.sum() - FOUR_PI) < 1e-13 * FOUR_PI
    assert np.allclose(np.linalg.norm(s, axis=1), 1.0, atol=1e-15)
    if table == "1d":
        assert abs((w * s[:, 0]).sum()) < 1e-13 * FOUR_PI
        assert abs((w * s[:, 0] ** 2).sum() - FOUR_PI / 3) < 1e-13 * FOUR_PI
        return
    assert np.abs((w[:, None] * s).sum(0)).max() < 1e-13 * FOUR_PI
    second = np.einsum("d,da,db->ab", w, s, s)
    tol = 1e-13 * FOUR_PI if table == "3d" else 2e-3 * FOUR_PI  # GL-in-theta is not exact for s s^T
    assert np.abs(second - np.eye(3) * FOUR_PI / 3).max() < tol
    # 16 directions per octant, closed under the three mirror flips with equal weights
    octs = (s[:, 0] < 0) * 1 + (s[:, 1] < 0) * 2 + (s[:, 2] < 0) * 4
    assert np.all(np.bincount(octs, minlength=8) == len(w) // 8)
    for a in range(3):
        t = s.copy()
        t[:, a] *= -1
        for d in range(len(w)):
            m = np.where(np.abs(s - t[d]).max(1) < 1e-12)[0]
            assert len(m) == 1 and abs(w[m[0]] - w[d]) < 1e-15


def test_pi_face_is_discrete_hemisphere_sum():
    p = W.config(2, grid=(4, 4, 4))
    r = oracle.RefSolver(p)
    for f in range(6):
        a, side = divmod(f, 2)
        sn = (1 if side else -1) * p.s[:, a]
        assert abs(r.pi_face(f) - (p.w * np.where(sn < 0, -sn, 0)).sum()) < 1e-14
        assert 0.99 * np.pi < r.pi_face(f) < 1.02 * np.pi   # G10: close to, not equal to, pi


# ---------------------------------------------------------------- P2a
def test_ballistic_limit():
    """Kn >> 1: dT -> (dT_h + dT_c)/2 everywhere (jumps at both walls),
    q -> C v (dT_h - dT_c) S1 / 4pi with S1 = sum_{mu>0} w mu."""
    dTh, dTc = 0.7, -0.2
    p = film(200, 100e-9, tau=1e-6, dTh=dTh, dTc=dTc)  # MFP 6.4 mm, Kn = 6.4e4
    r = oracle.RefSolver(p, diagnostics=True)
    r.iterate(60)
    T = r.temperature().ravel()
    assert np.abs(T - 0.5 * (dTh + dTc)).max() < 3e-5 * (dTh - dTc)
    S1 = (p.w * np.clip(p.s[:, 0], 0, None)).sum()
    F = r.face_flux()[1].ravel()
    expected = 1.6e6 * 6400.0 * (dTh - dTc) * S1 / FOUR_PI
    assert np.abs(F / expected - 1).max() < 1e-4
    assert abs(S1 / np.pi - 1.00303) < 1e-5  # 16-pt GL half-range first moment


# ---------------------------------------------------------------- P2b
def test_diffusive_limit_closed_form_keff():
    """Kn << 1: in the bulk dT is exactly linear and the face flux obeys
    F = -k_eff dT/dx, k_eff = (C v L/3)(1 + (3/4)(S1/pi)(dx/L)), L = v tau
    (first-order-upwind numerical diffusion; -> C v^2 tau/3 as dx/L -> 0)."""
    C, v, n_mu = 1.6e6, 6400.0, 8
    L = 100e-9
    for nx in (100, 200):
        tau = (L / 100) / v          # MFP = L/100, Kn = 0.01
        p = film(nx, L, C=C, v=v, tau=tau, n_mu=n_mu)
        r = oracle.RefSolver(p, diagnostics=True)
        x = (np.arange(nx) + 0.5) / nx
        r.set_temperature(0.5 - x)
        for _ in range(400):
            r.iterate(250)
            if r.residual()[0] < 1e-14:
                break
        T = r.temperature().ravel()
        F = r.face_flux()[1].ravel()
        bulk = slice(nx // 4, 3 * nx // 4)
        slope = np.diff(T[bulk]) / p.dx
        assert np.abs(slope / slope.mean() - 1).max() < 1e-9          # exactly linear in the bulk
        Lam = v * tau
        S1 = (p.w * np.clip(p.s[:, 0], 0, None)).sum()
        keff = C * v * Lam / 3 * (1 + 0.75 * (S1 / np.pi) * (p.dx / Lam))
        assert abs(F[bulk].mean() / (-keff * slope.mean()) - 1) < 1e-9
        assert np.abs(F / F.mean() - 1).max() < 1e-10                 # P3 flux constancy
    # and k_eff -> C v^2 tau / 3 as dx/Lambda -> 0
    assert keff / (C * v * Lam / 3) < 1.0 + 0.76 * 1.01 * (p.dx / Lam)


# ---------------------------------------------------------------- P2c
def nystrom_slab(tauL, panels=60, order=8):
    """Radiative equilibrium between black parallel plates (gray medium):
    theta(t) = 1/2 [E2(t) + int_0^tauL theta(t') E1(|t-t'|) dt'],
    psi = q / (Eb1 - Eb2) = 1 - 2 int_0^tauL theta(t) E2(t) dt   (hot wall at t = 0).
    Singularity subtraction: int E1(|t-t'|) dt' = 2 - E2(t) - E2(tauL - t)."""
    xg, wg = np.polynomial.legendre.leggauss(order)
    edges = np.linspace(0, tauL, panels + 1)
    t = np.concatenate([(a + b) / 2 + (b - a) / 2 * xg for a, b in zip(edges[:-1], edges[1:])])
    wt = np.concatenate([(b - a) / 2 * wg for a, b in zip(edges[:-1], edges[1:])])
    n = len(t)
    dist = np.abs(t[:, None] - t[None, :])
    K = np.zeros((n, n))
    off = ~np.eye(n, dtype=bool)
    K[off] = expn(1, dist[off])
    Kw = K * wt[None, :]
    total = 2 - expn(2, t) - expn(2, tauL - t)
    A = np.eye(n) - 0.5 * (Kw - np.diag(Kw.sum(1)) + np.diag(total))
    theta = np.linalg.solve(A, 0.5 * expn(2, t))
    psi = 1 - 2 * (wt * theta * expn(2, t)).sum()
    return t, theta, psi


def test_kn1_matches_integral_equation():
    t, theta, psi = nystrom_slab(1.0)
    # the Nystrom reference is itself pinned by two textbook facts (Heaslet & Warming tables /
    # the slip-corrected diffusion asymptote psi -> (4/3)/(tauL + 2*0.710446)), then by 0.5532+-3e-4
    assert abs(nystrom_slab(0.1)[2] - 0.9157) < 1e-4
    assert abs(nystrom_slab(10.0, panels=200)[2] - (4 / 3) / (10 + 1.42089)) < 1e-5
    assert abs(psi - 0.5532) < 3e-4
    C, v, tau = 1.6e6, 6400.0, 15.6e-12
    L = v * tau                                 # L / MFP = 1 exactly
    errs = []
    for nx, n_mu in ((200, 16), (800, 32)):
        p = film(nx, L, n_mu=n_mu)
        r = oracle.RefSolver(p, diagnostics=True)
        r.iterate(120)
        F = r.face_flux()[1].ravel()
        ratio = F.mean() / (C * v * 1.0 / 4)
        errs.append(abs(ratio - psi))
        x = (np.arange(nx) + 0.5) / nx
        th = (r.temperature().ravel() + 0.5)   # (T - Tc)/(Th - Tc)
        assert np.abs(th - np.interp(x, t, theta)).max() < (4e-3 if nx == 200 else 1.2e-3)
    assert errs[0] < 3e-3 and errs[1] < 1e-3 and errs[1] < errs[0]   # first-order convergence


def test_config0_antisymmetric_and_golden():
    p = W.config(0)
    r = oracle.RefSolver(p, diagnostics=True)
    r.iterate(p.n_iter)
    T = r.temperature().ravel()
    assert np.abs(T + T[::-1]).max() < 1e-13                 # P7 antisymmetry about mid-plane
    assert r.residual() == (0.0, 0.0)                        # machine fixed point (harness tolerates 0)
    F = r.face_flux()[1].ravel()
    assert np.abs(F / F.mean() - 1).max() < 1e-12            # P3
    g = np.loadtxt(os.path.join(os.path.dirname(__file__), "golden", "cfg0_kn1_film.txt"))
    assert np.abs(T - g[:, 1]).max() < 1e-13
    assert np.abs(r.heat_flux()[0].ravel() - g[:, 2]).max() < 1e-13 * np.abs(g[:, 2]).max()
