"""Seeded problem generators (inputs only; no solver arithmetic).

Every array produced here is passed unchanged to both the CPU oracle and the
CUDA library, so PRNG identity between the two never matters.
"""
from __future__ import annotations

from dataclasses import dataclass, field, replace
from typing import List, Optional, Tuple

import numpy as np

MASTER_SEED = 250323657  # arxiv 2503.23657

# numeric codes of the C-ABI enums (include/bte.h and oracle/bte_ref.h each
# declare their own copy; these are plain integers, not shared code)
BC_ISOTHERMAL, BC_DIFFUSE, BC_SPECULAR, BC_PERIODIC = 0, 1, 2, 3
FP64, FP32_STORE_FP64_ACC = 0, 1

CONFIG_NAMES = [
    "cfg0_1d_gray_film",
    "cfg1_2d_nongray_hotspot",
    "cfg2_3d_cube_diffuse",
    "cfg3_finfet_voxels",
    "cfg4_large_slab",
]


@dataclass
class Problem:
    """Plain-array description of one BTE problem (SURVEY.md 8(b) `bte_problem`)."""
    name: str
    nx: int
    ny: int
    nz: int
    dim: int
    dx: float
    dy: float
    dz: float
    C: np.ndarray          # [B]  J/m^3K
    v: np.ndarray          # [B]  m/s
    tau: np.ndarray        # [B]  s
    s: np.ndarray          # [D,3] unit vectors
    w: np.ndarray          # [D]   weights, sum = 4*pi
    face_bc: List[Tuple[int, float]]      # x-,x+,y-,y+,z-,z+ : (type, dT_wall)
    interface_bc: Tuple[int, float] = (BC_DIFFUSE, 0.0)
    mask: Optional[np.ndarray] = None     # uint8 [nz,ny,nx] (x fastest), 1 = solid
    Q: Optional[np.ndarray] = None        # float64 [nz,ny,nx], W/m^3
    precision: int = FP64
    n_iter: int = 50                      # iteration count used for parity
    notes: str = ""

    @property
    def n_cells(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def n_solid(self) -> int:
        return self.n_cells if self.mask is None else int(self.mask.sum())

    @property
    def updates_per_sweep(self) -> int:
        return self.n_solid * len(self.C) * len(self.w)

    def with_precision(self, precision: int) -> "Problem":
        return replace(self, precision=precision)


# ----------------------------------------------------------------------------
# tables
# ----------------------------------------------------------------------------
def band_table(n_bands: int = 15, seed: int = MASTER_SEED):
    """v log-uniform [1e3,8e3] m/s, tau log-uniform [1e-12,1e-9] s
    (all v drawn first, then all tau), C_b = 1.6e6 * b^2 / sum(b^2)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    v = np.exp(rng.uniform(np.log(1e3), np.log(8e3), n_bands))
    tau = np.exp(rng.uniform(np.log(1e-12), np.log(1e-9), n_bands))
    b = np.arange(1, n_bands + 1, dtype=np.float64)
    C = 1.6e6 * b * b / np.sum(b * b)
    return C, v, tau


def quadrature_3d(n_polar: int = 8, n_azimuth: int = 16):
    """Gauss-Legendre in mu = cos(theta) on [-1,1] (polar axis z) x uniform
    azimuth phi_k = (k+1/2) 2pi/n_azimuth (Eq. 14; reading G6)."""
    mu, wmu = np.polynomial.legendre.leggauss(n_polar)
    phi = (np.arange(n_azimuth) + 0.5) * (2.0 * np.pi / n_azimuth)
    s = np.empty((n_polar * n_azimuth, 3))
    w = np.empty(n_polar * n_azimuth)
    n = 0
    for m, wm in zip(mu, wmu):
        st = np.sqrt(max(0.0, 1.0 - m * m))
        for p in phi:
            s[n] = (st * np.cos(p), st * np.sin(p), m)
            w[n] = wm * (2.0 * np.pi / n_azimuth)
            n += 1
    return s, w


def quadrature_1d(n_mu: int = 16):
    """1-D slab table: s = (mu, sqrt(1-mu^2), 0), w = 2 pi w_GL (azimuthal symmetry)."""
    mu, wmu = np.polynomial.legendre.leggauss(n_mu)
    s = np.stack([mu, np.sqrt(1.0 - mu * mu), np.zeros_like(mu)], axis=1)
    return s, 2.0 * np.pi * wmu


def quadrature_gl_theta_octant(n_theta: int = 4, n_phi: int = 4):
    """The paper's own variant: [n_theta, n_phi] Gauss-Legendre in
    theta AND phi per octant, weight sin(theta), polar axis x,
    s = (cos t, sin t cos p, sin t sin p).  Sum of weights is 4 pi only to
    quadrature accuracy, so weights are rescaled to sum exactly to 4 pi."""
    xt, wt = np.polynomial.legendre.leggauss(n_theta)
    xp, wp = np.polynomial.legendre.leggauss(n_phi)
    s, w = [], []
    for it in range(2):
        t0 = it * np.pi / 2
        for ip in range(4):
            p0 = ip * np.pi / 2
            for a, wa in zip(xt, wt):
                th = t0 + (a + 1.0) * np.pi / 4
                for b, wb in zip(xp, wp):
                    ph = p0 + (b + 1.0) * np.pi / 4
                    s.append((np.cos(th), np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph)))
                    w.append(wa * wb * (np.pi / 4) ** 2 * np.sin(th))
    s = np.array(s)
    w = np.array(w)
    w *= 4.0 * np.pi / w.sum()
    return s, w


# ----------------------------------------------------------------------------
# fields
# ----------------------------------------------------------------------------
def _centres(n, d):
    return (np.arange(n) + 0.5) * d


def _gaussian(nx, ny, nz, dx, dy, dz, centre, sigma, peak):
    x = _centres(nx, dx)[None, None, :]
    y = _centres(ny, dy)[None, :, None]
    z = _centres(nz, dz)[:, None, None]
    r2 = (x - centre[0]) ** 2 + (y - centre[1]) ** 2
    if nz > 1 or centre[2] is not None:
        r2 = r2 + (z - (centre[2] if centre[2] is not None else 0.0)) ** 2
    return peak * np.exp(-r2 / (2.0 * sigma * sigma)) * np.ones((nz, ny, nx))


# ----------------------------------------------------------------------------
# the five configs of BASELINE.json
# ----------------------------------------------------------------------------
def config(k: int, grid: Optional[Tuple[int, int, int]] = None, precision: Optional[int] = None) -> Problem:
    """Config k of BASELINE.json. `grid=(nx,ny,nz)` keeps the physical size and
    changes only the resolution (shrunken replicas for fast parity tests)."""
    if k == 0:
        nx = 200 if grid is None else grid[0]
        L = 100e-9
        s, w = quadrature_1d(16)
        p = Problem(
            name=CONFIG_NAMES[0], nx=nx, ny=1, nz=1, dim=1, dx=L / nx, dy=1.0, dz=1.0,
            C=np.array([1.6e6]), v=np.array([6400.0]), tau=np.array([15.6e-12]),
            s=s, w=w,
            face_bc=[(BC_ISOTHERMAL, +0.5), (BC_ISOTHERMAL, -0.5)] + [(BC_SPECULAR, 0.0)] * 4,
            precision=FP64, n_iter=200,
            notes="1-D gray film, Kn=1 (MFP 99.84 nm over L=100 nm)")
    elif k == 1:
        nx, ny, _ = (200, 200, 1) if grid is None else grid
        Lx = Ly = 400e-9
        C, v, tau = band_table()
        s, w = quadrature_3d()
        dx, dy = Lx / nx, Ly / ny
        Q = _gaussian(nx, ny, 1, dx, dy, 1.0, (200e-9, 360e-9, None), 20e-9, 1e18)
        p = Problem(
            name=CONFIG_NAMES[1], nx=nx, ny=ny, nz=1, dim=2, dx=dx, dy=dy, dz=1.0,
            C=C, v=v, tau=tau, s=s, w=w,
            face_bc=[(BC_SPECULAR, 0.0), (BC_SPECULAR, 0.0), (BC_ISOTHERMAL, 0.0),
                     (BC_SPECULAR, 0.0), (BC_SPECULAR, 0.0), (BC_SPECULAR, 0.0)],
            Q=Q, precision=FP64, n_iter=50,
            notes="2-D film, hotspot 40 nm below the top (y+) face; y- isothermal")
    elif k == 2:
        nx, ny, nz = (64, 64, 64) if grid is None else grid
        L = 500e-9
        C, v, tau = band_table()
        s, w = quadrature_3d()
        Q = np.full((nz, ny, nx), 1e17)
        p = Problem(
            name=CONFIG_NAMES[2], nx=nx, ny=ny, nz=nz, dim=3, dx=L / nx, dy=L / ny, dz=L / nz,
            C=C, v=v, tau=tau, s=s, w=w,
            face_bc=[(BC_DIFFUSE, 0.0)] * 4 + [(BC_ISOTHERMAL, 0.0), (BC_DIFFUSE, 0.0)],
            Q=Q, precision=FP64, n_iter=50,
            notes="3-D cube, uniform source; z- isothermal, other five diffuse")
    elif k == 3:
        nx, ny, nz = (128, 64, 64) if grid is None else grid
        Lx, Ly, Lz = 256e-9, 128e-9, 128e-9
        dx, dy, dz = Lx / nx, Ly / ny, Lz / nz
        C, v, tau = band_table()
        s, w = quadrature_3d()
        # substrate z < 40/64 Lz; fin 27/64 <= y < 37/64 of Ly above it, full x length
        kz = int(round(nz * 40 / 64))
        j0 = int(round(ny * 27 / 64))
        j1 = max(j0 + 1, int(round(ny * 37 / 64)))
        mask = np.zeros((nz, ny, nx), dtype=np.uint8)
        mask[:kz, :, :] = 1
        mask[kz:, j0:j1, :] = 1
        Q = _gaussian(nx, ny, nz, dx, dy, dz, (128e-9, 64e-9, 116e-9), 6e-9, 5e18) * mask
        p = Problem(
            name=CONFIG_NAMES[3], nx=nx, ny=ny, nz=nz, dim=3, dx=dx, dy=dy, dz=dz,
            C=C, v=v, tau=tau, s=s, w=w,
            face_bc=[(BC_PERIODIC, 0.0), (BC_PERIODIC, 0.0), (BC_DIFFUSE, 0.0),
                     (BC_DIFFUSE, 0.0), (BC_ISOTHERMAL, 0.0), (BC_DIFFUSE, 0.0)],
            interface_bc=(BC_DIFFUSE, 0.0), mask=mask, Q=Q,
            precision=FP32_STORE_FP64_ACC, n_iter=50,
            notes="FinFET-like voxels: substrate + one fin; x periodic; interfaces diffuse")
    elif k == 4:
        nx, ny, nz = (256, 128, 128) if grid is None else grid
        Lx, Ly, Lz = 512e-9, 256e-9, 256e-9
        dx, dy, dz = Lx / nx, Ly / ny, Lz / nz
        C, v, tau = band_table()
        s, w = quadrature_3d()
        rng = np.random.default_rng([MASTER_SEED, 4])
        Q = np.zeros((nz, ny, nx))
        for _ in range(3):
            c = rng.uniform(0.2, 0.8, 3) * np.array([Lx, Ly, Lz])
            peak = 10.0 ** rng.uniform(17.0, 18.0)
            Q += _gaussian(nx, ny, nz, dx, dy, dz, tuple(c), 10e-9, peak)
        p = Problem(
            name=CONFIG_NAMES[4], nx=nx, ny=ny, nz=nz, dim=3, dx=dx, dy=dy, dz=dz,
            C=C, v=v, tau=tau, s=s, w=w,
            face_bc=[(BC_SPECULAR, 0.0)] * 4 + [(BC_ISOTHERMAL, 0.0), (BC_DIFFUSE, 0.0)],
            Q=Q, precision=FP32_STORE_FP64_ACC, n_iter=5,
            notes="large slab, 3 hotspots; z- isothermal, sides specular, top diffuse")
    else:
        raise ValueError(f"no config {k}")
    if precision is not None:
        p.precision = precision
    return p


# ----------------------------------------------------------------------------
# randomised small problems for parity / property tests
# ----------------------------------------------------------------------------
def random_problem(seed: int, dim: int = 3, shape: Tuple[int, int, int] = (7, 6, 5),
                   n_bands: int = 3, masked: bool = True, periodic_axis: Optional[int] = None,
                   bc_types: Tuple[int, ...] = (BC_ISOTHERMAL, BC_DIFFUSE, BC_SPECULAR),
                   interface_type: int = BC_DIFFUSE, n_polar: int = 4, n_azimuth: int = 8,
                   precision: int = FP64) -> Problem:
    """A small random problem: random mask, random BC types per face, random source.
    At least one face is isothermal so a steady state exists."""
    rng = np.random.default_rng([MASTER_SEED, 1000 + seed])
    nx, ny, nz = shape
    if dim < 3:
        nz = 1
    if dim < 2:
        ny = 1
    C, v, tau = band_table(n_bands, seed=MASTER_SEED + 17 * seed + 1)
    if dim == 1:
        s, w = quadrature_1d(2 * n_polar)
    else:
        s, w = quadrature_3d(n_polar, n_azimuth)
    L = 10.0 ** rng.uniform(-8.0, -6.5)
    dx, dy, dz = L / nx, L / max(ny, 1) * rng.uniform(0.7, 1.4), L / max(nz, 1) * rng.uniform(0.7, 1.4)
    face_bc = []
    for f in range(6):
        t = int(rng.choice(bc_types))
        face_bc.append((t, float(rng.uniform(-1, 1)) if t == BC_ISOTHERMAL else 0.0))
    iso_face = int(rng.integers(0, 2 * dim))
    face_bc[iso_face] = (BC_ISOTHERMAL, float(rng.uniform(-1, 1)))
    if periodic_axis is not None and periodic_axis < dim:
        if iso_face // 2 == periodic_axis:
            other = (periodic_axis + 1) % dim if dim > 1 else None
            if other is not None:
                face_bc[2 * other] = (BC_ISOTHERMAL, float(rng.uniform(-1, 1)))
        face_bc[2 * periodic_axis] = (BC_PERIODIC, 0.0)
        face_bc[2 * periodic_axis + 1] = (BC_PERIODIC, 0.0)
    for f in range(2 * dim, 6):
        face_bc[f] = (BC_SPECULAR, 0.0)
    mask = None
    if masked:
        mask = (rng.uniform(size=(nz, ny, nx)) > 0.2).astype(np.uint8)
        mask[nz // 2, ny // 2, nx // 2] = 1
    Q = rng.uniform(0.0, 1e17, size=(nz, ny, nx))
    if mask is not None:
        Q = Q * mask
    it = (interface_type, float(rng.uniform(-1, 1)) if interface_type == BC_ISOTHERMAL else 0.0)
    return Problem(name=f"random_{seed}_d{dim}", nx=nx, ny=ny, nz=nz, dim=dim, dx=dx, dy=dy, dz=dz,
                   C=C, v=v, tau=tau, s=s, w=w, face_bc=face_bc, interface_bc=it,
                   mask=mask, Q=Q, precision=precision, n_iter=10)
