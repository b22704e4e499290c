/* oracle/bte_ref.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU reference of the hot path of arxiv 2503.23657 (JAX-BTE):
 * nongray RTA phonon BTE in energy-deviation form, source iteration with an
 * upwind finite-volume discrete-ordinates sweep per (band, direction) and the
 * lattice-temperature update from energy conservation.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load this library.  It shares no code, header or table
 * with the CUDA path (include/bte.h, paper_2503_23657_b200/csrc): this header
 * declares its OWN problem struct on purpose.
 *
 * All pointers are HOST pointers.  Layout everywhere: x fastest,
 * idx = i + nx*(j + ny*k).
 */
#ifndef BTE_REF_H
#define BTE_REF_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct bte_ref_solver bte_ref_solver;

/* boundary-condition codes: Eq. 5 (isothermal), Eq. 6 (diffuse), Eq. 7 (specular),
 * PAPER.md:190-207; periodic is BASELINE.json configs[3]. */
enum { BTE_REF_ISOTHERMAL = 0, BTE_REF_DIFFUSE = 1, BTE_REF_SPECULAR = 2, BTE_REF_PERIODIC = 3 };

typedef struct { int32_t type; double dT_wall; } bte_ref_bc;

typedef struct {
  int32_t nx, ny, nz, dim;      /* dim = number of active axes (1: x; 2: x,y; 3: x,y,z) */
  double dx, dy, dz;            /* metres */
  const uint8_t *solid_mask;    /* nx*ny*nz, 1 = solid; NULL = all solid */
  int32_t n_bands;
  const double *C, *v, *tau;    /* [n_bands] J/m^3K, m/s, s */
  int32_t n_dirs;
  const double *s;              /* [n_dirs][3] unit vectors */
  const double *w;              /* [n_dirs], sum = 4 pi */
  bte_ref_bc face_bc[6];        /* x-, x+, y-, y+, z-, z+ */
  bte_ref_bc interface_bc;      /* every solid/void face */
  const double *Q;              /* nx*ny*nz W/m^3, NULL = 0 */
  int32_t diagnostics;          /* 1: keep the full intensity field + face fluxes (small grids) */
  int32_t literal_one_over_pi;  /* 1: divide diffuse inflow by pi (Eq. 6 literally) instead of the
                                   discrete Pi_f (reading G10); for the leak demonstration only */
} bte_ref_problem;

/* returns 0 on success, nonzero on invalid input (codes mirror SURVEY.md 8(b)) */
int  bte_ref_create(const bte_ref_problem *p, bte_ref_solver **out);
void bte_ref_destroy(bte_ref_solver *h);
/* worker threads over BANDS (results are bit-identical for any count: per-band
 * partial moments are combined in band order afterwards). default 1. */
void bte_ref_set_threads(bte_ref_solver *h, int32_t n);
/* visit (band,direction) pairs of a band in a permuted order (reading G9 test);
 * perm = permutation of [0,n_dirs), NULL resets */
int  bte_ref_set_dir_order(bte_ref_solver *h, const int32_t *perm);
int  bte_ref_iterate(bte_ref_solver *h, int32_t n);
int  bte_ref_get_temperature(const bte_ref_solver *h, double *out /*[nx*ny*nz]*/);
int  bte_ref_get_heat_flux(const bte_ref_solver *h, double *out /*[3][nx*ny*nz]*/);
int  bte_ref_residual(const bte_ref_solver *h, double *eps_T, double *eps_q);
int64_t bte_ref_updates_per_sweep(const bte_ref_solver *h);
int64_t bte_ref_iterations_done(const bte_ref_solver *h);
int  bte_ref_set_temperature(bte_ref_solver *h, const double *dT /*[nx*ny*nz]*/);

/* diagnostics (need diagnostics=1) */
int  bte_ref_get_intensity(const bte_ref_solver *h, double *out /*[n_bands][n_dirs][nx*ny*nz]*/);
/* outward energy flux density (W/m^2) through face f (x-,x+,y-,y+,z-,z+) of every cell, from the
 * LAST sweep: sum_b v_b sum_d w_d (s_d.n) e_face, e_face = cell value if s_d.n>0 (G13) else the
 * upwind value actually used (neighbour or boundary inflow). out[6][nx*ny*nz]; 0 on void cells. */
int  bte_ref_face_flux(const bte_ref_solver *h, double *out);
/* same, per band: out[n_bands][6][nx*ny*nz] */
int  bte_ref_face_flux_band(const bte_ref_solver *h, double *out);
/* total power (W) leaving through boundary faces of each type: out[4] indexed by BC code
 * (periodic faces net to ~0 at convergence). Uses the last sweep's face fluxes. */
int  bte_ref_boundary_power(const bte_ref_solver *h, double *out);
/* discrete hemispherical normaliser Pi_f for face f (0..5): sum_{s.n<0} w |s.n|  (G10) */
double bte_ref_pi_face(const bte_ref_solver *h, int32_t face);

#ifdef __cplusplus
}
#endif
#endif
