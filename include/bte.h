/* include/bte.h -- C-ABI boundary of the B200-native phonon-BTE sweep library.
 *
 * What it computes (arxiv 2503.23657 "JAX-BTE", /root/reference/PAPER.md):
 * the forward solver's hot path -- nongray RTA phonon BTE in energy-deviation form
 * (Eq. 15) advanced by source iteration (steps 1-4):
 * every iteration runs an upwind finite-volume discrete-ordinates sweep for every
 * (band, direction) (exact solve of Eq. 20 with the first-order A of Eq. 21,
 * PAPER.md:270-279, on a Cartesian / voxel-masked grid), accumulates the 0th/1st
 * angular moments inside the sweep, then updates the lattice temperature (Eq. 16,
 * PAPER.md:244-247), the heat flux (Eq. 4) and the residuals (Eq. 23,
 * PAPER.md:299-304).  Boundary inflow follows Eq. 5-7 plus a
 * periodic wrap, always taken from the previous iteration (lagged store).
 *
 * Conventions
 *  - all functions are extern "C", return a bte_status, never throw, never abort;
 *  - arrays are x fastest: idx = i + nx*(j + ny*k);
 *  - "host" / "device" in a comment says where a pointer must live;
 *  - OWNERSHIP: the caller owns the device workspace and every output buffer and keeps
 *    them alive until bte_destroy; host input arrays are copied during bte_create and may
 *    be freed afterwards; the library calls no cudaMalloc after bte_create returns and none
 *    on the hot path (it allocates nothing on the device at all: everything lives in the
 *    caller's workspace);
 *  - cuda_stream is a cudaStream_t passed as void* (NULL = legacy default stream);
 *  - a handle is not thread-safe; different handles are independent, but handles that
 *    iterate concurrently on different streams of one device are NOT supported (they share
 *    one __constant__ coefficient bank, re-uploaded in stream order by bte_iterate);
 *  - there is no CPU fallback: without a CUDA device every compute entry point returns
 *    BTE_ERR_CUDA.
 */
#ifndef BTE_H
#define BTE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct bte_solver bte_solver; /* opaque */

typedef enum {
  BTE_OK = 0,
  BTE_ERR_INVALID_ARG = 1, /* sizes <= 0, C/v/tau <= 0, non-unit s, unpaired PERIODIC, dim/nz mismatch,
                              no solid cell, interface_bc PERIODIC, NULL where a pointer is required */
  BTE_ERR_QUADRATURE = 2,  /* |sum w - 4pi| > 1e-6*4pi; with a SPECULAR face: |sum w s| > 1e-9*4pi, or an axis
                              reflection that does not map the direction set onto itself (equal weights) */
  BTE_ERR_WORKSPACE = 3,   /* workspace NULL, misaligned (256 B) or smaller than bte_workspace_bytes */
  BTE_ERR_CUDA = 4,        /* any CUDA runtime error (bte_last_cuda_error gives the code) */
  BTE_ERR_UNSUPPORTED = 5, /* valid problem outside this build: SPECULAR interface_bc; coefficient table
                              larger than the constant bank (non-mirror-symmetric quadrature x many bands) */
  BTE_ERR_TOO_LARGE = 6    /* bte_residual_static only: n_cells > BTE_STATIC_MAX_CELLS */
} bte_status;

/* Eq. 5 / Eq. 6 / Eq. 7; PERIODIC: BASELINE.json configs[3] */
typedef enum { BTE_BC_ISOTHERMAL = 0, BTE_BC_DIFFUSE = 1, BTE_BC_SPECULAR = 2, BTE_BC_PERIODIC = 3 } bte_bc_type;

/* BTE_FP64: everything fp64.  BTE_FP32_STORE_FP64_ACC (reading G15, as built): cell inputs, tables,
 * recurrence, wavefront buffers and the lagged boundary store are fp32.  Moments: on the fast path
 * (bte_kernel_path == 2) the sum over the 16 directions and all bands of ONE OCTANT is fp32 (register partial sums
 * per band group, added group by group into an fp32 per-octant accumulator, the hemispherical partial sums of
 * diffuse interfaces likewise); on the generic path only the sum over <= 16 directions of one (octant, band) item is
 * fp32.  The sums over octants and cells (residual norms), the diffuse-face sums over octants and the dT division
 * are fp64 on both paths.  Tested against the fp64 oracle at 1e-4 (measured 1e-7 ... 1e-6). */
typedef enum { BTE_FP64 = 0, BTE_FP32_STORE_FP64_ACC = 1 } bte_precision;

typedef struct { int32_t type; double dT_wall; } bte_bc; /* dT_wall [K] used by ISOTHERMAL only */

typedef struct {
  int32_t nx, ny, nz, dim;   /* dim=1: x only (ny=nz=1); 2: x,y (nz=1); 3: x,y,z */
  double dx, dy, dz;         /* metres; only the first `dim` are used */
  const uint8_t *solid_mask; /* host, nx*ny*nz, 1 = solid; NULL = all solid */
  int32_t n_bands;
  const double *C, *v, *tau; /* host, [n_bands]; J/m^3K, m/s, s; all > 0 */
  int32_t n_dirs;
  const double *s;           /* host, [n_dirs][3] unit vectors */
  const double *w;           /* host, [n_dirs], sum = 4 pi */
  bte_bc face_bc[6];         /* x-, x+, y-, y+, z-, z+ ; PERIODIC must be set on both faces of an axis */
  bte_bc interface_bc;       /* every solid/void face inside the box (ISOTHERMAL or DIFFUSE) */
  const double *Q;           /* host, nx*ny*nz, W/m^3; NULL = 0 */
  int32_t precision;         /* bte_precision */
} bte_problem;

/* Bytes of device workspace bte_create needs for this problem; 0 if the problem is invalid. */
size_t bte_workspace_bytes(const bte_problem *p);

/* Validate, build the sweep schedule, upload tables into d_workspace (device, 256-B aligned,
 * >= bte_workspace_bytes), initialise dT = 0 and the lagged store = 0.  Synchronises the stream
 * before returning.  *out is untouched on failure. */
bte_status bte_create(const bte_problem *p, void *d_workspace, size_t bytes, void *cuda_stream, bte_solver **out);

/* n source iterations (sweep of all (band,direction) + moments + dT/q/residual update), asynchronous
 * on cuda_stream; n >= 0. */
bte_status bte_iterate(bte_solver *h, int32_t n, void *cuda_stream);

/* dT [K] (deviation from the reference temperature) per cell, fp64 in both precisions, void cells 0.
 * d_out: device, [nx*ny*nz]. Asynchronous on cuda_stream. */
bte_status bte_get_temperature(bte_solver *h, double *d_out, void *cuda_stream);
/* q [W/m^2], cell-centred (Eq. 4). d_out: device, [3][nx*ny*nz]. Asynchronous. */
bte_status bte_get_heat_flux(bte_solver *h, double *d_out, void *cuda_stream);
/* Overwrite dT (restart / tests). d_in: device, [nx*ny*nz]. Asynchronous. */
bte_status bte_set_temperature(bte_solver *h, const double *d_in, void *cuda_stream);

/* eps_T, eps_q of the last iteration (Eq. 23; normalised by max|dT|, max|q| over
 * solid cells; 0/0 -> 0, x/0 -> +inf; +inf before the first iteration). Host outputs (may be NULL).
 * SYNCHRONISES the stream last used by bte_iterate. */
bte_status bte_residual(bte_solver *h, double *eps_T, double *eps_q);

/* Whole-path convenience with HOST buffers (used for end-to-end timing): uploads Q (host, [nx*ny*nz],
 * may be NULL = keep); if reset != 0 sets dT and the lagged store back to 0 and the iteration count to 0;
 * runs n iterations; downloads dT (host [nx*ny*nz]) and q (host [3][nx*ny*nz]; may be NULL).
 * Synchronous (returns after the downloads completed). */
bte_status bte_solve_host(bte_solver *h, const double *Q_host, int32_t n, int32_t reset, double *dT_host,
                          double *q_host, void *cuda_stream);

/* Measurement aid: record a CUDA-event pair around the sweep kernel of the next max_launches iterations
 * (on the stream bte_iterate is given); 0 switches it off. bte_get_sweep_timing synchronises on the last
 * recorded event, returns the summed device time [ms] and the number of launches covered, and re-arms. */
bte_status bte_set_sweep_timing(bte_solver *h, int32_t max_launches);
bte_status bte_get_sweep_timing(bte_solver *h, double *total_ms, int64_t *launches);

int64_t bte_updates_per_sweep(const bte_solver *h); /* solid cells * n_bands * n_dirs */
int64_t bte_iterations_done(const bte_solver *h);
int32_t bte_kernel_launches_per_iteration(const bte_solver *h);
/* Which sweep kernel serves this problem: 2 = fast path (3-D with even ny and nz, or 2-D with even ny -- run as a
 * slab of two identical layers without z coupling; all-solid or voxel-masked; 16 directions in each octant with
 * mirror-symmetric |s|, w tables; <= 16 bands), 1 = generic path (everything else: 1-D, odd ny / nz, other
 * quadratures).  Both compute the same iteration; bte_set_option(BTE_OPT_FORCE_GENERIC, 1) forces 1 for testing. */
int32_t bte_kernel_path(const bte_solver *h);
/* schedule facts for reporting: out[0]=work units per sweep, [1]=CTAs launched, [2]=threads per CTA,
 * [3]=wavefront steps summed over units, [4]=thread-slot updates issued per sweep (occupancy
 * denominator: useful updates / this), [5]=bytes of workspace in use */
void bte_schedule_info(const bte_solver *h, int64_t out[6]);
/* Host-only view of the plan bte_create would build (no CUDA call): out[0] = kernel path (1 / 2), [1] = work
 * units per sweep, [2] = 1 if the ticket order is topological (every unit comes after the units it follows, and
 * each dependency points at the right neighbour tile / band group) when simulated for `resident_ctas` CTAs,
 * [3] = wavefront steps per unit, [4] = warps per CTA, [5] = band groups, [6] = 1 if voxel-masked, [7] = workspace
 * bytes.  Returns the status bte_create would return for an invalid problem. */
bte_status bte_plan_info(const bte_problem *p, int32_t resident_ctas, int64_t out[8]);
void bte_destroy(bte_solver *h);
const char *bte_status_string(bte_status s);
/* Last CUDA runtime error code seen by any entry point of this process (any thread); 0 = none. */
int32_t bte_last_cuda_error(void);

/* Test / tuning hook: process-wide options consulted by bte_workspace_bytes / bte_create / bte_plan_info (handles
 * already created are not affected).  The library never reads the environment.  value 0 = default.
 *   BTE_OPT_FORCE_GENERIC   1: use the generic kernels for every problem
 *   BTE_OPT_WARPS           2 | 4 | 8: warps per CTA of the fast path (default: by nz)
 *   BTE_OPT_PUBLISH_PERIOD  4 | 8 | 16 | 32: steps between progress publications of a unit (default: 4 if nx < 224, 8 if nx < 256, else 16)
 *   BTE_OPT_START_SLACK     1..256: extra steps a unit lets the units it follows get ahead before it starts
 *   BTE_OPT_SCHEDULE        1: ticket order = band groups of one (tile, octant) consecutively instead of the simulated
 *                           list schedule (experiment on L2 reuse; same results, different timing)
 * Returns BTE_ERR_INVALID_ARG for an unknown option. */
typedef enum { BTE_OPT_FORCE_GENERIC = 0, BTE_OPT_WARPS = 1, BTE_OPT_PUBLISH_PERIOD = 2, BTE_OPT_START_SLACK = 3,
               BTE_OPT_SCHEDULE = 4, BTE_OPT_COUNT_ = 5 } bte_option;
bte_status bte_set_option(int32_t option, int32_t value);

/* Allocation-free stopping test, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving
 * loops, harnesses that forbid it) and so cannot hold a bte_solver workspace: eps_T, eps_q of Eq. 23 (
 * N = solid cells, maxima over solid cells of the NEW snapshot, |q| magnitudes; 0/0 -> 0, x/0 -> +inf) between two
 * snapshots the caller holds -- the numbers bte_residual reports when the snapshots are bte_get_temperature /
 * bte_get_heat_flux taken before and after one bte_iterate(h, 1, .).
 *   d_dT_new, d_dT_old: device, [n_cells];  d_q_new, d_q_old: device, [3][n_cells];
 *   d_solid_mask: device, [n_cells], 1 = solid, or NULL = all solid;  d_eps: device, [2] = {eps_T, eps_q}.
 * One memset node + one kernel, asynchronous on cuda_stream; calls no cudaMalloc / cudaFree and no allocating library
 * routine.  The per-block partial sums live in a file-scope __device__ array of the library (164 096 B, held by every
 * GPU that loads the library until the process exits; its address is resolved once per device by the first call made
 * with that device current).  LIMIT: n_cells <= BTE_STATIC_MAX_CELLS, else BTE_ERR_TOO_LARGE and nothing is launched.
 * All calls on one device share that array: calls that may overlap on the GPU (different streams or threads) race --
 * serialise them.  The result does not depend on what an earlier call left in the array. */
#define BTE_STATIC_MAX_CELLS (1 << 24) /* 16 777 216 cells (configs[4] has 256*128*128 = 4 194 304) */
bte_status bte_residual_static(const double *d_dT_new, const double *d_dT_old, const double *d_q_new,
                               const double *d_q_old, const uint8_t *d_solid_mask, int64_t n_cells, double *d_eps,
                               void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif
