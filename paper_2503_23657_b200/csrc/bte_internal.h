// Internal definitions shared by the host setup (bte_api.cu) and the kernels (bte_kernels.cu).
// Product code: shares nothing with oracle/.
#pragma once
#include <cstddef>
#include <cstdint>

#define BTE_P 16        // direction slots per work item (one band x <=16 directions of one octant)
#define BTE_TY 32       // tile rows along y' = lanes of a warp
#define BTE_MAX_TZ 16   // tile rows along z' = warps of a CTA
#define BTE_NCOEF 8     // per slot: inv, ax, ay, az, w, w|sx|, w|sy|, w|sz|
#define BTE_CONST_BYTES 61440

// cell code bits (octant independent): bit0 solid; bit 1+f set if the neighbour across face f
// (x-,x+,y-,y+,z-,z+) is a solid/void interface (or a periodic wrap onto a void cell).
#define BTE_CODE_SOLID 1

struct BteUnit {          // one work unit of the sweep: (octant, item, tile)
  int32_t oct, item, ty, tz;
  int32_t dep_y, dep_z, dep_prev;   // unit ids that must be complete first, -1 = none
  int32_t coef_off;                 // offset (in values) of this item's 16x8 coefficient block
  int32_t band, chunk;
};

struct BteOct {           // per direction octant
  int32_t sx, sy, sz;     // +1 / -1 sweep orientation per axis
  int32_t cls;            // (sx<0) | (sy<0)<<1 : which skewed copy of the cell arrays it reads
  int32_t nitems, nchunk; // items = n_bands * nchunk
  int32_t active;
  int32_t pad;
  double *M;              // [4][NS] moment partials of this octant (skewed class layout)
  void *xpl, *ypl, *zpl;  // face planes (see bte_kernels.cu for the layouts)
};

struct BteDev {           // passed by value to every kernel
  int32_t nx, ny, nz, dim;
  int32_t nty, ntz, TZ, NU, nyp;    // tiles along y', z'; warps per CTA; nx+31; nty*32
  int32_t B, n_units, has_y, has_z;
  int32_t nHslot, n_iface, fp32, n_dirs;
  int64_t NS, ncell, nsolid;
  double inv_sumCtau;
  void *dT_sk[4];         // T  [NS]   lattice temperature deviation, skewed copies per class
  void *Q_sk[4];          // T  [NS]   Q / sum C
  uint8_t *code_sk[4];    // u8 [NS]
  uint8_t *code;          // u8 [ncell] physical layout
  double *dT, *q, *qmag;  // fp64 physical layout outputs [ncell], [3][ncell], [ncell]
  double *Qphys;          // fp64 [ncell] source (kept for bte_solve_host re-skew)
  int32_t *iface;         // [6][ncell] interface-face id or -1 (NULL if no interface faces)
  void *Gi;               // T  [n_iface][B] interface inflow of this iteration
  double *Hpart;          // [n_iface][B][nHslot] outgoing hemispherical partial sums
  int32_t *iface_info;    // [n_iface] : face code f (0..5)
  const int32_t *item_coef; // [8][max_items] coefficient-block offset of (octant, item)
  void *Gf;               // T diffuse box-face inflow [sum_f B*na*nb]
  int32_t max_items, pad2;
  BteOct oct[8];
  BteUnit *units;
  int32_t *done;          // [n_units] epoch stamps
  int32_t *ticket;        // [1]
  double *band;           // [4][B]: C/4pi, C tau/(4pi sumC), 1/tau, v
  double *red;            // residual partials [4][n_red_blocks] + final [4]
  int32_t n_red_blocks, epoch;
  int32_t face_type[6];
  double face_dT[6];
  double Pi_face[6];
  int32_t iface_type, pad1;
  double iface_dT;
};
