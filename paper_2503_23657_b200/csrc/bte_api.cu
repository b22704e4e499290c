// Host side of the B200 phonon-BTE sweep library: validation, sweep schedule, workspace
// carve-up and the extern "C" entry points declared in include/bte.h.
// Product code: shares nothing with oracle/.  No CPU fallback: every compute entry point
// needs a CUDA device.
#include "../../include/bte.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <map>
#include <new>
#include <queue>
#include <string>
#include <vector>

#include "bte_kernels.cuh"

#include <atomic>
static std::atomic<int> g_last_cuda{0};   // process-wide: bte_last_cuda_error() may be called from any thread
// Process-wide test / tuning options (bte_set_option): the product never reads the environment.
static std::atomic<int> g_opt[BTE_OPT_COUNT_];
#define CK(call)                                                       \
  do {                                                                 \
    cudaError_t e_ = (call);                                           \
    if (e_ != cudaSuccess) { g_last_cuda.store((int)e_); return BTE_ERR_CUDA; } \
  } while (0)

namespace {

const double kFourPi = 12.566370614359172953850573533118;

struct Plan {
  BteDev dev{};                          // geometry part filled by build_plan, pointers by carve()
  std::vector<uint8_t> code;             // [ncell]
  std::vector<int32_t> iface, iface_info, iface_cell;
  std::vector<double> Q;                 // [ncell]
  std::vector<double> band;              // [4][B]
  std::vector<double> coef;              // unique coefficient blocks, 16x8 doubles each
  std::vector<int32_t> item_coef;        // [8][max_items]
  std::vector<BteUnit> units;
  double sumC = 0;
  int nthreads = 32;
  size_t smem = 0;
  int64_t steps_total = 0;
  // workspace offsets
  size_t total = 0, state_begin = 0, state_end = 0;
  bool any_diffuse_face = false;
  size_t gf_elems = 0;
  // fast path (bte_sweep2.cuh)
  bool v2 = false, masked2 = false;
  int layers = 1;                        // 2: a 2-D problem run as a two-layer 3-D slab on the fast path
  int64_t user_ncell = 0, user_nsolid = 0;
  std::vector<uint32_t> codeP[4];
  Bte2Dev d2{};
  std::vector<Bte2Unit> units2;
  Bte2Coefs<float> cf32{};
  Bte2Coefs<double> cf64{};
  size_t smem2 = 0;
  size_t x2_chunks = 0, y2_chunks = 0, z2_chunks = 0, y2_slot = 0, z2_slot = 0;
  size_t xpl_elems[8]{}, ypl_elems[8]{}, zpl_elems[8]{};
};

size_t align_up(size_t x) { return (x + 255) & ~size_t(255); }

bte_status build_plan_impl(const bte_problem *p, Plan &pl) {
  if (!p) return BTE_ERR_INVALID_ARG;
  if (p->nx < 1 || p->ny < 1 || p->nz < 1 || p->dim < 1 || p->dim > 3) return BTE_ERR_INVALID_ARG;
  if ((p->dim < 3 && p->nz != 1) || (p->dim < 2 && p->ny != 1)) return BTE_ERR_INVALID_ARG;
  if (p->n_bands < 1 || p->n_dirs < 1 || !p->C || !p->v || !p->tau || !p->s || !p->w) return BTE_ERR_INVALID_ARG;
  if (p->precision != BTE_FP64 && p->precision != BTE_FP32_STORE_FP64_ACC) return BTE_ERR_INVALID_ARG;
  const double delta[3] = {p->dx, p->dy, p->dz};
  for (int a = 0; a < p->dim; ++a)
    if (!(delta[a] > 0.0) || !std::isfinite(delta[a])) return BTE_ERR_INVALID_ARG;
  const int B = p->n_bands, D = p->n_dirs;
  for (int b = 0; b < B; ++b)
    if (!(p->C[b] > 0) || !(p->v[b] > 0) || !(p->tau[b] > 0)) return BTE_ERR_INVALID_ARG;
  double sw = 0;
  for (int d = 0; d < D; ++d) {
    const double *s = p->s + 3 * d;
    if (std::fabs(s[0] * s[0] + s[1] * s[1] + s[2] * s[2] - 1.0) > 1e-9) return BTE_ERR_INVALID_ARG;
    if (!(p->w[d] >= 0)) return BTE_ERR_INVALID_ARG;
    sw += p->w[d];
  }
  if (std::fabs(sw - kFourPi) > 1e-6 * kFourPi) return BTE_ERR_QUADRATURE;
  for (int a = 0; a < p->dim; ++a) {
    const int t0 = p->face_bc[2 * a].type, t1 = p->face_bc[2 * a + 1].type;
    if (t0 < 0 || t0 > 3 || t1 < 0 || t1 > 3) return BTE_ERR_INVALID_ARG;
    if ((t0 == BTE_BC_PERIODIC) != (t1 == BTE_BC_PERIODIC)) return BTE_ERR_INVALID_ARG;
  }
  if (p->interface_bc.type == BTE_BC_PERIODIC || p->interface_bc.type < 0 || p->interface_bc.type > 3)
    return BTE_ERR_INVALID_ARG;

  BteDev &dv = pl.dev;
  dv.nx = p->nx; dv.ny = p->ny; dv.nz = p->nz; dv.dim = p->dim;
  dv.B = B; dv.n_dirs = D;
  dv.fp32 = p->precision == BTE_FP32_STORE_FP64_ACC;
  dv.has_y = p->dim >= 2; dv.has_z = p->dim >= 3;
  dv.TZ = dv.has_z ? (p->nz > 8 ? 16 : 8) : 1;
  dv.nty = (p->ny + 31) / 32; dv.ntz = (p->nz + dv.TZ - 1) / dv.TZ;
  dv.NU = p->nx + 31; dv.nyp = dv.nty * 32;
  dv.ncell = (int64_t)p->nx * p->ny * p->nz;
  dv.NS = (int64_t)p->nz * dv.nty * dv.NU * 32;
  pl.nthreads = 32 * dv.TZ;
  const size_t tsz = dv.fp32 ? 4 : 8;
  pl.smem = (size_t)(2 * (dv.TZ + 1) * BTE_P * 32 + 2 * dv.TZ * BTE_P) * tsz;

  // ---- cells: solid mask, interface bits, interface faces
  const int64_t N = dv.ncell;
  const int n[3] = {p->nx, p->ny, p->nz};
  pl.code.assign((size_t)N, 0);
  int64_t nsolid = 0;
  for (int64_t c = 0; c < N; ++c) {
    const bool s = p->solid_mask ? p->solid_mask[c] != 0 : true;
    pl.code[c] = s ? BTE_CODE_SOLID : 0;
    nsolid += s;
  }
  if (nsolid == 0) return BTE_ERR_INVALID_ARG;
  dv.nsolid = nsolid;
  std::vector<int32_t> iface;
  if (p->solid_mask) iface.assign((size_t)6 * N, -1);
  int32_t nif = 0;
  if (p->solid_mask) {
    for (int k = 0; k < n[2]; ++k) for (int j = 0; j < n[1]; ++j) for (int i = 0; i < n[0]; ++i) {
      const int64_t c = i + (int64_t)n[0] * (j + (int64_t)n[1] * k);
      if (!(pl.code[c] & BTE_CODE_SOLID)) continue;
      const int ijk[3] = {i, j, k};
      for (int f = 0; f < 2 * p->dim; ++f) {
        const int a = f >> 1;
        int u[3] = {i, j, k};
        u[a] = ijk[a] + ((f & 1) ? 1 : -1);
        if (u[a] < 0 || u[a] >= n[a]) {
          if (p->face_bc[f].type != BTE_BC_PERIODIC) continue;   // box face: handled by ghost planes
          u[a] = (u[a] + n[a]) % n[a];
        }
        const int64_t uc = u[0] + (int64_t)n[0] * (u[1] + (int64_t)n[1] * u[2]);
        if (pl.code[uc] & BTE_CODE_SOLID) continue;
        pl.code[c] |= (uint8_t)(2 << f);
        iface[(size_t)f * N + c] = nif++;
        pl.iface_info.push_back(f);
        pl.iface_cell.push_back((int32_t)c);
      }
    }
  }
  dv.n_iface = nif;
  if (nif > 0) {
    if (p->interface_bc.type == BTE_BC_SPECULAR) return BTE_ERR_UNSUPPORTED;
    pl.iface.swap(iface);
  }
  dv.iface_type = p->interface_bc.type; dv.iface_dT = p->interface_bc.dT_wall;
  for (int f = 0; f < 6; ++f) {
    dv.face_type[f] = p->face_bc[f].type; dv.face_dT[f] = p->face_bc[f].dT_wall;
    const int a = f >> 1;
    const double ns = (f & 1) ? 1.0 : -1.0;
    double Pi = 0;
    for (int d = 0; d < D; ++d) { const double sn = ns * p->s[3 * d + a]; if (sn < 0) Pi -= p->w[d] * sn; }
    dv.Pi_face[f] = Pi;
    if (f < 2 * p->dim && p->face_bc[f].type == BTE_BC_DIFFUSE) pl.any_diffuse_face = true;
  }
  pl.Q.assign((size_t)N, 0.0);
  if (p->Q) for (int64_t c = 0; c < N; ++c) pl.Q[c] = p->Q[c];

  // ---- bands
  double sumC = 0, sumCt = 0;
  for (int b = 0; b < B; ++b) { sumC += p->C[b]; sumCt += p->C[b] / p->tau[b]; }
  pl.sumC = sumC;
  dv.inv_sumCtau = 1.0 / sumCt;
  pl.band.assign((size_t)4 * B, 0.0);
  for (int b = 0; b < B; ++b) {
    pl.band[b] = p->C[b] / kFourPi;                              // e0 = C dT / 4pi (Eq. 16)
    pl.band[B + b] = p->C[b] * p->tau[b] / kFourPi;              // x (Q / sumC): tau Q_b / 4pi (Eq. 11, 15)
    pl.band[2 * B + b] = 1.0 / p->tau[b];
    pl.band[3 * B + b] = p->v[b];
  }

  // ---- directions -> octants, canonical order inside an octant (by |s|), 16-slot chunks
  std::vector<int> od[8];
  for (int d = 0; d < D; ++d) {
    const double *s = p->s + 3 * d;
    od[(s[0] < 0) | ((s[1] < 0) << 1) | ((s[2] < 0) << 2)].push_back(d);
  }
  auto key = [&](int d, int a) { return std::llround(std::fabs(p->s[3 * d + a]) * 1e11); };
  for (int o = 0; o < 8; ++o)
    std::sort(od[o].begin(), od[o].end(), [&](int x, int y) {
      for (int a = 0; a < 3; ++a) if (key(x, a) != key(y, a)) return key(x, a) < key(y, a);
      return x < y;
    });
  {   // a SPECULAR face needs a first moment that vanishes (Eq. 7 conserves energy only then): |sum w s| <= 1e-9 * 4 pi
    bool any_spec = false;
    for (int f = 0; f < 2 * p->dim; ++f) any_spec = any_spec || p->face_bc[f].type == BTE_BC_SPECULAR;
    if (any_spec) {
      double m1[3] = {0, 0, 0};
      for (int d = 0; d < D; ++d) for (int c = 0; c < 3; ++c) m1[c] += p->w[d] * p->s[3 * d + c];
      if (std::sqrt(m1[0] * m1[0] + m1[1] * m1[1] + m1[2] * m1[2]) > 1e-9 * kFourPi) return BTE_ERR_QUADRATURE;
    }
  }
  for (int a = 0; a < p->dim; ++a) {
    if (p->face_bc[2 * a].type != BTE_BC_SPECULAR && p->face_bc[2 * a + 1].type != BTE_BC_SPECULAR) continue;
    for (int o = 0; o < 8; ++o) {
      const std::vector<int> &A = od[o], &M = od[o ^ (1 << a)];
      if (A.size() != M.size()) return BTE_ERR_QUADRATURE;
      for (size_t q = 0; q < A.size(); ++q) {
        for (int c = 0; c < 3; ++c)
          if (std::fabs(std::fabs(p->s[3 * A[q] + c]) - std::fabs(p->s[3 * M[q] + c])) > 1e-12) return BTE_ERR_QUADRATURE;
        if (std::fabs(p->w[A[q]] - p->w[M[q]]) > 1e-12 * kFourPi) return BTE_ERR_QUADRATURE;
      }
    }
  }
  int max_items = 1, max_chunk = 1;
  for (int o = 0; o < 8; ++o) {
    BteOct &O = dv.oct[o];
    O.sx = (o & 1) ? -1 : 1; O.sy = (o & 2) ? -1 : 1; O.sz = (o & 4) ? -1 : 1;
    O.cls = o & 3;
    O.active = !od[o].empty();
    O.nchunk = ((int)od[o].size() + BTE_P - 1) / BTE_P;
    O.nitems = O.nchunk * B;
    max_items = std::max(max_items, O.nitems);
    max_chunk = std::max(max_chunk, O.nchunk);
  }
  dv.max_items = max_items;
  dv.nHslot = 4 * max_chunk;
  pl.item_coef.assign((size_t)8 * max_items, 0);
  for (int o = 0; o < 8; ++o) {
    const BteOct &O = dv.oct[o];
    for (int b = 0; b < B; ++b) for (int c = 0; c < O.nchunk; ++c) {
      double blk[BTE_P * BTE_NCOEF];
      std::memset(blk, 0, sizeof blk);
      const double Lam = p->v[b] * p->tau[b];
      for (int q = 0; q < BTE_P; ++q) {
        const size_t pos = (size_t)c * BTE_P + q;
        if (pos >= od[o].size()) break;
        const int d = od[o][pos];
        double ca[3] = {0, 0, 0}, sum = 1.0;
        for (int a = 0; a < p->dim; ++a) { ca[a] = Lam * std::fabs(p->s[3 * d + a]) / delta[a]; sum += ca[a]; }
        const double inv = 1.0 / sum;     // row i of Eq. 21 scaled by tau: (1 + sum_a c_a) e = rhs + sum_a c_a e_up
        double *r = blk + q * BTE_NCOEF;
        r[0] = inv; r[1] = ca[0] * inv; r[2] = ca[1] * inv; r[3] = ca[2] * inv;
        r[4] = p->w[d];
        for (int a = 0; a < 3; ++a) r[5 + a] = p->w[d] * std::fabs(p->s[3 * d + a]);
      }
      // reuse an existing block that agrees to rounding (mirrored direction cosines differ in the last bits)
      int32_t off = -1;
      for (size_t e = 0; e + BTE_P * BTE_NCOEF <= pl.coef.size() && off < 0; e += BTE_P * BTE_NCOEF) {
        bool eq = true;
        for (int c = 0; c < BTE_P * BTE_NCOEF && eq; ++c)
          eq = std::fabs(pl.coef[e + c] - blk[c]) <= 1e-13 * std::max(std::fabs(blk[c]), 1e-300);
        if (eq) off = (int32_t)e;
      }
      if (off < 0) {
        off = (int32_t)pl.coef.size();
        pl.coef.insert(pl.coef.end(), blk, blk + BTE_P * BTE_NCOEF);
      }
      pl.item_coef[(size_t)o * max_items + b * O.nchunk + c] = off;
    }
  }
  const bool const_overflow = pl.coef.size() * tsz > BTE_CONST_BYTES;   // only the generic path keeps the table in c_coef

  // ---- work units in ticket (topological) order: key = item + ty + tz
  struct Key { int key, o, item, ty, tz; };
  std::vector<Key> ks;
  for (int o = 0; o < 8; ++o) {
    if (!dv.oct[o].active) continue;
    for (int it = 0; it < dv.oct[o].nitems; ++it)
      for (int ty = 0; ty < dv.nty; ++ty) for (int tz = 0; tz < dv.ntz; ++tz) ks.push_back({it + ty + tz, o, it, ty, tz});
  }
  std::stable_sort(ks.begin(), ks.end(), [](const Key &a, const Key &b) { return a.key < b.key; });
  std::vector<int32_t> idmap((size_t)8 * max_items * dv.nty * dv.ntz, -1);
  auto slot = [&](int o, int it, int ty, int tz) { return (((size_t)o * max_items + it) * dv.nty + ty) * dv.ntz + tz; };
  for (size_t u = 0; u < ks.size(); ++u) idmap[slot(ks[u].o, ks[u].item, ks[u].ty, ks[u].tz)] = (int32_t)u;
  pl.units.resize(ks.size());
  for (size_t u = 0; u < ks.size(); ++u) {
    const Key &k = ks[u];
    BteUnit &U = pl.units[u];
    U.oct = k.o; U.item = k.item; U.ty = k.ty; U.tz = k.tz;
    U.band = k.item / dv.oct[k.o].nchunk; U.chunk = k.item % dv.oct[k.o].nchunk;
    U.coef_off = pl.item_coef[(size_t)k.o * max_items + k.item];
    U.dep_y = k.ty > 0 ? idmap[slot(k.o, k.item, k.ty - 1, k.tz)] : -1;
    U.dep_z = k.tz > 0 ? idmap[slot(k.o, k.item, k.ty, k.tz - 1)] : -1;
    U.dep_prev = k.item > 0 ? idmap[slot(k.o, k.item - 1, k.ty, k.tz)] : -1;
  }
  dv.n_units = (int32_t)pl.units.size();
  pl.steps_total = (int64_t)pl.units.size() * (dv.nx + 31 + dv.TZ - 1);

  // ---- workspace carve-up (offsets only; pointers are set in bind())
  pl.gf_elems = 0;
  for (int f = 0; f < 2 * p->dim; ++f) {
    const int a = f >> 1;
    const int64_t na = a == 0 ? p->ny : p->nx, nb = a == 2 ? p->ny : p->nz;
    pl.gf_elems += (size_t)na * nb * B;
  }
  for (int o = 0; o < 8; ++o) {
    const BteOct &O = dv.oct[o];
    if (!O.active) continue;
    pl.xpl_elems[o] = (size_t)2 * O.nitems * BTE_P * dv.nz * dv.nyp;
    pl.ypl_elems[o] = dv.has_y ? (size_t)(dv.nty + 1) * O.nitems * dv.nz * dv.nx * BTE_P : 0;
    pl.zpl_elems[o] = dv.has_z ? (size_t)(dv.ntz + 1) * O.nitems * dv.nty * dv.NU * BTE_P * 32 : 0;
  }
  dv.n_red_blocks = (int)std::min<int64_t>((N + 255) / 256, 148 * 16);

  // ---- fast path: 3-D, all solid, 16 directions in each of the 8 octants with identical |s|, w tables
  // (mirror-symmetric quadrature), <= 16 bands.  Anything else runs the generic kernels above.
  bool v2 = p->dim == 3 && B <= BTE2_MAXB && p->nx <= 60000 && p->ny % 2 == 0 && p->nz % 2 == 0 && N < (int64_t)1 << 31;   // (32-bit cell index in the update kernel)
  pl.masked2 = nsolid != N;
  if (g_opt[BTE_OPT_FORCE_GENERIC].load() == 1) v2 = false;
  for (int o = 0; o < 8 && v2; ++o) {
    if ((int)od[o].size() != BTE2_P) v2 = false;
    for (int b = 0; b < B && v2; ++b) {   // same table up to rounding of the mirrored direction cosines
      const double *x = pl.coef.data() + pl.item_coef[(size_t)o * max_items + b], *y = pl.coef.data() + pl.item_coef[b];
      for (int c = 0; c < BTE_P * BTE_NCOEF && v2; ++c)
        if (std::fabs(x[c] - y[c]) > 1e-12 * std::max(std::fabs(y[c]), 1e-300)) v2 = false;
    }
  }
  pl.v2 = v2;
  if (!v2 && const_overflow) return BTE_ERR_UNSUPPORTED;
  if (v2) {
    Bte2Dev &d = pl.d2;
    int W = p->nz >= 48 ? 8 : (p->nz <= 4 ? 2 : 4);   // 2 warps: thin slabs (the two-layer form of 2-D problems)
    { const int w = g_opt[BTE_OPT_WARPS].load(); if (w == 2 || w == 4 || w == 8) W = w; }
    d.nx = p->nx; d.ny = p->ny; d.nz = p->nz; d.B = B; d.W = W;
    d.nty = (p->ny + 63) / 64; d.ntz = (p->nz + 2 * W - 1) / (2 * W); d.NU = p->nx + 31;
    d.nsteps = p->nx + 31 + W - 1;
    // publication period of a unit's progress (measured, profiles/README.md): short and medium rows gain from frequent
    // publication (the units behind start and follow more closely: configs 1-3 -6 ... -8 %), long rows from fewer fences
    d.pub_mask = (p->nx < 224 ? BTE2_PUB / 2 : (p->nx < 256 ? BTE2_PUB : 2 * BTE2_PUB)) - 1; d.slack = BTE2_SLACK;
    { const int v = g_opt[BTE_OPT_PUBLISH_PERIOD].load(); if (v == 4 || v == 8 || v == 16 || v == 32) d.pub_mask = v - 1; }
    { const int v = g_opt[BTE_OPT_START_SLACK].load(); if (v > 0 && v <= 256) d.slack = v; }
    d.NS = (int64_t)p->nz * d.nty * d.NU * 64;
    d.ncell = N; d.src_mod = N; d.inv_sumCtau = dv.inv_sumCtau;
    const int NBmax = dv.fp32 ? 2 : 1, G = (B + NBmax - 1) / NBmax;
    for (int b = 0; b < B; ++b) {
      const double *blk = pl.coef.data() + pl.item_coef[b];
      for (int q = 0; q < BTE2_P; ++q) {
        const double *r = blk + q * BTE_NCOEF;
        double k[8] = {r[0], r[1], r[2], r[3], r[4] / p->tau[b], p->v[b] * r[5], p->v[b] * r[6], p->v[b] * r[7]};
        for (int c = 0; c < 8; ++c) { pl.cf64.k[b][c][q] = k[c]; pl.cf32.k[b][c][q] = (float)k[c]; }
        if (b == 0) for (int a = 0; a < 3; ++a) d.wsa[q][a] = r[5 + a];
      }
      pl.cf64.bc[b][0] = pl.band[b]; pl.cf64.bc[b][1] = pl.band[B + b];
      pl.cf32.bc[b][0] = (float)pl.band[b]; pl.cf32.bc[b][1] = (float)pl.band[B + b];
    }
    for (int f = 0; f < 6; ++f) {
      d.face_type[f] = dv.face_type[f]; d.Pi_face[f] = dv.Pi_face[f];
      for (int b = 0; b < B; ++b) d.face_e0[f][b] = pl.band[b] * dv.face_dT[f];
    }
    for (int o = 0; o < 8; ++o) {
      d.oct[o].sx = (o & 1) ? -1 : 1; d.oct[o].sy = (o & 2) ? -1 : 1; d.oct[o].sz = (o & 4) ? -1 : 1;
      d.oct[o].cls = o & 3;
    }
    // units in ticket order (g, ty, tz, octant): every dependency has a smaller index
    auto uid = [&](int g, int ty, int tz, int o) { return ((g * d.nty + ty) * d.ntz + tz) * 8 + o; };
    pl.units2.resize((size_t)G * d.nty * d.ntz * 8);
    for (int g = 0; g < G; ++g) for (int ty = 0; ty < d.nty; ++ty) for (int tz = 0; tz < d.ntz; ++tz) for (int o = 0; o < 8; ++o) {
      Bte2Unit &U = pl.units2[uid(g, ty, tz, o)];
      U.oct = o; U.g = g; U.ty = ty; U.tz = tz;
      U.dep_y = ty > 0 ? uid(g, ty - 1, tz, o) : -1;
      U.dep_z = tz > 0 ? uid(g, ty, tz - 1, o) : -1;
      U.dep_prev = g > 0 ? uid(g - 1, ty, tz, o) : -1;
      U.b0 = g * NBmax; U.nb = std::min(NBmax, B - U.b0);
    }
    d.n_iface = nif; d.iface_type = p->interface_bc.type;
    for (int b = 0; b < B; ++b) { d.iface_e0[b] = pl.band[b] * p->interface_bc.dT_wall; d.ivband[b] = 1.0 / p->v[b]; }
    if (pl.masked2) {
      const size_t NPp = (size_t)(p->nz / 2) * d.nty * d.NU * 32;
      for (int cl = 0; cl < 4; ++cl) {
        pl.codeP[cl].assign(NPp, 0u);
        for (int k = 0; k < p->nz; ++k) for (int j = 0; j < p->ny; ++j) for (int i = 0; i < p->nx; ++i) {
          const int ipc = (cl & 1) ? p->nx - 1 - i : i, jpc = (cl & 2) ? p->ny - 1 - j : j;
          const int ty = jpc >> 6, J = (jpc & 63) >> 1;
          const size_t idx = (((size_t)(k >> 1) * d.nty + ty) * d.NU + (ipc + J)) * 32 + J;
          const uint32_t byte = pl.code[(size_t)i + (size_t)p->nx * (j + (size_t)p->ny * k)];
          pl.codeP[cl][idx] |= byte << (8 * ((j & 1) + 2 * (k & 1)));
        }
      }
    }
    d.n_units = (int32_t)pl.units2.size();
    const size_t nch = BTE2_P * tsz / 16;
    pl.x2_chunks = (size_t)d.ntz * d.nty * B * W * 2 * 2 * nch * 32;
    pl.y2_slot = (size_t)d.ntz * B * W * d.nx * 2 * nch;
    pl.z2_slot = (size_t)d.nty * B * d.NU * 2 * nch * 32;
    pl.y2_chunks = (size_t)(d.nty + 2) * pl.y2_slot;
    pl.z2_chunks = (size_t)(d.ntz + 2) * pl.z2_slot;
    int64_t off = 0;
    for (int f = 0; f < 6; ++f) {
      const int a = f >> 1;
      const int64_t na = a == 0 ? p->ny : p->nx, nb = a == 2 ? p->ny : p->nz;
      d.gf_off[f] = off; off += na * nb * B;
    }
    d.gf_off[6] = off;
    pl.steps_total = (int64_t)pl.units2.size() * d.nsteps;
  }
  return BTE_OK;
}

// 2-D problems (dim 2, nz 1) have no z coupling; on the fast path they run as a 3-D slab of two identical layers
// with a z spacing so large that the z coefficient vanishes (c_z = v tau |s_z| / dz -> 0), isothermal z faces
// whose inflow is then multiplied by 0.  Layer 0 is what the caller sees; the second layer is redundant work
// (not counted in bte_updates_per_sweep) that buys the tiled, register-resident sweep instead of the generic one.
bte_status build_plan(const bte_problem *p, Plan &pl) {
  bte_status st = build_plan_impl(p, pl);
  pl.user_ncell = pl.dev.ncell; pl.user_nsolid = pl.dev.nsolid;
  if (st != BTE_OK || pl.v2 || p->dim != 2 || p->ny % 2 != 0) return st;
  if (g_opt[BTE_OPT_FORCE_GENERIC].load() == 1) return st;
  const size_t N = (size_t)p->nx * p->ny;
  std::vector<uint8_t> mask2;
  std::vector<double> Q2;
  bte_problem q = *p;
  q.dim = 3; q.nz = 2; q.dz = 1e300;
  q.face_bc[4].type = q.face_bc[5].type = BTE_BC_ISOTHERMAL;
  q.face_bc[4].dT_wall = q.face_bc[5].dT_wall = 0.0;
  if (p->solid_mask) { mask2.assign(p->solid_mask, p->solid_mask + N); mask2.insert(mask2.end(), p->solid_mask, p->solid_mask + N); q.solid_mask = mask2.data(); }
  if (p->Q) { Q2.assign(p->Q, p->Q + N); Q2.insert(Q2.end(), p->Q, p->Q + N); q.Q = Q2.data(); }
  Plan p3;
  if (build_plan_impl(&q, p3) == BTE_OK && p3.v2) {
    p3.layers = 2; p3.user_ncell = pl.dev.ncell; p3.user_nsolid = pl.dev.nsolid;
    pl = std::move(p3);
  }
  return BTE_OK;
}

// Assign device pointers inside the workspace. Returns total bytes needed.
size_t bind(Plan &pl, unsigned char *ws) {
  BteDev &dv = pl.dev;
  const size_t tsz = dv.fp32 ? 4 : 8;
  size_t off = 0;
  auto take = [&](size_t bytes) { void *p = ws ? ws + off : nullptr; off = align_up(off + bytes); return p; };
  const size_t N = (size_t)dv.ncell, NS = (size_t)dv.NS;
  dv.code = (uint8_t *)take(N);
  dv.Qphys = (double *)take(N * 8);
  if (!pl.v2) {
    for (int c = 0; c < 4; ++c) dv.code_sk[c] = (uint8_t *)take(NS);
    for (int c = 0; c < 4; ++c) dv.Q_sk[c] = take(NS * tsz);
    dv.iface = dv.n_iface ? (int32_t *)take((size_t)6 * N * 4) : nullptr;
    dv.iface_info = dv.n_iface ? (int32_t *)take((size_t)dv.n_iface * 4) : nullptr;
  }
  if (pl.v2) {
    Bte2Dev &d = pl.d2;
    const size_t NS2 = (size_t)d.NS;
    d.units = (const Bte2Unit *)take(pl.units2.size() * sizeof(Bte2Unit));
    if (pl.masked2) {
      d.code = dv.code;
      for (int c = 0; c < 4; ++c) d.codeP[c] = (const uint32_t *)take((size_t)(dv.nz / 2) * d.nty * d.NU * 32 * 4);
      d.iface = d.n_iface ? (const int32_t *)take((size_t)6 * N * 4) : nullptr;
      d.iface_info = d.n_iface ? (const int32_t *)take((size_t)d.n_iface * 4) : nullptr;
      d.iface_cell = d.n_iface ? (const int32_t *)take((size_t)d.n_iface * 4) : nullptr;
    } else {
      d.code = nullptr; d.iface = nullptr; d.iface_info = nullptr; d.iface_cell = nullptr;
      for (int c = 0; c < 4; ++c) d.codeP[c] = nullptr;
    }
    pl.state_begin = off;
    d.Gi = d.n_iface ? take((size_t)d.n_iface * d.B * tsz) : nullptr;
    d.Hd = (d.n_iface && d.iface_type == 1) ? take((size_t)6 * N * d.B * 4 * tsz) : nullptr;
    d.prog = (int32_t *)take((size_t)d.n_units * 4);
    d.ticket = (int32_t *)take(256);
    dv.red = (double *)take((size_t)(4 * dv.n_red_blocks + 4) * 8);
    dv.dT = (double *)take(N * 8);
    dv.q = (double *)take(3 * N * 8);
    dv.qmag = (double *)take(N * 8);
    d.Gf = take(std::max<size_t>(pl.gf_elems, 1) * tsz);
    for (int o = 0; o < 8; ++o) {
      d.oct[o].M = take(NS2 * 4 * tsz);
      d.oct[o].xin = take(pl.x2_chunks * 16); d.oct[o].xout = take(2 * pl.x2_chunks * 16);
      d.oct[o].ypl = take(pl.y2_chunks * 16); d.oct[o].zpl = take(pl.z2_chunks * 16);
    }
    pl.state_end = off;
    for (int c = 0; c < 4; ++c) d.dTQ[c] = take(NS2 * 2 * tsz);
    d.dT = dv.dT; d.q = dv.q; d.qmag = dv.qmag; d.red = dv.red; d.n_red_blocks = dv.n_red_blocks;
    pl.total = off;
    return off;
  }
  dv.item_coef = (const int32_t *)take((size_t)8 * dv.max_items * 4);
  dv.units = (BteUnit *)take((size_t)dv.n_units * sizeof(BteUnit));
  dv.band = (double *)take((size_t)4 * dv.B * 8);
  // ---- state (reset to 0 by bte_solve_host)
  pl.state_begin = off;
  dv.done = (int32_t *)take((size_t)dv.n_units * 4);
  dv.ticket = (int32_t *)take(256);
  dv.red = (double *)take((size_t)(4 * dv.n_red_blocks + 4) * 8);
  for (int c = 0; c < 4; ++c) dv.dT_sk[c] = take(NS * tsz);
  dv.dT = (double *)take(N * 8);
  dv.q = (double *)take(3 * N * 8);
  dv.qmag = (double *)take(N * 8);
  dv.Gi = dv.n_iface ? take((size_t)dv.n_iface * dv.B * tsz) : nullptr;
  dv.Hpart = dv.n_iface ? (double *)take((size_t)dv.n_iface * dv.B * dv.nHslot * 8) : nullptr;
  dv.Gf = take(std::max<size_t>(pl.gf_elems, 1) * tsz);
  for (int o = 0; o < 8; ++o) {
    BteOct &O = dv.oct[o];
    if (!O.active) { O.M = nullptr; O.xpl = O.ypl = O.zpl = nullptr; continue; }
    O.M = (double *)take(4 * NS * 8);
    O.xpl = take(pl.xpl_elems[o] * tsz);
    O.ypl = pl.ypl_elems[o] ? take(pl.ypl_elems[o] * tsz) : nullptr;
    O.zpl = pl.zpl_elems[o] ? take(pl.zpl_elems[o] * tsz) : nullptr;
  }
  pl.state_end = off;
  pl.total = off;
  return off;
}

// Ticket order of the fast path = start order of a list schedule simulated on `slots` resident CTAs:
// a unit may start once every unit it follows is lag + BTE2_SLACK steps ahead, so that the per-step
// dependency polls of the kernel (which stay in place for correctness) almost never have to wait.
void order_units2(Plan &pl, int slots) {
  std::vector<Bte2Unit> &U = pl.units2;
  const int n = (int)U.size(), W = pl.d2.W, nsteps = pl.d2.nsteps;
  const int NBmax = pl.dev.fp32 ? 2 : 1;
  std::vector<double> start(n, -1.0), steptime(n);
  std::vector<int> ndep(n, 0), order;
  std::vector<std::vector<int>> succ(n);
  for (int u = 0; u < n; ++u) {
    steptime[u] = (double)U[u].nb / NBmax;
    const int deps[3] = {U[u].dep_y, U[u].dep_z, U[u].dep_prev};
    for (int d : deps) if (d >= 0) { ++ndep[u]; succ[d].push_back(u); }
  }
  auto allowed = [&](int u) {
    const int deps[3] = {U[u].dep_y, U[u].dep_z, U[u].dep_prev};
    const int lag[3] = {33, W + 1, 1};
    double a = 0;
    for (int k = 0; k < 3; ++k)
      if (deps[k] >= 0) a = std::max(a, start[deps[k]] + (lag[k] + (pl.dev.fp32 ? BTE2_DIST(W, float) : BTE2_DIST(W, double)) + pl.d2.slack + pl.d2.pub_mask + 1) * steptime[deps[k]]);
    return a;
  };
  typedef std::pair<double, int> Key;
  std::priority_queue<Key, std::vector<Key>, std::greater<Key>> ready, freeslot;
  for (int u = 0; u < n; ++u) if (ndep[u] == 0) ready.push({0.0, u});
  for (int k = 0; k < std::max(slots, 1); ++k) freeslot.push({0.0, k});
  order.reserve(n);
  if (g_opt[BTE_OPT_SCHEDULE].load() == 1) {
    // "gang" order (experiment): the band groups of one (tile, octant) take consecutive tickets, tiles in (ty, tz) order
    // -- topological, and group g + 1 trails group g on the same tile by the publication period (L2 reuse of the
    // accumulator rows and cell inputs of the tile)
    std::vector<int> idx(n);
    for (int u = 0; u < n; ++u) idx[u] = u;
    std::stable_sort(idx.begin(), idx.end(), [&](int a, int b) {
      const Bte2Unit &A = U[a], &B = U[b];
      if (A.ty != B.ty) return A.ty < B.ty;
      if (A.tz != B.tz) return A.tz < B.tz;
      if (A.oct != B.oct) return A.oct < B.oct;
      return A.g < B.g;
    });
    order = idx;
    while (!ready.empty()) ready.pop();
  }
  while (!ready.empty()) {
    const Key f = freeslot.top(); freeslot.pop();
    const Key r = ready.top(); ready.pop();
    const int u = r.second;
    start[u] = std::max(f.first, r.first);
    freeslot.push({start[u] + nsteps * steptime[u], f.second});
    order.push_back(u);
    for (int v : succ[u]) if (--ndep[v] == 0) ready.push({allowed(v), v});
  }
  std::vector<int> newid(n);
  for (int k = 0; k < n; ++k) newid[order[k]] = k;
  std::vector<Bte2Unit> out(n);
  for (int k = 0; k < n; ++k) {
    Bte2Unit x = U[order[k]];
    if (x.dep_y >= 0) x.dep_y = newid[x.dep_y];
    if (x.dep_z >= 0) x.dep_z = newid[x.dep_z];
    if (x.dep_prev >= 0) x.dep_prev = newid[x.dep_prev];
    out[k] = x;
  }
  U.swap(out);
}

}  // namespace

struct bte_solver {
  Plan pl;
  unsigned char *ws = nullptr;
  std::vector<unsigned char> coef_bytes;   // coefficient table in the compute type, for c_coef
  cudaStream_t last_stream = nullptr;
  int64_t iters = 0;
  int sweep_grid = 1, num_sms = 148;
  int launches_per_iter = 0;
  // optional device timing of the sweep kernel (bte_set_sweep_timing)
  bool timing = false;
  std::vector<cudaEvent_t> ev;             // pairs (start, stop)
  size_t ev_used = 0;
};

namespace {

template <typename T>
bte_status launch_skew(bte_solver *h, const double *src, double scale, int which, cudaStream_t st) {
  const int64_t N = h->pl.dev.ncell;
  const int grid = (int)std::min<int64_t>((N + 255) / 256, 148 * 16);
  bte_skew_kernel<T><<<grid, 256, 0, st>>>(h->pl.dev, src, scale, which);
  CK(cudaGetLastError());
  return BTE_OK;
}

template <typename T>
bte_status launch_skew2(bte_solver *h, const double *src, double scale, int which, cudaStream_t st) {
  const int64_t N = h->pl.dev.ncell;
  const int grid = (int)std::min<int64_t>((N + 255) / 256, 148 * 16);
  bte2_skew_kernel<T><<<grid, 256, 0, st>>>(h->pl.d2, src, scale, which);
  CK(cudaGetLastError());
  return BTE_OK;
}

bte_status skew(bte_solver *h, const double *src, double scale, int which, cudaStream_t st) {
  if (h->pl.v2) {
    if (which == 2) return BTE_OK;   // no cell codes on the fast path
    return h->pl.dev.fp32 ? launch_skew2<float>(h, src, scale, which, st) : launch_skew2<double>(h, src, scale, which, st);
  }
  return h->pl.dev.fp32 ? launch_skew<float>(h, src, scale, which, st) : launch_skew<double>(h, src, scale, which, st);
}

template <typename T, int W>
void launch_sweep2(bte_solver *h, const Bte2Coefs<T> &cf, cudaStream_t st) {
  if (h->pl.masked2) bte2_sweep_kernel<T, W, true><<<h->sweep_grid, W * 32, h->pl.smem2, st>>>(h->pl.d2, cf);
  else bte2_sweep_kernel<T, W, false><<<h->sweep_grid, W * 32, h->pl.smem2, st>>>(h->pl.d2, cf);
}

template <typename T>
bte_status iterate2_T(bte_solver *h, int n, const Bte2Coefs<T> &cf, cudaStream_t st) {
  Plan &pl = h->pl;
  Bte2Dev &d = pl.d2;
  const int bgrid = h->num_sms * 8;
  for (int it = 0; it < n; ++it) {
    const int ep = (int)(h->iters % 30000) + 1;
    if (ep == 1 && h->iters > 0) CK(cudaMemsetAsync(d.prog, 0, (size_t)d.n_units * 4, st));
    d.epoch = ep;
    d.fill_iso = h->iters == 0;
    {   // ghost planes to fill: diffuse faces every iteration, isothermal faces once (specular / periodic: none)
      const int NCHh = (int)(BTE2_P * (pl.dev.fp32 ? 4 : 8) / 16);
      const int64_t nseg[3] = {(int64_t)d.ny * d.nz * d.B * NCHh, (int64_t)d.nx * d.nz * d.B * NCHh, (int64_t)d.nx * d.ny * d.B * NCHh};
      d.gseg_n = 0; d.gseg_off[0] = 0;
      for (int o = 0; o < 8; ++o) for (int a = 0; a < 3; ++a) {
        const int sg = a == 0 ? d.oct[o].sx : (a == 1 ? d.oct[o].sy : d.oct[o].sz);
        const int type = d.face_type[2 * a + (sg > 0 ? 0 : 1)];
        if (type >= 2 || (type == 0 && !d.fill_iso)) continue;
        d.gseg_oa[d.gseg_n] = o * 3 + a;
        d.gseg_off[d.gseg_n + 1] = d.gseg_off[d.gseg_n] + nseg[a];
        ++d.gseg_n;
      }
    }
    {   // inflow sources / outflow buffers of this iteration (parity of the epoch)
      const size_t cur = (size_t)(ep & 1), prev = cur ^ 1;
      auto xo = [&](int o, size_t par) { return (char *)d.oct[o].xout + par * pl.x2_chunks * 16; };
      auto yo = [&](int o, size_t par) { return (char *)d.oct[o].ypl + ((size_t)d.nty + par) * pl.y2_slot * 16; };
      auto zo = [&](int o, size_t par) { return (char *)d.oct[o].zpl + ((size_t)d.ntz + par) * pl.z2_slot * 16; };
      for (int o = 0; o < 8; ++o) {
        Bte2Oct &O = d.oct[o];
        O.xdst = xo(o, cur); O.ydstN = yo(o, cur); O.zdstN = zo(o, cur);
        O.xprev = xo(o, prev); O.yprev = yo(o, prev); O.zprev = zo(o, prev);
        const int sg[3] = {O.sx, O.sy, O.sz};
        const void *ghost[3] = {O.xin, O.ypl, O.zpl};
        const void *src[3];
        for (int a = 0; a < 3; ++a) {
          const int type = d.face_type[2 * a + (sg[a] > 0 ? 0 : 1)];
          const int from = type == 2 ? (o ^ (1 << a)) : o;
          src[a] = type < 2 ? ghost[a] : (a == 0 ? (const void *)xo(from, prev) : (a == 1 ? (const void *)yo(from, prev) : (const void *)zo(from, prev)));
        }
        O.xsrc = src[0]; O.ysrc0 = src[1]; O.zsrc0 = src[2];
      }
    }
    if (pl.any_diffuse_face) bte2_gdiff_kernel<T><<<bgrid, 256, 0, st>>>(d);
    bte2_ghost_kernel<T><<<bgrid, 256, 0, st>>>(d);
    const bool tm = h->timing && h->ev_used + 2 <= h->ev.size();
    if (tm) CK(cudaEventRecord(h->ev[h->ev_used], st));
    if (d.W == 8) launch_sweep2<T, 8>(h, cf, st); else if (d.W == 4) launch_sweep2<T, 4>(h, cf, st); else launch_sweep2<T, 2>(h, cf, st);
    if (tm) { CK(cudaEventRecord(h->ev[h->ev_used + 1], st)); h->ev_used += 2; }
    bte2_update_kernel<T><<<pl.dev.n_red_blocks, 256, 0, st>>>(d);
    bte_final_kernel<<<1, 256, 0, st>>>(pl.dev);
    h->iters += 1;
    if (it == 0) CK(cudaGetLastError());   // a bad launch configuration shows up at once, not after n queued iterations
  }
  CK(cudaGetLastError());
  return BTE_OK;
}

template <typename T, int W>
bte_status setup_sweep2_W(bte_solver *h) {
  Plan &pl = h->pl;
  pl.smem2 = sizeof(Bte2Smem<T, sizeof(T) == 4 ? 2 : 1, W, BTE2_DIST(W, T)>);
  int occ = 0;
  if (pl.masked2) {
    CK(cudaFuncSetAttribute(bte2_sweep_kernel<T, W, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem2));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, bte2_sweep_kernel<T, W, true>, W * 32, pl.smem2));
  } else {
    CK(cudaFuncSetAttribute(bte2_sweep_kernel<T, W, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem2));
    CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, bte2_sweep_kernel<T, W, false>, W * 32, pl.smem2));
  }
  if (occ < 1) { g_last_cuda.store((int)cudaErrorLaunchOutOfResources); return BTE_ERR_CUDA; }
  h->sweep_grid = (int)std::min<int64_t>(pl.d2.n_units, (int64_t)h->num_sms * occ);
  pl.nthreads = W * 32;
  return BTE_OK;
}
template <typename T>
bte_status setup_sweep2(bte_solver *h) {
  return h->pl.d2.W == 8 ? setup_sweep2_W<T, 8>(h) : (h->pl.d2.W == 4 ? setup_sweep2_W<T, 4>(h) : setup_sweep2_W<T, 2>(h));
}

template <typename T>
bte_status iterate_T(bte_solver *h, int n, cudaStream_t st) {
  Plan &pl = h->pl;
  BteDev &dv = pl.dev;
  CK(cudaMemcpyToSymbolAsync(c_coef, h->coef_bytes.data(), h->coef_bytes.size(), 0, cudaMemcpyHostToDevice, st));
  const int bgrid = h->num_sms * 4;
  for (int it = 0; it < n; ++it) {
    dv.epoch = (int32_t)(h->iters + 1);
    if (pl.any_diffuse_face) bte_gdiff_kernel<T><<<bgrid, 256, 0, st>>>(dv);
    bte_ghost_kernel<T><<<bgrid, 256, 0, st>>>(dv);
    const bool tm = h->timing && h->ev_used + 2 <= h->ev.size();
    if (tm) CK(cudaEventRecord(h->ev[h->ev_used], st));
    bte_sweep_kernel<T><<<h->sweep_grid, pl.nthreads, pl.smem, st>>>(dv);
    if (tm) { CK(cudaEventRecord(h->ev[h->ev_used + 1], st)); h->ev_used += 2; }
    bte_update_kernel<T><<<dv.n_red_blocks, 256, 0, st>>>(dv);
    bte_final_kernel<<<1, 256, 0, st>>>(dv);
    h->iters += 1;
    if (it == 0) CK(cudaGetLastError());
  }
  CK(cudaGetLastError());
  return BTE_OK;
}

template <typename T>
bte_status setup_sweep(bte_solver *h) {
  Plan &pl = h->pl;
  CK(cudaFuncSetAttribute(bte_sweep_kernel<T>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl.smem));
  int occ = 0;
  CK(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, bte_sweep_kernel<T>, pl.nthreads, pl.smem));
  if (occ < 1) { g_last_cuda.store((int)cudaErrorLaunchOutOfResources); return BTE_ERR_CUDA; }
  h->sweep_grid = (int)std::min<int64_t>(pl.dev.n_units, (int64_t)h->num_sms * occ);
  return BTE_OK;
}

}  // namespace

extern "C" {

size_t bte_workspace_bytes(const bte_problem *p) {
  Plan pl;
  if (build_plan(p, pl) != BTE_OK) return 0;
  return bind(pl, nullptr);
}

bte_status bte_create(const bte_problem *p, void *d_workspace, size_t bytes, void *cuda_stream, bte_solver **out) {
  if (!out) return BTE_ERR_INVALID_ARG;
  bte_solver *h = new (std::nothrow) bte_solver();
  if (!h) return BTE_ERR_INVALID_ARG;
  bte_status st = build_plan(p, h->pl);
  if (st != BTE_OK) { delete h; return st; }
  const size_t need = bind(h->pl, nullptr);
  if (!d_workspace || (reinterpret_cast<uintptr_t>(d_workspace) & 255) || bytes < need) { delete h; return BTE_ERR_WORKSPACE; }
  h->ws = static_cast<unsigned char *>(d_workspace);
  bind(h->pl, h->ws);
  h->pl.d2.src_mod = h->pl.user_ncell;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  Plan &pl = h->pl;
  BteDev &dv = pl.dev;
  auto fail = [&](bte_status e) { delete h; return e; };
#define CKD(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { g_last_cuda.store((int)e_); return fail(BTE_ERR_CUDA); } } while (0)
  int devid = 0;
  CKD(cudaGetDevice(&devid));
  CKD(cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, devid));
  CKD(cudaMemsetAsync(h->ws, 0, need, s));
  if (pl.v2) st = dv.fp32 ? setup_sweep2<float>(h) : setup_sweep2<double>(h);
  else st = dv.fp32 ? setup_sweep<float>(h) : setup_sweep<double>(h);
  if (st != BTE_OK) return fail(st);
  CKD(cudaMemcpyAsync(dv.code, pl.code.data(), pl.code.size(), cudaMemcpyHostToDevice, s));
  CKD(cudaMemcpyAsync(dv.Qphys, pl.Q.data(), pl.Q.size() * 8, cudaMemcpyHostToDevice, s));
  if (pl.v2) {
    order_units2(pl, h->sweep_grid);
    CKD(cudaMemcpyAsync((void *)pl.d2.units, pl.units2.data(), pl.units2.size() * sizeof(Bte2Unit), cudaMemcpyHostToDevice, s));
    if (pl.masked2) {
      for (int c = 0; c < 4; ++c)
        CKD(cudaMemcpyAsync((void *)pl.d2.codeP[c], pl.codeP[c].data(), pl.codeP[c].size() * 4, cudaMemcpyHostToDevice, s));
      if (pl.d2.n_iface) {
        CKD(cudaMemcpyAsync((void *)pl.d2.iface, pl.iface.data(), pl.iface.size() * 4, cudaMemcpyHostToDevice, s));
        CKD(cudaMemcpyAsync((void *)pl.d2.iface_info, pl.iface_info.data(), pl.iface_info.size() * 4, cudaMemcpyHostToDevice, s));
        CKD(cudaMemcpyAsync((void *)pl.d2.iface_cell, pl.iface_cell.data(), pl.iface_cell.size() * 4, cudaMemcpyHostToDevice, s));
      }
    }
  } else {
    if (dv.n_iface) {
      CKD(cudaMemcpyAsync(dv.iface, pl.iface.data(), pl.iface.size() * 4, cudaMemcpyHostToDevice, s));
      CKD(cudaMemcpyAsync(dv.iface_info, pl.iface_info.data(), pl.iface_info.size() * 4, cudaMemcpyHostToDevice, s));
    }
    CKD(cudaMemcpyAsync((void *)dv.item_coef, pl.item_coef.data(), pl.item_coef.size() * 4, cudaMemcpyHostToDevice, s));
    CKD(cudaMemcpyAsync(dv.units, pl.units.data(), pl.units.size() * sizeof(BteUnit), cudaMemcpyHostToDevice, s));
    CKD(cudaMemcpyAsync(dv.band, pl.band.data(), pl.band.size() * 8, cudaMemcpyHostToDevice, s));
  }
  // coefficient table in the compute type
  if (dv.fp32) {
    h->coef_bytes.resize(pl.coef.size() * 4);
    float *f = reinterpret_cast<float *>(h->coef_bytes.data());
    for (size_t i = 0; i < pl.coef.size(); ++i) f[i] = (float)pl.coef[i];
    // unit offsets are in values, identical for both types
  } else {
    h->coef_bytes.resize(pl.coef.size() * 8);
    std::memcpy(h->coef_bytes.data(), pl.coef.data(), pl.coef.size() * 8);
  }

  st = skew(h, dv.Qphys, 0.0, 2, s);                       // cell codes -> skewed copies
  if (st == BTE_OK) st = skew(h, dv.Qphys, 1.0 / pl.sumC, 0, s);  // Q / sum C (Eq. 11)
  if (st != BTE_OK) return fail(st);
  CKD(cudaStreamSynchronize(s));
#undef CKD
  h->last_stream = s;
  h->launches_per_iter = 4 + (pl.any_diffuse_face ? 1 : 0);
  *out = h;
  return BTE_OK;
}

bte_status bte_iterate(bte_solver *h, int32_t n, void *cuda_stream) {
  if (!h || n < 0) return BTE_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  h->last_stream = s;
  if (n == 0) return BTE_OK;
  if (h->pl.v2) return h->pl.dev.fp32 ? iterate2_T<float>(h, n, h->pl.cf32, s) : iterate2_T<double>(h, n, h->pl.cf64, s);
  return h->pl.dev.fp32 ? iterate_T<float>(h, n, s) : iterate_T<double>(h, n, s);
}

bte_status bte_get_temperature(bte_solver *h, double *d_out, void *cuda_stream) {
  if (!h || !d_out) return BTE_ERR_INVALID_ARG;
  CK(cudaMemcpyAsync(d_out, h->pl.dev.dT, (size_t)h->pl.user_ncell * 8, cudaMemcpyDeviceToDevice,
                     static_cast<cudaStream_t>(cuda_stream)));
  return BTE_OK;
}

bte_status bte_get_heat_flux(bte_solver *h, double *d_out, void *cuda_stream) {
  if (!h || !d_out) return BTE_ERR_INVALID_ARG;
  for (int c = 0; c < 3; ++c)
    CK(cudaMemcpyAsync(d_out + c * h->pl.user_ncell, h->pl.dev.q + c * h->pl.dev.ncell, (size_t)h->pl.user_ncell * 8,
                       cudaMemcpyDeviceToDevice, static_cast<cudaStream_t>(cuda_stream)));
  return BTE_OK;
}

bte_status bte_set_temperature(bte_solver *h, const double *d_in, void *cuda_stream) {
  if (!h || !d_in) return BTE_ERR_INVALID_ARG;
  return skew(h, d_in, 1.0, 1, static_cast<cudaStream_t>(cuda_stream));
}

bte_status bte_residual(bte_solver *h, double *eps_T, double *eps_q) {
  if (!h) return BTE_ERR_INVALID_ARG;
  const double inf = std::numeric_limits<double>::infinity();
  double eT = inf, eq = inf;
  if (h->iters > 0) {
    double r[4];
    CK(cudaMemcpyAsync(r, h->pl.dev.red + 4 * h->pl.dev.n_red_blocks, 32, cudaMemcpyDeviceToHost, h->last_stream));
    CK(cudaStreamSynchronize(h->last_stream));
    const double n = (double)h->pl.dev.nsolid;
    const double rT = std::sqrt(r[0] / n), rq = std::sqrt(r[2] / n);
    eT = r[1] > 0 ? rT / r[1] : (rT == 0 ? 0.0 : inf);
    eq = r[3] > 0 ? rq / r[3] : (rq == 0 ? 0.0 : inf);
  } else {
    CK(cudaStreamSynchronize(h->last_stream));
  }
  if (eps_T) *eps_T = eT;
  if (eps_q) *eps_q = eq;
  return BTE_OK;
}

bte_status bte_set_sweep_timing(bte_solver *h, int32_t max_launches) {
  if (!h || max_launches < 0 || max_launches > 4096) return BTE_ERR_INVALID_ARG;
  for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
  h->ev.clear(); h->ev_used = 0; h->timing = max_launches > 0;
  for (int i = 0; i < 2 * max_launches; ++i) {
    cudaEvent_t e;
    CK(cudaEventCreate(&e));
    h->ev.push_back(e);
  }
  return BTE_OK;
}

bte_status bte_get_sweep_timing(bte_solver *h, double *total_ms, int64_t *launches) {
  if (!h) return BTE_ERR_INVALID_ARG;
  double tot = 0;
  if (h->ev_used) CK(cudaEventSynchronize(h->ev[h->ev_used - 1]));
  for (size_t i = 0; i + 1 < h->ev_used; i += 2) {
    float ms = 0;
    CK(cudaEventElapsedTime(&ms, h->ev[i], h->ev[i + 1]));
    tot += ms;
  }
  if (total_ms) *total_ms = tot;
  if (launches) *launches = (int64_t)(h->ev_used / 2);
  h->ev_used = 0;
  return BTE_OK;
}

bte_status bte_solve_host(bte_solver *h, const double *Q_host, int32_t n, int32_t reset, double *dT_host,
                          double *q_host, void *cuda_stream) {
  if (!h || n < 0 || !dT_host) return BTE_ERR_INVALID_ARG;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  Plan &pl = h->pl;
  BteDev &dv = pl.dev;
  if (Q_host) {
    CK(cudaMemcpyAsync(dv.Qphys, Q_host, (size_t)pl.user_ncell * 8, cudaMemcpyHostToDevice, s));
    bte_status st = skew(h, dv.Qphys, 1.0 / pl.sumC, 0, s);
    if (st != BTE_OK) return st;
  }
  if (reset) {
    CK(cudaMemsetAsync(h->ws + pl.state_begin, 0, pl.state_end - pl.state_begin, s));
    h->iters = 0;
    if (pl.v2) {   // dT = 0 into the skewed class copies the sweep reads
      bte_status st = skew(h, dv.dT, 1.0, 1, s);
      if (st != BTE_OK) return st;
    }
  }
  bte_status st = bte_iterate(h, n, cuda_stream);
  if (st != BTE_OK) return st;
  CK(cudaMemcpyAsync(dT_host, dv.dT, (size_t)pl.user_ncell * 8, cudaMemcpyDeviceToHost, s));
  if (q_host)
    for (int c = 0; c < 3; ++c)
      CK(cudaMemcpyAsync(q_host + c * pl.user_ncell, dv.q + c * dv.ncell, (size_t)pl.user_ncell * 8, cudaMemcpyDeviceToHost, s));
  CK(cudaStreamSynchronize(s));
  return BTE_OK;
}

bte_status bte_plan_info(const bte_problem *p, int32_t resident_ctas, int64_t out[8]) {
  if (!out) return BTE_ERR_INVALID_ARG;
  Plan pl;
  bte_status st = build_plan(p, pl);
  if (st != BTE_OK) return st;
  for (int i = 0; i < 8; ++i) out[i] = 0;
  out[0] = pl.v2 ? 2 : 1;
  out[7] = (int64_t)bind(pl, nullptr);
  if (!pl.v2) {
    out[1] = pl.dev.n_units; out[3] = pl.dev.nx + 31 + pl.dev.TZ - 1; out[4] = pl.dev.TZ;
    bool topo = true;
    for (size_t u = 0; u < pl.units.size(); ++u)
      for (int d : {pl.units[u].dep_y, pl.units[u].dep_z, pl.units[u].dep_prev}) topo = topo && d < (int)u;
    out[2] = topo;
    return BTE_OK;
  }
  order_units2(pl, std::max(resident_ctas, 1));
  bool topo = true, same = true;
  for (size_t u = 0; u < pl.units2.size(); ++u) {
    const Bte2Unit &U = pl.units2[u];
    for (int d : {U.dep_y, U.dep_z, U.dep_prev}) topo = topo && d < (int)u;
    if (U.dep_y >= 0) { const Bte2Unit &D = pl.units2[U.dep_y]; same = same && D.oct == U.oct && D.g == U.g && D.ty == U.ty - 1 && D.tz == U.tz; }
    if (U.dep_z >= 0) { const Bte2Unit &D = pl.units2[U.dep_z]; same = same && D.oct == U.oct && D.g == U.g && D.ty == U.ty && D.tz == U.tz - 1; }
    if (U.dep_prev >= 0) { const Bte2Unit &D = pl.units2[U.dep_prev]; same = same && D.oct == U.oct && D.g == U.g - 1 && D.ty == U.ty && D.tz == U.tz; }
  }
  out[1] = pl.d2.n_units; out[2] = topo && same; out[3] = pl.d2.nsteps; out[4] = pl.d2.W;
  out[5] = (pl.d2.B + (pl.dev.fp32 ? 2 : 1) - 1) / (pl.dev.fp32 ? 2 : 1);
  out[6] = pl.masked2;
  return BTE_OK;
}

int64_t bte_updates_per_sweep(const bte_solver *h) {
  if (!h) return 0;
  return h->pl.user_nsolid * h->pl.dev.B * (int64_t)h->pl.dev.n_dirs;
}
int64_t bte_iterations_done(const bte_solver *h) { return h ? h->iters : 0; }
int32_t bte_kernel_launches_per_iteration(const bte_solver *h) { return h ? h->launches_per_iter : 0; }
int32_t bte_kernel_path(const bte_solver *h) { return h ? (h->pl.v2 ? 2 : 1) : 0; }

void bte_schedule_info(const bte_solver *h, int64_t out[6]) {
  if (!h || !out) return;
  const Plan &pl = h->pl;
  out[0] = pl.v2 ? pl.d2.n_units : pl.dev.n_units;
  out[1] = h->sweep_grid;
  out[2] = pl.nthreads;
  out[3] = pl.steps_total;
  out[4] = pl.steps_total * pl.nthreads * BTE_P;
  if (pl.v2) {
    out[4] = 0;
    for (const Bte2Unit &u : pl.units2) out[4] += (int64_t)pl.d2.nsteps * pl.d2.W * 32 * 4 * BTE2_P * u.nb;
  }
  out[5] = (int64_t)pl.total;
}

void bte_destroy(bte_solver *h) {
  if (!h) return;
  for (cudaEvent_t e : h->ev) cudaEventDestroy(e);
  delete h;
}

const char *bte_status_string(bte_status s) {
  switch (s) {
    case BTE_OK: return "ok";
    case BTE_ERR_INVALID_ARG: return "invalid argument";
    case BTE_ERR_QUADRATURE: return "quadrature rejected";
    case BTE_ERR_WORKSPACE: return "workspace too small or misaligned";
    case BTE_ERR_CUDA: return "CUDA error";
    case BTE_ERR_UNSUPPORTED: return "unsupported problem";
    case BTE_ERR_TOO_LARGE: return "size beyond the static scratch array (n_cells > BTE_STATIC_MAX_CELLS)";
  }
  return "unknown";
}
int32_t bte_last_cuda_error(void) { return g_last_cuda.load(); }

bte_status bte_set_option(int32_t option, int32_t value) {
  if (option < 0 || option >= BTE_OPT_COUNT_) return BTE_ERR_INVALID_ARG;
  g_opt[option].store(value);
  return BTE_OK;
}

}  // extern "C"

// the allocation-free entry point (bte_residual_static) and its file-scope __device__ scratch array
#include "bte_static.cuh"
