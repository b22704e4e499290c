// oracle/bte_ref.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see bte_ref.h).
//
// Step-by-step fp64 CPU restatement of the source iteration of arxiv 2503.23657
// restricted to Cartesian / voxel-masked grids with first-order upwind faces
// (DESIGN.md "Readings").  No blocking, fusion or reordering
// beyond what the algorithm states:
//
//   for n = 1..:                                           PAPER.md:292-304 (steps 1-4)
//     for every band b, direction d:                       Eq. 20-21
//        nested k/j/i loops in upwind order: solve row i of A e = rhs, A from Eq. 21,
//        rhs = e0 + tau Q_b/4pi (Eq. 15 x tau; Q_b Eq. 11)
//     dT = sum_b sum_d w e/tau_b / sum_b C_b/tau_b          Eq. 16
//     q  = sum_b v_b sum_d w s e                            Eq. 4
//     eps_T, eps_q                                          Eq. 23
//
// Boundary inflow (Eq. 5-7, + periodic) is always taken from
// iteration n (reading G9: pure Jacobi lag, double-buffered store).
//
// Parity pins: tests/test_oracle_*.py (quadrature sums, ballistic/diffusive 1-D
// limits with the closed-form k_eff, Kn=1 integral-equation value, flux
// constancy, energy balance, linearity, symmetry, gray-equivalence, dense LU
// solves of Eq. 21 and of the coupled fixed point).
#include "bte_ref.h"

#include <algorithm>
#include <cmath>
#include <cstring>
#include <limits>
#include <thread>
#include <vector>

namespace {

const double FOUR_PI = 4.0 * 3.14159265358979323846264338327950288;
const double PI = 3.14159265358979323846264338327950288;

struct Face {
  int64_t cell;   // solid cell that owns the face
  int axis;       // 0,1,2
  int side;       // 0: minus side (outward normal -e_a), 1: plus side (+e_a)
  int type;       // BC code
  double dTw;     // isothermal wall deviation temperature
  int64_t partner;  // periodic: face id whose outgoing value flows in here
  int64_t slot;     // index into the lagged store, -1 for isothermal faces
};

}  // namespace

struct bte_ref_solver {
  int nx, ny, nz, dim;
  double delta[3];
  int64_t ncell, nsolid;
  int B, D;
  std::vector<uint8_t> solid;
  std::vector<double> C, v, tau, s, w, Q;
  bte_ref_bc face_bc[6], interface_bc;
  bool diag, literal_pi;
  int threads = 1;
  std::vector<int> dir_order;
  double sumC, sumCtau;
  double Pi_face[6];               // discrete hemispherical normaliser per face orientation
  std::vector<int> reflect[3];     // R_a(d)
  std::vector<int64_t> face_of;    // [6][ncell]: -1 interior solid neighbour, else face id
  std::vector<Face> faces;
  int64_t nslots = 0;
  std::vector<double> out_prev, out_next;  // [slot][B][D] cell-centre intensity at boundary faces
  std::vector<double> Gdiff;               // [face][B] diffuse inflow of this iteration
  std::vector<double> dT, q, qmag;         // [ncell], [3][ncell], [ncell]
  double eps_T = std::numeric_limits<double>::infinity();
  double eps_q = std::numeric_limits<double>::infinity();
  int64_t iters = 0;
  std::vector<double> intensity;           // diag: [B][D][ncell]
  std::vector<double> fflux;               // diag: [B][6][ncell]
};

namespace {

inline int64_t cidx(const bte_ref_solver *h, int i, int j, int k) {
  return (int64_t)i + (int64_t)h->nx * ((int64_t)j + (int64_t)h->ny * (int64_t)k);
}

// inflow value at boundary face f for (band b, direction d), from iteration n.
inline double inflow(const bte_ref_solver *h, const Face &f, int64_t fid, int b, int d) {
  switch (f.type) {
    case BTE_REF_ISOTHERMAL:  // Eq. 5: e = C T / 4pi (deviation form, G3)
      return h->C[b] * f.dTw / FOUR_PI;
    case BTE_REF_DIFFUSE:     // Eq. 6, PAPER.md:198 (discrete normalisation, G10)
      return h->Gdiff[(size_t)fid * h->B + b];
    case BTE_REF_SPECULAR:    // Eq. 7: s' = s - 2 n (s.n)
      return h->out_prev[((size_t)f.slot * h->B + b) * h->D + h->reflect[f.axis][d]];
    case BTE_REF_PERIODIC: {  // BASELINE.json configs[3]: outflow of the opposite face
      const Face &g = h->faces[(size_t)f.partner];
      return h->out_prev[((size_t)g.slot * h->B + b) * h->D + d];
    }
  }
  return 0.0;
}

// All directions of one band. A0 = sum_d w e, A1[a] = sum_d w s_a e  (per cell).
void sweep_band(bte_ref_solver *h, int b, double *A0, double *A1, double *e) {
  const int64_t N = h->ncell;
  const int nx = h->nx, ny = h->ny, nz = h->nz;
  const int64_t stride[3] = {1, nx, (int64_t)nx * ny};
  std::fill(A0, A0 + N, 0.0);
  std::fill(A1, A1 + 3 * N, 0.0);
  const double Cb = h->C[b], vb = h->v[b], taub = h->tau[b];
  const double Lambda = vb * taub;
  double *ff = h->diag ? &h->fflux[(size_t)b * 6 * N] : nullptr;
  if (ff) std::fill(ff, ff + 6 * N, 0.0);
  for (int dd = 0; dd < h->D; ++dd) {
    const int d = h->dir_order.empty() ? dd : h->dir_order[dd];
    const double *sd = &h->s[3 * (size_t)d];
    const double wd = h->w[d];
    double c[3];
    int sg[3];
    for (int a = 0; a < 3; ++a) {
      sg[a] = (sd[a] >= 0.0) ? +1 : -1;  // G14: s_a == 0 -> +1, coefficient 0
      c[a] = (a < h->dim) ? Lambda * std::fabs(sd[a]) / h->delta[a] : 0.0;
    }
    for (int kk = 0; kk < nz; ++kk) {
      const int k = sg[2] > 0 ? kk : nz - 1 - kk;
      for (int jj = 0; jj < ny; ++jj) {
        const int j = sg[1] > 0 ? jj : ny - 1 - jj;
        for (int ii = 0; ii < nx; ++ii) {
          const int i = sg[0] > 0 ? ii : nx - 1 - ii;
          const int64_t id = cidx(h, i, j, k);
          if (!h->solid[id]) { e[id] = 0.0; continue; }
          // rhs = e0 + tau_b Q_b / 4pi, Q_b = C_b Q / sum C  (Eq. 11, 15)
          const double rhs = (Cb / FOUR_PI) * (h->dT[id] + taub * h->Q[id] / h->sumC);
          double num = rhs, den = 1.0;
          for (int a = 0; a < h->dim; ++a) {
            const int upside = sg[a] > 0 ? 2 * a : 2 * a + 1;
            const int64_t fid = h->face_of[(size_t)upside * N + id];
            double eup;
            if (fid < 0) eup = e[id - sg[a] * stride[a]];
            else eup = inflow(h, h->faces[(size_t)fid], fid, b, d);
            num += c[a] * eup;
            den += c[a];
            if (ff) {  // incoming part of the outward flux through the upwind face
              ff[(size_t)upside * N + id] += vb * wd * (-std::fabs(sd[a])) * eup;
            }
          }
          const double val = num / den;  // row i of A e = rhs, A from Eq. 21 (x tau)
          e[id] = val;
          if (ff) {
            for (int a = 0; a < h->dim; ++a) {
              const int downside = sg[a] > 0 ? 2 * a + 1 : 2 * a;
              ff[(size_t)downside * N + id] += vb * wd * std::fabs(sd[a]) * val;  // G13
            }
          }
        }
      }
    }
    for (int64_t id = 0; id < N; ++id) {
      if (!h->solid[id]) continue;
      A0[id] += wd * e[id];
      A1[id] += wd * sd[0] * e[id];
      A1[N + id] += wd * sd[1] * e[id];
      A1[2 * N + id] += wd * sd[2] * e[id];
    }
    // step 5: outgoing cell-centre values at boundary faces -> store^{n+1}
    for (size_t f = 0; f < h->faces.size(); ++f) {
      const Face &F = h->faces[f];
      if (F.slot < 0) continue;
      h->out_next[((size_t)F.slot * h->B + b) * h->D + d] = e[F.cell];
    }
    if (h->diag) {
      std::memcpy(&h->intensity[((size_t)b * h->D + d) * N], e, sizeof(double) * N);
    }
  }
}

void one_iteration(bte_ref_solver *h) {
  const int64_t N = h->ncell;
  // diffuse inflow G_{f,b} = H^n_{f,b} / Pi_f,  H = sum_{s.n>0} w (s.n) e^n  (Eq. 6, G10)
  for (size_t f = 0; f < h->faces.size(); ++f) {
    const Face &F = h->faces[f];
    if (F.type != BTE_REF_DIFFUSE) continue;
    const double nsign = F.side ? +1.0 : -1.0;
    const double Pi_f = h->literal_pi ? PI : h->Pi_face[2 * F.axis + F.side];
    for (int b = 0; b < h->B; ++b) {
      double H = 0.0;
      for (int d = 0; d < h->D; ++d) {
        const double sn = nsign * h->s[3 * (size_t)d + F.axis];
        if (sn > 0.0) H += h->w[d] * sn * h->out_prev[((size_t)F.slot * h->B + b) * h->D + d];
      }
      h->Gdiff[f * h->B + b] = H / Pi_f;
    }
  }
  std::vector<double> M0(N, 0.0), qn(3 * N, 0.0);
  const int T = std::max(1, std::min(h->threads, h->B));
  std::vector<std::vector<double>> A0(T, std::vector<double>(N)), A1(T, std::vector<double>(3 * N)),
      E(T, std::vector<double>(N));
  for (int b0 = 0; b0 < h->B; b0 += T) {
    const int nb = std::min(T, h->B - b0);
    if (nb == 1) {
      sweep_band(h, b0, A0[0].data(), A1[0].data(), E[0].data());
    } else {
      std::vector<std::thread> th;
      for (int t = 0; t < nb; ++t)
        th.emplace_back(sweep_band, h, b0 + t, A0[t].data(), A1[t].data(), E[t].data());
      for (auto &x : th) x.join();
    }
    for (int t = 0; t < nb; ++t) {  // combine in band order (bit-identical for any T)
      const int b = b0 + t;
      const double it = 1.0 / h->tau[b], vb = h->v[b];
      for (int64_t id = 0; id < N; ++id) M0[id] += it * A0[t][id];
      for (int64_t id = 0; id < 3 * N; ++id) qn[id] += vb * A1[t][id];
    }
  }
  // Eq. 16 and Eq. 23
  double sT = 0.0, mT = 0.0, sq = 0.0, mq = 0.0;
  for (int64_t id = 0; id < N; ++id) {
    if (!h->solid[id]) continue;
    const double Tn = M0[id] / h->sumCtau;
    const double dlt = Tn - h->dT[id];
    sT += dlt * dlt;
    mT = std::max(mT, std::fabs(Tn));
    h->dT[id] = Tn;
    const double qm = std::sqrt(qn[id] * qn[id] + qn[N + id] * qn[N + id] + qn[2 * N + id] * qn[2 * N + id]);
    const double dq = qm - h->qmag[id];
    sq += dq * dq;
    mq = std::max(mq, qm);
    h->qmag[id] = qm;
  }
  h->q.swap(qn);
  const double rT = std::sqrt(sT / (double)h->nsolid), rq = std::sqrt(sq / (double)h->nsolid);
  const double inf = std::numeric_limits<double>::infinity();
  h->eps_T = (mT > 0.0) ? rT / mT : (rT == 0.0 ? 0.0 : inf);
  h->eps_q = (mq > 0.0) ? rq / mq : (rq == 0.0 ? 0.0 : inf);
  h->out_prev.swap(h->out_next);
  h->iters += 1;
}

}  // namespace

extern "C" {

int bte_ref_create(const bte_ref_problem *p, bte_ref_solver **out) {
  if (!p || !out) return 1;
  if (p->nx < 1 || p->ny < 1 || p->nz < 1 || p->dim < 1 || p->dim > 3) return 1;
  if (p->dim < 3 && p->nz != 1) return 1;
  if (p->dim < 2 && p->ny != 1) return 1;
  if (p->n_bands < 1 || p->n_dirs < 1 || !p->C || !p->v || !p->tau || !p->s || !p->w) return 1;
  if (!(p->dx > 0) || (p->dim > 1 && !(p->dy > 0)) || (p->dim > 2 && !(p->dz > 0))) return 1;
  for (int b = 0; b < p->n_bands; ++b)
    if (!(p->C[b] > 0) || !(p->v[b] > 0) || !(p->tau[b] > 0)) return 1;
  auto *h = new bte_ref_solver();
  h->nx = p->nx; h->ny = p->ny; h->nz = p->nz; h->dim = p->dim;
  h->delta[0] = p->dx; h->delta[1] = p->dy; h->delta[2] = p->dz;
  h->ncell = (int64_t)p->nx * p->ny * p->nz;
  h->B = p->n_bands; h->D = p->n_dirs;
  h->C.assign(p->C, p->C + h->B); h->v.assign(p->v, p->v + h->B); h->tau.assign(p->tau, p->tau + h->B);
  h->s.assign(p->s, p->s + 3 * (size_t)h->D); h->w.assign(p->w, p->w + h->D);
  h->solid.assign((size_t)h->ncell, 1);
  if (p->solid_mask) for (int64_t i = 0; i < h->ncell; ++i) h->solid[i] = p->solid_mask[i] ? 1 : 0;
  h->nsolid = 0;
  for (int64_t i = 0; i < h->ncell; ++i) h->nsolid += h->solid[i];
  if (h->nsolid == 0) { delete h; return 1; }
  h->Q.assign((size_t)h->ncell, 0.0);
  if (p->Q) std::copy(p->Q, p->Q + h->ncell, h->Q.begin());
  for (int f = 0; f < 6; ++f) h->face_bc[f] = p->face_bc[f];
  h->interface_bc = p->interface_bc;
  h->diag = p->diagnostics != 0;
  h->literal_pi = p->literal_one_over_pi != 0;
  // quadrature checks (SURVEY.md 8(b) error behaviour)
  double sw = 0, swx[3] = {0, 0, 0};
  for (int d = 0; d < h->D; ++d) {
    const double *sd = &h->s[3 * (size_t)d];
    const double n2 = sd[0] * sd[0] + sd[1] * sd[1] + sd[2] * sd[2];
    if (std::fabs(n2 - 1.0) > 1e-9) { delete h; return 1; }
    sw += h->w[d];
    for (int a = 0; a < 3; ++a) swx[a] += h->w[d] * sd[a];
  }
  if (std::fabs(sw - FOUR_PI) > 1e-6 * FOUR_PI) { delete h; return 2; }
  // periodic pairs / interface type
  for (int a = 0; a < 3; ++a) {
    const bool pm = h->face_bc[2 * a].type == BTE_REF_PERIODIC, pp = h->face_bc[2 * a + 1].type == BTE_REF_PERIODIC;
    if (a < h->dim && pm != pp) { delete h; return 1; }
  }
  if (h->interface_bc.type == BTE_REF_PERIODIC) { delete h; return 1; }
  for (int f = 0; f < 2 * h->dim; ++f)
    if (h->face_bc[f].type < 0 || h->face_bc[f].type > 3) { delete h; return 1; }
  h->sumC = 0; h->sumCtau = 0;
  for (int b = 0; b < h->B; ++b) { h->sumC += h->C[b]; h->sumCtau += h->C[b] / h->tau[b]; }
  for (int a = 0; a < 3; ++a)
    for (int side = 0; side < 2; ++side) {
      const double nsign = side ? +1.0 : -1.0;
      double P = 0;
      for (int d = 0; d < h->D; ++d) {
        const double sn = nsign * h->s[3 * (size_t)d + a];
        if (sn < 0) P += h->w[d] * (-sn);
      }
      h->Pi_face[2 * a + side] = P;
    }
  // reflection maps R_a(d): flip component a
  bool need_reflect[3] = {false, false, false};
  for (int a = 0; a < h->dim; ++a) {
    if (h->face_bc[2 * a].type == BTE_REF_SPECULAR || h->face_bc[2 * a + 1].type == BTE_REF_SPECULAR) need_reflect[a] = true;
    if (h->interface_bc.type == BTE_REF_SPECULAR && p->solid_mask) need_reflect[a] = true;
  }
  for (int a = 0; a < 3; ++a) {
    h->reflect[a].assign(h->D, -1);
    for (int d = 0; d < h->D; ++d) {
      double t[3] = {h->s[3 * (size_t)d], h->s[3 * (size_t)d + 1], h->s[3 * (size_t)d + 2]};
      t[a] = -t[a];
      for (int g = 0; g < h->D; ++g) {
        const double *sg = &h->s[3 * (size_t)g];
        if (std::fabs(sg[0] - t[0]) < 1e-12 && std::fabs(sg[1] - t[1]) < 1e-12 && std::fabs(sg[2] - t[2]) < 1e-12 &&
            std::fabs(h->w[g] - h->w[d]) < 1e-12 * FOUR_PI) { h->reflect[a][d] = g; break; }
      }
      if (need_reflect[a] && h->reflect[a][d] < 0) { delete h; return 2; }
    }
  }
  if ((need_reflect[0] || need_reflect[1] || need_reflect[2]) &&
      std::sqrt(swx[0] * swx[0] + swx[1] * swx[1] + swx[2] * swx[2]) > 1e-9 * FOUR_PI) { delete h; return 2; }
  // enumerate boundary faces (outer box + solid/void)
  const int64_t N = h->ncell;
  const int n[3] = {h->nx, h->ny, h->nz};
  h->face_of.assign((size_t)6 * N, -1);
  std::vector<int64_t> wrapped_cell;  // for periodic faces: the cell whose outflow enters
  for (int k = 0; k < h->nz; ++k) for (int j = 0; j < h->ny; ++j) for (int i = 0; i < h->nx; ++i) {
    const int64_t id = cidx(h, i, j, k);
    if (!h->solid[id]) continue;
    const int ijk[3] = {i, j, k};
    for (int a = 0; a < h->dim; ++a) for (int side = 0; side < 2; ++side) {
      int u[3] = {i, j, k};
      u[a] = ijk[a] + (side ? +1 : -1);
      bte_ref_bc bc; bool boundary = false; int64_t wc = -1;
      if (u[a] < 0 || u[a] >= n[a]) {
        boundary = true;
        bc = h->face_bc[2 * a + side];
        if (bc.type == BTE_REF_PERIODIC) {
          u[a] = (u[a] + n[a]) % n[a];
          const int64_t uid = cidx(h, u[0], u[1], u[2]);
          if (h->solid[uid]) wc = uid; else bc = h->interface_bc;
        }
      } else if (!h->solid[cidx(h, u[0], u[1], u[2])]) {
        boundary = true;
        bc = h->interface_bc;
      }
      if (!boundary) continue;
      Face F; F.cell = id; F.axis = a; F.side = side; F.type = bc.type; F.dTw = bc.dT_wall; F.partner = -1;
      F.slot = (bc.type == BTE_REF_ISOTHERMAL) ? -1 : h->nslots++;
      h->face_of[(size_t)(2 * a + side) * N + id] = (int64_t)h->faces.size();
      h->faces.push_back(F);
      wrapped_cell.push_back(wc);
    }
  }
  for (size_t f = 0; f < h->faces.size(); ++f) {
    Face &F = h->faces[f];
    if (F.type != BTE_REF_PERIODIC) continue;
    // inflow through (cell, axis, side) = outflow of the wrapped cell through its opposite side
    F.partner = h->face_of[(size_t)(2 * F.axis + (1 - F.side)) * N + wrapped_cell[f]];
    if (F.partner < 0) { delete h; return 1; }
  }
  h->out_prev.assign((size_t)h->nslots * h->B * h->D, 0.0);  // store^0 = 0 (e^0 = C dT^0/4pi = 0)
  h->out_next.assign((size_t)h->nslots * h->B * h->D, 0.0);
  h->Gdiff.assign(h->faces.size() * (size_t)h->B, 0.0);
  h->dT.assign((size_t)N, 0.0); h->q.assign((size_t)3 * N, 0.0); h->qmag.assign((size_t)N, 0.0);
  if (h->diag) {
    h->intensity.assign((size_t)h->B * h->D * N, 0.0);
    h->fflux.assign((size_t)h->B * 6 * N, 0.0);
  }
  *out = h;
  return 0;
}

void bte_ref_destroy(bte_ref_solver *h) { delete h; }
void bte_ref_set_threads(bte_ref_solver *h, int32_t n) { if (h) h->threads = n < 1 ? 1 : n; }

int bte_ref_set_dir_order(bte_ref_solver *h, const int32_t *perm) {
  if (!h) return 1;
  h->dir_order.clear();
  if (!perm) return 0;
  std::vector<int> seen(h->D, 0);
  for (int d = 0; d < h->D; ++d) { if (perm[d] < 0 || perm[d] >= h->D || seen[perm[d]]++) return 1; }
  h->dir_order.assign(perm, perm + h->D);
  return 0;
}

int bte_ref_iterate(bte_ref_solver *h, int32_t n) {
  if (!h || n < 0) return 1;
  for (int i = 0; i < n; ++i) one_iteration(h);
  return 0;
}

int bte_ref_get_temperature(const bte_ref_solver *h, double *out) {
  if (!h || !out) return 1;
  std::copy(h->dT.begin(), h->dT.end(), out);
  return 0;
}
int bte_ref_get_heat_flux(const bte_ref_solver *h, double *out) {
  if (!h || !out) return 1;
  std::copy(h->q.begin(), h->q.end(), out);
  return 0;
}
int bte_ref_residual(const bte_ref_solver *h, double *eT, double *eq) {
  if (!h) return 1;
  if (eT) *eT = h->eps_T;
  if (eq) *eq = h->eps_q;
  return 0;
}
int64_t bte_ref_updates_per_sweep(const bte_ref_solver *h) { return h ? h->nsolid * h->B * h->D : 0; }
int64_t bte_ref_iterations_done(const bte_ref_solver *h) { return h ? h->iters : 0; }
int bte_ref_set_temperature(bte_ref_solver *h, const double *dT) {
  if (!h || !dT) return 1;
  for (int64_t i = 0; i < h->ncell; ++i) h->dT[i] = h->solid[i] ? dT[i] : 0.0;
  return 0;
}
int bte_ref_get_intensity(const bte_ref_solver *h, double *out) {
  if (!h || !out || !h->diag) return 1;
  std::copy(h->intensity.begin(), h->intensity.end(), out);
  return 0;
}
int bte_ref_face_flux_band(const bte_ref_solver *h, double *out) {
  if (!h || !out || !h->diag) return 1;
  std::copy(h->fflux.begin(), h->fflux.end(), out);
  return 0;
}
int bte_ref_face_flux(const bte_ref_solver *h, double *out) {
  if (!h || !out || !h->diag) return 1;
  const size_t n6 = (size_t)6 * h->ncell;
  std::fill(out, out + n6, 0.0);
  for (int b = 0; b < h->B; ++b)
    for (size_t i = 0; i < n6; ++i) out[i] += h->fflux[(size_t)b * n6 + i];
  return 0;
}
int bte_ref_boundary_power(const bte_ref_solver *h, double *out) {
  if (!h || !out || !h->diag) return 1;
  for (int t = 0; t < 4; ++t) out[t] = 0.0;
  const int64_t N = h->ncell;
  const double area[3] = {(h->dim > 1 ? h->delta[1] : 1.0) * (h->dim > 2 ? h->delta[2] : 1.0),
                          h->delta[0] * (h->dim > 2 ? h->delta[2] : 1.0),
                          h->delta[0] * (h->dim > 1 ? h->delta[1] : 1.0)};
  for (const Face &F : h->faces) {
    double fl = 0.0;
    for (int b = 0; b < h->B; ++b) fl += h->fflux[((size_t)b * 6 + 2 * F.axis + F.side) * N + F.cell];
    out[F.type] += fl * area[F.axis];
  }
  return 0;
}
double bte_ref_pi_face(const bte_ref_solver *h, int32_t face) {
  return (h && face >= 0 && face < 6) ? h->Pi_face[face] : 0.0;
}

}  // extern "C"
