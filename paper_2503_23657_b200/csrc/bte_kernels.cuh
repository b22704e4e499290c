// Device code of the B200 phonon-BTE sweep library (included once by bte_api.cu).
//
// Kernels:
//   bte_gdiff_kernel   diffuse-wall hemispherical sums H/Pi of the previous sweep (Eq. 6)
//   bte_ghost_kernel   fills the inflow ("ghost") face planes of every octant from the lagged
//                      outflow planes according to the BC type (Eq. 5-7 + periodic)
//   bte_sweep_kernel   (a)+(b): persistent, ticket-scheduled tile dataflow; each CTA sweeps an
//                      x-pencil tile for the <=16 directions of one (octant, band) item with a
//                      lane-skewed wavefront; intensity lives in registers / shared memory only;
//                      0th/1st moments are accumulated in the same loop
//   bte_update_kernel  (c): sums octant partials -> dT, q, residual partials, re-skews dT
//   bte_final_kernel   final fixed-order reduction of the residual partials
#pragma once
#include <cuda_runtime.h>

#include "bte_internal.h"

__constant__ __align__(16) unsigned char c_coef[BTE_CONST_BYTES];

// ------------------------------------------------------------------ layouts
// skewed cell index of class cls (bit0: x flipped, bit1: y flipped), physical k
__device__ __forceinline__ int64_t sk_index(const BteDev &P, int cls, int i, int j, int k) {
  const int ip = (cls & 1) ? P.nx - 1 - i : i;
  const int jp = (cls & 2) ? P.ny - 1 - j : j;
  const int ty = jp >> 5, J = jp & 31;
  return (((int64_t)k * P.nty + ty) * P.NU + (ip + J)) * 32 + J;
}
// face planes of one octant (oriented coordinates i', j', k'); `n` = items of that octant
__device__ __forceinline__ int64_t xpl_index(const BteDev &P, int n, int side, int item, int p, int kp, int jp) {
  return ((((int64_t)side * n + item) * BTE_P + p) * P.nz + kp) * P.nyp + jp;
}
__device__ __forceinline__ int64_t ypl_index(const BteDev &P, int n, int ty, int item, int kp, int ip, int p) {
  return ((((int64_t)ty * n + item) * P.nz + kp) * P.nx + ip) * BTE_P + p;
}
__device__ __forceinline__ int64_t zpl_index(const BteDev &P, int n, int tz, int item, int ty, int u, int p, int J) {
  return (((((int64_t)tz * n + item) * P.nty + ty) * P.NU + u) * BTE_P + p) * 32 + J;
}

template <typename T> __device__ __forceinline__ T ld_cg(const T *p) { return __ldcg(p); }

__device__ __forceinline__ int ld_acquire(const int *p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release(int *p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}

// ------------------------------------------------------------------ sweep
// One CTA = TZ warps x 32 lanes. Thread (J = lane, K = warp) owns the x-row (j' = 32 ty + J,
// k' = TZ tz + K) of its tile and marches i' = t - J - K (lane/warp-skewed wavefront):
//   x-upwind : its own register (carry[p])
//   y-upwind : lane J-1's carry via __shfl_up (lane 0: inflow y-plane staged in shared memory)
//   z-upwind : warp K-1's values of the previous step via shared memory (warp 0: inflow z-plane)
// so the (band x direction) intensity never goes to HBM; only tile faces do (L2-resident hand-off
// to the downstream tile, or the lagged boundary store at box faces).
template <typename T>
__global__ void __launch_bounds__(BTE_MAX_TZ * 32) bte_sweep_kernel(const __grid_constant__ BteDev P) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int TZ = P.TZ;
  T *zbuf = reinterpret_cast<T *>(smem_raw);                   // [2][TZ+1][16][32]
  T *ybuf = zbuf + 2 * (TZ + 1) * BTE_P * 32;                  // [2][TZ][16]
  __shared__ int s_unit;
  const int tid = threadIdx.x, J = tid & 31, K = tid >> 5, nthr = blockDim.x;
  const unsigned FULL = 0xffffffffu;

  for (;;) {
    if (tid == 0) {
      const int tk = atomicAdd(P.ticket, 1);
      s_unit = tk;
      if (tk < P.n_units) {
        const BteUnit *U = P.units + tk;
        const int d0 = U->dep_y, d1 = U->dep_z, d2 = U->dep_prev;
        if (d0 >= 0) while (ld_acquire(P.done + d0) != P.epoch) __nanosleep(64);
        if (d1 >= 0) while (ld_acquire(P.done + d1) != P.epoch) __nanosleep(64);
        if (d2 >= 0) while (ld_acquire(P.done + d2) != P.epoch) __nanosleep(64);
      }
    }
    __syncthreads();
    const int unit = s_unit;
    if (unit >= P.n_units) break;
    const BteUnit un = P.units[unit];
    const BteOct &O = P.oct[un.oct];
    const int item = un.item, ty = un.ty, tz = un.tz, b = un.band, nit = O.nitems;
    const T *ck = reinterpret_cast<const T *>(c_coef) + un.coef_off;
    const int jp = ty * 32 + J, kp = tz * TZ + K;
    const bool rowvalid = (jp < P.ny) && (kp < P.nz);
    const int j = rowvalid ? (O.sy > 0 ? jp : P.ny - 1 - jp) : 0;
    const int k = rowvalid ? (O.sz > 0 ? kp : P.nz - 1 - kp) : 0;
    const int jlast = min(P.ny, (ty + 1) * 32) - 1 - ty * 32;
    const int klast = min(P.nz, (tz + 1) * TZ) - 1 - tz * TZ;
    const int64_t rowbase = (((int64_t)k * P.nty + ty) * P.NU) * 32 + J;
    const T *dTs = reinterpret_cast<const T *>(P.dT_sk[O.cls]);
    const T *Qs = reinterpret_cast<const T *>(P.Q_sk[O.cls]);
    const uint8_t *cds = P.code_sk[O.cls];
    T *xpl = reinterpret_cast<T *>(O.xpl);
    T *ypl = reinterpret_cast<T *>(O.ypl);
    T *zpl = reinterpret_cast<T *>(O.zpl);
    double *M = O.M;
    const T cb = (T)P.band[b], tb = (T)P.band[P.B + b];
    const double invtau = P.band[2 * P.B + b], vb = P.band[3 * P.B + b];
    const double qsx = vb * O.sx, qsy = vb * O.sy, qsz = vb * O.sz;
    // face codes of the upwind / downwind sides of this octant
    const int fux = O.sx > 0 ? 0 : 1, fuy = O.sy > 0 ? 2 : 3, fuz = O.sz > 0 ? 4 : 5;
    const int upmask = (2 << fux) | (P.has_y ? (2 << fuy) : 0) | (P.has_z ? (2 << fuz) : 0);
    const int dnmask = (2 << (fux ^ 1)) | (P.has_y ? (2 << (fuy ^ 1)) : 0) | (P.has_z ? (2 << (fuz ^ 1)) : 0);

    T carry[BTE_P];
#pragma unroll
    for (int p = 0; p < BTE_P; ++p)
      carry[p] = rowvalid ? ld_cg(xpl + xpl_index(P, nit, 0, item, p, kp, jp)) : (T)0;

    const int nsteps = P.nx + 31 + TZ - 1;
    // ---- prologue: stage inflow planes for step 0 into parity 0, prefetch cell inputs of step 0
    const int zper = (BTE_P * 32) / nthr;  // z-plane elements per thread per step (1 or 2) when has_z
    T zpf[2] = {(T)0, (T)0};
    T ypf = (T)0;
    if (P.has_z) {
      for (int e = 0; e < zper; ++e) {
        const int el = tid + e * nthr;
        zbuf[el] = ld_cg(zpl + zpl_index(P, nit, tz, item, ty, 0, el >> 5, el & 31));
      }
    }
    if (P.has_y && J < BTE_P) {
      const int ip0 = 0 - K;
      ybuf[K * BTE_P + J] = (kp < P.nz && ip0 >= 0 && ip0 < P.nx)
                                ? ld_cg(ypl + ypl_index(P, nit, ty, item, kp, ip0, J)) : (T)0;
    }
    int code_n = 0;
    T dT_n = (T)0, Q_n = (T)0;
    {
      const int ip = 0 - J - K;
      if (rowvalid && ip >= 0 && ip < P.nx) {
        const int64_t idx = rowbase + (int64_t)(0 - K) * 32;
        code_n = cds[idx]; dT_n = dTs[idx]; Q_n = Qs[idx];
      }
    }
    __syncthreads();

    for (int t = 0; t < nsteps; ++t) {
      const int cur = t & 1, nxt = cur ^ 1;
      const int ip = t - J - K;
      const bool act = rowvalid && ip >= 0 && ip < P.nx;
      const int code = code_n;
      const T dTv = dT_n, Qv = Q_n;
      const int64_t idx = rowbase + (int64_t)(t - K) * 32;
      // ---- prefetch for step t+1
      {
        const int ipn = ip + 1;
        code_n = 0;
        if (rowvalid && ipn >= 0 && ipn < P.nx) {
          code_n = cds[idx + 32]; dT_n = dTs[idx + 32]; Q_n = Qs[idx + 32];
        }
        if (P.has_z && t + 1 < P.NU) {
#pragma unroll
          for (int e = 0; e < 2; ++e)
            if (e < zper) {
              const int el = tid + e * nthr;
              zpf[e] = ld_cg(zpl + zpl_index(P, nit, tz, item, ty, t + 1, el >> 5, el & 31));
            }
        }
        if (P.has_y && J < BTE_P) {
          const int ipy = t + 1 - K;
          ypf = (kp < P.nz && ipy >= 0 && ipy < P.nx) ? ld_cg(ypl + ypl_index(P, nit, ty, item, kp, ipy, J)) : (T)0;
        }
      }
      const bool solid = act && (code & BTE_CODE_SOLID);
      double mold0 = 0, mold1 = 0, mold2 = 0, mold3 = 0;
      if (solid && item > 0) {
        mold0 = ld_cg(M + idx); mold1 = ld_cg(M + P.NS + idx);
        mold2 = ld_cg(M + 2 * P.NS + idx); mold3 = ld_cg(M + 3 * P.NS + idx);
      }
      // ---- interface (solid/void) inflow: rare path
      const bool ux = solid && (code & (2 << fux)), uy = solid && P.has_y && (code & (2 << fuy)),
                 uz = solid && P.has_z && (code & (2 << fuz));
      T gx = (T)0, gy = (T)0, gz = (T)0;
      int64_t cphys = 0;
      if (solid && (code & (upmask | dnmask))) {
        const int i = O.sx > 0 ? ip : P.nx - 1 - ip;
        cphys = (int64_t)i + (int64_t)P.nx * (j + (int64_t)P.ny * k);
        const T *Gi = reinterpret_cast<const T *>(P.Gi);
        if (ux) gx = Gi[(int64_t)P.iface[(int64_t)fux * P.ncell + cphys] * P.B + b];
        if (uy) gy = Gi[(int64_t)P.iface[(int64_t)fuy * P.ncell + cphys] * P.B + b];
        if (uz) gz = Gi[(int64_t)P.iface[(int64_t)fuz * P.ncell + cphys] * P.B + b];
      }
      const T r = cb * dTv + tb * Qv;
      T m0 = (T)0, m1 = (T)0, m2 = (T)0, m3 = (T)0;
      const T *zin = zbuf + (cur * (TZ + 1) + K) * (BTE_P * 32) + J;
      T *zout = zbuf + (nxt * (TZ + 1) + K + 1) * (BTE_P * 32) + J;
      const T *yin = ybuf + (cur * TZ + K) * BTE_P;
#pragma unroll
      for (int p = 0; p < BTE_P; ++p) {
        T ex = carry[p];
        T ey = __shfl_up_sync(FULL, ex, 1);
        if (J == 0) ey = yin[p];
        T ez = P.has_z ? zin[p * 32] : (T)0;
        if (!P.has_y) ey = (T)0;
        if (ux) ex = gx;
        if (uy) ey = gy;
        if (uz) ez = gz;
        T e = r * ck[p * BTE_NCOEF + 0];
        e = fma(ck[p * BTE_NCOEF + 1], ex, e);
        e = fma(ck[p * BTE_NCOEF + 2], ey, e);
        e = fma(ck[p * BTE_NCOEF + 3], ez, e);
        e = solid ? e : (T)0;
        if (act) carry[p] = e;
        m0 = fma(ck[p * BTE_NCOEF + 4], e, m0);
        m1 = fma(ck[p * BTE_NCOEF + 5], e, m1);
        m2 = fma(ck[p * BTE_NCOEF + 6], e, m2);
        m3 = fma(ck[p * BTE_NCOEF + 7], e, m3);
        if (P.has_z) zout[p * 32] = carry[p];
      }
      if (solid) {   // (b): moments of this item into the octant partial (plain RMW: one owner)
        M[idx] = mold0 + invtau * (double)m0;
        M[P.NS + idx] = mold1 + qsx * (double)m1;
        M[2 * P.NS + idx] = mold2 + qsy * (double)m2;
        M[3 * P.NS + idx] = mold3 + qsz * (double)m3;
      }
      // ---- outflow faces (tile hand-off / lagged boundary store)
      if (act) {
        if (P.has_y && J == jlast) {
          T *dst = ypl + ypl_index(P, nit, ty + 1, item, kp, ip, 0);
#pragma unroll
          for (int p = 0; p < BTE_P; ++p) dst[p] = carry[p];
        }
        if (P.has_z && K == klast) {
#pragma unroll
          for (int p = 0; p < BTE_P; ++p) zpl[zpl_index(P, nit, tz + 1, item, ty, t - K, p, J)] = carry[p];
        }
        if (ip == P.nx - 1) {
#pragma unroll
          for (int p = 0; p < BTE_P; ++p) xpl[xpl_index(P, nit, 1, item, p, kp, jp)] = carry[p];
        }
        // outgoing hemispherical partial sums at solid/void faces (diffuse interface, Eq. 6)
        if (solid && (code & dnmask)) {
          const int slot_base = un.chunk * 4;
          for (int a = 0; a < P.dim; ++a) {
            const int fd = 2 * a + ((a == 0 ? O.sx : (a == 1 ? O.sy : O.sz)) > 0 ? 1 : 0);
            if (!(code & (2 << fd))) continue;
            double h = 0.0;
#pragma unroll
            for (int p = 0; p < BTE_P; ++p) h += (double)ck[p * BTE_NCOEF + 5 + a] * (double)carry[p];
            // slot: the two sign bits of the other axes
            const int bx = O.sx < 0, by = O.sy < 0, bz = O.sz < 0;
            const int s2 = (a == 0) ? (by | (bz << 1)) : (a == 1 ? (bx | (bz << 1)) : (bx | (by << 1)));
            const int64_t fid = P.iface[(int64_t)fd * P.ncell + cphys];
            P.Hpart[(fid * P.B + b) * P.nHslot + slot_base + s2] = h;
          }
        }
      }
      // ---- stage the inflow planes of step t+1
      if (P.has_z) {
#pragma unroll
        for (int e = 0; e < 2; ++e)
          if (e < zper) zbuf[nxt * (TZ + 1) * (BTE_P * 32) + tid + e * nthr] = zpf[e];
      }
      if (P.has_y && J < BTE_P) ybuf[(nxt * TZ + K) * BTE_P + J] = ypf;
      __syncthreads();
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) st_release(P.done + unit, P.epoch);
  }
}

// ------------------------------------------------------------------ boundary kernels
// Coordinates of face f (0..5 = x-,x+,y-,y+,z-,z+): transverse physical cell (ta, tb):
//   x faces: (j,k);  y faces: (i,k);  z faces: (i,j).  G layout: Gf[f][b][tb][ta].
struct BteFaceGeom { int na, nb; };
__device__ __forceinline__ BteFaceGeom face_geom(const BteDev &P, int f) {
  BteFaceGeom g;
  if (f < 2) { g.na = P.ny; g.nb = P.nz; }
  else if (f < 4) { g.na = P.nx; g.nb = P.nz; }
  else { g.na = P.nx; g.nb = P.ny; }
  return g;
}

// value of octant o's OUTFLOW plane on axis a at physical boundary cell (i,j,k), item, slot p
template <typename T>
__device__ __forceinline__ T outflow_value(const BteDev &P, int o, int a, int item, int p, int i, int j, int k) {
  const BteOct &O = P.oct[o];
  const int ip = O.sx > 0 ? i : P.nx - 1 - i, jp = O.sy > 0 ? j : P.ny - 1 - j, kp = O.sz > 0 ? k : P.nz - 1 - k;
  if (a == 0) return ld_cg(reinterpret_cast<const T *>(O.xpl) + xpl_index(P, O.nitems, 1, item, p, kp, jp));
  if (a == 1) return ld_cg(reinterpret_cast<const T *>(O.ypl) + ypl_index(P, O.nitems, P.nty, item, kp, ip, p));
  return ld_cg(reinterpret_cast<const T *>(O.zpl) +
               zpl_index(P, O.nitems, P.ntz, item, jp >> 5, ip + (jp & 31), p, jp & 31));
}

// G_{f,b}(cell) = (1/Pi_f) sum_{s.n>0} w (s.n) e^n   for DIFFUSE box faces (Eq. 6, reading G10)
template <typename T>
__global__ void bte_gdiff_kernel(const __grid_constant__ BteDev P) {
  T *Gf = reinterpret_cast<T *>(P.Gf);
  const T *ckall = reinterpret_cast<const T *>(c_coef);
  int64_t base = 0;
  for (int f = 0; f < 2 * P.dim; ++f) {
    const BteFaceGeom g = face_geom(P, f);
    const int64_t nf = (int64_t)g.na * g.nb * P.B;
    if (P.face_type[f] == 1) {
      const int a = f >> 1, side = f & 1;
      for (int64_t e = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; e < nf; e += (int64_t)gridDim.x * blockDim.x) {
        const int ta = (int)(e % g.na), tb = (int)((e / g.na) % g.nb), b = (int)(e / ((int64_t)g.na * g.nb));
        int i, j, k;
        if (a == 0) { i = side ? P.nx - 1 : 0; j = ta; k = tb; }
        else if (a == 1) { j = side ? P.ny - 1 : 0; i = ta; k = tb; }
        else { k = side ? P.nz - 1 : 0; i = ta; j = tb; }
        double H = 0.0;
        for (int o = 0; o < 8; ++o) {
          const BteOct &O = P.oct[o];
          if (!O.active) continue;
          const int sg = a == 0 ? O.sx : (a == 1 ? O.sy : O.sz);
          if ((sg > 0) != (side == 1)) continue;  // outgoing octants only
          for (int c = 0; c < O.nchunk; ++c) {
            const int item = b * O.nchunk + c;
            const T *ck = ckall + P.item_coef[o * P.max_items + item];
            for (int p = 0; p < BTE_P; ++p)
              H += (double)ck[p * BTE_NCOEF + 5 + a] * (double)outflow_value<T>(P, o, a, item, p, i, j, k);
          }
        }
        Gf[base + e] = (T)(H / P.Pi_face[f]);
      }
    }
    base += nf;
  }
}

// Fill the inflow (ghost) plane of every active octant on every active axis, and the interface
// inflow table Gi, from the lagged outflow of the previous iteration.
template <typename T>
__global__ void bte_ghost_kernel(const __grid_constant__ BteDev P) {
  const T *Gf = reinterpret_cast<const T *>(P.Gf);
  const int64_t gtid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x, gstride = (int64_t)gridDim.x * blockDim.x;
  int64_t gbase[6];
  {
    int64_t acc = 0;
    for (int f = 0; f < 6; ++f) {
      gbase[f] = acc;
      if (f < 2 * P.dim) { const BteFaceGeom g = face_geom(P, f); acc += (int64_t)g.na * g.nb * P.B; }
    }
  }
  for (int o = 0; o < 8; ++o) {
    const BteOct &O = P.oct[o];
    if (!O.active) continue;
    for (int a = 0; a < P.dim; ++a) {
      const int sg = a == 0 ? O.sx : (a == 1 ? O.sy : O.sz);
      const int f = 2 * a + (sg > 0 ? 0 : 1);     // physical face the octant enters through
      const int type = P.face_type[f];
      const BteFaceGeom g = face_geom(P, f);
      const int64_t n = (int64_t)g.na * g.nb * O.nitems * BTE_P;
      for (int64_t e = gtid; e < n; e += gstride) {
        // x faces iterate (j fastest), others (p fastest) to follow the plane layouts
        int ta, tb, item, p;
        if (a == 0) {
          ta = (int)(e % g.na); tb = (int)((e / g.na) % g.nb);
          p = (int)((e / ((int64_t)g.na * g.nb)) % BTE_P); item = (int)(e / ((int64_t)g.na * g.nb * BTE_P));
        } else {
          p = (int)(e % BTE_P); ta = (int)((e / BTE_P) % g.na); tb = (int)((e / ((int64_t)BTE_P * g.na)) % g.nb);
          item = (int)(e / ((int64_t)BTE_P * g.na * g.nb));
        }
        int i, j, k;
        if (a == 0) { i = (f & 1) ? P.nx - 1 : 0; j = ta; k = tb; }
        else if (a == 1) { j = (f & 1) ? P.ny - 1 : 0; i = ta; k = tb; }
        else { k = (f & 1) ? P.nz - 1 : 0; i = ta; j = tb; }
        const int b = item / O.nchunk;
        T val;
        if (type == 0) val = (T)(P.band[b] * P.face_dT[f]);                       // Eq. 5
        else if (type == 1) val = Gf[gbase[f] + ((int64_t)b * g.nb + tb) * g.na + ta];  // Eq. 6
        else if (type == 2) val = outflow_value<T>(P, o ^ (1 << a), a, item, p, i, j, k);  // Eq. 7
        else {                                                                    // periodic
          int i2 = i, j2 = j, k2 = k;
          if (a == 0) i2 = P.nx - 1 - i; else if (a == 1) j2 = P.ny - 1 - j; else k2 = P.nz - 1 - k;
          val = outflow_value<T>(P, o, a, item, p, i2, j2, k2);
        }
        const int ip = O.sx > 0 ? i : P.nx - 1 - i, jp = O.sy > 0 ? j : P.ny - 1 - j, kp = O.sz > 0 ? k : P.nz - 1 - k;
        if (a == 0) reinterpret_cast<T *>(O.xpl)[xpl_index(P, O.nitems, 0, item, p, kp, jp)] = val;
        else if (a == 1) reinterpret_cast<T *>(O.ypl)[ypl_index(P, O.nitems, 0, item, kp, ip, p)] = val;
        else reinterpret_cast<T *>(O.zpl)[zpl_index(P, O.nitems, 0, item, jp >> 5, ip + (jp & 31), p, jp & 31)] = val;
      }
    }
  }
  // interface faces
  T *Gi = reinterpret_cast<T *>(P.Gi);
  const int64_t ni = (int64_t)P.n_iface * P.B;
  for (int64_t e = gtid; e < ni; e += gstride) {
    const int64_t fid = e / P.B;
    const int b = (int)(e % P.B);
    if (P.iface_type == 0) { Gi[e] = (T)(P.band[b] * P.iface_dT); continue; }
    double H = 0.0;
    for (int s = 0; s < P.nHslot; ++s) H += P.Hpart[e * P.nHslot + s];
    Gi[e] = (T)(H / P.Pi_face[P.iface_info[fid]]);
  }
  if (gtid == 0) *P.ticket = 0;
}

// ------------------------------------------------------------------ (c) update + residual
__device__ __forceinline__ void block_reduce4(double &a, double &b, double &c, double &d) {
  // a, c: sums; b, d: maxima.  Fixed-order tree -> deterministic.
  __shared__ double sh[4][32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  for (int off = 16; off > 0; off >>= 1) {
    a += __shfl_down_sync(0xffffffffu, a, off);
    c += __shfl_down_sync(0xffffffffu, c, off);
    b = fmax(b, __shfl_down_sync(0xffffffffu, b, off));
    d = fmax(d, __shfl_down_sync(0xffffffffu, d, off));
  }
  if (lane == 0) { sh[0][w] = a; sh[1][w] = b; sh[2][w] = c; sh[3][w] = d; }
  __syncthreads();
  if (w == 0) {
    a = lane < nw ? sh[0][lane] : 0.0; b = lane < nw ? sh[1][lane] : 0.0;
    c = lane < nw ? sh[2][lane] : 0.0; d = lane < nw ? sh[3][lane] : 0.0;
    for (int off = 16; off > 0; off >>= 1) {
      a += __shfl_down_sync(0xffffffffu, a, off);
      c += __shfl_down_sync(0xffffffffu, c, off);
      b = fmax(b, __shfl_down_sync(0xffffffffu, b, off));
      d = fmax(d, __shfl_down_sync(0xffffffffu, d, off));
    }
  }
}

// dT^{n+1} = M0 / sum(C/tau) (Eq. 16), q = M1 (Eq. 4), residual partial sums (Eq. 23);
// re-skews dT into the four class layouts the next sweep reads.
template <typename T>
__global__ void __launch_bounds__(256) bte_update_kernel(const __grid_constant__ BteDev P) {
  double sT = 0, mT = 0, sq = 0, mq = 0;
  for (int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; c < P.ncell; c += (int64_t)gridDim.x * blockDim.x) {
    if (!(P.code[c] & BTE_CODE_SOLID)) continue;
    const int i = (int)(c % P.nx), j = (int)((c / P.nx) % P.ny), k = (int)(c / ((int64_t)P.nx * P.ny));
    int64_t sk[4];
#pragma unroll
    for (int cl = 0; cl < 4; ++cl) sk[cl] = sk_index(P, cl, i, j, k);
    double m0 = 0, m1 = 0, m2 = 0, m3 = 0;
#pragma unroll
    for (int o = 0; o < 8; ++o) {
      if (!P.oct[o].active) continue;
      const double *M = P.oct[o].M;
      const int64_t id = sk[o & 3];
      m0 += ld_cg(M + id); m1 += ld_cg(M + P.NS + id); m2 += ld_cg(M + 2 * P.NS + id); m3 += ld_cg(M + 3 * P.NS + id);
    }
    const double Tn = m0 * P.inv_sumCtau;
    const double dlt = Tn - P.dT[c];
    sT += dlt * dlt; mT = fmax(mT, fabs(Tn));
    P.dT[c] = Tn;
    P.q[c] = m1; P.q[P.ncell + c] = m2; P.q[2 * P.ncell + c] = m3;
    const double qm = sqrt(m1 * m1 + m2 * m2 + m3 * m3);
    const double dq = qm - P.qmag[c];
    sq += dq * dq; mq = fmax(mq, qm);
    P.qmag[c] = qm;
#pragma unroll
    for (int cl = 0; cl < 4; ++cl) reinterpret_cast<T *>(P.dT_sk[cl])[sk[cl]] = (T)Tn;
  }
  block_reduce4(sT, mT, sq, mq);
  if (threadIdx.x == 0) {
    P.red[blockIdx.x] = sT; P.red[P.n_red_blocks + blockIdx.x] = mT;
    P.red[2 * P.n_red_blocks + blockIdx.x] = sq; P.red[3 * P.n_red_blocks + blockIdx.x] = mq;
  }
}

__global__ void __launch_bounds__(256) bte_final_kernel(const __grid_constant__ BteDev P) {
  double sT = 0, mT = 0, sq = 0, mq = 0;
  for (int e = threadIdx.x; e < P.n_red_blocks; e += blockDim.x) {
    sT += P.red[e]; mT = fmax(mT, P.red[P.n_red_blocks + e]);
    sq += P.red[2 * P.n_red_blocks + e]; mq = fmax(mq, P.red[3 * P.n_red_blocks + e]);
  }
  block_reduce4(sT, mT, sq, mq);
  if (threadIdx.x == 0) {
    double *out = P.red + 4 * P.n_red_blocks;
    out[0] = sT; out[1] = mT; out[2] = sq; out[3] = mq;
  }
}

// ------------------------------------------------------------------ layout helpers
// physical fp64 field -> four skewed class copies (scaled); used for Q/sumC, dT and the cell codes
template <typename T>
__global__ void bte_skew_kernel(const __grid_constant__ BteDev P, const double *src, double scale, int which) {
  for (int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; c < P.ncell; c += (int64_t)gridDim.x * blockDim.x) {
    const int i = (int)(c % P.nx), j = (int)((c / P.nx) % P.ny), k = (int)(c / ((int64_t)P.nx * P.ny));
    const bool solid = P.code[c] & BTE_CODE_SOLID;
    for (int cl = 0; cl < 4; ++cl) {
      const int64_t id = sk_index(P, cl, i, j, k);
      if (which == 2) { P.code_sk[cl][id] = P.code[c]; continue; }
      const T v = solid ? (T)(src[c] * scale) : (T)0;
      if (which == 0) reinterpret_cast<T *>(P.Q_sk[cl])[id] = v;
      else reinterpret_cast<T *>(P.dT_sk[cl])[id] = v;
    }
    if (which == 1) { P.dT[c] = solid ? src[c] : 0.0; }
  }
}

#include "bte_sweep2.cuh"
