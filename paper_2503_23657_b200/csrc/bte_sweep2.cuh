// Fast path of the B200 phonon-BTE sweep: 3-D, even ny / nz, all-solid or voxel-masked, 16 directions per
// octant, mirror-symmetric quadrature, <= 16 bands.  DESIGN.md section 6.
//
// Mapping.  One CTA = W warps sweeps one tile = 64 (y') x 2W (z') rows along x' for one octant and
// one band group (NB = 1 or 2 bands x 16 directions).  Thread (J = lane, K = warp) owns the 2x2
// row patch j' = 64 ty + 2J + {0,1}, k' = 2W tz + 2K + {0,1} and marches i' = t - J - K
// (lane/warp-skewed wavefront), so that
//   x-upwind  = its own register (carry),
//   y-upwind  = its own patch row jj=0, or lane J-1's jj=1 row of the previous step (one SHFL),
//   z-upwind  = its own patch row kk=0, or warp K-1's kk=1 row of the previous step (16-byte
//               shared-memory exchange, double buffered),
// i.e. 64 NB updates per thread and step need 32 NB shuffles and 16 NB 16-byte LDS/STS.  The
// recurrence/moment coefficients are warp-uniform kernel parameters (constant bank -> uniform
// registers), so an update is 8 FMA-pipe instructions with two vector-register operands each.
// The (band x direction) intensity lives in registers only; tile faces go through L2-resident
// planes (hand-off to the downstream tile, or the lagged boundary store at box faces).
//
// Scheduling.  Persistent CTAs take tickets in a topological unit order.  Dependencies between
// tiles are tracked per STEP, not per tile: every unit publishes its step count (release store)
// every BTE2_PUB steps, and the downstream tile in y / z (and the previous band group on the same
// tile, which owns the moment accumulator before it) only has to stay 32 / W / 1 steps behind.
#pragma once
#include <cuda_runtime.h>

#include <type_traits>

#include "bte_internal.h"

#define BTE2_P 16         // directions per octant
#define BTE2_MAXB 16      // bands in the parameter table
#define BTE2_PUB 8        // progress is published every PUB steps
#define BTE2_DIST(W, T) (sizeof(T) == 4 ? 2 : 1)   // cp.async prefetch distance in steps (shared-memory budget; >= 1 + BTE2_MDIST)
#define BTE2_MDIST(T) (sizeof(T) == 4 ? 1 : 0)   // same for the moment accumulator (fp64: fetched in the step that adds to it)
#ifndef BTE2_SPLITBAR
#define BTE2_SPLITBAR 1   // 0: plain __syncthreads per step (config 4 sweep 5.23 ms instead of 4.89 ms)
#endif
#define BTE2_SLACK 0      // extra steps a unit lets the units it follows get ahead before it starts
// timing experiments only (-DBTE2_ENABLE_DBG + env BTE_V2_DBG): the product build compiles the switches out
#ifdef BTE2_ENABLE_DBG
#define BTE2_DBGBIT(P, bit) ((P).dbg & (bit))
#else
#define BTE2_DBGBIT(P, bit) 0
#endif

template <typename T> struct alignas(16) Bte2Coefs {   // kernel parameter (constant bank 0)
  T k[BTE2_MAXB][8][BTE2_P];   // [band][inv, ax, ay, az, w/tau, v w|sx|, v w|sy|, v w|sz|][direction]
  T bc[BTE2_MAXB][2];          // C/4pi, C tau/(4pi sumC)
};

struct Bte2Unit {
  int32_t oct, g, ty, tz;
  int32_t dep_y, dep_z, dep_prev;   // unit ids (same octant) or -1
  int32_t b0, nb;                   // first band, bands in this group (1 or 2)
  int32_t pad[3];
};

struct Bte2Oct {
  int32_t sx, sy, sz, cls;
  void *M;                  // T [NS][4]   moment accumulator of this octant (skewed class layout)
  void *xin, *xout;         // x face planes: inflow ghost plane; outflow, two buffers (iteration parity)
  void *ypl, *zpl;          // y / z face planes: slot 0 = inflow ghost plane, slots 1..n-1 = hand-off between tiles,
                            // slots n, n+1 = outflow of the last tile row (lagged boundary store), two buffers
  // set by the host for every iteration (epoch parity): where this octant's sweep reads its box-face inflow
  // (its ghost plane for isothermal / diffuse faces; for specular / periodic faces directly the outflow buffer
  // the mirrored / same octant wrote in the PREVIOUS iteration -- same layout, so no copy is needed) and which
  // outflow buffers it writes (dst) / the boundary kernels read (prev)
  const void *xsrc, *ysrc0, *zsrc0;
  void *xdst, *ydstN, *zdstN;
  const void *xprev, *yprev, *zprev;
};

struct Bte2Dev {
  int32_t nx, ny, nz, B;
  int32_t W, nty, ntz, NU;          // warps per CTA; tiles along y', z'; nx + 31
  int32_t nsteps, n_units, epoch, dbg;   // dbg: timing experiments only (BTE_V2_DBG), 0 in production
  int64_t NS;                       // nz * nty * NU * 64
  void *dTQ[4];                     // T2 [NS]: (dT, Q / sum C) per x/y-flip class
  Bte2Oct oct[8];
  const Bte2Unit *units;
  int32_t *prog;                    // [n_units] epoch << 16 | steps published
  int32_t *ticket;
  // boundary conditions (box faces x-,x+,y-,y+,z-,z+) and the update kernel
  int32_t face_type[6];
  double face_e0[6][BTE2_MAXB];     // isothermal inflow C_b dT_w / 4pi (Eq. 5)
  double Pi_face[6];                // discrete hemispherical normaliser (reading G10)
  double wsa[BTE2_P][3];            // w_p |s_p,a|
  void *Gf;                         // T diffuse inflow [f][b][tb][ta]
  int64_t gf_off[7];                // offsets of the 6 faces in Gf, [6] = total
  double *dT, *q, *qmag, *red;      // fp64 outputs in physical layout; residual partials
  int32_t n_red_blocks, pub_mask;   // progress is published when (t & pub_mask) == pub_mask
  int32_t slack, fill_iso;          // fill_iso: (re)write the constant isothermal ghost planes (first iteration only)
  // ghost planes to fill in this iteration: (octant, axis) segments and their offsets in one flat index space
  int32_t gseg_n, gseg_oa[24];
  int64_t gseg_off[25];
  int64_t ncell, src_mod;            // src_mod: cells of the caller's field (2-D problems run as two layers)
  double inv_sumCtau;
  // voxel masks (all null / 0 when every cell is solid).  Cell byte: bit0 solid, bit 1+f: the neighbour across
  // face f (x-,x+,y-,y+,z-,z+) is a solid/void interface (or a periodic wrap onto a void cell).
  const uint8_t *code;              // [ncell] physical layout
  const uint32_t *codeP[4];         // per x/y-flip class: the 4 cell bytes of a thread's 2x2 patch, byte (j&1) + 2 (k&1),
                                    // index ((kz * nty + ty) * NU + (i' + J)) * 32 + J, kz = physical k / 2
  const int32_t *iface;             // [6][ncell] interface-face id or -1
  const int32_t *iface_info;        // [n_iface] face code f
  void *Gi;                         // T [n_iface][B] interface inflow of this iteration (Eq. 5 / Eq. 6)
  void *Hd;                         // T [6][ncell][B][4] outgoing hemispherical partial sums per face, cell, band and
                                    // outgoing-octant slot (dense, touched at interface faces only: no id look-up in the sweep)
  const int32_t *iface_cell;        // [n_iface] physical cell of the face
  int32_t n_iface, iface_type;
  double iface_e0[BTE2_MAXB];       // isothermal interface inflow C_b dT_w / 4pi
  double ivband[BTE2_MAXB];         // 1 / group velocity (undoes the v_b in the moment coefficients)
};

// ------------------------------------------------------------------ layouts (host + device)
template <typename T> struct alignas(16) Bte2Chunk { T v[16 / sizeof(T)]; };   // 4 floats / 2 doubles
template <typename T> struct alignas(2 * sizeof(T)) Bte2Pair { T x, y; };
template <typename T> struct alignas(16) Bte2Mom { T v[4]; };

#define BTE2_HD __host__ __device__ __forceinline__

// skewed cell index: oriented i', j' of the class, physical k
BTE2_HD int64_t sk2_index(int nty, int NU, int ip, int jp, int k) {
  const int ty = jp >> 6, r = jp & 63, J = r >> 1, jj = r & 1;
  return ((((int64_t)k * nty + ty) * NU + (ip + J)) * 2 + jj) * 32 + J;
}
// x planes: [tile][b][K][kk][jj][chunk][J], chunk = p / CP
template <typename T>
BTE2_HD int64_t xpl2_index(const Bte2Dev &P, int ty, int tz, int b, int K, int kk, int jj, int ch, int J) {
  constexpr int NCH = BTE2_P * sizeof(T) / 16;
  return ((((((int64_t)(tz * P.nty + ty) * P.B + b) * P.W + K) * 2 + kk) * 2 + jj) * NCH + ch) * 32 + J;
}
// y planes: [slot][tz][b][K][i'][kk][chunk]
template <typename T>
BTE2_HD int64_t ypl2_index(const Bte2Dev &P, int slot, int tz, int b, int K, int ip, int kk, int ch) {
  constexpr int NCH = BTE2_P * sizeof(T) / 16;
  return (((((int64_t)(slot * P.ntz + tz) * P.B + b) * P.W + K) * P.nx + ip) * 2 + kk) * NCH + ch;
}
// z planes: [slot][ty][b][u][jj][chunk][J], u = i' + J
template <typename T>
BTE2_HD int64_t zpl2_index(const Bte2Dev &P, int slot, int ty, int b, int u, int jj, int ch, int J) {
  constexpr int NCH = BTE2_P * sizeof(T) / 16;
  return (((((int64_t)(slot * P.nty + ty) * P.B + b) * P.NU + u) * 2 + jj) * NCH + ch) * 32 + J;
}

#ifdef __CUDACC__
// ------------------------------------------------------------------ device helpers
__device__ __forceinline__ int ld_acquire_gpu(const int *p) {
  int v;
  asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ int ld_relaxed_gpu(const int *p) {
  int v;
  asm volatile("ld.relaxed.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_gpu(int *p, int v) {
  asm volatile("st.release.gpu.global.s32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
template <int BYTES>
__device__ __forceinline__ void cp_async(unsigned d, const void *gsrc) {   // d: shared-window address
  if (BYTES == 16) asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
  else if (BYTES == 8) asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(d), "l"(gsrc) : "memory");
  else if (BYTES == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

// split CTA barrier (BTE2_SPLITBAR): arrive once the step's shared-memory traffic is done, wait after the moment store
__device__ __forceinline__ unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t *b, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(b)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t *b) { asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(b)) : "memory"); }
__device__ __forceinline__ void mbar_wait(uint64_t *b, unsigned parity) {
  asm volatile(
      "{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nbra LAB_WAIT;\nDONE:\n}" ::"r"(smem_u32(b)),
      "r"(parity)
      : "memory");
}

template <typename T> __device__ __forceinline__ Bte2Chunk<T> ldcg_chunk(const Bte2Chunk<T> *p) {
  const float4 v = __ldcg(reinterpret_cast<const float4 *>(p));
  Bte2Chunk<T> r;
  memcpy(&r, &v, 16);
  return r;
}
// packed pairs of directions: fp32 uses the sm_100 two-wide FMA (FFMA2: two FMAs per issue slot, which frees
// issue slots for the non-FMA instructions of the step); fp64 is two scalar DFMAs.
// Measured on B200 (csrc/microbench_fma_forms.cu, profiles/r01_fma_forms_microbench.txt): FFMA2 with two vector-register
// operands and a uniform-register pair (the form used here) runs at the full FMA rate, 124.6 of 128 FMA/clk/SM.
template <typename T> struct Bte2V2;
template <> struct Bte2V2<float> { typedef float2 t; };
template <> struct Bte2V2<double> { typedef double2 t; };
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ double2 fma2(double2 a, double2 b, double2 c) { return make_double2(fma(a.x, b.x, c.x), fma(a.y, b.y, c.y)); }
__device__ __forceinline__ double2 mul2(double2 a, double2 b) { return make_double2(a.x * b.x, a.y * b.y); }
// moment accumulation m += w * e over a pair: fp32 keeps even / odd partial sums (one FFMA2), fp64 one sum
__device__ __forceinline__ void acc2(float2 &m, float2 w, float2 e) { m = __ffma2_rn(w, e, m); }
__device__ __forceinline__ void acc2(double2 &m, double2 w, double2 e) { m.x = fma(w.x, e.x, m.x); m.x = fma(w.y, e.y, m.x); }
__device__ __forceinline__ float2 mk2(float a, float b) { return make_float2(a, b); }
__device__ __forceinline__ double2 mk2(double a, double b) { return make_double2(a, b); }
template <typename T> __device__ __forceinline__ T shfl_up1(T v);
template <> __device__ __forceinline__ float shfl_up1<float>(float v) { return __shfl_up_sync(0xffffffffu, v, 1); }
template <> __device__ __forceinline__ double shfl_up1<double>(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }

// shared-memory carve-up of one CTA.  D = prefetch distance in steps (ring of D+1 buffers).
template <typename T, int NB, int W, int D> struct Bte2Smem {
  static constexpr int CP = 16 / sizeof(T);            // directions per 16-byte chunk
  static constexpr int NCH = BTE2_P / CP;              // chunks per band
  static constexpr int NC = NB * NCH;                  // chunks per row and step
  typedef Bte2Chunk<T> Ch;
  Ch zex[2][W][2][NC][32];           // [parity][K][jj][chunk][lane]: kk=1 rows of warp K, read by warp K+1 / copied out
  Ch zin0[D + 1][2][NC][32];         // staged z inflow plane of warp 0
  Ch ybuf[D + 1][W][2][NC];          // [ring][warp][kk][chunk]: y inflow of lane 0
  Ch yst[2][W][2 * NC];              // [parity][warp][kk*NC + chunk]: jj=1 rows of lane Jl, copied out one step later
  Bte2Mom<T> mold[BTE2_MDIST(T) + 1][2][2][W * 32];  // [ring][kk][jj][tid] previous content of the moment accumulator
  Bte2Pair<T> inp[D + 1][2][2][W * 32];    // [ring][kk][jj][tid] (dT, Q/sumC) of the cell
  uint32_t codes[D + 1][W * 32];           // [ring][tid] cell bytes of the thread's patch (masked grids only)
};

// ------------------------------------------------------------------ one unit = (octant, band group, tile)
template <typename T, int NB, int W, int D, bool MASKED>
__device__ __forceinline__ void bte2_run_unit(const Bte2Dev &P, const Bte2Coefs<T> &CF, const Bte2Unit &un,
                                              unsigned char *smem_raw, int unit, uint64_t *stepbar, unsigned &bpar) {
  typedef Bte2Smem<T, NB, W, D> SM;
  SM *S = reinterpret_cast<SM *>(smem_raw);
  constexpr int CP = SM::CP, NCH = SM::NCH, NC = SM::NC, NT = W * 32, R = D + 1;
  // the accumulator rows of step t + 1 + MDIST are prefetched right after ensure(t + D) (split barrier): their publication
  // upstream is only known if D >= 1 + MDIST
  static_assert(D >= 1 + BTE2_MDIST(T), "prefetch distance too short for the accumulator prefetch");
  typedef Bte2Chunk<T> Ch;
  const unsigned FULL = 0xffffffffu;
  const int tid = threadIdx.x, J = tid & 31, K = tid >> 5;
  const Bte2Oct &O = P.oct[un.oct];
  const int ty = un.ty, tz = un.tz, b0 = un.b0;
  const int jp0 = ty * 64 + 2 * J, kp0 = tz * 2 * W + 2 * K;
  // ny and nz are even on this path (host check): a patch is valid or invalid as a whole, and the last
  // valid row of a tile is always the jj = 1 / kk = 1 row of lane Jl / warp Kl
  const bool vthread = (jp0 < P.ny) && (kp0 < P.nz);
  const int Jl = (min(P.ny, (ty + 1) * 64) - 1 - ty * 64) >> 1, Kl = (min(P.nz, (tz + 1) * 2 * W) - 1 - tz * 2 * W) >> 1;
  const bool first = un.dep_prev < 0;                  // first band group of this octant: M is written, not added to
  const int ebase = P.epoch << 16;
  // shared-window address for cp.async (hoisting one base address out of the step loop measured slower in fp32)
  auto saddr = [&](const void *ptr) { return (unsigned)__cvta_generic_to_shared(ptr); };

  const Ch *xin = reinterpret_cast<const Ch *>(O.xsrc);
  Ch *xout = reinterpret_cast<Ch *>(O.xdst);
  Bte2Mom<T> *M = reinterpret_cast<Bte2Mom<T> *>(O.M);
  const Bte2Pair<T> *dTQ = reinterpret_cast<const Bte2Pair<T> *>(P.dTQ[O.cls]);

  // cell index of row (jj,kk) at step t: cbase[kk] + jj*32 + (t - K) * 64
  int64_t cbase[2];
#pragma unroll
  for (int kk = 0; kk < 2; ++kk) {
    const int kp = kp0 + kk, k = vthread ? (O.sz > 0 ? kp : P.nz - 1 - kp) : 0;
    cbase[kk] = (((int64_t)k * P.nty + ty) * P.NU) * 64 + J - (int64_t)K * 64;
  }
  // voxel mask: patch-code stream of this thread, face indices of this octant
  const int fu[3] = {O.sx > 0 ? 0 : 1, O.sy > 0 ? 2 : 3, O.sz > 0 ? 4 : 5};      // upwind faces x, y, z
  const uint32_t *cpsrc = nullptr;
  if (MASKED) {
    const int kz = (vthread ? (O.sz > 0 ? kp0 : P.nz - 2 - kp0) : 0) >> 1;
    cpsrc = P.codeP[O.cls] + (((int64_t)kz * P.nty + ty) * P.NU) * 32 + J - (int64_t)K * 32;
  }
  // plane pointers of this thread at step 0; all advance by a constant stride per step
  //   z inflow staging: element e = tid + q*NT of the [b][jj][ch][lane] block of step u
  const Ch *zsrc = (tz == 0 ? reinterpret_cast<const Ch *>(O.zsrc0) : reinterpret_cast<const Ch *>(O.zpl) + zpl2_index<T>(P, tz, 0, 0, 0, 0, 0, 0)) +
                   zpl2_index<T>(P, 0, ty, b0, 0, 0, 0, 0);
  const int64_t zstep = 2 * NCH * 32, zband = (int64_t)P.NU * 2 * NCH * 32;
  Ch *zdst = (tz == P.ntz - 1 ? reinterpret_cast<Ch *>(O.zdstN) : reinterpret_cast<Ch *>(O.zpl) + zpl2_index<T>(P, tz + 1, 0, 0, 0, 0, 0, 0)) +
             zpl2_index<T>(P, 0, ty, b0, 0, 0, 0, 0);
  //   y planes: lane l < 2*NC of warp K loads chunk (b, kk, ch) of the cell i' = t - K
  const int yb = J / (2 * NCH), ykk = (J / NCH) & 1, ych = J % NCH;
  const Ch *ysrc = (ty == 0 ? reinterpret_cast<const Ch *>(O.ysrc0) : reinterpret_cast<const Ch *>(O.ypl) + ypl2_index<T>(P, ty, 0, 0, 0, 0, 0, 0)) +
                   ypl2_index<T>(P, 0, tz, b0 + (J < 2 * NC ? yb : 0), K, 0, ykk, ych) - (int64_t)K * 2 * NCH;
  Ch *ydst = (ty == P.nty - 1 ? reinterpret_cast<Ch *>(O.ydstN) : reinterpret_cast<Ch *>(O.ypl) + ypl2_index<T>(P, ty + 1, 0, 0, 0, 0, 0, 0)) +
             ypl2_index<T>(P, 0, tz, b0 + (J < 2 * NC ? yb : 0), K, 0, ykk, ych);

  // ---- progress of the units this one follows: three poller threads keep the last value seen in a register
  // the three pollers and the publisher sit in different warps: their memory round trips overlap instead of adding up
  // in warp 0 (every other warp waits for the slowest one at the step barrier)
  constexpr int ROLE1 = (1 % W) * 32 + 1 / W, ROLE2 = (2 % W) * 32 + 2 / W, ROLEP = (3 % W) * 32 + 3 / W;
  const int mydep = tid == 0 ? un.dep_y : (tid == ROLE1 ? un.dep_z : (tid == ROLE2 ? un.dep_prev : -1));
  const int mylag = tid == 0 ? 33 : (tid == ROLE1 ? W + 1 : 1);
  int seen = 0, peek = 0;
  auto ensure = [&](int t1) {          // everything step t1 reads from other units has been published
    if (mydep >= 0 && !BTE2_DBGBIT(P, 4)) {
      // the peek is a relaxed load (asynchronous: no L1 invalidation behind it); a publication it shows is then
      // acquired properly, once per publication instead of once per step
      if (peek - ebase > seen) seen = max(seen, ld_acquire_gpu(P.prog + mydep) - ebase);
      if (seen < t1 + mylag) {
        int v;
        while ((v = ld_acquire_gpu(P.prog + mydep) - ebase) < t1 + mylag) __nanosleep(64);
        seen = v;
      }
    }
  };

  // ---- previous content of the moment accumulator for step t1 (own commit group, one step ahead)
  auto prefetch_m = [&](int t1) {
    const int ip1 = t1 - J - K;
    if (!first && !BTE2_DBGBIT(P, 2) && vthread && ip1 >= 0 && ip1 < P.nx) {
#pragma unroll
      for (int kk = 0; kk < 2; ++kk)
#pragma unroll
        for (int jj = 0; jj < 2; ++jj) {
          const int64_t ci = cbase[kk] + jj * 32 + (int64_t)t1 * 64;
#pragma unroll
          for (int h = 0; h < (int)sizeof(Bte2Mom<T>) / 16; ++h)
            cp_async<16>(saddr(&S->mold[t1 % (BTE2_MDIST(T) + 1)][kk][jj][tid]) + 16 * h, reinterpret_cast<const char *>(M + ci) + 16 * h);
        }
    }
  };
  // ---- outflow faces of step t1 (staged in shared memory by the step) -> global planes, coalesced
  auto copy_out = [&](int t1) {
    const int par = (t1 & 1) ^ 1;                      // buffer the step wrote
    if (!BTE2_DBGBIT(P, 1) && kp0 < P.nz) {
      const int ipl = t1 - Jl - K;                     // cell lane Jl of this warp finished in step t1
      if (J < 2 * NC && ipl >= 0 && ipl < P.nx) ydst[(int64_t)ipl * 2 * NCH] = S->yst[par][K][ykk * NC + yb * NCH + ych];
    }
    const int ul = t1 - Kl;
    if (!BTE2_DBGBIT(P, 1) && ul >= 0 && ul < P.NU) {
#pragma unroll
      for (int q = 0; q < (2 * NC * 32) / NT; ++q) {
        const int e = tid + q * NT, b = e / (2 * NCH * 32), rem = e % (2 * NCH * 32);
        zdst[b * zband + ul * zstep + rem] = (&S->zex[par][Kl][0][b * NCH][0])[(rem / (NCH * 32)) * (NC * 32) + (rem % (NCH * 32))];
      }
    }
  };
  // ---- asynchronous prefetch (global -> shared) of everything step t1 consumes
  auto prefetch = [&](int t1, int rb) {                // rb = t1 % R, the ring slot of step t1
    const int ip1 = t1 - J - K;
    if (vthread && ip1 >= 0 && ip1 < P.nx) {
#pragma unroll
      for (int kk = 0; kk < 2; ++kk) {
#pragma unroll
          for (int jj = 0; jj < 2; ++jj) {
            const int64_t ci = cbase[kk] + jj * 32 + (int64_t)t1 * 64;
            cp_async<sizeof(Bte2Pair<T>)>(saddr(&S->inp[rb][kk][jj][tid]), dTQ + ci);
          }
        }
    }
    if (MASKED && vthread && ip1 >= 0 && ip1 < P.nx) cp_async<4>(saddr(&S->codes[rb][tid]), cpsrc + (int64_t)t1 * 32);
    if (t1 < P.NU && !BTE2_DBGBIT(P, 8)) {
#pragma unroll
      for (int q = 0; q < (2 * NC * 32) / NT; ++q) {
        const int e = tid + q * NT, b = e / (2 * NCH * 32), rem = e % (2 * NCH * 32);
        cp_async<16>(saddr(&S->zin0[rb][0][b * NCH][0] + (rem / (NCH * 32)) * (NC * 32) + (rem % (NCH * 32))), zsrc + b * zband + t1 * zstep + rem);
      }
    }
    {
      const int ipy = t1 - K;
      if (J < 2 * NC && ipy >= 0 && ipy < P.nx) cp_async<16>(saddr(&S->ybuf[rb][K][ykk][yb * NCH + ych]), ysrc + (int64_t)t1 * 2 * NCH);
    }
  };

  // ---- x inflow -> carry registers (kept untouched by a thread until its first active step)
  typedef typename Bte2V2<T>::t V2;
  V2 c[2][2][NB * BTE2_P / 2];                        // [jj][kk][(b*16 + p) / 2]: pairs of directions
#pragma unroll
  for (int kk = 0; kk < 2; ++kk)
#pragma unroll
    for (int jj = 0; jj < 2; ++jj)
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
          const Ch v = ldcg_chunk<T>(xin + xpl2_index<T>(P, ty, tz, b0 + b, K, kk, jj, ch, J));
#pragma unroll
          for (int q = 0; q < CP; q += 2) c[jj][kk][(b * BTE2_P + ch * CP + q) / 2] = mk2(v.v[q], v.v[q + 1]);
        }

  ensure(D + P.slack);
  __syncthreads();
#pragma unroll
  for (int t1 = 0; t1 < D; ++t1) {
    if (t1 == 0 && BTE2_MDIST(T) == 1) prefetch_m(0);
    prefetch(t1, t1); cp_async_commit();
  }
#if BTE2_SPLITBAR
  prefetch_m(BTE2_MDIST(T)); cp_async_commit();        // steady state: issued in the barrier window of the previous step
#endif
  cp_async_wait<D - 1>();
  __syncthreads();

  T bcx[NB], bcy[NB];
#pragma unroll
  for (int b = 0; b < NB; ++b) { bcx[b] = CF.bc[b0 + b][0]; bcy[b] = CF.bc[b0 + b][1]; }

  // one (band, chunk) of the 2x2 patch: FAST = every lane of the warp is active (no predication)
  auto chunk = [&](auto fastc, int b, int ch, const V2 (&r)[2][2], V2 (&m)[2][2][4], int rb, int cur, bool act,
                   const Ch *__restrict__ zrd, Ch *__restrict__ zwr) {
    constexpr bool FAST = decltype(fastc)::value;
    constexpr int NP = CP / 2;                         // direction pairs per chunk
    const int h0 = (b * BTE2_P + ch * CP) / 2, cn = b * NCH + ch;
    // y inflow: lane J-1's jj=1 rows of the previous step; lane 0: the staged plane
    V2 yin[2][NP];
#pragma unroll
    for (int kk = 0; kk < 2; ++kk)
#pragma unroll
      for (int q = 0; q < NP; ++q) yin[kk][q] = mk2(shfl_up1<T>(c[1][kk][h0 + q].x), shfl_up1<T>(c[1][kk][h0 + q].y));
    if (J == 0) {
#pragma unroll
      for (int kk = 0; kk < 2; ++kk) {
        const Ch v = S->ybuf[rb][K][kk][cn];
#pragma unroll
        for (int q = 0; q < NP; ++q) yin[kk][q] = mk2(v.v[2 * q], v.v[2 * q + 1]);
      }
    }
    // z inflow: warp K-1's kk=1 rows of the previous step, or the staged plane for warp 0
    const Ch z0 = zrd[cn * 32], z1 = zrd[(NC + cn) * 32];
    if (FAST || act) {
      Ch o0, o1;
#pragma unroll
      for (int q = 0; q < NP; ++q) {
        const int p = ch * CP + 2 * q;
        const T(&kb)[8][BTE2_P] = CF.k[b0 + b];
        const V2 inv = mk2(kb[0][p], kb[0][p + 1]), ax = mk2(kb[1][p], kb[1][p + 1]), ay = mk2(kb[2][p], kb[2][p + 1]),
                 az = mk2(kb[3][p], kb[3][p + 1]);
        const V2 w0 = mk2(kb[4][p], kb[4][p + 1]), w1 = mk2(kb[5][p], kb[5][p + 1]), w2 = mk2(kb[6][p], kb[6][p + 1]),
                 w3 = mk2(kb[7][p], kb[7][p + 1]);
        const V2 zq0 = mk2(z0.v[2 * q], z0.v[2 * q + 1]), zq1 = mk2(z1.v[2 * q], z1.v[2 * q + 1]);
        V2 e00 = mul2(r[0][0], inv); e00 = fma2(ax, c[0][0][h0 + q], e00); e00 = fma2(ay, yin[0][q], e00); e00 = fma2(az, zq0, e00);
        V2 e10 = mul2(r[1][0], inv); e10 = fma2(ax, c[1][0][h0 + q], e10); e10 = fma2(az, zq1, e10); e10 = fma2(ay, e00, e10);
        V2 e01 = mul2(r[0][1], inv); e01 = fma2(ax, c[0][1][h0 + q], e01); e01 = fma2(ay, yin[1][q], e01); e01 = fma2(az, e00, e01);
        V2 e11 = mul2(r[1][1], inv); e11 = fma2(ax, c[1][1][h0 + q], e11); e11 = fma2(ay, e01, e11); e11 = fma2(az, e10, e11);
        c[0][0][h0 + q] = e00; c[1][0][h0 + q] = e10; c[0][1][h0 + q] = e01; c[1][1][h0 + q] = e11;
        o0.v[2 * q] = e01.x; o0.v[2 * q + 1] = e01.y; o1.v[2 * q] = e11.x; o1.v[2 * q + 1] = e11.y;
        acc2(m[0][0][0], w0, e00); acc2(m[0][0][1], w1, e00); acc2(m[0][0][2], w2, e00); acc2(m[0][0][3], w3, e00);
        acc2(m[1][0][0], w0, e10); acc2(m[1][0][1], w1, e10); acc2(m[1][0][2], w2, e10); acc2(m[1][0][3], w3, e10);
        acc2(m[0][1][0], w0, e01); acc2(m[0][1][1], w1, e01); acc2(m[0][1][2], w2, e01); acc2(m[0][1][3], w3, e01);
        acc2(m[1][1][0], w0, e11); acc2(m[1][1][1], w1, e11); acc2(m[1][1][2], w2, e11); acc2(m[1][1][3], w3, e11);
      }
      zwr[cn * 32] = o0; zwr[(NC + cn) * 32] = o1;
    }
  };

  // the same (band, chunk) on a patch that contains void cells or solid/void interface faces: every cell
  // takes its upwind values through selects (interface inflow g instead of the neighbour) and void cells hold 0.
  // cb[c] = code byte, g[c][axis] = interface inflow of cell c = A (0,0), B (1,0), C (0,1), D (1,1).
  auto chunk_masked = [&](int b, int ch, const V2 (&r)[2][2], V2 (&m)[2][2][4], int rb, bool act, const uint32_t (&cb)[4],
                          const T (&g)[4][3], const Ch *__restrict__ zrd, Ch *__restrict__ zwr) {
    constexpr int NP = CP / 2;
    const int h0 = (b * BTE2_P + ch * CP) / 2, cn = b * NCH + ch;
    V2 yin[2][NP];
#pragma unroll
    for (int kk = 0; kk < 2; ++kk)
#pragma unroll
      for (int q = 0; q < NP; ++q) yin[kk][q] = mk2(shfl_up1<T>(c[1][kk][h0 + q].x), shfl_up1<T>(c[1][kk][h0 + q].y));
    if (J == 0) {
#pragma unroll
      for (int kk = 0; kk < 2; ++kk) {
        const Ch v = S->ybuf[rb][K][kk][cn];
#pragma unroll
        for (int q = 0; q < NP; ++q) yin[kk][q] = mk2(v.v[2 * q], v.v[2 * q + 1]);
      }
    }
    const Ch z0 = zrd[cn * 32], z1 = zrd[(NC + cn) * 32];
    if (!act) return;                                  // (shuffles above stay warp-convergent)
    auto up = [&](uint32_t code, int axis, T gv, V2 v) { return (code >> (1 + fu[axis])) & 1u ? mk2(gv, gv) : v; };
    auto keep = [&](uint32_t code, V2 v) { return (code & 1u) ? v : mk2((T)0, (T)0); };
    Ch o0, o1;
#pragma unroll
    for (int q = 0; q < NP; ++q) {
      const int p = ch * CP + 2 * q;
      const T(&kb)[8][BTE2_P] = CF.k[b0 + b];
      const V2 inv = mk2(kb[0][p], kb[0][p + 1]), ax = mk2(kb[1][p], kb[1][p + 1]), ay = mk2(kb[2][p], kb[2][p + 1]),
               az = mk2(kb[3][p], kb[3][p + 1]);
      const V2 w0 = mk2(kb[4][p], kb[4][p + 1]), w1 = mk2(kb[5][p], kb[5][p + 1]), w2 = mk2(kb[6][p], kb[6][p + 1]),
               w3 = mk2(kb[7][p], kb[7][p + 1]);
      const V2 zq0 = mk2(z0.v[2 * q], z0.v[2 * q + 1]), zq1 = mk2(z1.v[2 * q], z1.v[2 * q + 1]);
      V2 e00 = mul2(r[0][0], inv); e00 = fma2(ax, up(cb[0], 0, g[0][0], c[0][0][h0 + q]), e00);
      e00 = fma2(ay, up(cb[0], 1, g[0][1], yin[0][q]), e00); e00 = fma2(az, up(cb[0], 2, g[0][2], zq0), e00); e00 = keep(cb[0], e00);
      V2 e10 = mul2(r[1][0], inv); e10 = fma2(ax, up(cb[1], 0, g[1][0], c[1][0][h0 + q]), e10);
      e10 = fma2(az, up(cb[1], 2, g[1][2], zq1), e10); e10 = fma2(ay, up(cb[1], 1, g[1][1], e00), e10); e10 = keep(cb[1], e10);
      V2 e01 = mul2(r[0][1], inv); e01 = fma2(ax, up(cb[2], 0, g[2][0], c[0][1][h0 + q]), e01);
      e01 = fma2(ay, up(cb[2], 1, g[2][1], yin[1][q]), e01); e01 = fma2(az, up(cb[2], 2, g[2][2], e00), e01); e01 = keep(cb[2], e01);
      V2 e11 = mul2(r[1][1], inv); e11 = fma2(ax, up(cb[3], 0, g[3][0], c[1][1][h0 + q]), e11);
      e11 = fma2(ay, up(cb[3], 1, g[3][1], e01), e11); e11 = fma2(az, up(cb[3], 2, g[3][2], e10), e11); e11 = keep(cb[3], e11);
      c[0][0][h0 + q] = e00; c[1][0][h0 + q] = e10; c[0][1][h0 + q] = e01; c[1][1][h0 + q] = e11;
      o0.v[2 * q] = e01.x; o0.v[2 * q + 1] = e01.y; o1.v[2 * q] = e11.x; o1.v[2 * q + 1] = e11.y;
      acc2(m[0][0][0], w0, e00); acc2(m[0][0][1], w1, e00); acc2(m[0][0][2], w2, e00); acc2(m[0][0][3], w3, e00);
      acc2(m[1][0][0], w0, e10); acc2(m[1][0][1], w1, e10); acc2(m[1][0][2], w2, e10); acc2(m[1][0][3], w3, e10);
      acc2(m[0][1][0], w0, e01); acc2(m[0][1][1], w1, e01); acc2(m[0][1][2], w2, e01); acc2(m[0][1][3], w3, e01);
      acc2(m[1][1][0], w0, e11); acc2(m[1][1][1], w1, e11); acc2(m[1][1][2], w2, e11); acc2(m[1][1][3], w3, e11);
    }
    zwr[cn * 32] = o0; zwr[(NC + cn) * 32] = o1;
  };

  int rb = 0, rbp = R - 1;                             // ring slots of step t and of step t - 1 (= step t + D)
  for (int t = 0; t < P.nsteps; ++t) {
    const int cur = t & 1;
    const int ip = t - J - K;
    const bool act = vthread && ip >= 0 && ip < P.nx;
#if !BTE2_SPLITBAR
    prefetch_m(t + BTE2_MDIST(T));
    cp_async_commit();
#endif
    prefetch(t + D, rbp);
    cp_async_commit();
    if (t > 0) copy_out(t - 1);
    if (mydep >= 0 && seen < t + 1 + D + mylag) peek = ld_relaxed_gpu(P.prog + mydep);   // consumed by ensure() below

    V2 m[2][2][4];                                     // moment partial sums of even / odd directions
#pragma unroll
    for (int a = 0; a < 2; ++a)
#pragma unroll
      for (int b = 0; b < 2; ++b)
#pragma unroll
        for (int q = 0; q < 4; ++q) m[a][b][q] = mk2((T)0, (T)0);

    Bte2Pair<T> in[2][2];
#pragma unroll
    for (int kk = 0; kk < 2; ++kk)
#pragma unroll
      for (int jj = 0; jj < 2; ++jj) in[jj][kk] = S->inp[rb][kk][jj][tid];

    // masked grids: code bytes of the patch, oriented cell (jj,kk) -> byte (physical parities)
    uint32_t cb[4] = {1u, 1u, 1u, 1u};
    bool plain = true, live = act;                     // live: the patch holds at least one solid cell
    if (MASKED) {
      const uint32_t code = act ? S->codes[rb][tid] : 0x01010101u;
      plain = code == 0x01010101u;
      live = act && (code & 0x01010101u) != 0;
#pragma unroll
      for (int cc = 0; cc < 4; ++cc) {
        const int jj = cc & 1, kk = cc >> 1, pj = O.sy > 0 ? jj : 1 - jj, pk = O.sz > 0 ? kk : 1 - kk;
        cb[cc] = (code >> (8 * (pj + 2 * pk))) & 0xffu;
      }
    }
    const bool fast = __all_sync(FULL, act && plain);
    const bool slowmask = MASKED && __any_sync(FULL, live && !plain);
    const Ch *__restrict__ zrd = K == 0 ? &S->zin0[rb][0][0][J] : &S->zex[cur][K - 1][0][0][J];
    Ch *__restrict__ zwr = &S->zex[cur ^ 1][K][0][0][J];
    // warps without a valid row (ragged last z tile; 3 of 4 warps of a two-layer 2-D slab) and warps that are
    // entirely before their first or after their last cell skip the arithmetic (they still stage and synchronise)
    if (__any_sync(FULL, act))
#pragma unroll
    for (int b = 0; b < NB; ++b) {
      V2 r[2][2];
#pragma unroll
      for (int kk = 0; kk < 2; ++kk)
#pragma unroll
        for (int jj = 0; jj < 2; ++jj) {
          const T rv = fma(bcx[b], in[jj][kk].x, bcy[b] * in[jj][kk].y);
          r[jj][kk] = mk2(rv, rv);
        }
      if (MASKED && slowmask) {
        // physical cell indices of the patch, interface inflow per cell and axis (Eq. 5 / Eq. 6, lagged)
        int64_t cph[4];
        T g[4][3];
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          const int jj = cc & 1, kk = cc >> 1;
          const int i = O.sx > 0 ? ip : P.nx - 1 - ip, j = O.sy > 0 ? jp0 + jj : P.ny - 1 - jp0 - jj,
                    k = O.sz > 0 ? kp0 + kk : P.nz - 1 - kp0 - kk;
          cph[cc] = (int64_t)i + (int64_t)P.nx * (j + (int64_t)P.ny * k);
#pragma unroll
          for (int a = 0; a < 3; ++a) {
            g[cc][a] = (T)0;
            if (live && (cb[cc] & 1u) && ((cb[cc] >> (1 + fu[a])) & 1u))
              g[cc][a] = (P.iface_type == 0 || BTE2_DBGBIT(P, 64)) ? (T)P.iface_e0[b0 + b]
                                           : reinterpret_cast<const T *>(P.Gi)[(int64_t)__ldg(P.iface + (int64_t)fu[a] * P.ncell + cph[cc]) * P.B + b0 + b];
          }
        }
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) chunk_masked(b, ch, r, m, rb, live, cb, g, zrd, zwr);
        {
          // outgoing hemispherical partial sums at solid/void faces (diffuse interface, Eq. 6)
          uint32_t anydn = 0;
#pragma unroll
          for (int cc = 0; cc < 4; ++cc)
            if (cb[cc] & 1u) anydn |= cb[cc] & ((2u << (fu[0] ^ 1)) | (2u << (fu[1] ^ 1)) | (2u << (fu[2] ^ 1)));
          if (P.iface_type == 1 && live && anydn != 0 && !BTE2_DBGBIT(P, 128)) {
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
              const int jj = cc & 1, kk = cc >> 1;
              if (!(cb[cc] & 1u)) continue;
#pragma unroll
              for (int a = 0; a < 3; ++a) {
                const int fd = fu[a] ^ 1;
                if (!((cb[cc] >> (1 + fd)) & 1u)) continue;
                // sum_p w_p |s_p,a| e_p in the compute type with the moment coefficients v_b w |s_a| (<= 16 terms of
                // one sign pattern), divided by v_b; the sum over the 4 outgoing octants is fp64 (ghost kernel)
                // The first band of the group gets it for free: it IS the cell's first-moment partial sum so far.
                V2 hs = mk2((T)0, (T)0);
                if (b == 0) hs = m[jj][kk][1 + a];
                else {
#pragma unroll
                  for (int q = 0; q < BTE2_P / 2; ++q)
                    hs = fma2(mk2(CF.k[b0 + b][5 + a][2 * q], CF.k[b0 + b][5 + a][2 * q + 1]), c[jj][kk][b * (BTE2_P / 2) + q], hs);
                }
                const int bx = O.sx < 0, by = O.sy < 0, bz = O.sz < 0;
                const int s2 = a == 0 ? (by | (bz << 1)) : (a == 1 ? (bx | (bz << 1)) : (bx | (by << 1)));
                reinterpret_cast<T *>(P.Hd)[(((int64_t)fd * P.ncell + cph[cc]) * P.B + b0 + b) * 4 + s2] = (hs.x + hs.y) * (T)P.ivband[b0 + b];
              }
            }
          }
        }
      } else if (fast && !MASKED) {   // (the masked kernel does without this copy of the arithmetic: at ~10,000 instructions
                                      // it is bound by instruction fetch, and dropping it took config 3 from 2.47 to 2.24 ms)
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) chunk(std::true_type{}, b, ch, r, m, rb, cur, true, zrd, zwr);
      } else {
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) chunk(std::false_type{}, b, ch, r, m, rb, cur, live, zrd, zwr);
      }
    }

    if (BTE2_MDIST(T) == 0) cp_async_wait<D - 1>();   // the accumulator content fetched in THIS step has landed
#if BTE2_SPLITBAR
    cp_async_wait<D - 1>();            // everything step t+1 reads has landed
    if (mydep >= 0) ensure(t + 1 + D);    // ... and what step t+1 prefetches has been published upstream
    mbar_arrive(stepbar);              // this thread's shared-memory reads and writes of step t are done
#endif
    if (act) {
      // (b) moments of this band group into the octant accumulator (one owner per cell and group)
#pragma unroll
      for (int kk = 0; kk < 2; ++kk)
        if (!BTE2_DBGBIT(P, 2)) {
#pragma unroll
          for (int jj = 0; jj < 2; ++jj) {
            if (MASKED && !(cb[jj + 2 * kk] & 1u)) continue;      // void cell
            Bte2Mom<T> o;
            if (first) {
#pragma unroll
              for (int q = 0; q < 4; ++q) o.v[q] = m[jj][kk][q].x + m[jj][kk][q].y;
            } else {
              const Bte2Mom<T> old = S->mold[t % (BTE2_MDIST(T) + 1)][kk][jj][tid];
#pragma unroll
              for (int q = 0; q < 4; ++q) o.v[q] = old.v[q] + (m[jj][kk][q].x + m[jj][kk][q].y);
            }
            M[cbase[kk] + jj * 32 + (int64_t)t * 64] = o;
          }
        }
      // y outflow rows (jj = 1 of lane Jl) -> staging buffer; written to the plane by copy_out() next step
      if (J == Jl) {
#pragma unroll
        for (int b = 0; b < NB; ++b)
#pragma unroll
          for (int kk = 0; kk < 2; ++kk)
#pragma unroll
            for (int ch = 0; ch < NCH; ++ch) {
              Ch o;
#pragma unroll
              for (int q = 0; q < CP; q += 2) {
                const V2 v = c[1][kk][(b * BTE2_P + ch * CP + q) / 2];
                o.v[q] = v.x; o.v[q + 1] = v.y;
              }
              S->yst[cur ^ 1][K][kk * NC + b * NCH + ch] = o;
            }
      }
    }
#if BTE2_SPLITBAR
    // accumulator rows of the step after next: their publication upstream is known since the previous barrier
    // (ensure(t + D) covers step t + 1 + MDIST because D >= 1 + MDIST), and the ring slot was read just above
    prefetch_m(t + 1 + BTE2_MDIST(T));
    cp_async_commit();
    mbar_wait(stepbar, bpar);          // every thread has arrived: the moment store above overlapped the wait
    bpar ^= 1u;
    __syncwarp();                      // yst rows written after the arrive are read by this warp's copy_out next step
#else
    cp_async_wait<D - 1>();            // everything step t+1 reads has landed
    if (mydep >= 0) ensure(t + 1 + D);    // ... and what step t+1 prefetches has been published upstream
    __syncthreads();
#endif
    if ((t & P.pub_mask) == P.pub_mask && tid == ROLEP) {   // faces and moments of steps < t are in global memory
      __threadfence();
      st_release_gpu(P.prog + unit, ebase + t);
    }
    rbp = rb;
    rb = rb + 1 == R ? 0 : rb + 1;
  }
  cp_async_wait<0>();
  copy_out(P.nsteps - 1);

  // ---- x outflow (carries are final: a thread stops updating them after its last active step)
#pragma unroll
  for (int kk = 0; kk < 2; ++kk)
#pragma unroll
    for (int jj = 0; jj < 2; ++jj)
#pragma unroll
      for (int b = 0; b < NB; ++b)
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) {
          Ch o;
#pragma unroll
          for (int q = 0; q < CP; q += 2) {
            const V2 v = c[jj][kk][(b * BTE2_P + ch * CP + q) / 2];
            o.v[q] = v.x; o.v[q + 1] = v.y;
          }
          xout[xpl2_index<T>(P, ty, tz, b0 + b, K, kk, jj, ch, J)] = o;
        }
  __threadfence();
  __syncthreads();
  if (tid == 0) st_release_gpu(P.prog + unit, ebase + 0xffff);
}

template <typename T, int W, bool MASKED>
__global__ void __launch_bounds__(W * 32) bte2_sweep_kernel(const __grid_constant__ Bte2Dev P,
                                                            const __grid_constant__ Bte2Coefs<T> CF) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NBMAX = sizeof(T) == 4 ? 2 : 1, D = BTE2_DIST(W, T);
  __shared__ int s_unit;
  __shared__ uint64_t s_stepbar;
  unsigned bpar = 0;
  if (BTE2_SPLITBAR && threadIdx.x == 0) mbar_init(&s_stepbar, W * 32);
  for (;;) {
    __syncthreads();
    if (threadIdx.x == 0) s_unit = atomicAdd(P.ticket, 1);
    __syncthreads();
    const int unit = s_unit;
    if (unit >= P.n_units) break;
    const Bte2Unit un = P.units[unit];
    if (NBMAX == 2 && un.nb == 2) bte2_run_unit<T, NBMAX, W, D, MASKED>(P, CF, un, smem_raw, unit, &s_stepbar, bpar);
    else bte2_run_unit<T, 1, W, D, MASKED>(P, CF, un, smem_raw, unit, &s_stepbar, bpar);
  }
}

// ------------------------------------------------------------------ boundary kernels (v2 layouts)
// chunk holding direction p of band b on the face plane of octant o, axis a, at oriented cell (ip,jp,kp);
// side 0 = inflow plane, 1 = outflow plane
template <typename T>
__device__ __forceinline__ Bte2Chunk<T> *bte2_plane_chunk(const Bte2Dev &P, int o, int a, int side, int b, int ch,
                                                          int ip, int jp, int kp) {
  const Bte2Oct &O = P.oct[o];
  if (a == 0) {
    const int ty = jp >> 6, J = (jp & 63) >> 1, jj = jp & 1, tz = kp / (2 * P.W), K = (kp % (2 * P.W)) >> 1, kk = kp & 1;
    return reinterpret_cast<Bte2Chunk<T> *>(side ? const_cast<void *>(O.xprev) : O.xin) + xpl2_index<T>(P, ty, tz, b, K, kk, jj, ch, J);
  }
  if (a == 1) {
    const int tz = kp / (2 * P.W), K = (kp % (2 * P.W)) >> 1, kk = kp & 1;
    return reinterpret_cast<Bte2Chunk<T> *>(side ? const_cast<void *>(O.yprev) : O.ypl) + ypl2_index<T>(P, 0, tz, b, K, ip, kk, ch);
  }
  const int ty = jp >> 6, J = (jp & 63) >> 1, jj = jp & 1;
  return reinterpret_cast<Bte2Chunk<T> *>(side ? const_cast<void *>(O.zprev) : O.zpl) + zpl2_index<T>(P, 0, ty, b, ip + J, jj, ch, J);
}

struct Bte2Face { int na, nb; };
__device__ __forceinline__ Bte2Face bte2_face(const Bte2Dev &P, int a) {
  Bte2Face g;
  if (a == 0) { g.na = P.ny; g.nb = P.nz; } else if (a == 1) { g.na = P.nx; g.nb = P.nz; } else { g.na = P.nx; g.nb = P.ny; }
  return g;
}
// oriented coordinates of the boundary cell (ta, tb) of face axis a for octant o
__device__ __forceinline__ void bte2_face_cell(const Bte2Dev &P, int o, int a, int side_phys, int ta, int tb, int &ip, int &jp, int &kp) {
  const Bte2Oct &O = P.oct[o];
  int i, j, k;
  if (a == 0) { i = side_phys ? P.nx - 1 : 0; j = ta; k = tb; }
  else if (a == 1) { j = side_phys ? P.ny - 1 : 0; i = ta; k = tb; }
  else { k = side_phys ? P.nz - 1 : 0; i = ta; j = tb; }
  ip = O.sx > 0 ? i : P.nx - 1 - i; jp = O.sy > 0 ? j : P.ny - 1 - j; kp = O.sz > 0 ? k : P.nz - 1 - k;
}

// G_{f,b}(cell) = (1/Pi_f) sum_{s.n>0} w (s.n) e^n for DIFFUSE box faces (Eq. 6, reading G10)
template <typename T>
__global__ void bte2_gdiff_kernel(const __grid_constant__ Bte2Dev P) {
  constexpr int CP = 16 / sizeof(T), NCH = BTE2_P / CP;
  T *Gf = reinterpret_cast<T *>(P.Gf);
  // one flat index space over the entries of all six faces (all faces in flight at once)
  for (int64_t eg = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; eg < P.gf_off[6]; eg += (int64_t)gridDim.x * blockDim.x) {
    int f = 0;
    while (f < 5 && eg >= P.gf_off[f + 1]) ++f;
    if (P.face_type[f] != 1) continue;
    const int a = f >> 1, side = f & 1;
    const Bte2Face g = bte2_face(P, a);
    const int64_t e = eg - P.gf_off[f];
    const int ta = (int)(e % g.na), tb = (int)((e / g.na) % g.nb), b = (int)(e / ((int64_t)g.na * g.nb));
    double H = 0.0;
#pragma unroll
    for (int o = 0; o < 8; ++o) {
      const Bte2Oct &O = P.oct[o];
      const int sg = a == 0 ? O.sx : (a == 1 ? O.sy : O.sz);
      if ((sg > 0) != (side == 1)) continue;          // outgoing octants only
      int ip, jp, kp;
      bte2_face_cell(P, o, a, side, ta, tb, ip, jp, kp);
      Bte2Chunk<T> v[NCH];
#pragma unroll
      for (int ch = 0; ch < NCH; ++ch) v[ch] = ldcg_chunk<T>(bte2_plane_chunk<T>(P, o, a, 1, b, ch, ip, jp, kp));
#pragma unroll
      for (int ch = 0; ch < NCH; ++ch)
#pragma unroll
        for (int q = 0; q < CP; ++q) H += P.wsa[ch * CP + q][a] * (double)v[ch].v[q];
    }
    Gf[eg] = (T)(H / P.Pi_face[f]);
  }
}

// Fill the inflow ghost planes of isothermal (Eq. 5) and diffuse (Eq. 6) box faces.  Specular (Eq. 7) and periodic
// faces need none: their inflow IS another outflow plane of the previous iteration (Bte2Oct::xsrc / ysrc0 / zsrc0).
template <typename T>
__global__ void bte2_ghost_kernel(const __grid_constant__ Bte2Dev P) {
  constexpr int CP = 16 / sizeof(T), NCH = BTE2_P / CP;
  const T *Gf = reinterpret_cast<const T *>(P.Gf);
  const int64_t gtid = blockIdx.x * (int64_t)blockDim.x + threadIdx.x, gstride = (int64_t)gridDim.x * blockDim.x;
  // one flat index space over the (octant, axis) ghost planes that need filling: all of them concurrently
  for (int64_t eg = gtid; eg < P.gseg_off[P.gseg_n]; eg += gstride) {
    int sgi = 0;
    while (sgi + 1 < P.gseg_n && eg >= P.gseg_off[sgi + 1]) ++sgi;
    const int o = P.gseg_oa[sgi] / 3, a = P.gseg_oa[sgi] % 3;
    const int64_t e = eg - P.gseg_off[sgi];
    const Bte2Oct &O = P.oct[o];
    const int sg = a == 0 ? O.sx : (a == 1 ? O.sy : O.sz);
    const int side = sg > 0 ? 0 : 1, f = 2 * a + side;   // physical face the octant enters through
    const int type = P.face_type[f];                     // 0 isothermal (Eq. 5) or 1 diffuse (Eq. 6)
    const Bte2Face g = bte2_face(P, a);
    // thread order follows the plane layouts so that writes coalesce: x planes [..][chunk][J]: j fastest;
    // y planes [..][i'][kk][chunk]: chunk, then i; z planes [..][u][jj][chunk][J]: j fastest, then chunk, then i
    int ta, tb, ch;
    if (a == 0) { ta = (int)(e % g.na); ch = (int)((e / g.na) % NCH); tb = (int)((e / ((int64_t)g.na * NCH)) % g.nb); }
    else if (a == 1) { ch = (int)(e % NCH); ta = (int)((e / NCH) % g.na); tb = (int)((e / ((int64_t)g.na * NCH)) % g.nb); }
    else { tb = (int)(e % g.nb); ch = (int)((e / g.nb) % NCH); ta = (int)((e / ((int64_t)g.nb * NCH)) % g.na); }
    const int b = (int)(e / ((int64_t)g.na * NCH * g.nb));
    int ip, jp, kp;
    bte2_face_cell(P, o, a, side, ta, tb, ip, jp, kp);
    Bte2Chunk<T> v;
    if (type == 0) {
#pragma unroll
      for (int q = 0; q < CP; ++q) v.v[q] = (T)P.face_e0[f][b];
    } else {
      const T gv = Gf[P.gf_off[f] + ((int64_t)b * g.nb + tb) * g.na + ta];
#pragma unroll
      for (int q = 0; q < CP; ++q) v.v[q] = gv;
    }
    *bte2_plane_chunk<T>(P, o, a, 0, b, ch, ip, jp, kp) = v;
  }
  // interface faces: G = C dT_w / 4pi (isothermal) or (sum of the 4 outgoing octants' partial sums) / Pi_f (diffuse)
  T *Gi = reinterpret_cast<T *>(P.Gi);
  const int64_t ni = (int64_t)P.n_iface * P.B;
  for (int64_t e = gtid; e < ni; e += gstride) {
    const int64_t fid = e / P.B;
    const int b = (int)(e % P.B);
    if (P.iface_type == 0) { Gi[e] = (T)P.iface_e0[b]; continue; }
    double H = 0.0;
    const T *hp = reinterpret_cast<const T *>(P.Hd) + (((int64_t)P.iface_info[fid] * P.ncell + P.iface_cell[fid]) * P.B + b) * 4;
    for (int sl = 0; sl < 4; ++sl) H += (double)hp[sl];
    Gi[e] = (T)(H / P.Pi_face[P.iface_info[fid]]);
  }
  if (gtid == 0) *P.ticket = 0;
}

// ------------------------------------------------------------------ (c) update + residual, v2 layouts
// dT^{n+1} = M0 / sum(C/tau) (Eq. 16), q = M1 (Eq. 4), residual partial sums (Eq. 23); octant partials are
// summed in fp64 in a fixed order; dT is written back into the four skewed class copies the sweep reads.
template <typename T>
__global__ void __launch_bounds__(256, 4) bte2_update_kernel(const __grid_constant__ Bte2Dev P) {
  double sT = 0, mT = 0, sq = 0, mq = 0;
  // 32-bit cell index (host check: ncell < 2^31): the 64-bit divisions of the first version kept the XU pipe half busy
  const unsigned ncell = (unsigned)P.ncell, nxu = (unsigned)P.nx, nyu = (unsigned)P.ny;
  for (unsigned c = blockIdx.x * blockDim.x + threadIdx.x; c < ncell; c += gridDim.x * blockDim.x) {
    if (P.code && !(P.code[c] & 1)) continue;          // void cell: dT, q stay 0
    const unsigned row = c / nxu;
    const int i = (int)(c - row * nxu), k = (int)(row / nyu), j = (int)(row - (unsigned)k * nyu);
    int64_t sk[4];
#pragma unroll
    for (int cl = 0; cl < 4; ++cl)
      sk[cl] = sk2_index(P.nty, P.NU, (cl & 1) ? P.nx - 1 - i : i, (cl & 2) ? P.ny - 1 - j : j, k);
    double m0 = 0, m1 = 0, m2 = 0, m3 = 0;
#pragma unroll
    for (int o = 0; o < 8; ++o) {
      const Bte2Oct &O = P.oct[o];
      const Bte2Mom<T> *Mp = reinterpret_cast<const Bte2Mom<T> *>(O.M) + sk[o & 3];
      T v[4];
      if (sizeof(T) == 4) {
        const float4 x = __ldcg(reinterpret_cast<const float4 *>(Mp));
        memcpy(v, &x, 16);
      } else {
        const double2 x = __ldcg(reinterpret_cast<const double2 *>(Mp)), y = __ldcg(reinterpret_cast<const double2 *>(Mp) + 1);
        memcpy(v, &x, 16); memcpy(reinterpret_cast<char *>(v) + 16, &y, 16);
      }
      m0 += (double)v[0]; m1 += O.sx * (double)v[1]; m2 += O.sy * (double)v[2]; m3 += O.sz * (double)v[3];
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
    for (int cl = 0; cl < 4; ++cl) reinterpret_cast<Bte2Pair<T> *>(P.dTQ[cl])[sk[cl]].x = (T)Tn;
  }
  block_reduce4(sT, mT, sq, mq);
  if (threadIdx.x == 0) {
    P.red[blockIdx.x] = sT; P.red[P.n_red_blocks + blockIdx.x] = mT;
    P.red[2 * P.n_red_blocks + blockIdx.x] = sq; P.red[3 * P.n_red_blocks + blockIdx.x] = mq;
  }
}

// physical fp64 field -> the four skewed class copies: which = 0: Q * scale -> .y ; 1: dT -> .x (and P.dT)
template <typename T>
__global__ void bte2_skew_kernel(const __grid_constant__ Bte2Dev P, const double *src, double scale, int which) {
  for (int64_t c = blockIdx.x * (int64_t)blockDim.x + threadIdx.x; c < P.ncell; c += (int64_t)gridDim.x * blockDim.x) {
    const int i = (int)(c % P.nx), j = (int)((c / P.nx) % P.ny), k = (int)(c / ((int64_t)P.nx * P.ny));
    for (int cl = 0; cl < 4; ++cl) {
      Bte2Pair<T> *d = reinterpret_cast<Bte2Pair<T> *>(P.dTQ[cl]) +
                       sk2_index(P.nty, P.NU, (cl & 1) ? P.nx - 1 - i : i, (cl & 2) ? P.ny - 1 - j : j, k);
      const bool solid = !P.code || (P.code[c] & 1);    // void cells hold 0 (bte.h: "void cells 0")
      if (which == 0) d->y = (T)(src[c % P.src_mod] * scale); else d->x = solid ? (T)src[c % P.src_mod] : (T)0;
    }
    if (which == 1) P.dT[c] = (!P.code || (P.code[c] & 1)) ? src[c % P.src_mod] : 0.0;
  }
}
#endif  // __CUDACC__
