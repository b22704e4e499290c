// Warp-specialised variant of the fast sweep (same tiles, layouts, arithmetic and dependency protocol as
// bte_sweep2.cuh).  One CTA = W compute warps + 4 helper warps:
//   compute warp K : arithmetic of its 2x2 row patches, z exchange with warp K-1 / K+1 through shared memory,
//                    outflow faces and moments stored straight from registers; never polls, never prefetches inputs;
//   helper warp h  : serves compute warps h and h + 4: polls the progress flags of the units this one follows,
//                    cp.async-prefetches everything a step consumes (cell inputs, mask codes, y / z inflow rows)
//                    R - 1 steps ahead into a ring of R slots, and publishes the progress of its compute warps.
// Hand-shakes are mbarriers in shared memory: full[K][slot] (helper's copies have landed: cp.async.mbarrier.arrive),
// cdone[K][slot] (compute warp K finished the step that used the slot: its stores are issued, the slot is free) and the
// CTA-wide split step barrier of the compute warps (every arithmetic(t) before any arithmetic(t + 1)).
// Progress is published per WARP (prog[unit * W + K]) so that no CTA-wide agreement is needed to publish.
#pragma once
#include "bte_sweep2.cuh"

#ifdef __CUDACC__
#define BTE3_HELPERS 4                                 // helper warps (one warpgroup, so that setmaxnreg applies)
#define BTE3_THREADS(W) ((W) * 32 + BTE3_HELPERS * 32)
#define BTE3_ELAG 2   // a helper makes sure of step t + ELAG before it loads step t: the compute warp prefetches the
                      // accumulator rows of step t + 1 + MDIST on its own once it has seen full(t)

template <typename T, int NB, int W, int R> struct Bte3Smem {
  static constexpr int CP = 16 / sizeof(T);
  static constexpr int NCH = BTE2_P / CP;
  static constexpr int NC = NB * NCH;
  typedef Bte2Chunk<T> Ch;
  Ch zex[2][W][2][NC][32];           // [parity][K][jj][chunk][lane]: kk=1 rows of warp K, read by warp K+1 / copied out by warp Kl itself
  Ch yst[2][W][2 * NC];              // [parity][warp][kk*NC + chunk]: jj=1 rows of lane Jl, copied out by the warp one step later
  Ch zin0[R][2][NC][32];             // staged z inflow plane of warp 0
  Ch ybuf[R][W][2][NC];              // [ring][warp][kk][chunk]: y inflow of lane 0
  Bte2Mom<T> mold[BTE2_MDIST(T) + 1][2][2][W * 32];  // previous content of the moment accumulator (compute warps' own cp.async)
  Bte2Pair<T> inp[R][2][2][W * 32];  // [ring][kk][jj][tid] (dT, Q/sumC) of the cell
  uint32_t codes[R][W * 32];         // [ring][tid] cell bytes of the thread's patch (masked grids only)
};
template <int W, int R> struct Bte3Bars {
  uint64_t full[W][R], cdone[W][R], step;
};

// helper-side wait: sleeps between probes so that the probes (shared-memory pipe) do not compete with the SHFL / LDS /
// STS traffic of the compute warps
__device__ __forceinline__ void mbar_wait_polite(uint64_t *b, unsigned parity) {
  asm volatile(
      "{\n.reg .pred P1;\nLAB_WAIT:\nmbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n@P1 bra DONE;\nnanosleep.u32 256;\nbra LAB_WAIT;\nDONE:\n}" ::"r"(smem_u32(b)),
      "r"(parity)
      : "memory");
}
__device__ __forceinline__ void cp_async_mbar_arrive_noinc(uint64_t *b) {
  asm volatile("cp.async.mbarrier.arrive.noinc.shared::cta.b64 [%0];" ::"r"(smem_u32(b)) : "memory");
}

// ------------------------------------------------------------------ compute warps: one unit
template <typename T, int NB, int W, int R, bool MASKED>
__device__ __forceinline__ void bte3_compute_unit(const Bte2Dev &P, const Bte2Coefs<T> &CF, const Bte2Unit &un,
                                                  unsigned char *smem_raw, Bte3Bars<W, R> *BR, const int K, unsigned &bpar,
                                                  unsigned &g) {
  typedef Bte3Smem<T, NB, W, R> SM;
  SM *S = reinterpret_cast<SM *>(smem_raw);
  constexpr int CP = SM::CP, NCH = SM::NCH, NC = SM::NC, MD = BTE2_MDIST(T);
  typedef Bte2Chunk<T> Ch;
  const unsigned FULL = 0xffffffffu;
  const int J = threadIdx.x & 31, tid = K * 32 + J;
  const Bte2Oct &O = P.oct[un.oct];
  const int ty = un.ty, tz = un.tz, b0 = un.b0;
  const int jp0 = ty * 64 + 2 * J, kp0 = tz * 2 * W + 2 * K;
  const bool vthread = (jp0 < P.ny) && (kp0 < P.nz);
  const int Jl = (min(P.ny, (ty + 1) * 64) - 1 - ty * 64) >> 1, Kl = (min(P.nz, (tz + 1) * 2 * W) - 1 - tz * 2 * W) >> 1;
  const bool first = un.dep_prev < 0;                  // first band group of this octant: M is written, not added to
  const bool lastK = K == Kl;                          // this warp's kk=1 rows are the tile's z outflow
  auto saddr = [&](const void *ptr) { return (unsigned)__cvta_generic_to_shared(ptr); };

  const Ch *xin = reinterpret_cast<const Ch *>(O.xsrc);
  Ch *xout = reinterpret_cast<Ch *>(O.xdst);
  Bte2Mom<T> *M = reinterpret_cast<Bte2Mom<T> *>(O.M);

  // cell index of row (jj,kk) at step t: cbase[kk] + jj*32 + (t - K) * 64
  int64_t cbase[2];
#pragma unroll
  for (int kk = 0; kk < 2; ++kk) {
    const int kp = kp0 + kk, k = vthread ? (O.sz > 0 ? kp : P.nz - 1 - kp) : 0;
    cbase[kk] = (((int64_t)k * P.nty + ty) * P.NU) * 64 + J - (int64_t)K * 64;
  }
  const int fu[3] = {O.sx > 0 ? 0 : 1, O.sy > 0 ? 2 : 3, O.sz > 0 ? 4 : 5};      // upwind faces x, y, z
  // outflow planes: z rows [b][u][jj][ch][lane] are copied out of zex by warp Kl itself (every lane the chunks it
  // wrote), y rows [b][K][i'][kk][ch] are staged by lane Jl and copied out by the warp one step later
  const int64_t zstep = 2 * NCH * 32, zband = (int64_t)P.NU * 2 * NCH * 32;
  Ch *zdl = (tz == P.ntz - 1 ? reinterpret_cast<Ch *>(O.zdstN) : reinterpret_cast<Ch *>(O.zpl) + zpl2_index<T>(P, tz + 1, 0, 0, 0, 0, 0, 0)) +
            zpl2_index<T>(P, 0, ty, b0, 0, 0, 0, J) - (int64_t)K * zstep;
  const int yb = J / (2 * NCH), ykk = (J / NCH) & 1, ych = J % NCH;     // lane l < 2 NC copies chunk (b, kk, ch) of the y outflow
  Ch *ydl = (ty == P.nty - 1 ? reinterpret_cast<Ch *>(O.ydstN) : reinterpret_cast<Ch *>(O.ypl) + ypl2_index<T>(P, ty + 1, 0, 0, 0, 0, 0, 0)) +
            ypl2_index<T>(P, 0, tz, b0 + (J < 2 * NC ? yb : 0), K, 0, ykk, ych) - (int64_t)(Jl + K) * 2 * NCH;

  // ---- previous content of the moment accumulator for step t1 (this thread's own cp.async group)
  auto prefetch_m = [&](int t1) {
    const int ip1 = t1 - J - K;
    if (!first && vthread && ip1 >= 0 && ip1 < P.nx) {
#pragma unroll
      for (int kk = 0; kk < 2; ++kk)
#pragma unroll
        for (int jj = 0; jj < 2; ++jj) {
          const int64_t ci = cbase[kk] + jj * 32 + (int64_t)t1 * 64;
#pragma unroll
          for (int h = 0; h < (int)sizeof(Bte2Mom<T>) / 16; ++h)
            cp_async<16>(saddr(&S->mold[t1 % (MD + 1)][kk][jj][tid]) + 16 * h, reinterpret_cast<const char *>(M + ci) + 16 * h);
        }
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

  T bcx[NB], bcy[NB];
#pragma unroll
  for (int b = 0; b < NB; ++b) { bcx[b] = CF.bc[b0 + b][0]; bcy[b] = CF.bc[b0 + b][1]; }

  // one (band, chunk) of the 2x2 patch: FAST = every lane of the warp is active (no predication)
  auto chunk = [&](auto fastc, int b, int ch, const V2 (&r)[2][2], V2 (&m)[2][2][4], int rb, bool act,
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

  // the helper has made sure of the dependencies of steps <= ELAG before it filled the slot of step 0
  mbar_wait(&BR->full[K][g % R], (g / R) & 1u);
  if (MD == 1) { prefetch_m(0); cp_async_commit(); }
  prefetch_m(MD); cp_async_commit();

  for (int t = 0; t < P.nsteps; ++t) {
    const int cur = t & 1;
    const unsigned gs = g + t;
    const int rb = (int)(gs % R);
    const int ip = t - J - K;
    const bool act = vthread && ip >= 0 && ip < P.nx;
    if (t > 0) {
      mbar_wait(&BR->full[K][rb], (gs / R) & 1u);      // inputs of step t have landed
      mbar_wait(&BR->step, bpar);                      // every compute warp is done with arithmetic(t - 1)
      bpar ^= 1u;
    }

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
        T g4[4][3];
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
          const int jj = cc & 1, kk = cc >> 1;
          const int i = O.sx > 0 ? ip : P.nx - 1 - ip, j = O.sy > 0 ? jp0 + jj : P.ny - 1 - jp0 - jj,
                    k = O.sz > 0 ? kp0 + kk : P.nz - 1 - kp0 - kk;
          cph[cc] = (int64_t)i + (int64_t)P.nx * (j + (int64_t)P.ny * k);
#pragma unroll
          for (int a = 0; a < 3; ++a) {
            g4[cc][a] = (T)0;
            if (live && (cb[cc] & 1u) && ((cb[cc] >> (1 + fu[a])) & 1u))
              g4[cc][a] = P.iface_type == 0 ? (T)P.iface_e0[b0 + b]
                                            : reinterpret_cast<const T *>(P.Gi)[(int64_t)__ldg(P.iface + (int64_t)fu[a] * P.ncell + cph[cc]) * P.B + b0 + b];
          }
        }
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) chunk_masked(b, ch, r, m, rb, live, cb, g4, zrd, zwr);
        {
          // outgoing hemispherical partial sums at solid/void faces (diffuse interface, Eq. 6)
          uint32_t anydn = 0;
#pragma unroll
          for (int cc = 0; cc < 4; ++cc)
            if (cb[cc] & 1u) anydn |= cb[cc] & ((2u << (fu[0] ^ 1)) | (2u << (fu[1] ^ 1)) | (2u << (fu[2] ^ 1)));
          if (P.iface_type == 1 && live && anydn != 0) {
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
              const int jj = cc & 1, kk = cc >> 1;
              if (!(cb[cc] & 1u)) continue;
#pragma unroll
              for (int a = 0; a < 3; ++a) {
                const int fd = fu[a] ^ 1;
                if (!((cb[cc] >> (1 + fd)) & 1u)) continue;
                // sum_p w_p |s_p,a| e_p in the compute type with the moment coefficients v_b w |s_a| (<= 16 terms of
                // one sign pattern), divided by v_b; the sum over the 4 outgoing octants is fp64 (ghost kernel).
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
      } else if (fast) {
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) chunk(std::true_type{}, b, ch, r, m, rb, true, zrd, zwr);
      } else {
#pragma unroll
        for (int ch = 0; ch < NCH; ++ch) chunk(std::false_type{}, b, ch, r, m, rb, live, zrd, zwr);
      }
    }

    mbar_arrive(&BR->step);            // this thread's shared-memory reads and writes of step t are done
    cp_async_wait<MD>();               // the accumulator rows of step t (this thread's own copies) have landed
    if (act) {
      // (b) moments of this band group into the octant accumulator (one owner per cell and group)
#pragma unroll
      for (int kk = 0; kk < 2; ++kk) {
#pragma unroll
        for (int jj = 0; jj < 2; ++jj) {
          if (MASKED && !(cb[jj + 2 * kk] & 1u)) continue;      // void cell
          Bte2Mom<T> o;
          if (first) {
#pragma unroll
            for (int q = 0; q < 4; ++q) o.v[q] = m[jj][kk][q].x + m[jj][kk][q].y;
          } else {
            const Bte2Mom<T> old = S->mold[t % (MD + 1)][kk][jj][tid];
#pragma unroll
            for (int q = 0; q < 4; ++q) o.v[q] = old.v[q] + (m[jj][kk][q].x + m[jj][kk][q].y);
          }
          M[cbase[kk] + jj * 32 + (int64_t)t * 64] = o;
        }
      }
    }
    if (act && J == Jl) {              // y outflow rows (jj = 1 of lane Jl) -> staging buffer
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
            S->yst[cur][K][kk * NC + b * NCH + ch] = o;
          }
    }
    if (lastK) {                       // z outflow of the tile: this warp's own rows of step t, zex -> plane
      const int ul = t - K;
      if (ul >= 0 && ul < P.NU) {
#pragma unroll
        for (int q = 0; q < 2 * NC; ++q) {
          const int b = q / (2 * NCH), rem = q % (2 * NCH);
          zdl[b * zband + (int64_t)t * zstep + rem * 32] = S->zex[cur ^ 1][K][rem / NCH][b * NCH + rem % NCH][J];
        }
      }
    }
    __syncwarp();
    {                                  // y outflow of step t: staged row -> plane (lanes < 2 NC, one chunk each)
      const int ipl = t - Jl - K;
      if (kp0 < P.nz && J < 2 * NC && ipl >= 0 && ipl < P.nx) ydl[(int64_t)t * 2 * NCH] = S->yst[cur][K][ykk * NC + yb * NCH + ych];
    }
    // accumulator rows of step t + 1 + MD: the helper knew them published when it filled the slot of step t
    prefetch_m(t + 1 + MD);
    cp_async_commit();
    __syncwarp();
    if (J == 0) mbar_arrive(&BR->cdone[K][rb]);        // the stores of step t are issued, its ring slot is free
  }
  g += (unsigned)P.nsteps;
  cp_async_wait<0>();
  mbar_wait(&BR->step, bpar);                          // (keeps the barrier's phase in step with bpar across units)
  bpar ^= 1u;

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
}

// ------------------------------------------------------------------ helper warps: one unit
// Helper warp h serves compute warps K = h and h + BTE3_HELPERS (if < W).  Lane l loads what compute lane l of that
// warp consumes.  Pollers: lanes 0 / 1 hold the progress of dep_y / dep_prev for the first warp served, lanes 2 / 3
// for the second one, lane 4 the progress of dep_z (helper of warp 0 only).
template <typename T, int NB, int W, int R, bool MASKED>
__device__ __forceinline__ void bte3_helper_unit(const Bte2Dev &P, const Bte2Unit &un, unsigned char *smem_raw,
                                                 Bte3Bars<W, R> *BR, const int unit, const int h, unsigned &g) {
  typedef Bte3Smem<T, NB, W, R> SM;
  SM *S = reinterpret_cast<SM *>(smem_raw);
  constexpr int NCH = SM::NCH, NC = SM::NC, NSRV = (W + BTE3_HELPERS - 1) / BTE3_HELPERS;
  typedef Bte2Chunk<T> Ch;
  const int J = threadIdx.x & 31;
  const Bte2Oct &O = P.oct[un.oct];
  const int ty = un.ty, tz = un.tz, b0 = un.b0;
  const int ebase = P.epoch << 16;
  auto saddr = [&](const void *ptr) { return (unsigned)__cvta_generic_to_shared(ptr); };
  const Bte2Pair<T> *dTQ = reinterpret_cast<const Bte2Pair<T> *>(P.dTQ[O.cls]);
  const Ch *zsrc = (tz == 0 ? reinterpret_cast<const Ch *>(O.zsrc0) : reinterpret_cast<const Ch *>(O.zpl) + zpl2_index<T>(P, tz, 0, 0, 0, 0, 0, 0)) +
                   zpl2_index<T>(P, 0, ty, b0, 0, 0, 0, J);
  const int64_t zstep = 2 * NCH * 32, zband = (int64_t)P.NU * 2 * NCH * 32;
  const int yb = J / (2 * NCH), ykk = (J / NCH) & 1, ych = J % NCH;
  const Ch *ybase = ty == 0 ? reinterpret_cast<const Ch *>(O.ysrc0) : reinterpret_cast<const Ch *>(O.ypl) + ypl2_index<T>(P, ty, 0, 0, 0, 0, 0, 0);

  // ---- pollers
  const int pk = J < 4 ? h + (J >> 1) * BTE3_HELPERS : 0;            // compute warp the lane polls for
  int mydep = -1, mylag = 0;
  if (J < 4 && pk < W) { mydep = (J & 1) ? un.dep_prev : un.dep_y; mylag = (J & 1) ? 1 : 33; if (mydep >= 0) mydep = mydep * W + pk; }
  if (J == 4 && h == 0 && un.dep_z >= 0) { mydep = un.dep_z * W + (W - 1); mylag = W + 1; }
  const int psrv = J == 4 ? 0 : (J >> 1);                            // index (0 / 1) of the warp served this lane polls for
  int seen = 0;
  auto ensure = [&](int s, int t1) {   // everything step t1 of served warp s reads from other units has been published
    if (mydep >= 0 && psrv == s && seen < t1 + mylag) {
      int v;
      while ((v = ld_acquire_gpu(P.prog + mydep) - ebase) < t1 + mylag) __nanosleep(32);
      seen = v;
    }
    __syncwarp();
  };

  for (int t = 0; t < P.nsteps; ++t) {
    const unsigned gs = g + t;
    const int rb = (int)(gs % R);
#pragma unroll
    for (int s = 0; s < NSRV; ++s) {
      const int K = h + s * BTE3_HELPERS;
      if (K >= W) break;
      if (gs >= (unsigned)R) {
        mbar_wait_polite(&BR->cdone[K][rb], ((gs / R) - 1u) & 1u);   // compute warp K finished step gs - R: the slot is free
        const int sd = t - R;                                         // ... a step of this unit if >= 0
        if (sd >= 0 && (sd & P.pub_mask) == P.pub_mask && J == 0) {   // faces and moments of steps <= sd are issued
          __threadfence();
          st_release_gpu(P.prog + unit * W + K, ebase + sd + 1);
        }
      }
      ensure(s, t + BTE3_ELAG);
      // ---- everything step t of compute warp K consumes -> ring slot rb
      const int kp0 = tz * 2 * W + 2 * K;
      const bool vthread = (ty * 64 + 2 * J < P.ny) && (kp0 < P.nz);
      const int ip1 = t - J - K;
      const int tid = K * 32 + J;
      if (vthread && ip1 >= 0 && ip1 < P.nx) {
#pragma unroll
        for (int kk = 0; kk < 2; ++kk) {
          const int kp = kp0 + kk, k = O.sz > 0 ? kp : P.nz - 1 - kp;
          const int64_t cb = (((int64_t)k * P.nty + ty) * P.NU) * 64 + J + (int64_t)(t - K) * 64;
#pragma unroll
          for (int jj = 0; jj < 2; ++jj) cp_async<sizeof(Bte2Pair<T>)>(saddr(&S->inp[rb][kk][jj][tid]), dTQ + cb + jj * 32);
        }
        if (MASKED) {
          const int kz = (O.sz > 0 ? kp0 : P.nz - 2 - kp0) >> 1;
          cp_async<4>(saddr(&S->codes[rb][tid]), P.codeP[O.cls] + (((int64_t)kz * P.nty + ty) * P.NU) * 32 + J + (int64_t)(t - K) * 32);
        }
      }
      if (K == 0 && t < P.NU) {
#pragma unroll
        for (int q = 0; q < 2 * NC; ++q) {             // lane J: the chunks (b, jj, ch) compute lane J reads
          const int b = q / (2 * NCH), rem = q % (2 * NCH);
          cp_async<16>(saddr(&S->zin0[rb][rem / NCH][b * NCH + rem % NCH][J]), zsrc + b * zband + t * zstep + rem * 32);
        }
      }
      {
        const int ipy = t - K;
        if (J < 2 * NC && ipy >= 0 && ipy < P.nx)
          cp_async<16>(saddr(&S->ybuf[rb][K][ykk][yb * NCH + ych]), ybase + ypl2_index<T>(P, 0, tz, b0 + yb, K, ipy, ykk, ych));
      }
      cp_async_mbar_arrive_noinc(&BR->full[K][rb]);    // completes (32 lanes) once this lane's copies have landed
    }
  }
  g += (unsigned)P.nsteps;
}

// ------------------------------------------------------------------ kernel
#define BTE3_RING(T) (BTE2_DIST(8, T) + 1)
template <typename T, int W, bool MASKED>
__global__ void __launch_bounds__(BTE3_THREADS(W), 1) bte3_sweep_kernel(const __grid_constant__ Bte2Dev P,
                                                                        const __grid_constant__ Bte2Coefs<T> CF) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  constexpr int NBMAX = sizeof(T) == 4 ? 2 : 1, R = BTE3_RING(T);
  __shared__ int s_unit;
  __shared__ Bte3Bars<W, R> s_bars;
  // the warp index through a shuffle: the compiler then knows it is warp-uniform, keeps the role branches and the
  // band-indexed coefficient addressing on the uniform datapath (FFMA2 with uniform-register operands)
  const int warp = __shfl_sync(0xffffffffu, (int)(threadIdx.x >> 5), 0);
  if (threadIdx.x == 0) {
    for (int k = 0; k < W; ++k)
      for (int r = 0; r < R; ++r) { mbar_init(&s_bars.full[k][r], 32); mbar_init(&s_bars.cdone[k][r], 1); }
    mbar_init(&s_bars.step, W * 32);
  }
  unsigned bpar = 0, g = 0;
  if (warp >= W) {
    if (W == 8) asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    for (;;) {
      __syncthreads();
      if (threadIdx.x == 0) s_unit = atomicAdd(P.ticket, 1);
      __syncthreads();
      const int unit = s_unit;
      if (unit >= P.n_units) break;
      const Bte2Unit un = P.units[unit];
      if (NBMAX == 2 && un.nb == 2) bte3_helper_unit<T, NBMAX, W, R, MASKED>(P, un, smem_raw, &s_bars, unit, warp - W, g);
      else bte3_helper_unit<T, 1, W, R, MASKED>(P, un, smem_raw, &s_bars, unit, warp - W, g);
      __syncthreads();                                 // the compute warps have stored their x outflow and fenced
      if ((threadIdx.x & 31) == 0)
        for (int K = warp - W; K < W; K += BTE3_HELPERS) st_release_gpu(P.prog + unit * W + K, (P.epoch << 16) + 0xffff);
    }
  } else {
    if (W == 8) asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
    for (;;) {
      __syncthreads();
      if (threadIdx.x == 0) s_unit = atomicAdd(P.ticket, 1);
      __syncthreads();
      const int unit = s_unit;
      if (unit >= P.n_units) break;
      const Bte2Unit un = P.units[unit];
      if (NBMAX == 2 && un.nb == 2) bte3_compute_unit<T, NBMAX, W, R, MASKED>(P, CF, un, smem_raw, &s_bars, warp, bpar, g);
      else bte3_compute_unit<T, 1, W, R, MASKED>(P, CF, un, smem_raw, &s_bars, warp, bpar, g);
      __syncthreads();
    }
  }
}
#endif  // __CUDACC__
