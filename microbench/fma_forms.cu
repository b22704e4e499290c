// Microbenchmark (not part of the library): FMA-pipe rate of the FFMA / FFMA2 operand forms the sweep uses, on sm_100a.
// Build + run:  nvcc -gencode arch=compute_100a,code=sm_100a -O3 -std=c++17 -o /tmp/fma_forms microbench/fma_forms.cu && /tmp/fma_forms
// Result on B200: profiles/r01_fma_forms_microbench.txt (every form with a uniform-register coefficient runs at the full 128 FMA/clk/SM).
#include <cstdio>
#include <cuda_runtime.h>
struct Coefs { float k[64]; };
#define NACC 16
#define ITERS 2000
template <int FORM>
__global__ void __launch_bounds__(256) kern(const __grid_constant__ Coefs CF, float *out, const float *vin) {
  float2 a[NACC];
#pragma unroll
  for (int i = 0; i < NACC; ++i) a[i] = make_float2(threadIdx.x * 1e-3f + i, i * 0.5f);
  float2 vr[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) vr[i] = make_float2(vin[(threadIdx.x + i) & 63], vin[(threadIdx.x + 2 * i + 1) & 63]);
  for (int it = 0; it < ITERS; ++it) {
#pragma unroll
    for (int j = 0; j < 8; ++j) {
#pragma unroll
      for (int i = 0; i < NACC; ++i) {
        if (FORM == 0) { a[i].x = fmaf(a[i].x, vr[j].x, vr[j].y); a[i].y = fmaf(a[i].y, vr[j].x, vr[j].y); }                  // FFMA RRR
        if (FORM == 1) { a[i].x = fmaf(a[i].x, CF.k[2 * j], vr[j].y); a[i].y = fmaf(a[i].y, CF.k[2 * j + 1], vr[j].y); }     // FFMA R,UR,R
        if (FORM == 2) a[i] = __ffma2_rn(a[i], vr[j], vr[(j + 1) & 7]);                                                       // FFMA2 RRR
        if (FORM == 3) a[i] = __ffma2_rn(a[i], make_float2(CF.k[2 * j], CF.k[2 * j + 1]), vr[j]);                             // FFMA2 R,URpair,R
        if (FORM == 4) a[i] = __ffma2_rn(a[i], make_float2(CF.k[j], CF.k[j]), vr[j]);                                         // FFMA2 R,UR broadcast,R
        if (FORM == 5) a[i] = __ffma2_rn(vr[j], make_float2(CF.k[2 * j], CF.k[2 * j + 1]), a[i]);                             // acc form: a += v*URpair
        if (FORM == 6) { a[i].x = fmaf(vr[j].x, CF.k[2 * j], a[i].x); a[i].y = fmaf(vr[j].y, CF.k[2 * j + 1], a[i].y); }      // acc form scalar UR
        if (FORM == 7) a[i] = __ffma2_rn(vr[j], make_float2(CF.k[j], CF.k[j]), a[i]);                                         // acc form: UR broadcast
      }
    }
  }
  float s = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += a[i].x + a[i].y;
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// dependent-issue latency: ONE warp per SM, one accumulator chain (each instruction needs the previous result)
template <int FORM>
__global__ void __launch_bounds__(32) lat(const __grid_constant__ Coefs CF, float *out, const float *vin, long long *cyc) {
  float2 a = make_float2(threadIdx.x * 1e-3f, 0.5f);
  const float2 v = make_float2(vin[threadIdx.x & 63], vin[(threadIdx.x + 1) & 63]);
  const long long t0 = clock64();
  for (int it = 0; it < ITERS; ++it) {
#pragma unroll
    for (int j = 0; j < 32; ++j) {
      if (FORM == 0) a.x = fmaf(a.x, CF.k[j], v.y);                                        // FFMA R,UR,R chain
      if (FORM == 1) a = __ffma2_rn(a, make_float2(CF.k[2 * (j & 7)], CF.k[2 * (j & 7) + 1]), v);   // FFMA2 R,URpair,R chain
      if (FORM == 2) a = __ffma2_rn(v, make_float2(CF.k[2 * (j & 7)], CF.k[2 * (j & 7) + 1]), a);   // FFMA2 accumulate chain
    }
  }
  const long long t1 = clock64();
  out[blockIdx.x * 32 + threadIdx.x] = a.x + a.y;
  if (threadIdx.x == 0 && blockIdx.x == 0) *cyc = t1 - t0;
}
template <int FORM> void runlat(const char *name, float *out, float *vin) {
  Coefs cf; for (int i = 0; i < 64; ++i) cf.k[i] = 0.5f + 1e-3f * i;
  long long *d, h = 0; cudaMalloc(&d, 8);
  lat<FORM><<<148, 32>>>(cf, out, vin, d); cudaDeviceSynchronize();
  cudaMemcpy(&h, d, 8, cudaMemcpyDeviceToHost);
  printf("%-28s dependent chain: %.2f cycles per instruction\n", name, (double)h / (ITERS * 32.0));
  cudaFree(d);
}

// FP64: DFMA throughput (register operands), same launch shape
__global__ void __launch_bounds__(256) kern64(double *out, const double *vin) {
  double a[NACC];
#pragma unroll
  for (int i = 0; i < NACC; ++i) a[i] = threadIdx.x * 1e-3 + i;
  const double x = vin[threadIdx.x & 31], y = vin[(threadIdx.x + 1) & 31];
  for (int it = 0; it < ITERS; ++it)
#pragma unroll
    for (int j = 0; j < 8; ++j)
#pragma unroll
      for (int i = 0; i < NACC; ++i) a[i] = fma(a[i], x, y);
  double s = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += a[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
void run64(int bps) {
  double *out, *vin; cudaMalloc(&out, 148 * 8 * 256 * 8); cudaMalloc(&vin, 256); cudaMemset(vin, 0, 256);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int grid = 148 * bps;
  kern64<<<grid, 256>>>(out, vin); cudaDeviceSynchronize();
  cudaEventRecord(e0);
  for (int r = 0; r < 5; ++r) kern64<<<grid, 256>>>(out, vin);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 5;
  const double fma = (double)grid * 256 * ITERS * 8.0 * NACC;
  printf("%-28s blocks/SM=%d: %.3f ms  %.1f FMA/clk/SM (at 1.965 GHz)\n", "DFMA  R,R,R", bps, ms, fma / (ms * 1e-3) / 148 / 1.965e9);
  cudaFree(out); cudaFree(vin);
}
template <int FORM> void run(const char *name, int blocks_per_sm, float *out, float *vin) {
  Coefs cf; for (int i = 0; i < 64; ++i) cf.k[i] = 0.5f + 1e-3f * i;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  int grid = 148 * blocks_per_sm;
  kern<FORM><<<grid, 256>>>(cf, out, vin); cudaDeviceSynchronize();
  cudaEventRecord(e0);
  for (int r = 0; r < 5; ++r) kern<FORM><<<grid, 256>>>(cf, out, vin);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1); ms /= 5;
  double fma = (double)grid * 256 * ITERS * 8.0 * NACC * 2;
  printf("%-28s blocks/SM=%d: %.3f ms  %.1f FMA/clk/SM (at 1.965 GHz)  err=%d\n", name, blocks_per_sm, ms, fma / (ms * 1e-3) / 148 / 1.965e9, (int)cudaGetLastError());
}
int main() {
  float *out, *vin; cudaMalloc(&out, 148 * 8 * 256 * 4); cudaMalloc(&vin, 256); cudaMemset(vin, 0, 256);
  for (int bps = 1; bps <= 2; ++bps) {
    run<0>("FFMA  R,R,R", bps, out, vin);
    run<1>("FFMA  R,UR,R", bps, out, vin);
    run<2>("FFMA2 R,R,R", bps, out, vin);
    run<3>("FFMA2 R,URpair,R", bps, out, vin);
    run<4>("FFMA2 R,URbcast,R", bps, out, vin);
    run<5>("FFMA2 acc+=R*URpair", bps, out, vin);
    run<6>("FFMA  acc+=R*UR", bps, out, vin);
    run<7>("FFMA2 acc+=R*URbcast", bps, out, vin);
  }
  run64(1); run64(2);
  runlat<0>("FFMA  R,UR,R", out, vin);
  runlat<1>("FFMA2 R,URpair,R", out, vin);
  runlat<2>("FFMA2 acc+=R*URpair", out, vin);
  return 0;
}
