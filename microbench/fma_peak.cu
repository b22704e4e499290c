// Bench-only object (NOT part of the product library): measures the plain-ALU FMA peak that bench.py reports the
// sweep against -- a register-only chain of the instruction forms the sweep issues, on every SM, timed with CUDA
// events.  fp32: FFMA2 (two FMAs per instruction) with a uniform-register coefficient pair; fp64: DFMA.
// extern "C" so that bench.py can call it through ctypes.  Built by microbench.build() (__graft_entry__.build()).
#include <cstdint>
#include <cuda_runtime.h>

struct PeakCoefs { float k[64]; };
#define NACC 16
#define ITERS 2000

__global__ void __launch_bounds__(256) peak_f32(const __grid_constant__ PeakCoefs CF, float *out, const float *vin) {
  float2 a[NACC];
#pragma unroll
  for (int i = 0; i < NACC; ++i) a[i] = make_float2(threadIdx.x * 1e-3f + i, i * 0.5f);
  float2 vr[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) vr[i] = make_float2(vin[(threadIdx.x + i) & 63], vin[(threadIdx.x + 2 * i + 1) & 63]);
  for (int it = 0; it < ITERS; ++it)
#pragma unroll
    for (int j = 0; j < 8; ++j)
#pragma unroll
      for (int i = 0; i < NACC; ++i) a[i] = __ffma2_rn(a[i], make_float2(CF.k[2 * j], CF.k[2 * j + 1]), vr[j]);
  float s = 0;
#pragma unroll
  for (int i = 0; i < NACC; ++i) s += a[i].x + a[i].y;
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void __launch_bounds__(256) peak_f64(double *out, const double *vin) {
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

// dtype: 0 = fp64 (DFMA), 1 = fp32 (FFMA2).  scratch: device memory, >= 2 MiB, zero-filled by the caller.
// Returns 0 on success and writes the achieved FMA/s (best of `reps` launches) and the number of SMs.
extern "C" int bte_measure_fma_peak(int dtype, void *scratch, void *cuda_stream, int reps, double *fma_per_s, int *num_sms) {
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return 1;
  const int grid = sms * 2;                                  // 2 x 256 threads per SM: 16 warps, 4 per scheduler
  char *base = static_cast<char *>(scratch);
  PeakCoefs cf;
  for (int i = 0; i < 64; ++i) cf.k[i] = 0.5f + 1e-3f * i;
  cudaEvent_t e0, e1;
  if (cudaEventCreate(&e0) != cudaSuccess || cudaEventCreate(&e1) != cudaSuccess) return 1;
  double best = 0;
  for (int r = 0; r < reps + 1; ++r) {                       // first launch = warm-up
    cudaEventRecord(e0, st);
    if (dtype == 1) peak_f32<<<grid, 256, 0, st>>>(cf, reinterpret_cast<float *>(base + (1 << 20)), reinterpret_cast<const float *>(base));
    else peak_f64<<<grid, 256, 0, st>>>(reinterpret_cast<double *>(base + (1 << 20)), reinterpret_cast<const double *>(base));
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) return 1;
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double fma = (double)grid * 256 * ITERS * 8.0 * NACC * (dtype == 1 ? 2 : 1);
    if (r > 0 && ms > 0) best = fma / (ms * 1e-3) > best ? fma / (ms * 1e-3) : best;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  if (cudaGetLastError() != cudaSuccess) return 1;
  if (fma_per_s) *fma_per_s = best;
  if (num_sms) *num_sms = sms;
  return 0;
}
