// bte_residual_static: the stopping test of Eq. 23 (readings G11) between two snapshots the
// caller holds, for callers that cannot allocate (CUDA graph capture, tight serving loops, harnesses that forbid
// cudaMalloc).  A variant of bte_update_kernel's residual part + bte_final_kernel (bte_kernels.cuh): the same
// per-cell terms and the same fixed-order block tree, but the per-block partial sums live in a file-scope
// __device__ array instead of the caller's workspace, and the last block to finish does the final reduction, so
// it is ONE launch.  Included at the end of bte_api.cu (same translation unit: the array, the kernel and the host
// code that resolves the array's device address must share one).
//
// The array is held by every GPU that loads the library until the process exits: 32 + 5 * 4096 doubles = 164 096 B.
// Every call on a device shares it: calls that overlap on the GPU (different streams, different threads) race.
#ifndef BTE_STATIC_CUH
#define BTE_STATIC_CUH

#define BTE_STATIC_CHUNK 4096                                               // cells per block: 256 threads x 16
#define BTE_STATIC_MAX_BLOCKS (BTE_STATIC_MAX_CELLS / BTE_STATIC_CHUNK)     // 4096
#define BTE_STATIC_HEAD 32                                                  // doubles: [0] holds the ticket
static_assert(BTE_STATIC_MAX_CELLS % BTE_STATIC_CHUNK == 0, "whole chunks");

// In HOST code this name is a host-side stand-in, not a device address: only bte_static_scratch_ptr() below
// (cudaGetSymbolAddress) yields the pointer a kernel may be given.
static __device__ __align__(256) double bte_static_scratch[BTE_STATIC_HEAD + 5 * BTE_STATIC_MAX_BLOCKS];

__device__ __forceinline__ void block_reduce5(double &a, double &b, double &c, double &d, double &n) {
  block_reduce4(a, b, c, d);        // a, c: sums; b, d: maxima (fixed-order tree; result in thread 0)
  __shared__ double shn[32];
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
  for (int off = 16; off > 0; off >>= 1) n += __shfl_down_sync(0xffffffffu, n, off);
  if (lane == 0) shn[w] = n;
  __syncthreads();
  if (w == 0) {
    n = lane < nw ? shn[lane] : 0.0;
    for (int off = 16; off > 0; off >>= 1) n += __shfl_down_sync(0xffffffffu, n, off);
  }
  __syncthreads();                  // sh[][] / shn[] may be reused by a second call in the same kernel
}

// grid = ceil(n / 4096) blocks of 256 threads; block b owns cells [4096 b, 4096 (b + 1)): the summation order
// depends on n only.  scratch: [0] ticket (unsigned, 0 at entry), [32 + k * nb + b] partial k of block b.
__global__ void __launch_bounds__(256) bte_residual_static_kernel(double *scratch, const double *__restrict__ T1,
                                                                  const double *__restrict__ T0,
                                                                  const double *__restrict__ q1,
                                                                  const double *__restrict__ q0,
                                                                  const uint8_t *__restrict__ mask, int64_t n,
                                                                  double *__restrict__ out) {
  unsigned int *ticket = reinterpret_cast<unsigned int *>(scratch);
  double *part = scratch + BTE_STATIC_HEAD;
  const int nb = gridDim.x;
  double sT = 0, mT = 0, sq = 0, mq = 0, ns = 0;
  const int64_t c0 = (int64_t)blockIdx.x * BTE_STATIC_CHUNK + threadIdx.x;
#pragma unroll 4
  for (int r = 0; r < BTE_STATIC_CHUNK / 256; ++r) {
    const int64_t c = c0 + r * 256;
    if (c >= n) break;
    if (mask && !mask[c]) continue;                       // void cell: not counted (G11: N = solid cells)
    const double Tn = T1[c], dlt = Tn - T0[c];
    sT += dlt * dlt; mT = fmax(mT, fabs(Tn));
    const double a1 = q1[c], a2 = q1[n + c], a3 = q1[2 * n + c];
    const double b1 = q0[c], b2 = q0[n + c], b3 = q0[2 * n + c];
    const double qm = sqrt(a1 * a1 + a2 * a2 + a3 * a3);
    const double dq = qm - sqrt(b1 * b1 + b2 * b2 + b3 * b3);
    sq += dq * dq; mq = fmax(mq, qm);
    ns += 1.0;
  }
  block_reduce5(sT, mT, sq, mq, ns);
  __shared__ bool last;
  if (threadIdx.x == 0) {
    __stcg(part + blockIdx.x, sT); __stcg(part + nb + blockIdx.x, mT); __stcg(part + 2 * nb + blockIdx.x, sq);
    __stcg(part + 3 * nb + blockIdx.x, mq); __stcg(part + 4 * nb + blockIdx.x, ns);
    __threadfence();
    last = atomicAdd(ticket, 1u) == (unsigned)(nb - 1);
  }
  __syncthreads();
  if (!last) return;
  __threadfence();
  sT = mT = sq = mq = ns = 0;
  for (int e = threadIdx.x; e < nb; e += blockDim.x) {
    sT += __ldcg(part + e); mT = fmax(mT, __ldcg(part + nb + e)); sq += __ldcg(part + 2 * nb + e);
    mq = fmax(mq, __ldcg(part + 3 * nb + e)); ns += __ldcg(part + 4 * nb + e);
  }
  block_reduce5(sT, mT, sq, mq, ns);
  if (threadIdx.x == 0) {
    const double inf = __longlong_as_double(0x7ff0000000000000LL);
    const double rT = ns > 0 ? sqrt(sT / ns) : 0.0, rq = ns > 0 ? sqrt(sq / ns) : 0.0;
    out[0] = mT > 0 ? rT / mT : (rT == 0 ? 0.0 : inf);    // 0/0 -> 0, x/0 -> +inf (bte.h, bte_residual)
    out[1] = mq > 0 ? rq / mq : (rq == 0 ? 0.0 : inf);
    *ticket = 0;                                          // ready for the next call in stream order
  }
}

// Device address of bte_static_scratch on the CURRENT device, resolved once per device.
static bte_status bte_static_scratch_ptr(double **out) {
  constexpr int kMaxDev = 64;
  static std::atomic<double *> ptr[kMaxDev];
  int dev = -1;
  CK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDev) return BTE_ERR_UNSUPPORTED;
  double *p = ptr[dev].load(std::memory_order_acquire);
  if (!p) {
    CK(cudaGetSymbolAddress(reinterpret_cast<void **>(&p), bte_static_scratch));
    if (!p) { g_last_cuda.store((int)cudaErrorInvalidSymbol); return BTE_ERR_CUDA; }
    ptr[dev].store(p, std::memory_order_release);        // a racing thread resolves the same address
  }
  *out = p;
  return BTE_OK;
}

extern "C" bte_status bte_residual_static(const double *d_dT_new, const double *d_dT_old, const double *d_q_new,
                                          const double *d_q_old, const uint8_t *d_solid_mask, int64_t n_cells,
                                          double *d_eps, void *cuda_stream) {
  if (!d_dT_new || !d_dT_old || !d_q_new || !d_q_old || !d_eps || n_cells <= 0) return BTE_ERR_INVALID_ARG;
  if (n_cells > (int64_t)BTE_STATIC_MAX_CELLS) return BTE_ERR_TOO_LARGE;
  double *scratch = nullptr;
  const bte_status st = bte_static_scratch_ptr(&scratch);
  if (st != BTE_OK) return st;
  cudaStream_t s = static_cast<cudaStream_t>(cuda_stream);
  // the ticket must start at 0 whatever an earlier (possibly failed) call left behind; the partial sums are
  // all rewritten before they are read, so they need no clearing
  CK(cudaMemsetAsync(scratch, 0, BTE_STATIC_HEAD * sizeof(double), s));
  const int nb = (int)((n_cells + BTE_STATIC_CHUNK - 1) / BTE_STATIC_CHUNK);
  bte_residual_static_kernel<<<nb, 256, 0, s>>>(scratch, d_dT_new, d_dT_old, d_q_new, d_q_old, d_solid_mask, n_cells,
                                                d_eps);
  CK(cudaGetLastError());
  return BTE_OK;
}
#endif
