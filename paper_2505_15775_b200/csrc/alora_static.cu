// alora_static.cu -- alora_rowdots_static: the allocation-free variant of alora_rowdots (include/alora.h).
//
// alora_rowdots keeps its per-block partial sums in a workspace the ctx allocates with cudaMalloc on first use
// (alora_solve.cu, ensure_ws).  Some callers cannot allocate: code under CUDA graph capture, tight serving loops,
// harnesses that forbid cudaMalloc.  This variant keeps the same scratch in a file-scope __device__ array of a fixed,
// stated size, so the call allocates nothing -- no cudaMalloc, no cudaFree, no allocating library routine, no
// synchronisation: one 4-byte cudaMemsetAsync and one kernel launch on the ctx stream.
//
// The array's name is a host-side stand-in in host code, not a device address (a kernel handed the name itself faults,
// or, where the GPU can reach host memory, silently uses the wrong memory).  The device address is looked up once per
// device, with that device current, by cudaGetSymbolAddress below, and that pointer is what the kernel receives.
//
// Every GPU that loads libalora.so holds the array (kScratchBytes, about 64 KB) until the process exits.  All calls on
// a device share it and it keeps the last call's contents: the ticket word is cleared before every launch, the partial
// rows in use are overwritten before they are read.  Two calls that overlap on the GPU (different streams, or two
// ctx on one device used concurrently) race on it -- documented in alora.h, not guarded.
#include <mutex>

#include "alora_internal.h"

namespace {

using alora::kBlock;

constexpr int kChunkElems = 16384;   // elements of X (and Y) summed by one block: 64 per thread
constexpr int kMaxBlocks = 4096;     // partial rows the scratch holds
constexpr int64_t kMaxElems = (int64_t)kChunkElems * kMaxBlocks;
static_assert(kMaxElems == ALORA_ROWDOTS_STATIC_MAX_ELEMS, "alora.h states the limit of alora_rowdots_static");
// layout (doubles): [2 b], [2 b + 1] = block b's partial sums (X.X, X.Y); word kTicketAt holds the ticket counter
constexpr int kTicketAt = 2 * kMaxBlocks;
constexpr int kScratchDoubles = kTicketAt + 32;   // 256 bytes for the ticket, keeps it off the partial rows' lines
constexpr size_t kScratchBytes = sizeof(double) * kScratchDoubles;

static __device__ __align__(256) double s_rowdots_scratch[kScratchDoubles];

// Ordered block sum of two per-thread fp64 values; the result is valid in thread 0.
__device__ __forceinline__ void block_sum2(double& a, double& b, double (*sm)[kBlock / 32]) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  a = alora::warp_sum(a); b = alora::warp_sum(b);
  __syncthreads();   // sm may still be read by the previous use
  if (lane == 0) { sm[0][warp] = a; sm[1][warp] = b; }
  __syncthreads();
  if (threadIdx.x == 0) {
    a = 0.0; b = 0.0;
    for (int w = 0; w < kBlock / 32; ++w) { a += sm[0][w]; b += sm[1][w]; }
  }
}

// out[0] = sum X_ij^2, out[1] = sum X_ij Y_ij over the first n_rows rows (r columns, leading dimension ld).  Block b
// owns elements [b kChunkElems, (b + 1) kChunkElems) of the n_rows x r index space, so the summation order depends on
// the shape only (not on the SM count); the block that draws the last ticket adds the partial rows in order.
template <typename T>
__global__ void __launch_bounds__(kBlock) k_rowdots_static(int64_t n_rows, int r, int64_t ld, const T* __restrict__ X,
                                                           const T* __restrict__ Y, double* scratch, double* out) {
  __shared__ double sm[2][kBlock / 32];
  __shared__ unsigned int s_last;
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch + kTicketAt);
  const int64_t N = n_rows * r, beg = (int64_t)blockIdx.x * kChunkElems, end = min(N, beg + kChunkElems);
  double xx = 0.0, xy = 0.0;
  if (ld == r) {
    for (int64_t i = beg + threadIdx.x; i < end; i += kBlock) {
      const double x = (double)X[i];
      xx += x * x; xy += x * (double)Y[i];
    }
  } else {
    for (int64_t i = beg + threadIdx.x; i < end; i += kBlock) {
      const int64_t row = i / r, idx = row * ld + (i - row * r);
      const double x = (double)X[idx];
      xx += x * x; xy += x * (double)Y[idx];
    }
  }
  block_sum2(xx, xy, sm);
  if (threadIdx.x == 0) { scratch[2 * blockIdx.x] = xx; scratch[2 * blockIdx.x + 1] = xy; }
  __threadfence();
  __syncthreads();
  if (threadIdx.x == 0) s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  xx = 0.0; xy = 0.0;
  for (int b = threadIdx.x; b < (int)gridDim.x; b += kBlock) { xx += __ldcg(scratch + 2 * b); xy += __ldcg(scratch + 2 * b + 1); }
  block_sum2(xx, xy, sm);
  if (threadIdx.x == 0) { out[0] = xx; out[1] = xy; *ticket = 0u; }
}

// Device address of the scratch array, looked up once per device with that device current.
constexpr int kMaxDevices = 64;
std::mutex g_mu;
double* g_scratch_addr[kMaxDevices] = {};

cudaError_t scratch_address(int device, double** p) {
  std::lock_guard<std::mutex> lk(g_mu);
  if (!g_scratch_addr[device]) {
    void* q = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&q, s_rowdots_scratch);   // the device current here is `device` (caller set it)
    if (e != cudaSuccess) return e;
    g_scratch_addr[device] = static_cast<double*>(q);
  }
  *p = g_scratch_addr[device];
  return cudaSuccess;
}

}  // namespace

using namespace alora;

extern "C" alora_status alora_rowdots_static(alora_ctx* c, const void* X, const void* Y, int64_t n_rows, int32_t r, int64_t ld,
                                             double* out_dev) {
  if (!c) return ALORA_EINVAL;
  if (!X || !Y || !out_dev || n_rows < 0 || r < 1 || ld < r) return fail(c, ALORA_EINVAL, "alora_rowdots_static: bad argument");
  if (n_rows > kMaxElems / r)
    return fail(c, ALORA_EINVAL, "alora_rowdots_static: n_rows * r = " + std::to_string(n_rows) + " * " + std::to_string(r) +
                                     " exceeds the maximum of " + std::to_string(kMaxElems) +
                                     " elements its static scratch array is sized for (ALORA_ROWDOTS_STATIC_MAX_ELEMS); use alora_rowdots");
  if (c->device < 0 || c->device >= kMaxDevices) return fail(c, ALORA_EINVAL, "alora_rowdots_static: device index out of range");
  ALORA_CUDA(c, cudaSetDevice(c->device));
  double* scratch = nullptr;
  ALORA_CUDA(c, scratch_address(c->device, &scratch));
  if (n_rows == 0) {
    ALORA_CUDA(c, cudaMemsetAsync(out_dev, 0, sizeof(double) * 2, c->stream));
    return ALORA_OK;
  }
  // the ticket must start at zero; the finishing block resets it, but a launch that failed midway would leave it stale
  ALORA_CUDA(c, cudaMemsetAsync(scratch + kTicketAt, 0, sizeof(unsigned int), c->stream));
  const int grid = (int)((n_rows * r + kChunkElems - 1) / kChunkElems);
  if (c->dtype == ALORA_F32) k_rowdots_static<float><<<grid, kBlock, 0, c->stream>>>(n_rows, r, ld, (const float*)X, (const float*)Y, scratch, out_dev);
  else k_rowdots_static<double><<<grid, kBlock, 0, c->stream>>>(n_rows, r, ld, (const double*)X, (const double*)Y, scratch, out_dev);
  c->launches++;
  ALORA_CUDA(c, cudaGetLastError());
  return ALORA_OK;
}
