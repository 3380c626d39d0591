// exx_energy_static (include/exx.h): the energy step of the hot path -- e_k = dv <tgt_k, vx_k>,
// E_x = 1/2 sum_k occ_tgt_k e_k (BASELINE.json north_star; R7) -- for callers that are not in a position to
// allocate device memory.
//
// Who that is: a host code that hands every byte of HBM to its own arena at start-up (an electronic-structure code
// sizes its orbital arrays to fill the card, so a later cudaMalloc simply fails), and a caller inside a time-critical
// loop that runs several streams at once (cudaMalloc and cudaFree synchronise the whole device and would stall all of
// them).  Every other compute call of this library needs a plan, whose creation allocates, and a caller-provided
// workspace; this one needs neither.  The per-block partial sums of the two-stage reduction -- the only memory the
// step touches beyond its inputs and outputs -- live in the fixed array below, which is part of the library image:
// every GPU that loads libexx.so holds EXX_ENERGY_STATIC_MAX_TGT * 64 doubles (2 MiB) from load until the process
// exits, whether the entry point is ever called or not.
//
// Same arithmetic as the energy step inside exx_apply (kernels_ref.cu: 64 blocks per target, warp-shuffle block sums,
// partials added in block order by one thread per target), written out again here so that no existing kernel or host
// path changes.  The file shares nothing with them but the status codes.
#include <cuda_runtime.h>

#include <mutex>

#include "exx.h"

namespace exx {
void note_cuda_error(cudaError_t e);  // exx_api.cu: what exx_status_string reports for EXX_ERR_CUDA
}

namespace {

constexpr int kBlocksPerTarget = 64;
constexpr int kThreads = 256;
constexpr int kMaxDevices = 64;

// The scratch.  In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address and must
// never be passed to a kernel as one; static_scratch() below turns it into the address valid on the current device.
static __device__ __align__(256) double g_energy_partials[(size_t)EXX_ENERGY_STATIC_MAX_TGT * kBlocksPerTarget];

std::mutex g_mutex;
double* g_scratch_of_device[kMaxDevices] = {};  // device address of g_energy_partials, per device ordinal

// Address of the scratch on the CURRENT device; resolved once per device (each device has its own copy of the array).
cudaError_t static_scratch(double** out) {
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(g_mutex);
  if (!g_scratch_of_device[dev]) {
    double* ptr = nullptr;
    e = cudaGetSymbolAddress((void**)&ptr, g_energy_partials);
    if (e != cudaSuccess) return e;
    if (!ptr) return cudaErrorInvalidSymbol;
    g_scratch_of_device[dev] = ptr;
  }
  *out = g_scratch_of_device[dev];
  return cudaSuccess;
}

__device__ __forceinline__ double warp_total(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// stage 1: block (b, k) writes the sum of tgt_k .* vx_k over its grid-stride share of the points to partial[k][b].
// Every slot [k < n_tgt][b < 64] is overwritten, so nothing left in the array by an earlier call is ever read.
__global__ void __launch_bounds__(kThreads) k_energy_static_partial(const double* __restrict__ tgt,
                                                                    const double* __restrict__ vx, long long n_points,
                                                                    double* __restrict__ partial) {
  const int k = blockIdx.y;
  const double* t = tgt + (long long)k * n_points;
  const double* v = vx + (long long)k * n_points;
  double acc = 0.0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n_points;
       i += (long long)gridDim.x * blockDim.x)
    acc = fma(t[i], v[i], acc);
  __shared__ double sh[kThreads / 32];
  acc = warp_total(acc);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x < 32) {
    double s = threadIdx.x < kThreads / 32 ? sh[threadIdx.x] : 0.0;
    s = warp_total(s);
    if (threadIdx.x == 0) partial[(long long)k * gridDim.x + blockIdx.x] = s;
  }
}

// stage 2, one block: e_k = dv * (partials of target k, block order); *ex = 1/2 sum_k occ_tgt_k e_k (overwritten)
__global__ void __launch_bounds__(kThreads) k_energy_static_final(const double* __restrict__ partial, int n_tgt, double dv,
                                                                  const double* __restrict__ occ_tgt,
                                                                  double* __restrict__ ex_k, double* __restrict__ ex) {
  double acc = 0.0;
  for (int k = threadIdx.x; k < n_tgt; k += blockDim.x) {
    double s = 0.0;
    for (int b = 0; b < kBlocksPerTarget; ++b) s += partial[(long long)k * kBlocksPerTarget + b];
    s *= dv;
    if (ex_k) ex_k[k] = s;
    if (occ_tgt) acc = fma(occ_tgt[k], s, acc);
  }
  __shared__ double sh[kThreads / 32];
  acc = warp_total(acc);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x < 32) {
    double s = threadIdx.x < kThreads / 32 ? sh[threadIdx.x] : 0.0;
    s = warp_total(s);
    if (threadIdx.x == 0 && ex) *ex = 0.5 * s;
  }
}

inline exx_status cuda_fail(cudaError_t e) {
  exx::note_cuda_error(e);
  return EXX_ERR_CUDA;
}

}  // namespace

extern "C" exx_status exx_energy_static(const double* d_tgt, const double* d_vx, const double* d_occ_tgt, int n_tgt,
                                        long long n_points, double dv, double* d_ex_k, double* d_ex, void* cuda_stream) {
  if (n_tgt < 0 || n_points < 1 || !(dv > 0.0) || (n_tgt > 0 && (!d_tgt || !d_vx)) || (d_ex && n_tgt > 0 && !d_occ_tgt))
    return EXX_ERR_INVALID_ARG;
  if (n_tgt > EXX_ENERGY_STATIC_MAX_TGT) return EXX_ERR_LIMIT;  // nothing enqueued, nothing touched
  if (!d_ex_k && !d_ex) return EXX_OK;
  double* partial = nullptr;
  cudaError_t e = static_scratch(&partial);
  if (e != cudaSuccess) return cuda_fail(e);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (n_tgt > 0) {
    k_energy_static_partial<<<dim3(kBlocksPerTarget, n_tgt), kThreads, 0, s>>>(d_tgt, d_vx, n_points, partial);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
  }
  k_energy_static_final<<<1, kThreads, 0, s>>>(partial, n_tgt, dv, d_occ_tgt, d_ex_k, d_ex);
  e = cudaGetLastError();
  if (e != cudaSuccess) return cuda_fail(e);
  return EXX_OK;
}
