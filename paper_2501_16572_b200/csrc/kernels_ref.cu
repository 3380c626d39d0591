// Reference variant (EXX_VARIANT_REFERENCE): one plain FP64 kernel per step of the hot path.
// Deliberately simple -- used to cross-check the fast variant on the GPU and as a fallback-free
// "second opinion" in the parity tests.  Also holds the kernels both variants share (energy, zero fill).
#include <cstdint>
#include <cstdlib>

#include "exx_internal.h"

namespace exx {
namespace {

// a1: rho_b(r) = psi_j(r) * tgt_k(r)   (Eq. 2 right-hand side; real => no conj)
__global__ void k_pair_density(const double* __restrict__ psi, const double* __restrict__ tgt,
                               BatchDesc bd, long long N, double* __restrict__ out) {
  const int b = blockIdx.y;
  const int j = bd.j0 + b % bd.nj, k = bd.k0 + b / bd.nj;
  const double* pj = psi + (long long)j * N;
  const double* tk = tgt + (long long)k * N;
  double* o = out + (long long)b * N;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N;
       i += (long long)gridDim.x * blockDim.x)
    o[i] = pj[i] * tk[i];
}

// a2/a4: one mode product along `axis`.  Data viewed as [outer][n][inner]; forward contracts with V^T
// (out[m] = sum_i V[i][m] in[i]), backward with V (out[i] = sum_m V[i][m] in[m]).  PAPER.md:96-98 (Eq. 11).
// a3 (optional): multiply the result by the table m (Eq. 16) -- only ever used on the
// last forward product, whose output index is the full eigen-space index.
__global__ void k_mode_product(const double* __restrict__ in, double* __restrict__ out,
                               const double* __restrict__ V, int n, long long inner, long long total,
                               bool forward, const double* __restrict__ mult, long long N) {
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const long long i_in = t % inner;
    const long long r = t / inner;
    const int m = (int)(r % n);
    const long long o = r / n;
    const double* src = in + o * n * inner + i_in;
    double acc = 0.0;
    if (forward) {
      for (int i = 0; i < n; ++i) acc = fma(V[(long long)i * n + m], src[i * inner], acc);
    } else {
      for (int i = 0; i < n; ++i) acc = fma(V[(long long)m * n + i], src[i * inner], acc);
    }
    if (mult) acc *= mult[t % N];
    out[t] = acc;
  }
}

// a5: vx_k(r) (-)= sum_b occ_j psi_j(r) phi_b(r), b ascending (PAPER.md:38 Eq. 1, :178 Eq. 19b).
// Streaming kernel: per grid point one read of phi_b and psi_j per pair, vx_k read-modify-written once per
// batch.  VEC = 2 uses 16-byte accesses (N even, 16-byte aligned buffers); UNROLL independent j per trip keep
// 2*UNROLL loads per thread in flight.  The sum over j runs in ascending order whatever the template
// arguments, so all instantiations give bitwise identical results.
template <int VEC, int UNROLL>
__global__ void __launch_bounds__(256) k_accumulate(const double* __restrict__ psi, const double* __restrict__ occ,
                                                    const double* __restrict__ phi, BatchDesc bd, bool first,
                                                    unsigned N, double* __restrict__ vx, bool sym) {
  const int kk = blockIdx.y;
  // sym (pair-symmetric apply): only the pairs j <= k of the rectangular batch contribute to vx_k
  const int nj = sym ? min(bd.nj, bd.k0 + kk - bd.j0 + 1) : bd.nj;
  if (nj <= 0) return;
  double* v = vx + (size_t)(bd.k0 + kk) * N;
  const double* oc = occ + bd.j0;
  const double* psi0 = psi + (size_t)bd.j0 * N;
  const double* phi0 = phi + (size_t)kk * bd.nj * N;
  const unsigned stride = gridDim.x * blockDim.x * VEC;
  for (unsigned i = (blockIdx.x * blockDim.x + threadIdx.x) * VEC; i < N; i += stride) {
    double acc[VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) acc[e] = first ? 0.0 : v[i + e];
    const double* pj = psi0 + i;
    const double* ph = phi0 + i;
    int jj = 0;
    for (; jj + UNROLL <= nj; jj += UNROLL) {
      double a[UNROLL][VEC], b[UNROLL][VEC];
#pragma unroll
      for (int u = 0; u < UNROLL; ++u) {
        if (VEC == 2) {
          const double2 x = *reinterpret_cast<const double2*>(pj + (size_t)u * N);
          const double2 y = *reinterpret_cast<const double2*>(ph + (size_t)u * N);
          a[u][0] = x.x; a[u][VEC - 1] = x.y; b[u][0] = y.x; b[u][VEC - 1] = y.y;
        } else {
          a[u][0] = pj[(size_t)u * N];
          b[u][0] = ph[(size_t)u * N];
        }
      }
#pragma unroll
      for (int u = 0; u < UNROLL; ++u) {
        const double o = oc[jj + u];
#pragma unroll
        for (int e = 0; e < VEC; ++e) acc[e] -= o * a[u][e] * b[u][e];
      }
      pj += (size_t)UNROLL * N;
      ph += (size_t)UNROLL * N;
    }
    for (; jj < nj; ++jj) {
      const double o = oc[jj];
#pragma unroll
      for (int e = 0; e < VEC; ++e) acc[e] -= o * pj[e] * ph[e];
      pj += N;
      ph += N;
    }
#pragma unroll
    for (int e = 0; e < VEC; ++e) v[i + e] = acc[e];
  }
}

// Pair-symmetric apply, the transposed contribution (phi_jk = phi_kj): for every j of the
// batch, vx_j(r) -= sum_{k in batch, k > j} occ_k psi_k(r) phi_jk(r), k ascending.  grid.y = nj.
template <int VEC>
__global__ void __launch_bounds__(256) k_accumulate_transposed(const double* __restrict__ psi,
                                                               const double* __restrict__ occ,
                                                               const double* __restrict__ phi, BatchDesc bd,
                                                               unsigned N, double* __restrict__ vx) {
  const int jj = blockIdx.y;
  const int j = bd.j0 + jj;
  int kk0 = j + 1 - bd.k0;  // first target of the batch with k > j
  if (kk0 < 0) kk0 = 0;
  if (kk0 >= bd.nk) return;
  double* v = vx + (size_t)j * N;
  const unsigned stride = gridDim.x * blockDim.x * VEC;
  for (unsigned i = (blockIdx.x * blockDim.x + threadIdx.x) * VEC; i < N; i += stride) {
    double acc[VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) acc[e] = v[i + e];
    for (int kk = kk0; kk < bd.nk; ++kk) {
      const double o = occ[bd.k0 + kk];
      const double* pk = psi + (size_t)(bd.k0 + kk) * N + i;
      const double* ph = phi + ((size_t)kk * bd.nj + jj) * N + i;
      if (VEC == 2) {
        const double2 x = *reinterpret_cast<const double2*>(pk);
        const double2 y = *reinterpret_cast<const double2*>(ph);
        acc[0] -= o * x.x * y.x;
        acc[VEC - 1] -= o * x.y * y.y;
      } else {
        acc[0] -= o * pk[0] * ph[0];
      }
    }
#pragma unroll
    for (int e = 0; e < VEC; ++e) v[i + e] = acc[e];
  }
}

// a6: per-target partial sums with warp shuffles, deterministic two-stage reduction.
constexpr int kEnergyBlocks = 64;
constexpr int kEnergyThreads = 256;

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__global__ void k_energy_partial(const double* __restrict__ tgt, const double* __restrict__ vx,
                                 long long N, double* __restrict__ partial) {
  const int k = blockIdx.y;
  const double* t = tgt + (long long)k * N;
  const double* v = vx + (long long)k * N;
  double acc = 0.0;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N;
       i += (long long)gridDim.x * blockDim.x)
    acc = fma(t[i], v[i], acc);
  __shared__ double sh[kEnergyThreads / 32];
  acc = warp_sum(acc);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x < 32) {
    double s = threadIdx.x < kEnergyThreads / 32 ? sh[threadIdx.x] : 0.0;
    s = warp_sum(s);
    if (threadIdx.x == 0) partial[(long long)k * gridDim.x + blockIdx.x] = s;
  }
}

// one block: e_k = dV * sum of the partials of target k (fixed order), E_x += 1/2 sum_k occ_k e_k
__global__ void k_energy_final(const double* __restrict__ partial, int nblk, int n_tgt, double dV,
                               const double* __restrict__ occ_tgt, double* __restrict__ ex_k,
                               double* __restrict__ ex) {
  double acc = 0.0;
  for (int k = threadIdx.x; k < n_tgt; k += blockDim.x) {
    double s = 0.0;
    for (int b = 0; b < nblk; ++b) s += partial[(long long)k * nblk + b];
    s *= dV;
    if (ex_k) ex_k[k] = s;
    if (occ_tgt) acc = fma(occ_tgt[k], s, acc);
  }
  __shared__ double sh[32];
  acc = warp_sum(acc);
  if ((threadIdx.x & 31) == 0) sh[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x < 32) {
    double s = threadIdx.x < (blockDim.x >> 5) ? sh[threadIdx.x] : 0.0;
    s = warp_sum(s);
    if (threadIdx.x == 0 && ex) *ex += 0.5 * s;  // caller zeroes *ex before the first chunk
  }
}

__global__ void k_zero(double* p, long long n) {
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < n;
       i += (long long)gridDim.x * blockDim.x)
    p[i] = 0.0;
}

inline int grid_for(long long work, int threads, int sm_count) {
  long long g = (work + threads - 1) / threads;
  const long long cap = (long long)sm_count * 16;
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  return (int)g;
}

}  // namespace

cudaError_t ref_pair_density(const exx_plan* p, const double* psi, const double* tgt, BatchDesc bd,
                             double* out, cudaStream_t s) {
  dim3 grid(grid_for(p->N, 256, p->sm_count), bd.nj * bd.nk);
  k_pair_density<<<grid, 256, 0, s>>>(psi, tgt, bd, p->N, out);
  return cudaGetLastError();
}

cudaError_t ref_mode_product(const exx_plan* p, int axis, bool forward, const double* in, double* out,
                             int nb, bool apply_mult, cudaStream_t s) {
  const int n = p->n[axis];
  const long long inner = axis == 0 ? 1 : (axis == 1 ? p->n[0] : (long long)p->n[0] * p->n[1]);
  const long long total = p->N * nb;
  k_mode_product<<<grid_for(total, 256, p->sm_count), 256, 0, s>>>(
      in, out, p->d_V[axis], n, inner, total, forward, apply_mult ? p->d_mult : nullptr, p->N);
  return cudaGetLastError();
}

cudaError_t ref_accumulate(const exx_plan* p, const double* psi, const double* occ, const double* phi,
                           BatchDesc bd, bool first, double* vx, cudaStream_t s, bool sym) {
  const unsigned N = (unsigned)p->N;
  const bool vec2 = (N % 2 == 0) && ((((uintptr_t)psi | (uintptr_t)phi | (uintptr_t)vx) & 15) == 0);
  if (vec2) {  // 16-byte loads and stores (the normal case: N even, buffers 16-byte aligned)
    dim3 grid(grid_for(p->N / 2, 256, p->sm_count), bd.nk);
    k_accumulate<2, 4><<<grid, 256, 0, s>>>(psi, occ, phi, bd, first, N, vx, sym);
  } else {
    dim3 grid(grid_for(p->N, 256, p->sm_count), bd.nk);
    k_accumulate<1, 4><<<grid, 256, 0, s>>>(psi, occ, phi, bd, first, N, vx, sym);
  }
  return cudaGetLastError();
}

cudaError_t sym_accumulate_transposed(const exx_plan* p, const double* psi, const double* occ, const double* phi,
                                      BatchDesc bd, double* vx, cudaStream_t s) {
  const unsigned N = (unsigned)p->N;
  const bool vec2 = (N % 2 == 0) && ((((uintptr_t)psi | (uintptr_t)phi | (uintptr_t)vx) & 15) == 0);
  if (vec2) {
    dim3 grid(grid_for(p->N / 2, 256, p->sm_count), bd.nj);
    k_accumulate_transposed<2><<<grid, 256, 0, s>>>(psi, occ, phi, bd, N, vx);
  } else {
    dim3 grid(grid_for(p->N, 256, p->sm_count), bd.nj);
    k_accumulate_transposed<1><<<grid, 256, 0, s>>>(psi, occ, phi, bd, N, vx);
  }
  return cudaGetLastError();
}

// ex_k_scratch: n_tgt * kEnergyBlocks doubles (carved from the caller's workspace)
cudaError_t energy(const exx_plan* p, const double* tgt, const double* vx, const double* occ_tgt,
                   int n_tgt, double* ex_k_scratch, double* ex_k, double* ex, cudaStream_t s, long long len) {
  if (n_tgt <= 0) return cudaSuccess;
  dim3 grid(kEnergyBlocks, n_tgt);
  // len: doubles per function (0 = N; the complex variant passes 2N for its two planes)
  k_energy_partial<<<grid, kEnergyThreads, 0, s>>>(tgt, vx, len > 0 ? len : p->N, ex_k_scratch);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_energy_final<<<1, 256, 0, s>>>(ex_k_scratch, kEnergyBlocks, n_tgt, p->h * p->h * p->h, occ_tgt,
                                   ex_k, ex);
  return cudaGetLastError();
}

cudaError_t zero_fill(const exx_plan* p, double* ptr, long long n, cudaStream_t s) {
  if (n <= 0) return cudaSuccess;
  k_zero<<<grid_for(n, 256, p->sm_count), 256, 0, s>>>(ptr, n);
  return cudaGetLastError();
}

}  // namespace exx
