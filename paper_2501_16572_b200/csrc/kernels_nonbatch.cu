// The NON-batch Kronecker solver of PAPER.md:74-78 (Eq. 8a/8b), kept as the comparison line of the paper's Fig. 2
// (SURVEY.md 8(f) NEXT-4): one linear system at a time, every frontal slice B(:,:,k) multiplied by V1^T and V2 in two
// small dense products, the stacked slices by V3, then the multiplier and the same back -- 4 n3 + 2 products per
// system, ONE KERNEL LAUNCH PER PRODUCT, exactly as the paper's implementation calls its math library once per
// product.  It is not the product path: the batch formalism (kernels_tma.cu, kernels_fused.cu) is, and bench.py
// --solver-sweep reports the two side by side.
#include "exx_internal.h"

namespace exx {
namespace {

// C(i,j) = [mult(i,j) *] sum_k A(i,k) B(k,j) with arbitrary element strides; 16x16 tiles in shared memory, plain DFMA.
__global__ void __launch_bounds__(256) k_small_product(const double* __restrict__ A, long long sai, long long sak,
                                                       const double* __restrict__ B, long long sbk, long long sbj,
                                                       double* __restrict__ C, long long sci, long long scj, int M,
                                                       int Nn, int K, const double* __restrict__ mult) {
  __shared__ double As[16][17], Bs[16][17];
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int i = blockIdx.x * 16 + tx, j = blockIdx.y * 16 + ty;
  double acc = 0.0;
  for (int k0 = 0; k0 < K; k0 += 16) {
    // As[kk][ii] = A(i0 + ii, k0 + kk); Bs[kk][jj] = B(k0 + kk, j0 + jj)
    const int ai = blockIdx.x * 16 + tx, ak = k0 + ty;
    As[ty][tx] = (ai < M && ak < K) ? A[ai * sai + ak * sak] : 0.0;
    const int bk = k0 + tx, bj = blockIdx.y * 16 + ty;
    Bs[tx][ty] = (bk < K && bj < Nn) ? B[bk * sbk + bj * sbj] : 0.0;
    __syncthreads();
#pragma unroll
    for (int kk = 0; kk < 16; ++kk) acc = fma(As[kk][tx], Bs[kk][ty], acc);
    __syncthreads();
  }
  if (i < M && j < Nn) {
    const long long o = i * sci + j * scj;
    C[o] = mult ? mult[o] * acc : acc;
  }
}

cudaError_t product(const double* A, long long sai, long long sak, const double* B, long long sbk, long long sbj,
                    double* C, long long sci, long long scj, int M, int Nn, int K, const double* mult, cudaStream_t s) {
  dim3 grid((M + 15) / 16, (Nn + 15) / 16);
  k_small_product<<<grid, 256, 0, s>>>(A, sai, sak, B, sbk, sbj, C, sci, scj, M, Nn, K, mult);
  return cudaGetLastError();
}

}  // namespace

// One right-hand side; buf0 / buf1: N doubles each; rhs == phi allowed (rhs is read by the first products only).
cudaError_t nonbatch_solve_one(exx_plan* p, const double* rhs, double* phi, double* buf0, double* buf1, cudaStream_t s,
                               long long* launches) {
  const int n1 = p->n[0], n2 = p->n[1], n3 = p->n[2];
  const long long plane = (long long)n1 * n2;
  const double *V1 = p->d_V[0], *V2 = p->d_V[1], *V3 = p->d_V[2];  // row-major [i][m]
  cudaError_t e;
  ProfScope ps(p, KC_MODE_PRODUCT, s);
  for (int k = 0; k < n3; ++k) {
    const double* Bk = rhs + plane * k;
    // T1(a,y) = sum_x V1[x][a] B_k(x,y)
    if ((e = product(V1, 1, n1, Bk, 1, n1, buf0 + plane * k, 1, n1, n1, n2, n1, nullptr, s)) != cudaSuccess) return e;
    // T2(a,b) = sum_y T1(a,y) V2[y][b]
    if ((e = product(buf0 + plane * k, 1, n1, V2, n2, 1, buf1 + plane * k, 1, n1, n1, n2, n2, nullptr, s)) != cudaSuccess)
      return e;
  }
  // X~((a,b),c) = f(Lambda~) (.) sum_k T2((a,b),k) V3[k][c]
  if ((e = product(buf1, 1, plane, V3, n3, 1, buf0, 1, plane, (int)plane, n3, n3, p->d_mult, s)) != cudaSuccess) return e;
  // Y3((a,b),k) = sum_c X~((a,b),c) V3[k][c]
  if ((e = product(buf0, 1, plane, V3, 1, n3, buf1, 1, plane, (int)plane, n3, n3, nullptr, s)) != cudaSuccess) return e;
  for (int k = 0; k < n3; ++k) {
    // U(x,b) = sum_a V1[x][a] Y3_k(a,b)
    if ((e = product(V1, n1, 1, buf1 + plane * k, 1, n1, buf0 + plane * k, 1, n1, n1, n2, n1, nullptr, s)) != cudaSuccess)
      return e;
    // X_k(x,y) = sum_b U(x,b) V2[y][b]
    if ((e = product(buf0 + plane * k, 1, n1, V2, 1, n2, phi + plane * k, 1, n1, n1, n2, n2, nullptr, s)) != cudaSuccess)
      return e;
  }
  *launches += 4LL * n3 + 2;
  return cudaSuccess;
}

}  // namespace exx
