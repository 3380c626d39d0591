// ACE tail and ACE application (Section III.A-B, Eqs. 17-20, 26-29; R15-R17).
//
//   M   = h^3 Psi^T W            (Eq. 20)        k_gram + k_gram_reduce      (the paper: cublasDgemm, Eq. 25)
//   A   = -(M + M^T)/2 = R R^T   (R16, R17)      k_ace_prepare, k_potrf_diag / k_potrf_panel / k_potrf_update
//                                                                            (the paper: cusolver dpotrf)
//   xi  = W R^-T                 (Eqs. 18, 26)   k_subst_op + k_expand per block of 64 orbitals
//                                                                            (the paper: cublasDtrsm)
//   chi = h^3 xi^T Phi           (Eq. 28)        k_gram + k_gram_reduce
//   V~ Phi = -xi chi             (Eqs. 27, 29)   k_expand
//
// A set of n grid functions is [n][N] with each function contiguous (include/exx.h), so the paper's tall
// matrices are stored transposed: "Psi^T W" is a product of two row-major [n][N] arrays contracted over the
// long index (k_gram, split over that index, partials reduced in a fixed order: bitwise reproducible), and
// "W R^-T" / "xi chi" are a small matrix times a very wide one (k_expand).  Both run on the FP64 tensor pipe
// (mma.sync.m8n8k4.f64 -> DMMA.8x8x4; tcgen05 has no FP64 kind on sm_100a), operands staged by cp.async into
// padded shared-memory tiles whose strides make the 8-byte fragment reads bank-conflict free.
#include <cstdint>

#include "exx_internal.h"

namespace exx {
namespace {

constexpr int kTile = 64;     // CTA tile: 64 x 64 outputs, four warps of 32 x 32
constexpr int kKC = 16;       // contraction indices per stage
constexpr int kStages = 4;  // measured: three stages (three CTAs per SM) gain 8-10 % at n = 64 but lose 5-10 % at n = 256
constexpr int kLdA = kKC + 4;    // stride of a [64][16] tile: == 4 (mod 16) doubles
constexpr int kLdB = kTile + 4;  // stride of a [16][64] tile: == 4 (mod 16) doubles
constexpr int kNB = 64;          // Cholesky / substitution block

__device__ __forceinline__ void dmma(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}
// asynchronous copy of `bytes` (0, 8 or 16) valid bytes into a 16- or 8-byte slot, the rest zero-filled
__device__ __forceinline__ void cp16(unsigned dst, const void* src, int bytes) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;\n" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp8(unsigned dst, const void* src, int bytes) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(dst), "l"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void cp_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

// ---- C_part[ks][i][j] = sum_{r in slice ks} A[i][r] B[j][r] ------------------------------------------
// A [ni][N], B [nj][N] row-major.  grid = (tiles_i * tiles_j, ksplit), 128 threads.  VEC = doubles per copy
// (2 needs N even and 16-byte aligned bases).
template <int VEC>
__global__ void __launch_bounds__(128)
    k_gram(const double* __restrict__ A, const double* __restrict__ B, int ni, int nj, long long N,
           long long slice, int tiles_j, double* __restrict__ part) {
  extern __shared__ __align__(16) double sm[];
  // stage s: A tile at sm + s*2*64*kLdA, B tile right behind it
  constexpr int kTileD = kTile * kLdA;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, q = lane & 3;
  const int wm = warp >> 1, wn = warp & 1;
  const int i0 = kTile * (blockIdx.x / tiles_j), j0 = kTile * (blockIdx.x % tiles_j);
  const long long r_begin = (long long)blockIdx.y * slice;
  const long long r_end = r_begin + slice < N ? r_begin + slice : N;
  const int nst = r_end > r_begin ? (int)((r_end - r_begin + kKC - 1) / kKC) : 0;
  const unsigned sm0 = (unsigned)__cvta_generic_to_shared(sm);

  auto load_stage = [&](int st, int buf) {
    const long long r0 = r_begin + (long long)st * kKC;
    constexpr int kPerRow = kKC / VEC;
    for (int c = tid; c < 2 * kTile * kPerRow; c += 128) {
      const int op = c / (kTile * kPerRow);
      const int rem = c - op * (kTile * kPerRow);
      const int row = rem / kPerRow, ch = rem - row * kPerRow;
      const long long r = r0 + (long long)ch * VEC;
      const int grow = (op ? j0 : i0) + row;
      const int nrow = op ? nj : ni;
      long long left = r_end - r;
      int bytes = (grow < nrow && left > 0) ? (left >= VEC ? 8 * VEC : 8 * (int)left) : 0;
      const double* src = (op ? B : A) + (bytes ? (long long)grow * N + r : 0);
      const unsigned dst = sm0 + 8u * (unsigned)(buf * 2 * kTileD + op * kTileD + row * kLdA + ch * VEC);
      if (VEC == 2) cp16(dst, src, bytes);
      else cp8(dst, src, bytes);
    }
  };

  double acc[4][4][2];
#pragma unroll
  for (int mt = 0; mt < 4; ++mt)
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

  for (int s = 0; s < kStages - 1; ++s) {
    if (s < nst) load_stage(s, s);
    cp_commit();
  }
  for (int st = 0; st < nst; ++st) {
    cp_wait<kStages - 2>();
    __syncthreads();  // stage st has landed for every thread; the buffer refilled below was consumed at st-1
    if (st + kStages - 1 < nst) load_stage(st + kStages - 1, (st + kStages - 1) % kStages);
    cp_commit();
    const double* sa = sm + (st % kStages) * 2 * kTileD + (wm * 32 + g) * kLdA + q;
    const double* sb = sm + (st % kStages) * 2 * kTileD + kTileD + (wn * 32 + g) * kLdA + q;
#pragma unroll
    for (int kk = 0; kk < kKC / 4; ++kk) {
      double af[4], bf[4];
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) af[mt] = sa[8 * mt * kLdA + 4 * kk];
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) bf[nt] = sb[8 * nt * kLdA + 4 * kk];
#pragma unroll
      for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) dmma(acc[mt][nt], af[mt], bf[nt]);
    }
  }
  cp_wait<0>();
  double* out = part + (long long)blockIdx.y * ni * nj;
#pragma unroll
  for (int mt = 0; mt < 4; ++mt) {
    const int i = i0 + wm * 32 + 8 * mt + g;
    if (i >= ni) continue;
#pragma unroll
    for (int nt = 0; nt < 4; ++nt)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int j = j0 + wn * 32 + 8 * nt + 2 * q + e;
        if (j < nj) out[(long long)i * nj + j] = acc[mt][nt][e];
      }
  }
}

// C[i][j] = alpha * sum_ks part[ks][i][j] in a fixed order (bitwise reproducible): a block of 256 threads handles 8
// entries; lane l of an entry's 32 lanes adds the slices l, l + 32, ... in ascending order, then the 32 lane sums are
// combined by a fixed shuffle tree.
__global__ void __launch_bounds__(256) k_gram_reduce(const double* __restrict__ part, int ksplit, long long nn, double alpha,
                                                     double* __restrict__ C) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  for (long long e = blockIdx.x * 8LL + w; e < nn; e += 8LL * gridDim.x) {
    double s = 0.0;
    for (int k = lane; k < ksplit; k += 32) s += part[(long long)k * nn + e];
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) s += __shfl_xor_sync(0xffffffffu, s, off);
    if (lane == 0) C[e] = alpha * s;
  }
}

// ---- Out[i][r] = alpha * sum_{k < nk} T[i][k] In_k[r] ------------------------------------------------
// T row-major [mi][ldt]; row k of the input is in_lo + k*N for k < ksel, in_hi + k*N otherwise (both [.][N]
// arrays indexed by the absolute k).  Out [mi][N].  grid = (ceil(N/64), ceil(mi/64)), 128 threads.
// Out may alias the input rows when mi <= 64: a CTA reads exactly the columns it writes and the block barrier
// before the epilogue orders every read before every write.
template <int VEC>
__global__ void __launch_bounds__(128)
    k_expand(const double* __restrict__ T, int ldt, int mi, int nk, const double* in_lo, const double* in_hi,
             int ksel, long long N, double alpha, double* Out) {
  extern __shared__ __align__(16) double sm[];
  constexpr int kTileT = kTile * kLdA;  // [64 i][16 k]
  constexpr int kTileI = kKC * kLdB;    // [16 k][64 r]
  constexpr int kStageD = kTileT + kTileI;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, q = lane & 3;
  const int wm = warp >> 1, wn = warp & 1;
  const long long r0 = (long long)blockIdx.x * kTile;
  const int i0 = blockIdx.y * kTile;
  const int nst = (nk + kKC - 1) / kKC;
  const unsigned sm0 = (unsigned)__cvta_generic_to_shared(sm);

  auto load_stage = [&](int st, int buf) {
    const int k0 = st * kKC;
    for (int c = tid; c < kTile * kKC; c += 128) {  // T tile, 8-byte copies (ldt is arbitrary)
      const int row = c / kKC, kc = c - row * kKC;
      const int i = i0 + row, k = k0 + kc;
      const int bytes = (i < mi && k < nk) ? 8 : 0;
      const double* src = T + (bytes ? (long long)i * ldt + k : 0);
      cp8(sm0 + 8u * (unsigned)(buf * kStageD + row * kLdA + kc), src, bytes);
    }
    constexpr int kPerRow = kTile / VEC;
    for (int c = tid; c < kKC * kPerRow; c += 128) {
      const int kr = c / kPerRow, ch = c - kr * kPerRow;
      const int k = k0 + kr;
      const long long r = r0 + (long long)ch * VEC;
      long long left = N - r;
      int bytes = (k < nk && left > 0) ? (left >= VEC ? 8 * VEC : 8 * (int)left) : 0;
      const double* base = k < ksel ? in_lo : in_hi;
      const double* src = base + (bytes ? (long long)k * N + r : 0);
      const unsigned dst = sm0 + 8u * (unsigned)(buf * kStageD + kTileT + kr * kLdB + ch * VEC);
      if (VEC == 2) cp16(dst, src, bytes);
      else cp8(dst, src, bytes);
    }
  };

  double acc[4][4][2];
#pragma unroll
  for (int mt = 0; mt < 4; ++mt)
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

  for (int s = 0; s < kStages - 1; ++s) {
    if (s < nst) load_stage(s, s);
    cp_commit();
  }
  for (int st = 0; st < nst; ++st) {
    cp_wait<kStages - 2>();
    __syncthreads();
    if (st + kStages - 1 < nst) load_stage(st + kStages - 1, (st + kStages - 1) % kStages);
    cp_commit();
    const double* sa = sm + (st % kStages) * kStageD + (wm * 32 + g) * kLdA + q;
    const double* sb = sm + (st % kStages) * kStageD + kTileT + q * kLdB + wn * 32 + g;
#pragma unroll
    for (int kk = 0; kk < kKC / 4; ++kk) {
      double af[4], bf[4];
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) af[mt] = sa[8 * mt * kLdA + 4 * kk];
#pragma unroll
      for (int nt = 0; nt < 4; ++nt) bf[nt] = sb[4 * kk * kLdB + 8 * nt];
#pragma unroll
      for (int mt = 0; mt < 4; ++mt)
#pragma unroll
        for (int nt = 0; nt < 4; ++nt) dmma(acc[mt][nt], af[mt], bf[nt]);
    }
  }
  cp_wait<0>();
  __syncthreads();  // in-place use: every read of this CTA's columns precedes every write
#pragma unroll
  for (int mt = 0; mt < 4; ++mt) {
    const int i = i0 + wm * 32 + 8 * mt + g;
    if (i >= mi) continue;
#pragma unroll
    for (int nt = 0; nt < 4; ++nt) {
      const long long r = r0 + wn * 32 + 8 * nt + 2 * q;
      double* dst = Out + (long long)i * N + r;
      const double x = alpha * acc[mt][nt][0], y = alpha * acc[mt][nt][1];
      if (VEC == 2) {
        if (r < N) *reinterpret_cast<double2*>(dst) = make_double2(x, y);  // N even: r+1 < N too
      } else {
        if (r < N) dst[0] = x;
        if (r + 1 < N) dst[1] = y;
      }
    }
  }
}

// ---- Cholesky of the small n x n matrix A = -(M + M^T)/2, blocked right-looking, block kNB ------------
// (row-major, lower triangle referenced and overwritten by R; the strict upper triangle is left alone)

__global__ void k_ace_prepare(const double* __restrict__ M, int n, double* __restrict__ A, int* info) {
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < (long long)n * n;
       e += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(e / n), j = (int)(e - (long long)i * n);
    A[e] = -0.5 * (M[e] + M[(long long)j * n + i]);
  }
  if (info && blockIdx.x == 0 && threadIdx.x == 0) *info = 0;
}

// One CTA: factor the diagonal block A[kb.., kb..] (nb <= 64), write R11 back, and write Tinv = R11^-1 (lower
// triangular, [kNB][kNB], zero above the diagonal).  A non-positive (or NaN) pivot sets *info = its 1-based index once;
// the factorisation continues and produces NaNs from there.
// Register-tiled: thread t owns row i = t % 64 and the 16 columns j == t / 64 (mod 4) of the block.  Right-looking step c:
// the owners of column c publish it (one double-buffered shared vector, one barrier per step), everybody subtracts
// l_i l_j from its own entries.  The inverse is the same scheme on the identity: step k publishes the finished row k of
// X and every row i > k subtracts R[i][k] X[k][:].  About 10 us for a 64 x 64 block (the shared-memory version with one
// thread per column of the inverse took 107 us and was the largest item of the ACE tail at n = 64).
__global__ void __launch_bounds__(256) k_potrf_diag(double* A, int n, int kb, int nb, double* Tinv, int* info) {
  __shared__ double Ls[kNB][kNB + 1];
  __shared__ double buf[2][kNB];
  __shared__ double rdiag[kNB];  // 1 / R[c][c]
  const int tid = threadIdx.x, i = tid & (kNB - 1), jq = tid >> 6;
  double a[16];
#pragma unroll
  for (int t = 0; t < 16; ++t) {
    const int j = 4 * t + jq;
    // rows and columns beyond nb: identity (keeps the padded part benign)
    a[t] = (i < nb && j <= i) ? A[(long long)(kb + i) * n + kb + j] : (i == j ? 1.0 : 0.0);
  }
  // column c = 4 cq + r lives in a[cq] of the threads with jq == r: cq unrolled so that every register index is static
#pragma unroll
  for (int cq = 0; cq < 16; ++cq) {
#pragma unroll 1
    for (int r = 0; r < 4; ++r) {
      const int c = 4 * cq + r;
      if (c < nb) {  // uniform
        double* cb = buf[c & 1];
        const bool owner = jq == r && i >= c;
        if (owner) cb[i] = a[cq];
        __syncthreads();
        const double piv = cb[c];
        if (tid == 0 && !(piv > 0.0) && info && *info == 0) *info = kb + c + 1;
        const double rd = rsqrt(piv), d = piv * rd;  // one reciprocal square root per step instead of a root and a division
        const double li = cb[i] * rd;
        if (i > c) {
#pragma unroll
          for (int t = cq; t < 16; ++t) {
            const int j = 4 * t + jq;
            if (j > c && j <= i) a[t] -= li * (cb[j] * rd);
          }
        }
        if (owner) {
          const double l = i == c ? d : li;
          a[cq] = l;
          Ls[i][c] = l;
          if (i == c) rdiag[c] = rd;
        }
      }
    }
  }
#pragma unroll
  for (int t = 0; t < 16; ++t) {
    const int j = 4 * t + jq;
    if (i < nb && j <= i) A[(long long)(kb + i) * n + kb + j] = a[t];
  }
  __syncthreads();  // Ls complete
  double x[16];
#pragma unroll
  for (int t = 0; t < 16; ++t) x[t] = (4 * t + jq == i) ? 1.0 : 0.0;
  for (int k = 0; k < nb; ++k) {
    double* rb = buf[k & 1];
    if (i == k) {
      const double r = rdiag[k];
#pragma unroll
      for (int t = 0; t < 16; ++t) {
        x[t] *= r;
        rb[4 * t + jq] = x[t];
      }
    }
    __syncthreads();
    if (i > k && i < nb) {
      const double lik = Ls[i][k];
#pragma unroll
      for (int t = 0; t < 16; ++t)
        if (4 * t + jq <= k) x[t] -= lik * rb[4 * t + jq];
    }
  }
#pragma unroll
  for (int t = 0; t < 16; ++t) {
    const int j = 4 * t + jq;
    Tinv[i * kNB + j] = (i < nb && j <= i) ? x[t] : 0.0;
  }
}

// Rows below the diagonal block: R21 = A21 R11^-T, i.e. R21[i][c] = sum_{t <= c} A21[i][t] Tinv[c][t].
// 16 rows per CTA, 256 threads.
__global__ void __launch_bounds__(256) k_potrf_panel(double* A, int n, int kb, int nb, const double* __restrict__ Tinv) {
  __shared__ double ti[kNB][kNB + 1];
  __shared__ double a[16][kNB + 1];
  const int tid = threadIdx.x;
  const int row0 = kb + nb + 16 * blockIdx.x;
  for (int e = tid; e < kNB * kNB; e += 256) ti[e / kNB][e % kNB] = Tinv[e];
  for (int e = tid; e < 16 * kNB; e += 256) {
    const int r = e / kNB, c = e % kNB;
    a[r][c] = (row0 + r < n && c < nb) ? A[(long long)(row0 + r) * n + kb + c] : 0.0;
  }
  __syncthreads();
  for (int e = tid; e < 16 * kNB; e += 256) {
    const int r = e / kNB, c = e % kNB;
    if (row0 + r < n && c < nb) {
      double acc = 0.0;
      for (int k = 0; k <= c; ++k) acc += a[r][k] * ti[c][k];
      A[(long long)(row0 + r) * n + kb + c] = acc;
    }
  }
}

// Trailing update, lower triangle only: A[i][j] -= sum_c R[i][kb+c] R[j][kb+c] for i, j >= kb+nb, j <= i.
// 32 x 32 outputs per CTA (grid = tiles x tiles; CTAs above the diagonal exit), 256 threads.
__global__ void __launch_bounds__(256) k_potrf_update(double* A, int n, int kb, int nb) {
  if (blockIdx.y > blockIdx.x) return;
  __shared__ double li[32][kNB + 1];
  __shared__ double lj[32][kNB + 1];
  const int tid = threadIdx.x;
  const int i0 = kb + nb + 32 * blockIdx.x, j0 = kb + nb + 32 * blockIdx.y;
  for (int e = tid; e < 32 * kNB; e += 256) {
    const int r = e / kNB, c = e % kNB;
    li[r][c] = (i0 + r < n && c < nb) ? A[(long long)(i0 + r) * n + kb + c] : 0.0;
    lj[r][c] = (j0 + r < n && c < nb) ? A[(long long)(j0 + r) * n + kb + c] : 0.0;
  }
  __syncthreads();
  for (int e = tid; e < 32 * 32; e += 256) {
    const int r = e / 32, c = e % 32;
    const int i = i0 + r, j = j0 + c;
    if (i < n && j <= i) {
      double acc = 0.0;
      for (int k = 0; k < nb; ++k) acc += li[r][k] * lj[c][k];
      A[(long long)i * n + j] -= acc;
    }
  }
}

// Substitution operator of block row B = [kb, kb+nb): xi_B = Tinv (W_B - R[B, <kb] xi_<kb) = G [xi_<kb ; W_B],
//   G[i][k] = -sum_{t <= i} Tinv[i][t] R[kb+t][k]  (k < kb),   G[i][kb+t] = Tinv[i][t].
// G is [kNB][ldg]; one thread per entry.
__global__ void k_subst_op(const double* __restrict__ R, int n, int kb, int nb, const double* __restrict__ Tinv,
                           double* __restrict__ G, int ldg) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int i = blockIdx.y;
  if (k >= kb + nb || i >= nb) return;
  double v;
  if (k >= kb) {
    v = Tinv[i * kNB + (k - kb)];
  } else {
    double acc = 0.0;
    for (int t = 0; t <= i; ++t) acc += Tinv[i * kNB + t] * R[(long long)(kb + t) * n + k];
    v = -acc;
  }
  G[(long long)i * ldg + k] = v;
}

// ---- complex (k-point) ACE: the small n x n work in complex arithmetic (cublasZgemm, zpotrf, Ztrsm) ---
// A set of n complex functions [n][2][N] is also a set of 2n real rows [2n][N] (row 2j = Re psi_j, row 2j+1 = Im psi_j),
// so the two big products run on the real kernels above with "embedded" shapes: the real Gram matrix G'[2n][2n] of the
// planes holds all four plane products of Psi^H W, and a complex combination out_i = sum_k T[i][k] in_k is the real
// k_expand with T'[(i,re)][(k,re)] = T'[(i,im)][(k,im)] = Re T, T'[(i,im)][(k,re)] = -T'[(i,re)][(k,im)] = Im T.
// Complex n x n matrices are row-major double2 (re, im).
constexpr int kNBc = 32;  // complex Cholesky / substitution block: 64 real rows, what k_expand's in-place rule allows

__device__ __forceinline__ double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
__device__ __forceinline__ double2 cmulc(double2 a, double2 b) {  // a * conj(b)
  return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}

// M[j][k] = (G[2j][2k] + G[2j+1][2k+1]) + i (G[2j][2k+1] - G[2j+1][2k])  (= h^3 sum conj(psi_j) w_k; G carries the h^3),
// A = -(M + M^H)/2.  Mout optional.
__global__ void k_ace_prepare_c(const double* __restrict__ G, int n, double2* __restrict__ A, double2* __restrict__ Mout,
                                int* info) {
  const long long ld = 2LL * n;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < (long long)n * n;
       e += (long long)gridDim.x * blockDim.x) {
    const long long j = e / n, k = e - j * n;
    const double mr = G[(2 * j) * ld + 2 * k] + G[(2 * j + 1) * ld + 2 * k + 1];
    const double mi = G[(2 * j) * ld + 2 * k + 1] - G[(2 * j + 1) * ld + 2 * k];
    const double tr = G[(2 * k) * ld + 2 * j] + G[(2 * k + 1) * ld + 2 * j + 1];   // M[k][j]
    const double ti = G[(2 * k) * ld + 2 * j + 1] - G[(2 * k + 1) * ld + 2 * j];
    if (Mout) Mout[e] = make_double2(mr, mi);
    A[e] = make_double2(-0.5 * (mr + tr), -0.5 * (mi - ti));
  }
  if (info && blockIdx.x == 0 && threadIdx.x == 0) *info = 0;
}

// One CTA: complex Cholesky of the diagonal block (nb <= 32), R11 written back (real positive diagonal), Tinv = R11^-1.
__global__ void __launch_bounds__(256) k_potrf_diag_c(double2* A, int n, int kb, int nb, double2* Tinv, int* info) {
  __shared__ double2 s[kNBc][kNBc + 1];
  const int tid = threadIdx.x;
  for (int e = tid; e < kNBc * kNBc; e += 256) {
    const int i = e / kNBc, j = e % kNBc;
    s[i][j] = (i < nb && j <= i) ? A[(long long)(kb + i) * n + kb + j] : make_double2(0.0, 0.0);
    Tinv[e] = make_double2(0.0, 0.0);
  }
  __syncthreads();
  for (int c = 0; c < nb; ++c) {
    if (tid == 0) {
      const double piv = s[c][c].x;
      if (!(piv > 0.0) && info && *info == 0) *info = kb + c + 1;
      s[c][c] = make_double2(sqrt(piv), 0.0);
    }
    __syncthreads();
    const double d = s[c][c].x;
    for (int i = c + 1 + tid; i < nb; i += 256) s[i][c] = make_double2(s[i][c].x / d, s[i][c].y / d);
    __syncthreads();
    const int m = nb - c - 1;
    for (int e = tid; e < m * m; e += 256) {
      const int i = c + 1 + e / m, j = c + 1 + e % m;
      if (j <= i) {
        const double2 t = cmulc(s[i][c], s[j][c]);
        s[i][j] = make_double2(s[i][j].x - t.x, s[i][j].y - t.y);
      }
    }
    __syncthreads();
  }
  for (int e = tid; e < kNBc * kNBc; e += 256) {
    const int i = e / kNBc, j = e % kNBc;
    if (i < nb && j <= i) A[(long long)(kb + i) * n + kb + j] = s[i][j];
  }
  if (tid < nb) {  // inverse by forward substitution, one column per thread
    const int col = tid;
    double2 x[kNBc];
    x[col] = make_double2(1.0 / s[col][col].x, 0.0);
    Tinv[col * kNBc + col] = x[col];
    for (int i = col + 1; i < nb; ++i) {
      double2 acc = make_double2(0.0, 0.0);
      for (int k = col; k < i; ++k) {
        const double2 t = cmul(s[i][k], x[k]);
        acc.x += t.x;
        acc.y += t.y;
      }
      x[i] = make_double2(-acc.x / s[i][i].x, -acc.y / s[i][i].x);
      Tinv[i * kNBc + col] = x[i];
    }
  }
}

// R21 = A21 R11^-H: R21[i][c] = sum_{t <= c} A21[i][t] conj(Tinv[c][t]).  16 rows per CTA.
__global__ void __launch_bounds__(256) k_potrf_panel_c(double2* A, int n, int kb, int nb, const double2* __restrict__ Tinv) {
  __shared__ double2 ti[kNBc][kNBc + 1];
  __shared__ double2 a[16][kNBc + 1];
  const int tid = threadIdx.x;
  const int row0 = kb + nb + 16 * blockIdx.x;
  for (int e = tid; e < kNBc * kNBc; e += 256) ti[e / kNBc][e % kNBc] = Tinv[e];
  for (int e = tid; e < 16 * kNBc; e += 256) {
    const int r = e / kNBc, c = e % kNBc;
    a[r][c] = (row0 + r < n && c < nb) ? A[(long long)(row0 + r) * n + kb + c] : make_double2(0.0, 0.0);
  }
  __syncthreads();
  for (int e = tid; e < 16 * kNBc; e += 256) {
    const int r = e / kNBc, c = e % kNBc;
    if (row0 + r < n && c < nb) {
      double2 acc = make_double2(0.0, 0.0);
      for (int k = 0; k <= c; ++k) {
        const double2 t = cmulc(a[r][k], ti[c][k]);
        acc.x += t.x;
        acc.y += t.y;
      }
      A[(long long)(row0 + r) * n + kb + c] = acc;
    }
  }
}

// Trailing update, lower triangle: A[i][j] -= sum_c R[i][kb+c] conj(R[j][kb+c]).  32 x 32 outputs per CTA.
__global__ void __launch_bounds__(256) k_potrf_update_c(double2* A, int n, int kb, int nb) {
  if (blockIdx.y > blockIdx.x) return;
  __shared__ double2 li[32][kNBc + 1];
  __shared__ double2 lj[32][kNBc + 1];
  const int tid = threadIdx.x;
  const int i0 = kb + nb + 32 * blockIdx.x, j0 = kb + nb + 32 * blockIdx.y;
  for (int e = tid; e < 32 * kNBc; e += 256) {
    const int r = e / kNBc, c = e % kNBc;
    li[r][c] = (i0 + r < n && c < nb) ? A[(long long)(i0 + r) * n + kb + c] : make_double2(0.0, 0.0);
    lj[r][c] = (j0 + r < n && c < nb) ? A[(long long)(j0 + r) * n + kb + c] : make_double2(0.0, 0.0);
  }
  __syncthreads();
  for (int e = tid; e < 32 * 32; e += 256) {
    const int r = e / 32, c = e % 32;
    const int i = i0 + r, j = j0 + c;
    if (i < n && j <= i) {
      double2 acc = make_double2(0.0, 0.0);
      for (int k = 0; k < nb; ++k) {
        const double2 t = cmulc(li[r][k], lj[c][k]);
        acc.x += t.x;
        acc.y += t.y;
      }
      double2 v = A[(long long)i * n + j];
      A[(long long)i * n + j] = make_double2(v.x - acc.x, v.y - acc.y);
    }
  }
}

// Substitution operator of block row B = [kb, kb+nb): conj(R) xi = W (functions as rows) gives
//   xi_B = conj(Tinv) (W_B - conj(R[B, <kb]) xi_<kb) = Gc [xi_<kb ; W_B],
//   Gc[i][k] = conj(-sum_{t <= i} Tinv[i][t] R[kb+t][k])  (k < kb),   Gc[i][kb+t] = conj(Tinv[i][t]),
// written as its real embedding G'[2 nb][ldg] (ldg >= 2 (kb + nb)).  One thread per complex entry.
__global__ void k_subst_op_c(const double2* __restrict__ R, int n, int kb, int nb, const double2* __restrict__ Tinv,
                             double* __restrict__ G, int ldg) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  const int i = blockIdx.y;
  if (k >= kb + nb || i >= nb) return;
  double2 v;
  if (k >= kb) {
    v = Tinv[i * kNBc + (k - kb)];
  } else {
    double2 acc = make_double2(0.0, 0.0);
    for (int t = 0; t <= i; ++t) {
      const double2 x = cmul(Tinv[i * kNBc + t], R[(long long)(kb + t) * n + k]);
      acc.x += x.x;
      acc.y += x.y;
    }
    v = make_double2(-acc.x, -acc.y);
  }
  const double gr = v.x, gi = -v.y;  // conj
  double* r0 = G + (long long)(2 * i) * ldg + 2 * k;
  double* r1 = r0 + ldg;
  r0[0] = gr;
  r0[1] = -gi;
  r1[0] = gi;
  r1[1] = gr;
}

// chi[j][a] = h^3 sum conj(xi_j) phi_a from the plane Gram matrix G[2m][2n] (rows: planes of phi, columns: planes of xi),
// written as the real embedding T'[2m][2n] of T[a][j] = chi[j][a].
__global__ void k_chi_embed(const double* __restrict__ G, int m, int n, double* __restrict__ T) {
  const long long ld = 2LL * n;
  for (long long e = blockIdx.x * (long long)blockDim.x + threadIdx.x; e < (long long)m * n;
       e += (long long)gridDim.x * blockDim.x) {
    const long long a = e / n, j = e - a * n;
    const double tr = G[(2 * a) * ld + 2 * j] + G[(2 * a + 1) * ld + 2 * j + 1];
    const double ti = G[(2 * a + 1) * ld + 2 * j] - G[(2 * a) * ld + 2 * j + 1];
    T[(2 * a) * ld + 2 * j] = tr;
    T[(2 * a) * ld + 2 * j + 1] = -ti;
    T[(2 * a + 1) * ld + 2 * j] = ti;
    T[(2 * a + 1) * ld + 2 * j + 1] = tr;
  }
}

struct GramSplit {
  int ksplit;
  long long slice;
};
inline GramSplit gram_split(int ni, int nj, long long N, int sm_count) {
  const long long tiles = (long long)((ni + kTile - 1) / kTile) * ((nj + kTile - 1) / kTile);
  long long want = (4LL * sm_count + tiles - 1) / tiles;
  const long long cap = N / 256 > 1 ? N / 256 : 1;
  if (want > cap) want = cap;
  if (want < 1) want = 1;
  long long slice = (N + want - 1) / want;
  slice = (slice + kKC - 1) / kKC * kKC;
  GramSplit g;
  g.slice = slice;
  g.ksplit = (int)((N + slice - 1) / slice);
  return g;
}

inline bool vec2_ok(long long N, const void* a, const void* b, const void* c) {
  return (N % 2 == 0) && ((((uintptr_t)a | (uintptr_t)b | (uintptr_t)c) & 15) == 0);
}

constexpr size_t kGramSmem = sizeof(double) * kStages * 2 * kTile * kLdA;
constexpr size_t kExpandSmem = sizeof(double) * kStages * (kTile * kLdA + kKC * kLdB);


// C[ni][nj] = alpha * A B^T over the grid index; part: ksplit*ni*nj doubles
cudaError_t gram(exx_plan* p, const double* A, int ni, const double* B, int nj, double alpha, double* part,
                 double* C, cudaStream_t s, long long* launches) {
  const long long N = p->N;
  const GramSplit gs = gram_split(ni, nj, N, p->sm_count);
  const int tiles_j = (nj + kTile - 1) / kTile;
  dim3 grid(((ni + kTile - 1) / kTile) * tiles_j, gs.ksplit);
  cudaError_t e;
  {
    ProfScope ps(p, KC_OTHER, s);
    if (vec2_ok(N, A, B, nullptr)) {
      static SmemOptIn opt;
      if ((e = opt.ensure(k_gram<2>, p->device, kGramSmem)) != cudaSuccess) return e;
      k_gram<2><<<grid, 128, kGramSmem, s>>>(A, B, ni, nj, N, gs.slice, tiles_j, part);
    } else {
      static SmemOptIn opt;
      if ((e = opt.ensure(k_gram<1>, p->device, kGramSmem)) != cudaSuccess) return e;
      k_gram<1><<<grid, 128, kGramSmem, s>>>(A, B, ni, nj, N, gs.slice, tiles_j, part);
    }
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  const long long nn = (long long)ni * nj;
  int blocks = (int)((nn + 7) / 8);
  if (blocks > 8 * p->sm_count) blocks = 8 * p->sm_count;
  k_gram_reduce<<<blocks, 256, 0, s>>>(part, gs.ksplit, nn, alpha, C);
  *launches += 2;
  return cudaGetLastError();
}

cudaError_t expand(exx_plan* p, const double* T, int ldt, int mi, int nk, const double* in_lo, const double* in_hi,
                   int ksel, double alpha, double* Out, cudaStream_t s, long long* launches) {
  const long long N = p->N;
  dim3 grid((unsigned)((N + kTile - 1) / kTile), (mi + kTile - 1) / kTile);
  cudaError_t e;
  ProfScope ps(p, KC_OTHER, s);
  if (vec2_ok(N, in_lo, in_hi, Out)) {
    static SmemOptIn opt;
    if ((e = opt.ensure(k_expand<2>, p->device, kExpandSmem)) != cudaSuccess) return e;
    k_expand<2><<<grid, 128, kExpandSmem, s>>>(T, ldt, mi, nk, in_lo, in_hi, ksel, N, alpha, Out);
  } else {
    static SmemOptIn opt;
    if ((e = opt.ensure(k_expand<1>, p->device, kExpandSmem)) != cudaSuccess) return e;
    k_expand<1><<<grid, 128, kExpandSmem, s>>>(T, ldt, mi, nk, in_lo, in_hi, ksel, N, alpha, Out);
  }
  *launches += 1;
  return cudaGetLastError();
}

}  // namespace

// ---- host entry points used by the C-ABI layer --------------------------------------------------------

// build: Gram partials | A -> R | inverses of the diagonal blocks | substitution operator | M
size_t ace_build_workspace_doubles(const exx_plan* p, int n) {
  const GramSplit gs = gram_split(n, n, p->N, p->sm_count);
  const size_t nblk = (size_t)(n + kNB - 1) / kNB;
  return (size_t)gs.ksplit * n * n + (size_t)n * n + nblk * kNB * kNB + (size_t)kNB * n + (size_t)n * n + 8;
}
// apply: Gram partials | chi^T
size_t ace_apply_workspace_doubles(const exx_plan* p, int n, int m) {
  const GramSplit gs = gram_split(m, n, p->N, p->sm_count);
  return (size_t)gs.ksplit * m * n + (size_t)m * n + 8;
}

// xi = W R^-T with R R^T = -(M + M^T)/2, M = h^3 Psi^T W.  xi may be w (in place).
cudaError_t ace_build(exx_plan* p, const double* psi, const double* w, int n, double* xi, double* M_out, int* info,
                      double* ws, cudaStream_t s, long long* launches) {
  const GramSplit gs = gram_split(n, n, p->N, p->sm_count);
  double* part = ws;
  double* A = part + (size_t)gs.ksplit * n * n;
  double* Tinv = A + (size_t)n * n;
  const size_t nblk = (size_t)(n + kNB - 1) / kNB;
  double* G = Tinv + nblk * kNB * kNB;
  double* M = M_out ? M_out : G + (size_t)kNB * n;
  const double dV = p->h * p->h * p->h;
  cudaError_t e;
  if ((e = gram(p, psi, n, w, n, dV, part, M, s, launches)) != cudaSuccess) return e;
  {
    int blocks = (int)(((long long)n * n + 255) / 256);
    if (blocks > 4 * p->sm_count) blocks = 4 * p->sm_count;
    k_ace_prepare<<<blocks, 256, 0, s>>>(M, n, A, info);
    ++*launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  {
    ProfScope ps(p, KC_OTHER, s);
    for (int kb = 0, b = 0; kb < n; kb += kNB, ++b) {
      const int nb = n - kb < kNB ? n - kb : kNB;
      double* Tb = Tinv + (size_t)b * kNB * kNB;
      k_potrf_diag<<<1, 256, 0, s>>>(A, n, kb, nb, Tb, info);
      ++*launches;
      const int below = n - kb - nb;
      if (below > 0) {
        k_potrf_panel<<<(below + 15) / 16, 256, 0, s>>>(A, n, kb, nb, Tb);
        const int t = (below + 31) / 32;
        k_potrf_update<<<dim3(t, t), 256, 0, s>>>(A, n, kb, nb);
        *launches += 2;
      }
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
  }
  for (int kb = 0, b = 0; kb < n; kb += kNB, ++b) {
    const int nb = n - kb < kNB ? n - kb : kNB;
    const double* Tb = Tinv + (size_t)b * kNB * kNB;
    k_subst_op<<<dim3((kb + nb + 127) / 128, nb), 128, 0, s>>>(A, n, kb, nb, Tb, G, n);
    ++*launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    // rows < kb come from xi (already final), the rows of the block itself from W
    if ((e = expand(p, G, n, nb, kb + nb, xi, w, kb, 1.0, xi + (size_t)kb * p->N, s, launches)) != cudaSuccess)
      return e;
  }
  return cudaSuccess;
}

// out = -xi (h^3 xi^T Phi): chi^T [m][n] by k_gram, then one k_expand.
cudaError_t ace_apply(exx_plan* p, const double* xi, int n, const double* phi, int m, double* out, double* ws,
                      cudaStream_t s, long long* launches) {
  const GramSplit gs = gram_split(m, n, p->N, p->sm_count);
  double* part = ws;
  double* chiT = part + (size_t)gs.ksplit * m * n;
  const double dV = p->h * p->h * p->h;
  cudaError_t e;
  if ((e = gram(p, phi, m, xi, n, dV, part, chiT, s, launches)) != cudaSuccess) return e;
  return expand(p, chiT, n, m, n, xi, xi, 0, -1.0, out, s, launches);
}

// ---- complex (k-point) ACE --------------------------------------------------------------------
// build: plane Gram partials | G' [2n][2n] | A (complex n x n) | inverses of the diagonal blocks | substitution operator
// (real embedding, [2 kNBc][2n]) | M (complex n x n)
size_t ace_build_c_workspace_doubles(const exx_plan* p, int n) {
  const GramSplit gs = gram_split(2 * n, 2 * n, p->N, p->sm_count);
  const size_t nblk = (size_t)(n + kNBc - 1) / kNBc;
  return (size_t)gs.ksplit * 4 * n * n + (size_t)4 * n * n + (size_t)2 * n * n + nblk * 2 * kNBc * kNBc +
         (size_t)2 * kNBc * 2 * n + (size_t)2 * n * n + 8;
}
// apply: plane Gram partials | G' [2m][2n] | T' [2m][2n]
size_t ace_apply_c_workspace_doubles(const exx_plan* p, int n, int m) {
  const GramSplit gs = gram_split(2 * m, 2 * n, p->N, p->sm_count);
  return (size_t)gs.ksplit * 4 * m * n + (size_t)8 * m * n + 8;
}

// xi = W R^-H with R R^H = -(M + M^H)/2, M = h^3 Psi^H W; psi, w, xi are [n][2][N].  xi may be w (in place).
cudaError_t ace_build_c(exx_plan* p, const double* psi, const double* w, int n, double* xi, double* M_out, int* info,
                        double* ws, cudaStream_t s, long long* launches) {
  const GramSplit gs = gram_split(2 * n, 2 * n, p->N, p->sm_count);
  double* part = ws;
  double* Gp = part + (size_t)gs.ksplit * 4 * n * n;
  double2* A = reinterpret_cast<double2*>(Gp + (size_t)4 * n * n);
  double2* Tinv = A + (size_t)n * n;
  const size_t nblk = (size_t)(n + kNBc - 1) / kNBc;
  double* G = reinterpret_cast<double*>(Tinv + nblk * kNBc * kNBc);
  double2* M = M_out ? reinterpret_cast<double2*>(M_out) : reinterpret_cast<double2*>(G + (size_t)2 * kNBc * 2 * n);
  const double dV = p->h * p->h * p->h;
  cudaError_t e;
  if ((e = gram(p, psi, 2 * n, w, 2 * n, dV, part, Gp, s, launches)) != cudaSuccess) return e;
  {
    int blocks = (int)(((long long)n * n + 255) / 256);
    if (blocks > 4 * p->sm_count) blocks = 4 * p->sm_count;
    k_ace_prepare_c<<<blocks, 256, 0, s>>>(Gp, n, A, M_out ? M : nullptr, info);
    ++*launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  {
    ProfScope ps(p, KC_OTHER, s);
    for (int kb = 0, b = 0; kb < n; kb += kNBc, ++b) {
      const int nb = n - kb < kNBc ? n - kb : kNBc;
      double2* Tb = Tinv + (size_t)b * kNBc * kNBc;
      k_potrf_diag_c<<<1, 256, 0, s>>>(A, n, kb, nb, Tb, info);
      ++*launches;
      const int below = n - kb - nb;
      if (below > 0) {
        k_potrf_panel_c<<<(below + 15) / 16, 256, 0, s>>>(A, n, kb, nb, Tb);
        const int t = (below + 31) / 32;
        k_potrf_update_c<<<dim3(t, t), 256, 0, s>>>(A, n, kb, nb);
        *launches += 2;
      }
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
    }
  }
  for (int kb = 0, b = 0; kb < n; kb += kNBc, ++b) {
    const int nb = n - kb < kNBc ? n - kb : kNBc;
    const double2* Tb = Tinv + (size_t)b * kNBc * kNBc;
    k_subst_op_c<<<dim3((kb + nb + 127) / 128, nb), 128, 0, s>>>(A, n, kb, nb, Tb, G, 2 * n);
    ++*launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
    // real rows < 2 kb come from xi (already final), the rows of the block itself from W
    if ((e = expand(p, G, 2 * n, 2 * nb, 2 * (kb + nb), xi, w, 2 * kb, 1.0, xi + (size_t)2 * kb * p->N, s, launches)) !=
        cudaSuccess)
      return e;
  }
  return cudaSuccess;
}

// out = -xi (h^3 xi^H Phi) for complex functions [.][2][N].
cudaError_t ace_apply_c(exx_plan* p, const double* xi, int n, const double* phi, int m, double* out, double* ws,
                        cudaStream_t s, long long* launches) {
  const GramSplit gs = gram_split(2 * m, 2 * n, p->N, p->sm_count);
  double* part = ws;
  double* Gp = part + (size_t)gs.ksplit * 4 * m * n;
  double* T = Gp + (size_t)4 * m * n;
  const double dV = p->h * p->h * p->h;
  cudaError_t e;
  if ((e = gram(p, phi, 2 * m, xi, 2 * n, dV, part, Gp, s, launches)) != cudaSuccess) return e;
  {
    int blocks = (int)(((long long)m * n + 255) / 256);
    if (blocks > 4 * p->sm_count) blocks = 4 * p->sm_count;
    k_chi_embed<<<blocks, 256, 0, s>>>(Gp, m, n, T);
    ++*launches;
    if ((e = cudaGetLastError()) != cudaSuccess) return e;
  }
  return expand(p, T, 2 * n, 2 * m, 2 * n, xi, xi, 0, -1.0, out, s, launches);
}

}  // namespace exx
