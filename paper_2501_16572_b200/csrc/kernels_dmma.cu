// Fast variant (EXX_VARIANT_FUSED_DMMA): mode products on the FP64 tensor pipe.
//
// Every mode product of Eq. 11 is a "small stationary matrix times a very wide
// matrix": out[:, c] = M in[:, c] with M = V^T (forward) or V (backward), n x n, n <= 128, and c running
// over N*n_c/n columns.  One persistent CTA per SM keeps V resident in shared memory for the whole
// launch and streams column tiles through a 2-stage cp.async pipeline; warps issue
// mma.sync.m8n8k4.f64 (SASS DMMA.8x8x4, measured 37.1 TFLOP/s on B200 = 128 flop/clk/SM) with
// MT x NT register blocking so that shared-memory operand traffic stays below 40 % of the LSU pipe.
//
// Two global<->tile mappings share the MMA core:
//   L-mode (axis y or z, contracted index strided by `inner`): tile = [k][w columns], columns are the
//           flattened (outer, inner) index, so there is no ragged waste except at the very end;
//   X-mode (axis x, contracted index contiguous): tile = [w rows][k], the transposed product
//           out^T = M in^T is computed, so the data rows are the MMA's N dimension.
// Results are stored straight from the accumulator fragments; all passes are in place.
//
// The paper's four data reorganisations (Eqs. 12-15) do not exist here: they are
// artefacts of calling a 2-D GEMM library and are replaced by the strided tile addressing above.
#include <cstdint>

#include "exx_internal.h"

namespace exx {
namespace {

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
  asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
               : "+d"(c[0]), "+d"(c[1])
               : "d"(a), "d"(b));
}

template <int BYTES>
__device__ __forceinline__ void cp_async(void* smem, const void* gmem) {
  const unsigned s = (unsigned)__cvta_generic_to_shared(smem);
  asm volatile("cp.async.ca.shared.global [%0], [%1], %2;\n" ::"r"(s), "l"(gmem), "n"(BYTES));
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N));
}

struct ModeArgs {
  const double* in;
  double* out;
  const double* V;      // row-major [i][m], n x n
  const double* mult;   // optional (L-mode only): multiplier table indexed [m*inner + i]
  int n;                // contracted extent
  int KT;               // ceil(n/4)
  int ldv;              // smem row stride of V (== 4 mod 8)
  int ldt;              // smem row stride of a data tile (== 4 mod 8)
  int fwd;              // 1: M = V^T, 0: M = V
  int inner;            // L-mode: length of the contiguous run below the contracted axis
  long long total;      // L-mode: number of columns (outer*inner); X-mode: number of rows
  int n_tiles;
};

// smem layout (doubles): [ V: R8 x ldv ][ stage0 ][ stage1 ],  R8 = roundup(n, 8)
template <int MT, int WR, int NT, int WC, bool XMODE, int VEC>
__global__ void __launch_bounds__(32 * WR * WC, 1) k_mode_dmma(const ModeArgs a) {
  constexpr int kThreads = 32 * WR * WC;
  constexpr int kW = 8 * NT * WC;
  extern __shared__ __align__(16) double smem[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, q = lane & 3;
  const int wr = warp % WR, wc = warp / WR;
  const int n = a.n, KT = a.KT, ldv = a.ldv, ldt = a.ldt;
  const int R8 = (n + 7) & ~7;
  double* Vs = smem;
  const int stage_elems = XMODE ? kW * ldt : 4 * KT * ldt;
  double* stage0 = Vs + R8 * ldv;

  // ---- one-time: zero everything (k-padding must be exact zeros), then stage V --------------------
  {
    const int tot = R8 * ldv + 2 * stage_elems;
    for (int i = tid; i < tot; i += kThreads) smem[i] = 0.0;
    __syncthreads();
    for (int i = tid; i < n * n; i += kThreads) {
      const int r = i / n, c = i - r * n;
      Vs[r * ldv + c] = a.V[i];
    }
  }

  // A operand (M): element (m,k) at Vs[m*a_sm + k*a_sk]
  const int a_sm = a.fwd ? 1 : ldv, a_sk = a.fwd ? ldv : 1;
  // B operand (data): element (k, col) at tile[k*b_sk + col*b_sn]
  const int b_sk = XMODE ? 1 : ldt, b_sn = XMODE ? ldt : 1;
  const int m_base = 8 * MT * wr, n_base = 8 * NT * wc;
  int mt_valid = 0;
#pragma unroll
  for (int mt = 0; mt < MT; ++mt) mt_valid += (m_base + 8 * mt < n) ? 1 : 0;
  const double* ap = Vs + (m_base + g) * a_sm + q * a_sk;

  auto load_tile = [&](int t, double* st) {
    if (XMODE) {
      // rows [t*kW, ...) of n contiguous doubles each; 16 threads per row
      const long long r0 = (long long)t * kW;
      const int rows = (int)((a.total - r0) < kW ? (a.total - r0) : kW);
      const double* src = a.in + r0 * n;
      const int trow = tid >> 4, tcol = (tid & 15) * VEC;
      for (int r = trow; r < rows; r += kThreads / 16)
        for (int c = tcol; c < n; c += 16 * VEC) cp_async<8 * VEC>(st + r * ldt + c, src + (long long)r * n + c);
    } else {
      // columns [t*kW, ...) of the flattened (outer, inner) index; each thread owns one column group
      constexpr int kCG = kW / VEC;             // column groups per row
      constexpr int kRowsPerPass = kThreads / kCG;
      static_assert(kThreads % kCG == 0, "thread/column mapping");
      const int cg = tid % kCG, k0 = tid / kCG;
      const long long cidx = (long long)t * kW + cg * VEC;
      if (cidx < a.total) {
        const long long o = cidx / a.inner;
        const int i = (int)(cidx - o * a.inner);
        const double* src = a.in + (o * n) * a.inner + i;
        double* dst = st + cg * VEC;
        for (int k = k0; k < n; k += kRowsPerPass) cp_async<8 * VEC>(dst + k * ldt, src + (long long)k * a.inner);
      }
    }
  };

  int t = blockIdx.x;
  int buf = 0;
  if (t < a.n_tiles) load_tile(t, stage0);
  cp_async_commit();
  __syncthreads();  // V staged (plain stores) before anyone reads it

  for (; t < a.n_tiles; t += gridDim.x) {
    double* cur = stage0 + buf * stage_elems;
    const int tn = t + gridDim.x;
    if (tn < a.n_tiles) load_tile(tn, stage0 + (buf ^ 1) * stage_elems);
    cp_async_commit();
    cp_async_wait<1>();
    __syncthreads();

    double acc[MT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    const double* bp = cur + (n_base + g) * b_sn + q * b_sk;
#pragma unroll 2
    for (int kt = 0; kt < KT; ++kt) {
      double af[MT], bf[NT];
#pragma unroll
      for (int mt = 0; mt < MT; ++mt)
        if (mt < mt_valid) af[mt] = ap[mt * 8 * a_sm + kt * 4 * a_sk];
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) bf[nt] = bp[nt * 8 * b_sn + kt * 4 * b_sk];
#pragma unroll
      for (int mt = 0; mt < MT; ++mt)
        if (mt < mt_valid) {
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], bf[nt]);
        }
    }

    // ---- epilogue: store accumulator fragments ------------------------------------------------------
    if (XMODE) {
      // C[m = a-index][col = row r]: out[(r0 + r) * n + m]
      const long long r0 = (long long)t * kW;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const long long r = r0 + n_base + 8 * nt + 2 * q + e;
          if (r < a.total) {
            double* dst = a.out + r * n;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
              const int m = m_base + 8 * mt + g;
              if (mt < mt_valid && m < n) dst[m] = acc[mt][nt][e];
            }
          }
        }
      }
    } else {
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        const long long cidx = (long long)t * kW + n_base + 8 * nt + 2 * q;
        if (VEC == 2) {
          if (cidx < a.total) {
            const long long o = cidx / a.inner;
            const int i = (int)(cidx - o * a.inner);
            double* dst = a.out + (o * n) * a.inner + i;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
              const int m = m_base + 8 * mt + g;
              if (mt < mt_valid && m < n) {
                double2 v = make_double2(acc[mt][nt][0], acc[mt][nt][1]);
                if (a.mult) {
                  const double2 mm = __ldg(reinterpret_cast<const double2*>(a.mult + (long long)m * a.inner + i));
                  v.x *= mm.x;
                  v.y *= mm.y;
                }
                *reinterpret_cast<double2*>(dst + (long long)m * a.inner) = v;
              }
            }
          }
        } else {
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const long long ce = cidx + e;
            if (ce < a.total) {
              const long long o = ce / a.inner;
              const int i = (int)(ce - o * a.inner);
              double* dst = a.out + (o * n) * a.inner + i;
#pragma unroll
              for (int mt = 0; mt < MT; ++mt) {
                const int m = m_base + 8 * mt + g;
                if (mt < mt_valid && m < n) {
                  double v = acc[mt][nt][e];
                  if (a.mult) v *= __ldg(a.mult + (long long)m * a.inner + i);
                  dst[(long long)m * a.inner] = v;
                }
              }
            }
          }
        }
      }
    }
    __syncthreads();  // everyone is done with `cur` before the next iteration's prefetch overwrites it
    buf ^= 1;
  }
  cp_async_wait<0>();
}

// ---- host side ------------------------------------------------------------------------------------

struct Shape {
  int MT, WR, NT, WC;
};

inline bool pick_shape(int n, Shape* s) {
  if (n <= 16) *s = {2, 1, 2, 8};
  else if (n <= 32) *s = {2, 2, 2, 4};
  else if (n <= 48) *s = {3, 2, 2, 4};
  else if (n <= 64) *s = {4, 2, 2, 4};
  else if (n <= 96) *s = {3, 4, 2, 2};
  else if (n <= 128) *s = {4, 4, 2, 2};
  else return false;
  return true;
}

struct Layout {
  int KT, ldv, ldt, R8, kW;
  size_t smem_bytes;
};

inline Layout make_layout(int n, const Shape& s, bool xmode) {
  Layout L;
  L.KT = (n + 3) / 4;
  L.R8 = (n + 7) & ~7;
  L.ldv = L.R8 + 4;
  L.kW = 8 * s.NT * s.WC;
  if (xmode) {
    const int k4 = 4 * L.KT;
    L.ldt = (k4 % 8 == 4) ? k4 : k4 + 4;
    L.smem_bytes = sizeof(double) * ((size_t)L.R8 * L.ldv + 2 * (size_t)L.kW * L.ldt);
  } else {
    L.ldt = L.kW + 4;
    L.smem_bytes = sizeof(double) * ((size_t)L.R8 * L.ldv + 2 * (size_t)4 * L.KT * L.ldt);
  }
  return L;
}

template <int MT, int WR, int NT, int WC>
cudaError_t launch_shape(bool xmode, int vec, const ModeArgs& a, int grid, size_t smem, cudaStream_t s) {
  constexpr int kThreads = 32 * WR * WC;
#define EXX_LAUNCH(XM, VC)                                                                              \
  do {                                                                                                  \
    auto kern = k_mode_dmma<MT, WR, NT, WC, XM, VC>;                                                    \
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
    if (e != cudaSuccess) return e;                                                                     \
    kern<<<grid, kThreads, smem, s>>>(a);                                                               \
    return cudaGetLastError();                                                                          \
  } while (0)
  if (xmode) {
    if (vec == 2) EXX_LAUNCH(true, 2);
    EXX_LAUNCH(true, 1);
  } else {
    if (vec == 2) EXX_LAUNCH(false, 2);
    EXX_LAUNCH(false, 1);
  }
#undef EXX_LAUNCH
  return cudaErrorUnknown;
}

// One mode product along `axis`, in place or out of place, nb right-hand sides.
cudaError_t fast_mode_product(const exx_plan* p, int axis, bool forward, const double* in, double* out,
                              int nb, bool apply_mult, cudaStream_t s) {
  const int n = p->n[axis];
  Shape sh;
  if (!pick_shape(n, &sh)) return cudaErrorNotSupported;
  const bool xmode = axis == 0;
  const Layout L = make_layout(n, sh, xmode);
  if (L.smem_bytes > (size_t)p->smem_optin) return cudaErrorNotSupported;
  ModeArgs a;
  a.in = in;
  a.out = out;
  a.V = p->d_V[axis];
  a.mult = apply_mult ? p->d_mult : nullptr;
  a.n = n;
  a.KT = L.KT;
  a.ldv = L.ldv;
  a.ldt = L.ldt;
  a.fwd = forward ? 1 : 0;
  const long long inner = axis == 1 ? p->n[0] : (long long)p->n[0] * p->n[1];
  a.inner = xmode ? 1 : (int)inner;
  a.total = p->N / n * nb;  // columns (L-mode) or rows (X-mode)
  const long long tiles = (a.total + L.kW - 1) / L.kW;
  if (tiles > 0x7fffffffLL) return cudaErrorNotSupported;
  a.n_tiles = (int)tiles;
  const bool aligned = (((uintptr_t)in | (uintptr_t)out) & 15) == 0 &&
                       (!apply_mult || ((uintptr_t)p->d_mult & 15) == 0);
  int vec = 1;
  if (aligned) {
    if (xmode) vec = (n % 2 == 0) ? 2 : 1;
    else vec = (inner % 2 == 0) ? 2 : 1;
  }
  const int grid = (int)(tiles < p->sm_count ? tiles : p->sm_count);
  if (sh.MT == 2 && sh.WR == 1) return launch_shape<2, 1, 2, 8>(xmode, vec, a, grid, L.smem_bytes, s);
  if (sh.MT == 2 && sh.WR == 2) return launch_shape<2, 2, 2, 4>(xmode, vec, a, grid, L.smem_bytes, s);
  if (sh.MT == 3 && sh.WR == 2) return launch_shape<3, 2, 2, 4>(xmode, vec, a, grid, L.smem_bytes, s);
  if (sh.MT == 4 && sh.WR == 2) return launch_shape<4, 2, 2, 4>(xmode, vec, a, grid, L.smem_bytes, s);
  if (sh.MT == 3 && sh.WR == 4) return launch_shape<3, 4, 2, 2>(xmode, vec, a, grid, L.smem_bytes, s);
  return launch_shape<4, 4, 2, 2>(xmode, vec, a, grid, L.smem_bytes, s);
}

}  // namespace

cudaError_t fast_init(exx_plan*) { return cudaSuccess; }
void fast_destroy(exx_plan*) {}

// Axes longer than 128 points do not fit the resident-V kernels; they run on the plain DFMA kernel
// (still CUDA, still in the library; stated in DESIGN.md).  buf1 is only needed in that case.
static cudaError_t one_product(exx_plan* p, int axis, bool fwd, double*& cur, double*& other, int nb,
                               bool mult, cudaStream_t s) {
  ProfScope ps(p, KC_MODE_PRODUCT, s);
  cudaError_t e = fast_mode_product(p, axis, fwd, cur, cur, nb, mult, s);
  if (e == cudaErrorNotSupported) {
    e = ref_mode_product(p, axis, fwd, cur, other, nb, mult, s);
    double* t = cur;
    cur = other;
    other = t;
  }
  return e;
}

cudaError_t fast_solve_batch(exx_plan* p, double* buf0, double* buf1, int nb, const FastArgs* fa,
                             cudaStream_t s, long long* launches) {
  cudaError_t e;
  double *cur = buf0, *other = buf1;
  if (fa) {
    {
      ProfScope ps(p, KC_PAIR_DENSITY, s);
      e = ref_pair_density(p, fa->psi, fa->tgt, fa->bd, cur, s);
    }
    if (e != cudaSuccess) return e;
    ++*launches;
  }
  if ((e = one_product(p, 0, true, cur, other, nb, false, s)) != cudaSuccess) return e;
  if ((e = one_product(p, 1, true, cur, other, nb, false, s)) != cudaSuccess) return e;
  if ((e = one_product(p, 2, true, cur, other, nb, true, s)) != cudaSuccess) return e;
  if ((e = one_product(p, 2, false, cur, other, nb, false, s)) != cudaSuccess) return e;
  if ((e = one_product(p, 1, false, cur, other, nb, false, s)) != cudaSuccess) return e;
  if ((e = one_product(p, 0, false, cur, other, nb, false, s)) != cudaSuccess) return e;
  *launches += 6;
  if (fa) {
    {
      ProfScope ps(p, KC_ACCUMULATE, s);
      e = ref_accumulate(p, fa->psi, fa->occ, cur, fa->bd, fa->first, fa->vx, s);
    }
    if (e != cudaSuccess) return e;
    ++*launches;
  } else if (cur != buf0) {
    e = cudaMemcpyAsync(buf0, cur, sizeof(double) * (size_t)p->N * nb, cudaMemcpyDeviceToDevice, s);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace exx
