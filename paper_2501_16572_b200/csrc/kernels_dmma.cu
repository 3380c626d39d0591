// Fast variant (EXX_VARIANT_FUSED_DMMA): mode products on the FP64 tensor pipe.
//
// Every mode product of Eq. 11 is "a small stationary matrix times a very wide one":
// out[:, c] = M in[:, c], M = V^T (forward) or V (backward), n x n with n <= 128, c running over
// N*n_c/n columns.  Design (measured facts in profiles/r1_dmma_issue_vs_occupancy.txt):
//   * mma.sync.m8n8k4.f64 lowers to DMMA.8x8x4; one warp per SM sub-partition with >= 2 independent
//     accumulators already saturates the pipe (37.1 TFLOP/s = 128 flop/clk/SM), every DMMA blocks its
//     warp for 16 issue cycles.  So the kernel is built from fully independent warps, 2 per
//     sub-partition, and everything that is not a DMMA must fit in the shadow of the other warp's DMMAs.
//   * V (<= 132 KB padded) is staged once per CTA in shared memory with a row stride == 4 (mod 8)
//     doubles, which makes both the V and the V^T fragment reads bank-conflict free.
//   * The data operand is never shared between warps: each element is used by exactly one warp (a warp
//     owns 8*NT columns for ALL n output rows), so every lane fetches exactly its own B-fragment elements
//     with 8-byte cp.async copies into a private D-deep ring of shared-memory slots (full 32 B sectors:
//     8 consecutive columns x 4 rows in L-mode, 4 consecutive x x 8 rows in X-mode).  cp.async groups,
//     not the register scoreboard, track completion; no block or warp barrier exists in the steady state.
//   * Accumulators (ceil(n/8) x NT tiles) live in registers; results are stored straight from the
//     fragments, so every pass runs in place.
// Fused into the passes: the pair density psi_j*tgt_k in the load path of the first product (a1), the
// multiplier f(Lambda~) in the store path of the last forward product (a3).
//
// Two global<->fragment mappings share the MMA core:
//   L-mode (axis y or z; contracted index strided by `inner`): columns = flattened (outer, inner) index;
//   X-mode (axis x; contracted index contiguous): the transposed product out^T = M in^T, columns = rows
//           of nx contiguous points, tiled per right-hand side.
//
// The paper's four data reorganisations (Eqs. 12-15) do not exist here: they are
// artefacts of calling a 2-D GEMM library and are replaced by the strided fragment addressing above.
#include <cstdint>
#include <cstdlib>

#include "exx_internal.h"

namespace exx {
namespace {

constexpr int kWarps = 8;
constexpr int kThreads = 32 * kWarps;
constexpr size_t kMinSmem = 117 * 1024;  // > half of the 227 KB per-SM limit
constexpr int kRing = 8;  // depth of the per-lane B-fragment ring (cp.async stages), in k-steps

__device__ __forceinline__ void dmma884(double (&c)[2], double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
      : "+d"(c[0]), "+d"(c[1])
      : "d"(a), "d"(b));
}
__device__ __forceinline__ double lds64(unsigned addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];\n" : "=d"(v) : "r"(addr));
  return v;
}
// 8-byte asynchronous global->shared copy; src_bytes = 0 writes zeros (used for k >= n and ragged tails).
// Completion is tracked by cp.async groups, not by the register scoreboard, so a D-deep ring really is
// D steps of latency tolerance (plain LDG prefetches shared scoreboard slots with the DMMAs and stalled).
__device__ __forceinline__ void cp_async8(unsigned smem_addr, const double* gmem, bool valid) {
  const int src_bytes = valid ? 8 : 0;
  asm volatile("cp.async.ca.shared.global [%0], [%1], 8, %2;\n" ::"r"(smem_addr), "l"(gmem), "r"(src_bytes)
               : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() {
  asm volatile("cp.async.wait_group %0;\n" ::"n"(N) : "memory");
}

// Exact n / d for n < 2^31 with a host-computed multiplier (d = 2^shift when mul == 0).
struct FastDiv {
  unsigned mul;
  int shift;
  unsigned d;
};
inline FastDiv make_fastdiv(unsigned d) {
  FastDiv f{0u, 0, d};
  if ((d & (d - 1)) == 0) {  // power of two (d >= 1)
    while ((1u << f.shift) < d) ++f.shift;
    return f;
  }
  int L = 0;
  while ((1ull << L) < d) ++L;  // ceil(log2 d)
  f.mul = (unsigned)(((1ull << (31 + L)) / d) + 1ull);
  f.shift = L - 1;
  return f;
}
__device__ __forceinline__ unsigned fast_div(unsigned n, const FastDiv& f) {
  return f.mul ? (__umulhi(n, f.mul) >> f.shift) : (n >> f.shift);
}

struct WArgs {
  const double* in;
  double* out;
  const double* V;     // zero-padded image [8*MTOT][8*MTOT+4] of the row-major eigenvector matrix
  const double* mult;  // optional (L-mode): table indexed [m*inner + i]
  const double* psi;   // PD only
  const double* tgt;   // PD only
  int n;
  int KT;                // ceil(n/4)
  int inner;             // L-mode: contiguous run below the contracted axis
  long long total;       // L-mode: number of columns (outer*inner)
  int rows_per_rhs;      // X-mode: N / nx
  int tiles_per_rhs;     // X-mode: ceil(rows_per_rhs / (8*NT))
  long long n_tiles;     // warp tiles in this launch
  long long N;           // points per right-hand side
  BatchDesc bd;          // PD only
  int vec2;              // L-mode: 16-byte stores are aligned
  FastDiv div_inner;     // L-mode: / inner
  FastDiv div_tiles;     // X-mode: / tiles_per_rhs
};

// MTOT = ceil(n/8) rounded up to a supported class, NT = column tiles (of 8) per warp.
template <int MTOT, int NT, bool XMODE, bool FWD, bool TWO>
__global__ void __launch_bounds__(kThreads, 1) k_mode_w(const WArgs a) {
  static_assert(!TWO || (XMODE && FWD) || (!XMODE && !FWD), "second stream: pair density (x fwd) or multiplier (z bwd)");
  static_assert((kRing & (kRing - 1)) == 0, "ring depth must be a power of two");
  constexpr int LDV = 8 * MTOT + 4;  // == 4 (mod 8): conflict-free for both fragment orientations
  extern __shared__ __align__(16) double Vs[];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, KT = a.KT;

  // ---- stage V once per CTA: the plan holds a zero-padded image in exactly this layout (k >= n must
  // contribute exact zeros), so staging is one burst of 16-byte asynchronous copies ----------------------
  {
    const unsigned vs0 = (unsigned)__cvta_generic_to_shared(Vs);
    for (int i = 2 * tid; i < 8 * MTOT * LDV; i += 2 * kThreads)
      asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(vs0 + 8u * i), "l"(a.V + i) : "memory");
    cp_async_commit();
    cp_async_wait<0>();
  }
  __syncthreads();
  // Programmatic dependent launch: everything above touched only the plan's constant V, so it overlaps
  // the tail of the previous pass; from here on we read that pass's output.
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  asm volatile("griddepcontrol.wait;\n" ::: "memory");

  // A fragment (M[m][k]) shared address for (mt, kt): base + mt*A_MT + kt*A_KT   (bytes)
  //   FWD: M[m][k] = V[k][m] -> Vs[(4kt+q)*LDV + 8mt+g];   BWD: M[m][k] = V[m][k] -> Vs[(8mt+g)*LDV + 4kt+q]
  constexpr unsigned A_MT = FWD ? 64u : 64u * LDV;
  constexpr unsigned A_KT = FWD ? 32u * LDV : 32u;
  const unsigned a_base = (unsigned)__cvta_generic_to_shared(Vs) + 8u * (FWD ? (q * LDV + g) : (g * LDV + q));

  // per-lane B-fragment ring: slot (d, nt, s) of this lane at ring_base + ((d*NT + nt)*NS + s)*256
  constexpr int NS = TWO ? 2 : 1;  // two streams are staged separately and multiplied on consumption
  constexpr unsigned kRingWarpBytes = kRing * NT * NS * 256u;
  const unsigned ring_base = (unsigned)__cvta_generic_to_shared(Vs) + 8u * (8 * MTOT * LDV) +
                             warp * kRingWarpBytes + lane * 8u;

  const long long gw = (long long)blockIdx.x * kWarps + warp;
  const long long gstride = (long long)gridDim.x * kWarps;
  const long long kstep = XMODE ? 4 : 4LL * a.inner;  // elements between consecutive k-steps

  // Per-lane source pointers of the B fragments of warp tile wt: element (k = 4kt+q, column 8nt+g).
  // TWO: a second stream with the same stride is multiplied in on consumption -- the target function in
  // X-mode (pair density, a1), the multiplier table in L-mode (a3, applied while loading the z-backward pass).
  auto setup = [&](long long wt, const double* (&bp)[NT], const double* (&tp)[NT], bool (&cv)[NT]) {
    if (XMODE) {
      const int rhs = (int)fast_div((unsigned)wt, a.div_tiles);
      const int rb = (int)wt - rhs * a.tiles_per_rhs;
      const double* base0 = nullptr;
      const double* base1 = nullptr;
      if (TWO) {
        const int j = a.bd.j0 + rhs % a.bd.nj, k = a.bd.k0 + rhs / a.bd.nj;
        base0 = a.psi + (long long)j * a.N;
        base1 = a.tgt + (long long)k * a.N;
      } else {
        base0 = a.in + (long long)rhs * a.N;
      }
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        const int rr = rb * 8 * NT + 8 * nt + g;
        cv[nt] = rr < a.rows_per_rhs;
        const int off = (cv[nt] ? rr : 0) * n + q;
        bp[nt] = base0 + off;
        tp[nt] = TWO ? base1 + off : nullptr;
      }
    } else {
      // columns wt*8NT + 8nt + g: one division for the first, the rest by stepping 8 with carry
      unsigned c = (unsigned)wt * (8 * NT) + g;               // host guarantees total < 2^31
      const unsigned cfirst = c < (unsigned)a.total ? c : 0u;
      unsigned o = fast_div(cfirst, a.div_inner);
      int i = (int)(cfirst - o * (unsigned)a.inner);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        cv[nt] = c < (unsigned)a.total;
        bp[nt] = a.in + ((long long)o * n + q) * a.inner + i;
        tp[nt] = TWO ? a.mult + (long long)q * a.inner + i : nullptr;
        c += 8;
        i += 8;
        while (i >= a.inner) {
          i -= a.inner;
          ++o;
        }
      }
    }
  };

  // ---- producer state: runs kRing k-steps ahead of the consumer, straight across tile boundaries ----------
  long long wt_i = gw;
  int kt_i = 0;
  const double* bp_i[NT];
  const double* tp_i[NT];
  bool cv_i[NT];
  if (wt_i < a.n_tiles) setup(wt_i, bp_i, tp_i, cv_i);
  // issue the copies of the producer's current k-step into ring stage `st` (always exactly one commit group)
  auto issue_next = [&](int st) {
    if (wt_i < a.n_tiles) {
      const unsigned slot = ring_base + st * (NT * NS * 256u);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        const bool ok = cv_i[nt] && (4 * kt_i + q < n);
        const long long off = ok ? kt_i * kstep : 0;
        cp_async8(slot + (nt * NS) * 256u, bp_i[nt] + off, ok);
        if (TWO) cp_async8(slot + (nt * NS + 1) * 256u, tp_i[nt] + off, ok);
      }
      if (++kt_i == KT) {
        kt_i = 0;
        wt_i += gstride;
        if (wt_i < a.n_tiles) setup(wt_i, bp_i, tp_i, cv_i);
      }
    }
    cp_async_commit();
  };
#pragma unroll
  for (int d = 0; d < kRing; ++d) issue_next(d);
  int stage = 0;

  for (long long wt = gw; wt < a.n_tiles; wt += gstride) {
    int rhs = 0, rb = 0;
    if (XMODE) {
      rhs = (int)fast_div((unsigned)wt, a.div_tiles);
      rb = (int)wt - rhs * a.tiles_per_rhs;
    }
    double acc[MTOT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

#pragma unroll 2
    for (int kt = 0; kt < KT; ++kt) {
      cp_async_wait<kRing - 1>();  // this step's group has landed (each lane reads only its own slots)
      const unsigned slot = ring_base + stage * (NT * NS * 256u);
      double bf[NT];
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        bf[nt] = lds64(slot + (nt * NS) * 256u);
        if (TWO) bf[nt] *= lds64(slot + (nt * NS + 1) * 256u);
      }
      double af[MTOT];
      const unsigned aaddr = a_base + kt * A_KT;
#pragma unroll
      for (int mt = 0; mt < MTOT; ++mt) af[mt] = lds64(aaddr + mt * A_MT);
#pragma unroll
      for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], bf[nt]);
      // refill this stage: the DMMAs above consumed bf, so the LDS of the stage have completed
      issue_next(stage);
      stage = (stage + 1) & (kRing - 1);
    }

    // ---- epilogue: C[m = 8mt+g][column 8nt + 2q + e] straight from the fragments --------------------------
    if (XMODE) {
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int rr = rb * 8 * NT + 8 * nt + 2 * q + e;
          if (rr < a.rows_per_rhs) {
            double* dst = a.out + (long long)rhs * a.N + (long long)rr * n + g;
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt)
              if (8 * mt + g < n) dst[8 * mt] = acc[mt][nt][e];
          }
        }
      }
    } else if (a.vec2) {
      // inner is even and c is even, so the pair (c, c+1) never straddles a row of the flattened index
      unsigned c = (unsigned)wt * (8 * NT) + 2 * q;
      const unsigned cfirst = c < (unsigned)a.total ? c : 0u;
      unsigned o = fast_div(cfirst, a.div_inner);
      int i = (int)(cfirst - o * (unsigned)a.inner);
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
        if (c < (unsigned)a.total) {
          double* dst = a.out + ((long long)o * n + g) * a.inner + i;
#pragma unroll
          for (int mt = 0; mt < MTOT; ++mt) {
            if (8 * mt + g < n)
              *reinterpret_cast<double2*>(dst + (long long)(8 * mt) * a.inner) =
                  make_double2(acc[mt][nt][0], acc[mt][nt][1]);
          }
        }
        c += 8;
        i += 8;
        while (i >= a.inner) {
          i -= a.inner;
          ++o;
        }
      }
    } else {
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) {
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const unsigned ce = (unsigned)wt * (8 * NT) + 8 * nt + 2 * q + e;
          if (ce < (unsigned)a.total) {
            const unsigned o = fast_div(ce, a.div_inner);
            const int i = (int)(ce - o * (unsigned)a.inner);
            double* dst = a.out + ((long long)o * n + g) * a.inner + i;
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt) {
              if (8 * mt + g < n) dst[(long long)(8 * mt) * a.inner] = acc[mt][nt][e];
            }
          }
        }
      }
    }
  }
}

// ---- host side ------------------------------------------------------------------------------------

// supported classes of ceil(n/8) and the columns-per-warp choice for each
inline bool pick_class(int n, int* mtot, int* nt) {
  const int need = (n + 7) / 8;
  if (need <= 2) { *mtot = 2; *nt = 4; }
  else if (need <= 4) { *mtot = 4; *nt = 4; }
  else if (need <= 6) { *mtot = 6; *nt = 4; }
  else if (need <= 8) { *mtot = 8; *nt = 2; }
  else if (need <= 12) { *mtot = 12; *nt = 2; }
  else if (need <= 15) { *mtot = 15; *nt = 2; }
  else if (need <= 16) { *mtot = 16; *nt = 2; }
  else return false;
  return true;
}

template <int MTOT, int NT>
cudaError_t launch_class(bool xmode, bool fwd, bool two, const WArgs& a, int grid, int device, cudaStream_t s) {
  constexpr size_t smem_v = sizeof(double) * 8 * MTOT * (8 * MTOT + 4);
#define EXX_LAUNCH(XM, FW, PDD)                                                                         \
  do {                                                                                                  \
    /* at least half of the SM's shared memory, so that exactly one CTA fits per SM: the work split      \
       assumes one persistent CTA per SM, and with programmatic dependent launch the block scheduler     \
       would otherwise double up early-launched CTAs on whichever SMs free up first */                  \
    const size_t smem_need = smem_v + (size_t)kWarps * kRing * NT * ((PDD) ? 2 : 1) * 256;              \
    const size_t smem = smem_need > kMinSmem ? smem_need : kMinSmem;                                    \
    auto kern = k_mode_w<MTOT, NT, XM, FW, PDD>;                                                        \
    static SmemOptIn opt; /* per instantiation and device */                                           \
    {                                                                                                   \
      cudaError_t e = opt.ensure(kern, device, smem);                                                   \
      if (e != cudaSuccess) return e;                                                                   \
    }                                                                                                   \
    cudaLaunchConfig_t cfg = {};                                                                        \
    cfg.gridDim = dim3(grid);                                                                           \
    cfg.blockDim = dim3(kThreads);                                                                      \
    cfg.dynamicSmemBytes = smem;                                                                        \
    cfg.stream = s;                                                                                     \
    cudaLaunchAttribute at[1];                                                                          \
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;                                      \
    at[0].val.programmaticStreamSerializationAllowed = 1;                                               \
    cfg.attrs = at;                                                                                     \
    cfg.numAttrs = 1;                                                                                   \
    return cudaLaunchKernelEx(&cfg, kern, a);                                                           \
  } while (0)
  if (xmode) {
    if (fwd && two) EXX_LAUNCH(true, true, true);
    if (fwd) EXX_LAUNCH(true, true, false);
    EXX_LAUNCH(true, false, false);
  } else {
    if (fwd) EXX_LAUNCH(false, true, false);
    if (two) EXX_LAUNCH(false, false, true);
    EXX_LAUNCH(false, false, false);
  }
#undef EXX_LAUNCH
  return cudaErrorUnknown;
}

// One mode product along `axis` for nb right-hand sides; in == out is allowed (and is the normal case).
// pd != nullptr (axis 0, forward only): the input is psi_j .* tgt_k formed on the fly.
// apply_mult (axis 2, backward only): the input is multiplied by f(Lambda~) while it is loaded.
cudaError_t fast_mode_product(const exx_plan* p, int axis, bool forward, const double* in, double* out,
                              int nb, bool apply_mult, const FastArgs* pd, cudaStream_t s) {
  const int n = p->n[axis];
  int mtot, nt;
  if (!pick_class(n, &mtot, &nt)) return cudaErrorNotSupported;
  const bool xmode = axis == 0;
  if (pd && !(xmode && forward)) return cudaErrorInvalidValue;
  if (apply_mult && !(axis == 2 && !forward)) return cudaErrorInvalidValue;
  const bool two = pd != nullptr || apply_mult;
  WArgs a{};
  a.in = in;
  a.out = out;
  a.V = p->d_Vpad[axis];
  a.mult = apply_mult ? p->d_mult : nullptr;
  a.psi = pd ? pd->psi : nullptr;
  a.tgt = pd ? pd->tgt : nullptr;
  if (pd) a.bd = pd->bd;
  a.n = n;
  a.KT = (n + 3) / 4;
  a.N = p->N;
  const int cols_per_tile = 8 * nt;
  if (xmode) {
    a.inner = 1;
    a.rows_per_rhs = (int)(p->N / n);
    a.tiles_per_rhs = (a.rows_per_rhs + cols_per_tile - 1) / cols_per_tile;
    a.total = (long long)a.rows_per_rhs * nb;
    a.n_tiles = (long long)a.tiles_per_rhs * nb;
    a.vec2 = 0;
  } else {
    const long long inner = axis == 1 ? p->n[0] : (long long)p->n[0] * p->n[1];
    a.inner = (int)inner;
    a.total = p->N / n * nb;
    a.n_tiles = (a.total + cols_per_tile - 1) / cols_per_tile;
    a.rows_per_rhs = 0;
    a.tiles_per_rhs = 1;
    const bool aligned = (((uintptr_t)out) & 15) == 0;
    a.vec2 = (aligned && inner % 2 == 0) ? 1 : 0;
  }
  a.div_inner = make_fastdiv((unsigned)a.inner);
  a.div_tiles = make_fastdiv((unsigned)a.tiles_per_rhs);
  if (a.n_tiles <= 0) return cudaSuccess;
  if (a.total >= (1LL << 31) - 64 || a.n_tiles >= (1LL << 31) - 64) return cudaErrorNotSupported;  // 32-bit tile math
  const long long ctas = (a.n_tiles + kWarps - 1) / kWarps;
  const int grid = (int)(ctas < p->sm_count ? ctas : p->sm_count);
  switch (mtot) {
    case 2: return launch_class<2, 4>(xmode, forward, two, a, grid, p->device, s);
    case 4: return launch_class<4, 4>(xmode, forward, two, a, grid, p->device, s);
    case 6: return launch_class<6, 4>(xmode, forward, two, a, grid, p->device, s);
    case 8: return launch_class<8, 2>(xmode, forward, two, a, grid, p->device, s);
    case 12: return launch_class<12, 2>(xmode, forward, two, a, grid, p->device, s);
    case 15: return launch_class<15, 2>(xmode, forward, two, a, grid, p->device, s);
    default: return launch_class<16, 2>(xmode, forward, two, a, grid, p->device, s);
  }
}

}  // namespace

// Upload, per axis, the zero-padded shared-memory image of V that k_mode_w stages verbatim.
cudaError_t fast_init(exx_plan* p) {
  for (int ax = 0; ax < 3; ++ax) {
    p->d_Vpad[ax] = nullptr;
    int mtot, nt;
    if (!pick_class(p->n[ax], &mtot, &nt)) continue;  // this axis runs on the plain kernel
    int same = -1;
    for (int b = 0; b < ax; ++b)
      if (p->d_V[b] == p->d_V[ax] && p->d_Vpad[b]) same = b;
    if (same >= 0) {
      p->d_Vpad[ax] = p->d_Vpad[same];
      continue;
    }
    const int n = p->n[ax], rows = 8 * mtot, ldv = 8 * mtot + 4;
    std::vector<double> img((size_t)rows * ldv, 0.0);
    for (int r = 0; r < n; ++r)
      for (int c = 0; c < n; ++c) img[(size_t)r * ldv + c] = p->h_V[ax][(size_t)r * n + c];
    cudaError_t e = cudaMalloc(&p->d_Vpad[ax], sizeof(double) * img.size());
    if (e != cudaSuccess) return e;
    e = cudaMemcpy(p->d_Vpad[ax], img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

void fast_destroy(exx_plan* p) {
  for (int ax = 0; ax < 3; ++ax) {
    bool shared = false;
    for (int b = 0; b < ax; ++b) shared |= (p->d_Vpad[b] == p->d_Vpad[ax]);
    if (!shared && p->d_Vpad[ax]) cudaFree(p->d_Vpad[ax]);
  }
  for (int ax = 0; ax < 3; ++ax) p->d_Vpad[ax] = nullptr;
}

// Axes longer than 128 points do not fit the resident-V kernels; they run on the plain DFMA kernel
// (still CUDA, still in the library; stated in DESIGN.md).  `scratch` is only needed in that case.
// The multiplier (a3) is applied by the z-forward store in the plain kernel and by the z-backward load
// in the DMMA kernel; `mult_pending` carries it from one to the other.
static cudaError_t one_product(exx_plan* p, int axis, bool fwd, const double* src, double*& cur, double*& other,
                               int nb, bool& mult_pending, cudaStream_t s) {
  static const int kPass[3][2] = {{PASS_XB, PASS_XF}, {PASS_YB, PASS_YF}, {PASS_ZB, PASS_Z}};
  ProfScope ps(p, KC_MODE_PRODUCT, s, kPass[axis][fwd ? 1 : 0]);
  const bool z_bwd = axis == 2 && !fwd;
  cudaError_t e = cudaErrorNotSupported;
  if (p->variant == EXX_VARIANT_FUSED_DMMA)
    e = tma_mode_product(p, axis, fwd, src, cur, nb, z_bwd && mult_pending, nullptr, s);
  if (e == cudaErrorNotSupported)
    e = fast_mode_product(p, axis, fwd, src, cur, nb, z_bwd && mult_pending, nullptr, s);
  if (e == cudaSuccess) {
    if (z_bwd) mult_pending = false;
    return e;
  }
  if (e != cudaErrorNotSupported) return e;
  const bool z_fwd = axis == 2 && fwd;
  if (src == cur) {
    e = ref_mode_product(p, axis, fwd, cur, other, nb, z_fwd, s);
    double* t = cur;
    cur = other;
    other = t;
  } else {
    e = ref_mode_product(p, axis, fwd, src, cur, nb, z_fwd, s);
  }
  if (z_fwd) mult_pending = false;
  return e;
}

// One batch: `src` holds nb right-hand sides (ignored when fa != nullptr: the pair densities are formed on
// the fly), `work` receives phi (src == work allowed), `scratch` is a second nb*N buffer used only by the
// plain-kernel fallback.  With fa, phi is then accumulated into vx (a5).
cudaError_t fast_solve_batch(exx_plan* p, const double* src, double* work, double* scratch, int nb,
                             const FastArgs* fa, cudaStream_t s, long long* launches) {
  cudaError_t e;
  double *cur = work, *other = scratch;
  bool first_done = false, mult_pending = true;
  const long long tma_before = p->tma_launches;
  // symmetric mode with the x axis: both x passes of the exchange apply on the reflection-adapted basis (decided here,
  // before the first pass writes the batch in that mode order)
  bool xsym = fa && fused_sym_mode(p) && sym_x_usable(p, cur, fa);
  if (fa) {
    // a1 fused into the first product: rho = psi_j .* tgt_k is formed in the load path
    {
      ProfScope ps(p, KC_MODE_PRODUCT, s, PASS_XF);
      e = cudaErrorNotSupported;
      if (xsym) {
        e = sym_xf(p, cur, nb, fa, s);
        if (e == cudaErrorNotSupported) xsym = false;
      }
      if (!xsym && p->variant == EXX_VARIANT_FUSED_DMMA) e = tma_mode_product(p, 0, true, nullptr, cur, nb, false, fa, s);
      if (e == cudaErrorNotSupported) e = fast_mode_product(p, 0, true, nullptr, cur, nb, false, fa, s);
      if (e == cudaErrorNotSupported) ps.cancel();  // nothing ran here: the plain pair density + x product below are recorded
    }
    if (e == cudaSuccess) {
      first_done = true;
    } else if (e == cudaErrorNotSupported) {
      ProfScope ps(p, KC_PAIR_DENSITY, s);
      e = ref_pair_density(p, fa->psi, fa->tgt, fa->bd, cur, s);
      ++*launches;
      src = cur;
    }
    if (e != cudaSuccess) return e;
  }
  // bare solver: both x passes on the reflection-adapted basis where the plan and the buffers allow it
  bool xsym_plain = !fa && p->variant == EXX_VARIANT_FUSED_DMMA && fused_sym_mode(p) && sym_x_usable_plain(p, src, cur, nb);
  if (xsym_plain) {
    ProfScope ps(p, KC_MODE_PRODUCT, s, PASS_XF);
    e = sym_xf_plain(p, src, cur, nb, s);
    if (e == cudaErrorNotSupported) {
      ps.cancel();
      xsym_plain = false;
    } else if (e != cudaSuccess) {
      return e;
    } else {
      first_done = true;
    }
  }
  if (!first_done && (e = one_product(p, 0, true, src, cur, other, nb, mult_pending, s)) != cudaSuccess) return e;
  // Symmetric mode: the y and z products on the reflection-adapted eigenbases, eigen-space data and
  // table in (even | odd) mode order.  Decided once per batch: it needs every remaining pass on the TMA kernels, which
  // the x-forward pass having run there (same buffer, same alignment rules) establishes.
  const bool sym = fused_sym_mode(p) && p->tma_launches > tma_before && (((uintptr_t)cur) & 15) == 0;
  auto y_product = [&](bool fwd) -> cudaError_t {
    if (sym) {
      ProfScope ps(p, KC_MODE_PRODUCT, s, fwd ? PASS_YF : PASS_YB);
      const cudaError_t ey = sym_mode_product_y(p, fwd, cur, nb, s);
      if (ey == cudaSuccess) return ey;
      ps.cancel();
      if (ey != cudaErrorNotSupported) return ey;  // NotSupported: the plan has no symmetric y axis, dense product below
    }
    return one_product(p, 1, fwd, cur, cur, other, nb, mult_pending, s);
  };
  if ((e = y_product(true)) != cudaSuccess) return e;
  // z-forward + multiplier + z-backward: one fused pass where k_mode_zz can run, else two passes
  e = cudaErrorNotSupported;
  if (p->variant == EXX_VARIANT_FUSED_DMMA) {
    ProfScope ps(p, KC_MODE_PRODUCT, s, PASS_Z);
    e = fused_zz(p, cur, cur, nb, s, (xsym || xsym_plain) ? 2 : sym ? 1 : 0);
    if (e != cudaSuccess) ps.cancel();
  }
  if (e == cudaSuccess) {
    mult_pending = false;
    *launches += 1;
  } else if (e == cudaErrorNotSupported && !sym) {
    if ((e = one_product(p, 2, true, cur, cur, other, nb, mult_pending, s)) != cudaSuccess) return e;
    if ((e = one_product(p, 2, false, cur, cur, other, nb, mult_pending, s)) != cudaSuccess) return e;
    *launches += 2;
  } else {
    return e;
  }
  if (mult_pending) return cudaErrorUnknown;  // cannot happen: same axis, same support decision
  if ((e = y_product(false)) != cudaSuccess) return e;
  *launches += 3;
  // x-backward + accumulate: one fused pass where k_mode_xacc can run
  if (fa && p->variant == EXX_VARIANT_FUSED_DMMA) {
    {
      ProfScope ps(p, KC_MODE_PRODUCT, s, PASS_XB);
      e = xsym ? sym_xacc(p, cur, nb, fa, s) : fused_xacc(p, cur, nb, fa, s);
      if (xsym && e == cudaErrorNotSupported) e = cudaErrorUnknown;  // the batch is in x-symmetric order: no fallback
      if (e != cudaSuccess) ps.cancel();
    }
    if (e == cudaSuccess && xsym && fa->sym) {
      // pair-symmetric apply: the same pass again with the orbitals as work items (vx_j -= sum_{k > j} occ_k psi_k phi_jk)
      ProfScope ps(p, KC_MODE_PRODUCT, s, PASS_XB2);
      e = sym_xacc(p, cur, nb, fa, s, 1);
      if (e != cudaSuccess) return e;
      *launches += 1;
    }
    if (e == cudaSuccess) {
      *launches += 1;
      return e;
    }
    if (e != cudaErrorNotSupported) return e;
  }
  if (xsym_plain) {  // the batch is in x-symmetric mode order: no fallback
    ProfScope ps(p, KC_MODE_PRODUCT, s, PASS_XB);
    e = sym_xb_plain(p, cur, nb, s);
    *launches += 1;
    return e == cudaErrorNotSupported ? cudaErrorUnknown : e;
  }
  if ((e = one_product(p, 0, false, cur, cur, other, nb, mult_pending, s)) != cudaSuccess) return e;
  *launches += 1;
  if (fa) {
    {
      ProfScope ps(p, KC_ACCUMULATE, s);
      e = ref_accumulate(p, fa->psi, fa->occ, cur, fa->bd, fa->first, fa->vx, s, fa->sym);
      if (e == cudaSuccess && fa->sym) {
        e = sym_accumulate_transposed(p, fa->psi, fa->occ, cur, fa->bd, fa->vx, s);
        ++*launches;
      }
    }
    if (e != cudaSuccess) return e;
    ++*launches;
  } else if (cur != work) {
    e = cudaMemcpyAsync(work, cur, sizeof(double) * (size_t)p->N * nb, cudaMemcpyDeviceToDevice, s);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

}  // namespace exx
