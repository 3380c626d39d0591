// Shared by the TMA-staged tensor-core kernels (kernels_tma.cu, kernels_fused.cu): PTX wrappers (DMMA, mbarrier, TMA
// box copies), exact integer division by a host-computed multiplier, and the host-side tensor-map cache and
// shared-memory images of the plan.  Everything has internal linkage (one copy per translation unit).
#pragma once
#include <cuda.h>  // CUtensorMap and its enums only; cuTensorMapEncodeTiled is resolved at run time

#include <cstdint>
#include <cstdlib>
#include <cstring>

#include "exx_internal.h"

namespace exx {

// state the plan keeps for the TMA-staged kernels (exx_plan::tma_state)
struct MapKey {
  const void* base;
  unsigned long long d0, d1, d2;
  unsigned b1;  // box rows (third box dimension 1)
  unsigned b0;  // box columns: 16, or 8 for the half-chunk tiles
  bool operator==(const MapKey& o) const {
    return base == o.base && d0 == o.d0 && d1 == o.d1 && d2 == o.d2 && b1 == o.b1 && b0 == o.b0;
  }
};
struct MapEntry {
  MapKey key;
  CUtensorMap map;
};

struct TmaState {
  double* d_img[3][2];  // [axis][0 = forward (V^T), 1 = backward (V)]
  bool img_owned[3][2];
  double* d_img_im[3][2];  // Bloch plans: images of the imaginary parts, forward = Im(V^H) = -Vi^T, backward = Vi
  double* d_img_c[3][2];   // Bloch axes with n <= 64: real embedding [[Mr, -Mi], [Mi, Mr]] for the single-launch complex product
  double* d_img_hc[2];     // y axis, nx == 8 (mod 16): L-mode images in the row order of the half-chunk tiles (HC)
  // reflection-adapted eigenbases ("symmetric mode").  z axis (k_mode_zz_sym): image over the half range,
  // number of even modes (0: not capable).  y axis (kernels_sym.cu): forward and backward images, their row order (hc),
  // the basis itself.  d_mult_sym: the multiplier table with the eigen index of every capable axis in (even | odd) order.
  double* d_img_zzs;
  int zs_nh;
  double* d_img_yf;
  double* d_img_yb;
  int ys_nh;
  bool ys_hc;
  std::vector<double> lam_ys, V_ys;
  double* d_mult_sym;
  // x axis (k_mode_xf_sym / k_mode_xacc_sym, exchange apply only): images, basis, and the table with x in that order too
  double* d_img_xf;
  double* d_img_xb;
  int xs_nh;
  std::vector<double> lam_xs, V_xs;
  double* d_mult_symx;
  double* d_img_zz_c;      // the same for a complex z axis with n <= 64 (embedding E = [[Vr, -Vi], [Vi, Vr]])
  double* d_img_zz;  // fused z-forward/z-backward kernel: one image of Vz serving both products (kernels_fused.cu)
  std::vector<MapEntry> cache;
};

namespace {

constexpr int kDepth = 2;  // ring depth in stages of 16 contraction indices (4 k-steps, >= 96 DMMAs each)

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
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
// Called by the elected lane right before it re-arms a ring slot and issues the TMA copies into it, after the
// __syncwarp that follows the warp's last reads of that slot: the proxy fence orders those generic-proxy reads before
// the async-proxy writes of the copies (the release half of the per-warp ring; the acquire half is the mbarrier wait).
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
  asm volatile("fence.proxy.async.shared::cta;\n" ::: "memory");
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
// Blocks until the phase with the given parity has completed.  A (very generously) bounded spin turns a lost
// transaction (a bug) into a trap instead of a hung GPU.
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
  unsigned done = 0;
  for (unsigned spin = 0; !done; ++spin) {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    if (spin > (1u << 30)) __trap();  // tens of seconds: far beyond any profiler replay or time-slicing delay
  }
}
__device__ __forceinline__ void tma_load_2d(unsigned dst, const CUtensorMap* tm, int c0, int c1, unsigned bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];\n" ::"r"(dst),
      "l"(tm), "r"(c0), "r"(c1), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void tma_load_3d(unsigned dst, const CUtensorMap* tm, int c0, int c1, int c2,
                                            unsigned bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];\n" ::"r"(
          dst),
      "l"(tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
      : "memory");
}

// Exact n / d for n < 2^31 with a host-computed multiplier (d = 2^shift when mul == 0).
struct FastDiv {
  unsigned mul;
  int shift;
};
inline FastDiv make_fastdiv(unsigned d) {
  FastDiv f{0u, 0};
  if ((d & (d - 1)) == 0) {
    while ((1u << f.shift) < d) ++f.shift;
    return f;
  }
  int L = 0;
  while ((1ull << L) < d) ++L;
  f.mul = (unsigned)(((1ull << (31 + L)) / d) + 1ull);
  f.shift = L - 1;
  return f;
}
__device__ __forceinline__ unsigned fast_div(unsigned n, const FastDiv& f) {
  return f.mul ? (__umulhi(n, f.mul) >> f.shift) : (n >> f.shift);
}

__device__ __forceinline__ bool elect_one() {
  unsigned pred;
  asm volatile("{\n .reg .pred p;\n elect.sync _|p, 0xffffffff;\n selp.u32 %0, 1, 0, p;\n}\n" : "=r"(pred));
  return pred != 0;
}
__device__ __forceinline__ void stg_v2(double* p, double x, double y) {
  asm volatile("st.global.v2.f64 [%0], {%1, %2};\n" ::"l"(p), "d"(x), "d"(y) : "memory");
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = [] {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qr) != cudaSuccess ||
        qr != cudaDriverEntryPointSuccess)
      p = nullptr;
    return (EncodeTiledFn)p;
  }();
  return fn;
}

// 2-D ([d1][d0]) or 3-D ([d2][d1][d0]) FP64 tensor, box {box_cols, box_rows(, 1)}, zero fill; the swizzle span equals the
// box width: 128 bytes for 16 columns, 64 bytes for 8.
cudaError_t get_map(TmaState* st, const void* base, unsigned long long d0, unsigned long long d1,
                    unsigned long long d2, unsigned box_rows, CUtensorMap* out, unsigned box_cols = 16) {
  const MapKey key{base, d0, d1, d2, box_rows, box_cols};
  for (const auto& e : st->cache)
    if (e.key == key) {
      *out = e.map;
      return cudaSuccess;
    }
  EncodeTiledFn fn = encode_fn();
  if (!fn) return cudaErrorNotSupported;
  const cuuint32_t rank = d2 ? 3 : 2;
  cuuint64_t gdim[3] = {d0, d1, d2 ? d2 : 1};
  cuuint64_t gstr[2] = {d0 * 8ull, d0 * d1 * 8ull};
  cuuint32_t box[3] = {box_cols, box_rows, 1u};
  cuuint32_t estr[3] = {1u, 1u, 1u};
  alignas(64) CUtensorMap m;
  const CUresult r = fn(&m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, rank, const_cast<void*>(base), gdim, gstr, box, estr,
                        CU_TENSOR_MAP_INTERLEAVE_NONE, box_cols == 8 ? CU_TENSOR_MAP_SWIZZLE_64B : CU_TENSOR_MAP_SWIZZLE_128B,
                        CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
                        CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return cudaErrorInvalidValue;
  if (st->cache.size() >= 64) st->cache.clear();
  st->cache.push_back(MapEntry{key, m});
  *out = m;
  return cudaSuccess;
}

inline bool aligned16(const void* p) { return (((uintptr_t)p) & 15) == 0; }

// k-steps of the ragged last stage (0 when n is a multiple of 16: every stage is a standard one)
inline int tail_ksteps(int n) { return (n % 16) ? (n % 16 + 3) / 4 : 0; }

// Contraction index (within its block of 16) that the lane with this q reads in k-step kk of stage s: the order in
// which the swizzled boxes deliver it in a standard stage, plain 4 kk + q in the ragged last stage.
inline int within_stage(bool xmode, int n, int s, int kk, int q, bool hc = false) {
  if ((n % 16) && s == (n + 15) / 16 - 1) return 4 * kk + q;
  if (hc) return (q & 1) + 4 * (q >> 1) + 2 * (kk & 1) + 8 * (kk >> 1);  // 8-column boxes, 64-byte rows
  return xmode ? ((q & 1) + 8 * (q >> 1) + 2 * kk) : (2 * q + (kk & 1) + 8 * (kk >> 1));
}

}  // namespace
}  // namespace exx
