// Mode products of the y axis on the reflection-adapted eigenbasis (plan_host.cpp symmetrize_axis).
// Every eigenvector of a real periodic or Dirichlet axis is even or odd under y -> mir(y), so
//     forward  (k_mode_lf_sym):  T[m] = sum_{y <= mir y} V[y][m] (f[y] +- f[mir y])     (+: even mode, -: odd mode)
//     backward (k_mode_lb_sym):  a[y] = sum_{m even} V[y][m] t[m],  b[y] = sum_{m odd} V[y][m] t[m],
//                                out[y] = a + b,  out[mir y] = a - b
// contract over half the range with two blocks of the matrix: about 55 % of the DMMAs of k_mode_t.  In eigen-space
// the modes are stored even block first (nh modes), then the odd block; the plan's "symmetric" multiplier table uses the
// same order.  Machinery as k_mode_t's L-mode (kernels_tma.cu): per-warp TMA rings, one persistent CTA per SM,
// programmatic dependent launch, 16-column chunks or (HC) 8-column half-chunks.  The forward kernel's stage is two boxes,
// rows [16 s, 16 s + 16) and the mirrored rows (row 15 - r of the second box is mir(16 s + r)).
#include <type_traits>

#include "tma_common.cuh"

namespace exx {
namespace {

struct SArgs {
  double* out;
  const double* V;
  int n;
  int nh;               // even modes = half-range points
  int Sh;               // forward: stages over the half range; backward: stages over the even modes
  int So;               // backward: stages over the odd modes
  int kk_last, kk_last_o;  // k-steps of the ragged last stage of the (even | half-range) block and of the odd block; 0: none
  int mir0, mirc, zfix;    // as k_mode_zz_sym
  unsigned n_tiles;
  int inner, cpo, outer;
  unsigned total_chunks;
  FastDiv div_cpo;
};

// box-row offset of (k-step kk, lane) inside a stage, and of its mirror image 15 - r, for 16-column boxes (128-byte rows,
// 128-byte swizzle; np = which 8-column half) and for 8-column boxes (64-byte rows, 64-byte swizzle)
__device__ __forceinline__ unsigned off16(unsigned r, unsigned np, unsigned g) {
  return 128u * r + 16u * ((4u * np + (g >> 1)) ^ (r & 7u)) + 8u * (g & 1);
}
__device__ __forceinline__ unsigned off8(unsigned r, unsigned g) {
  return 64u * r + 16u * ((g >> 1) ^ ((r >> 1) & 3u)) + 8u * (g & 1);
}
template <bool HC>
__device__ __forceinline__ unsigned row_of(int kk, int q, bool ragged) {
  if (ragged) return 4u * kk + q;
  return HC ? (unsigned)((q & 1) + 4 * (q >> 1) + 2 * (kk & 1) + 8 * (kk >> 1)) : (unsigned)(2 * q + (kk & 1) + 8 * (kk >> 1));
}

// ---------------------------------------------------------------------------------------------------------------
// forward
// ---------------------------------------------------------------------------------------------------------------
template <int MS, int NT, int WARPS, bool HC>
__global__ void __launch_bounds__(32 * WARPS, 1) k_mode_lf_sym(const __grid_constant__ CUtensorMap tm0, const SArgs a) {
  constexpr int MT = 2 * MS;
  constexpr int LDV = 8 * MT + 4;
  constexpr unsigned kS1 = 1024u * NT;
  constexpr unsigned kSlot = 2u * kS1;
  constexpr int CH = HC ? NT : NT / 2;
  constexpr int CW = HC ? 8 : 16;
  constexpr unsigned kBox = HC ? 1024u : 2048u;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, Sh = a.Sh;
  const unsigned smem0 = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned img_bytes = 8u * (16u * Sh) * LDV;
  for (unsigned i = 2 * tid; i < 16u * Sh * LDV; i += 2 * 32 * WARPS)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem0 + 8u * i), "l"(a.V + i) : "memory");
  asm volatile("cp.async.commit_group;\n" ::: "memory");
  const unsigned ring0 = (smem0 + img_bytes + 1023u) & ~1023u;
  const unsigned my_ring = ring0 + warp * (kDepth * kSlot);
  const unsigned my_bar = ring0 + WARPS * (kDepth * kSlot) + warp * (kDepth * 8u);
  const unsigned ctr_addr = ring0 + WARPS * (kDepth * kSlot) + WARPS * (kDepth * 8u);
  if (tid == 0) asm volatile("st.shared.u32 [%0], %1;\n" ::"r"(ctr_addr), "r"((unsigned)WARPS) : "memory");
  if (lane == 0) {
#pragma unroll
    for (int d = 0; d < kDepth; ++d) mbar_init(my_bar + 8u * d, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  asm volatile("griddepcontrol.wait;\n" ::: "memory");

  const unsigned tfirst = blockIdx.x + gridDim.x * warp;
  auto claim_tile = [&]() -> unsigned {
    unsigned i = 0;
    if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;\n" : "=r"(i) : "r"(ctr_addr) : "memory");
    i = __shfl_sync(0xffffffffu, i, 0);
    const unsigned long long t = (unsigned long long)blockIdx.x + (unsigned long long)gridDim.x * i;
    return t < a.n_tiles ? (unsigned)t : 0xffffffffu;
  };
  unsigned fifo[kDepth + 1];
  int fifo_n = 0;
  unsigned t_p = tfirst;
  int s_p = 0;
  int pc0[CH], pc2[CH];
  auto tile_coords = [&](unsigned t) {
#pragma unroll
    for (int ch = 0; ch < CH; ++ch) {
      const unsigned cc = t * CH + ch;
      if (cc < a.total_chunks) {
        const unsigned o = fast_div(cc, a.div_cpo);
        pc2[ch] = (int)o;
        pc0[ch] = CW * (int)(cc - o * (unsigned)a.cpo);
      } else {
        pc2[ch] = a.outer;
        pc0[ch] = 0;
      }
    }
  };
  auto produce = [&](int slot) {
    if (t_p >= a.n_tiles) return;
    const unsigned bar = my_bar + 8u * slot;
    const unsigned dst = my_ring + slot * kSlot;
    if (elect_one()) {
      mbar_expect_tx(bar, kSlot);
#pragma unroll
      for (int ch = 0; ch < CH; ++ch) {
        tma_load_3d(dst + kBox * ch, &tm0, pc0[ch], 16 * s_p, pc2[ch], bar);
        tma_load_3d(dst + kS1 + kBox * ch, &tm0, pc0[ch], a.mir0 - 16 * s_p, pc2[ch], bar);
      }
    }
    if (++s_p == Sh) {
      s_p = 0;
      t_p = claim_tile();
#pragma unroll
      for (int i = 0; i < kDepth + 1; ++i)
        if (i == fifo_n) fifo[i] = t_p;
      ++fifo_n;
      if (t_p < a.n_tiles) tile_coords(t_p);
    }
  };
  if (t_p < a.n_tiles) tile_coords(t_p);
#pragma unroll
  for (int d = 0; d < kDepth; ++d) produce(d);
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();

  unsigned a_lane_v = smem0 + 8u * (q * LDV + g);
  // standard stages: offsets of this lane's row and of its mirror image; HC: index kk; else index 2 (nt&1) + (kk&1)
  unsigned xo[4], xm[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (HC) {
      const unsigned r = row_of<true>(i, q, false);
      xo[i] = off8(r, g);
      xm[i] = kS1 + off8(15u - r, g);
    } else {
      const unsigned r = 2u * q + (i & 1);  // rows 0..7; k-steps 2, 3 add 8 rows
      xo[i] = off16(r, i >> 1, g);
      xm[i] = kS1 + off16(7u - r, i >> 1, g);
    }
  }

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  while (t < a.n_tiles) {
    double acc[MT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;
    // one stage of 16 half-range rows; `ragged` (the last stage when nh % 16 != 0: plain row order, kk_last k-steps) is a
    // compile-time flag so that the standard stages carry none of its address arithmetic
    auto do_stage = [&](int s, auto rag_c) {
      constexpr bool ragged = decltype(rag_c)::value;
      asm volatile("" : "+r"(a_lane_v), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
      mbar_wait(my_bar + 8u * slot, parity);
      const unsigned sb = my_ring + slot * kSlot;
      const unsigned aa = a_lane_v + (unsigned)s * (16u * LDV * 8u);
      const int zf = a.zfix - 16 * s;
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
        if (!ragged || kk < a.kk_last) {
          double be[NT], bo[NT];
          const int rowl = (int)row_of<HC>(kk, q, ragged);
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            unsigned oa, ob;
            if (HC) {
              if (!ragged) {
                oa = sb + 1024u * nt + xo[kk];
                ob = sb + 1024u * nt + xm[kk];
              } else {
                oa = sb + 1024u * nt + off8((unsigned)rowl, g);
                ob = sb + kS1 + 1024u * nt + off8(15u - (unsigned)rowl, g);
              }
            } else {
              if (!ragged) {
                oa = sb + xo[2 * (nt & 1) + (kk & 1)] + 2048u * (nt >> 1) + 1024u * (kk >> 1);
                ob = sb + xm[2 * (nt & 1) + (kk & 1)] + 2048u * (nt >> 1) + 1024u * (1 - (kk >> 1));
              } else {
                oa = sb + 2048u * (nt >> 1) + off16((unsigned)rowl, nt & 1, g);
                ob = sb + kS1 + 2048u * (nt >> 1) + off16(15u - (unsigned)rowl, nt & 1, g);
              }
            }
            const double va = lds64(oa);
            double vb = lds64(ob);
            if (rowl == zf) vb = 0.0;
            be[nt] = va + vb;
            bo[nt] = va - vb;
          }
          double af[MT];
#pragma unroll
          for (int mt = 0; mt < MT; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
          for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], mt < MS ? be[nt] : bo[nt]);
        }
      }
      __syncwarp();
      produce(slot);
      if (++slot == kDepth) {
        slot = 0;
        parity ^= 1u;
      }
    };
    {
      const int s_full = a.kk_last ? Sh - 1 : Sh;
      for (int s = 0; s < s_full; ++s) do_stage(s, std::false_type{});
      if (a.kk_last) do_stage(Sh - 1, std::true_type{});
    }
    // epilogue: C[mode 8 (mt % MS) + g of block mt / MS][column 8nt + 2q + e]; even modes -> rows 0.., odd modes -> rows nh..
    const long long rstep = a.inner;
#pragma unroll
    for (int ch = 0; ch < CH; ++ch) {
      const unsigned cc = t * CH + ch;
      if (cc < a.total_chunks) {
        const unsigned o = fast_div(cc, a.div_cpo);
        const int col0 = CW * (int)(cc - o * (unsigned)a.cpo) + 2 * q;
        double* base = a.out + (long long)o * n * a.inner + col0;
        const bool in0 = col0 < a.inner, in1 = !HC && col0 + 8 < a.inner;
#pragma unroll
        for (int mt = 0; mt < MT; ++mt) {
          const int blk = mt >= MS ? 1 : 0;
          const int ml = 8 * (mt - blk * MS) + g;
          if (ml < (blk ? n - a.nh : a.nh)) {
            double* ptr = base + (long long)(blk * a.nh + ml) * rstep;
            if (HC) {
              if (in0) stg_v2(ptr, acc[mt][ch][0], acc[mt][ch][1]);
            } else {
              if (in0) stg_v2(ptr, acc[mt][2 * ch < NT ? 2 * ch : 0][0], acc[mt][2 * ch < NT ? 2 * ch : 0][1]);
              if (in1) stg_v2(ptr + 8, acc[mt][2 * ch + 1 < NT ? 2 * ch + 1 : 0][0], acc[mt][2 * ch + 1 < NT ? 2 * ch + 1 : 0][1]);
            }
          }
        }
      }
    }
    t = fifo[0];
#pragma unroll
    for (int i = 0; i < kDepth; ++i) fifo[i] = fifo[i + 1];
    --fifo_n;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// backward
// ---------------------------------------------------------------------------------------------------------------
template <int MS, int NT, int WARPS, bool HC>
__global__ void __launch_bounds__(32 * WARPS, 1) k_mode_lb_sym(const __grid_constant__ CUtensorMap tm0, const SArgs a) {
  constexpr int LDV = 8 * MS + 4;
  constexpr unsigned kS1 = 1024u * NT;
  constexpr int CH = HC ? NT : NT / 2;
  constexpr int CW = HC ? 8 : 16;
  constexpr unsigned kBox = HC ? 1024u : 2048u;
  // a stage is up to SETS sets of 16 modes of one parity block: two halve the barrier waits per tile (-3 to -6 % from
  // 60 points per axis up); at 48 points, where a block is two sets and the pass is bound by HBM, one set measured 4 % faster
  constexpr int SETS = MS <= 3 ? 1 : 2;
  constexpr unsigned kSlot = SETS * kS1;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, SE = a.Sh, ST = a.Sh + a.So;
  const int SE2 = (SE + SETS - 1) / SETS, ST2 = SE2 + (ST - SE + SETS - 1) / SETS;  // stages of the even block / of a tile
  const unsigned smem0 = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned img_bytes = 8u * (16u * ST) * LDV;
  for (unsigned i = 2 * tid; i < 16u * ST * LDV; i += 2 * 32 * WARPS)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem0 + 8u * i), "l"(a.V + i) : "memory");
  asm volatile("cp.async.commit_group;\n" ::: "memory");
  const unsigned ring0 = (smem0 + img_bytes + 1023u) & ~1023u;
  const unsigned my_ring = ring0 + warp * (kDepth * kSlot);
  const unsigned my_bar = ring0 + WARPS * (kDepth * kSlot) + warp * (kDepth * 8u);
  const unsigned ctr_addr = ring0 + WARPS * (kDepth * kSlot) + WARPS * (kDepth * 8u);
  if (tid == 0) asm volatile("st.shared.u32 [%0], %1;\n" ::"r"(ctr_addr), "r"((unsigned)WARPS) : "memory");
  if (lane == 0) {
#pragma unroll
    for (int d = 0; d < kDepth; ++d) mbar_init(my_bar + 8u * d, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  asm volatile("griddepcontrol.wait;\n" ::: "memory");

  const unsigned tfirst = blockIdx.x + gridDim.x * warp;
  auto claim_tile = [&]() -> unsigned {
    unsigned i = 0;
    if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;\n" : "=r"(i) : "r"(ctr_addr) : "memory");
    i = __shfl_sync(0xffffffffu, i, 0);
    const unsigned long long t = (unsigned long long)blockIdx.x + (unsigned long long)gridDim.x * i;
    return t < a.n_tiles ? (unsigned)t : 0xffffffffu;
  };
  unsigned fifo[kDepth + 1];
  int fifo_n = 0;
  unsigned t_p = tfirst;
  int s_p = 0;
  int pc0[CH], pc2[CH];
  auto tile_coords = [&](unsigned t) {
#pragma unroll
    for (int ch = 0; ch < CH; ++ch) {
      const unsigned cc = t * CH + ch;
      if (cc < a.total_chunks) {
        const unsigned o = fast_div(cc, a.div_cpo);
        pc2[ch] = (int)o;
        pc0[ch] = CW * (int)(cc - o * (unsigned)a.cpo);
      } else {
        pc2[ch] = a.outer;
        pc0[ch] = 0;
      }
    }
  };
  auto produce = [&](int slot) {
    if (t_p >= a.n_tiles) return;
    const unsigned bar = my_bar + 8u * slot;
    const unsigned dst = my_ring + slot * kSlot;
    if (elect_one()) {
      const int blk = s_p < SE2 ? 0 : 1, b0 = SETS * (s_p - blk * SE2), cnt = blk ? ST - SE : SE;
      const int nbx = cnt - b0 < SETS ? cnt - b0 : SETS;
      mbar_expect_tx(bar, kS1 * (unsigned)nbx);
#pragma unroll
      for (int hh = 0; hh < SETS; ++hh)
        if (hh < nbx) {
          const int row = (blk ? a.nh : 0) + 16 * (b0 + hh);  // even modes: rows 0.., odd modes: rows nh..
#pragma unroll
          for (int ch = 0; ch < CH; ++ch) tma_load_3d(dst + kS1 * hh + kBox * ch, &tm0, pc0[ch], row, pc2[ch], bar);
        }
    }
    if (++s_p == ST2) {
      s_p = 0;
      t_p = claim_tile();
#pragma unroll
      for (int i = 0; i < kDepth + 1; ++i)
        if (i == fifo_n) fifo[i] = t_p;
      ++fifo_n;
      if (t_p < a.n_tiles) tile_coords(t_p);
    }
  };
  if (t_p < a.n_tiles) tile_coords(t_p);
#pragma unroll
  for (int d = 0; d < kDepth; ++d) produce(d);
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();

  unsigned a_lane_v = smem0 + 8u * (q * LDV + g);
  unsigned xo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (HC) xo[i] = off8(row_of<true>(i, q, false), g);
    else xo[i] = off16(2u * q + (i & 1), i >> 1, g);
  }

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  while (t < a.n_tiles) {
    double pa[MS][NT][2], pb[MS][NT][2];
#pragma unroll
    for (int mt = 0; mt < MS; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) pa[mt][nt][0] = pa[mt][nt][1] = pb[mt][nt][0] = pb[mt][nt][1] = 0.0;
    // one set of 16 modes (`ragged`, compile time: the last set of a block whose size is not a multiple of 16)
    auto box = [&](auto& acc, unsigned sb, int s, auto rag_c, int kk_last) {
      constexpr bool ragged = decltype(rag_c)::value;
      asm volatile("" : "+r"(a_lane_v), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
      const unsigned aa = a_lane_v + (unsigned)s * (16u * LDV * 8u);
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
        if (!ragged || kk < kk_last) {
          double bf[NT];
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            unsigned off;
            if (HC) off = sb + 1024u * nt + (ragged ? off8(4u * kk + q, g) : xo[kk]);
            else off = ragged ? sb + 2048u * (nt >> 1) + off16(4u * kk + q, nt & 1, g)
                              : sb + xo[2 * (nt & 1) + (kk & 1)] + 2048u * (nt >> 1) + 1024u * (kk >> 1);
            bf[nt] = lds64(off);
          }
          double af[MS];
#pragma unroll
          for (int mt = 0; mt < MS; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
          for (int mt = 0; mt < MS; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], bf[nt]);
        }
      }
    };
    // a parity block of `cnt` sets (image stages s0 ..): stages of two sets behind one barrier wait each
    auto block = [&](auto& acc, int s0, int cnt, int kk_last) {
      for (int b0 = 0; b0 < cnt; b0 += SETS) {
        const int nbx = cnt - b0 < SETS ? cnt - b0 : SETS;
        mbar_wait(my_bar + 8u * slot, parity);
        const unsigned sb = my_ring + slot * kSlot;
        if (SETS == 2 && nbx == 2) box(acc, sb, s0 + b0, std::false_type{}, 0);
        const unsigned sl = sb + kS1 * (unsigned)(nbx - 1);
        if (kk_last && b0 + nbx == cnt) box(acc, sl, s0 + b0 + nbx - 1, std::true_type{}, kk_last);
        else box(acc, sl, s0 + b0 + nbx - 1, std::false_type{}, 0);
        __syncwarp();
        produce(slot);
        if (++slot == kDepth) {
          slot = 0;
          parity ^= 1u;
        }
      }
    };
    block(pa, 0, SE, a.kk_last);
    block(pb, SE, ST - SE, a.kk_last_o);

    // epilogue: out[y] = a + b, out[mir y] = a - b for the half-range rows y = 8mt + g
#pragma unroll
    for (int ch = 0; ch < CH; ++ch) {
      const unsigned cc = t * CH + ch;
      if (cc < a.total_chunks) {
        const unsigned o = fast_div(cc, a.div_cpo);
        const int col0 = CW * (int)(cc - o * (unsigned)a.cpo) + 2 * q;
        double* base = a.out + (long long)o * n * a.inner + col0;
        const bool in0 = col0 < a.inner, in1 = !HC && col0 + 8 < a.inner;
#pragma unroll
        for (int mt = 0; mt < MS; ++mt) {
          const int y = 8 * mt + g;
          if (y < a.nh) {
            const int yb = a.mirc - y;
            const bool two = yb != y && yb < n;
            double* p0 = base + (long long)y * a.inner;
            double* p1 = base + (long long)yb * a.inner;
            constexpr int kZ = 0;
            const int n0 = HC ? ch : (2 * ch < NT ? 2 * ch : kZ), n1 = HC ? kZ : (2 * ch + 1 < NT ? 2 * ch + 1 : kZ);
            if (in0) {
              stg_v2(p0, pa[mt][n0][0] + pb[mt][n0][0], pa[mt][n0][1] + pb[mt][n0][1]);
              if (two) stg_v2(p1, pa[mt][n0][0] - pb[mt][n0][0], pa[mt][n0][1] - pb[mt][n0][1]);
            }
            if (in1) {
              stg_v2(p0 + 8, pa[mt][n1][0] + pb[mt][n1][0], pa[mt][n1][1] + pb[mt][n1][1]);
              if (two) stg_v2(p1 + 8, pa[mt][n1][0] - pb[mt][n1][0], pa[mt][n1][1] - pb[mt][n1][1]);
            }
          }
        }
      }
    }
    t = fifo[0];
#pragma unroll
    for (int i = 0; i < kDepth; ++i) fifo[i] = fifo[i + 1];
    --fifo_n;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// x axis.  k_mode_xf_sym: the x-forward product of the exchange apply -- pair density psi_j * tgt_k formed on the fly
// from two TMA streams (a1), each staged as rows x in [16 s, 16 s + 16) and the mirrored block, butterflied on the
// fragments -- on the reflection-adapted basis of the x axis.  Output rows hold the modes even block first.
// k_mode_xacc_sym: the x-backward product fused with the accumulate (k_mode_xacc, kernels_fused.cu) on the same basis:
// a = E t_even, b = O t_odd over the half range, phi[x] = a + b, phi[mir x] = a - b, and vx_k's tile kept in two
// accumulator sets (x and mir x); the psi_j tile arrives as a pair of boxes (x block and mirrored block).
// ---------------------------------------------------------------------------------------------------------------
struct XSArgs {
  double* out;         // xf: the batch buffer
  const double* V;
  const double* occ;   // xacc: occ + j0
  double* vx;          // xacc: vx + k0 * N
  int n, nh;
  int Sh, So;          // xf: Sh stages over the half range; xacc: Sh stages over the even modes, So over the odd modes
  int Sp;              // xacc: stages of the psi tile (half range)
  int kk_last, kk_last_o, kk_last_p;
  int mir0, mirc, zfix;
  unsigned n_tiles;
  int rows_per_rhs, tiles_per_rhs;
  // xacc: a work item is (row tile, item i < n_items) and loops over l in [max(0, i + c_lo), min(L, i + c_hi)): right-hand
  // side i stride_i + l stride_l of the batch, psi / occ of orbital p0 + l, result tile of vx function i.  Full apply and
  // the target side of the pair-symmetric apply: i = target, l = occupied orbital (j <= k: c_hi = k0 - j0 + 1); its
  // orbital side: i = orbital j, l = target k > j (c_lo = j0 - k0 + 1).
  int n_items, L, stride_i, stride_l, c_lo, c_hi, p0;
  int first;
  FastDiv div_tiles, div_nj, div_items;
  // xf with the pair density: tile t = (row tile, orbital, target) with the target index fastest, so that the tiles that
  // share a psi_j tile run back to back and find it in L2 (nb_rhs = nj nk right-hand sides, nkq = nk)
  FastDiv div_nb, div_nkq;
  int nb_rhs, nkq;
  BatchDesc bd;
};

// X-mode box ({16 x, rows}, 128-byte rows and swizzle): offset of (row 8nt + g, x) without the 1024 nt term
__device__ __forceinline__ unsigned offx(unsigned x, unsigned g) { return 128u * g + 16u * ((x >> 1) ^ g) + 8u * (x & 1); }

// PD: the right-hand side is the pair density psi_j * tgt_k formed from two TMA streams (exchange apply); without it the
// kernel reads nb right-hand sides from tm0 (the bare solver) and a stage is two boxes.
template <int MS, int NT, int WARPS, bool PD>
__global__ void __launch_bounds__(32 * WARPS, 1)
    k_mode_xf_sym(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1, const XSArgs a) {
  constexpr int MT = 2 * MS;
  constexpr int LDV = 8 * MT + 4;
  constexpr unsigned kBox = 1024u * NT;   // one {16 x, 8 NT rows} box
  constexpr unsigned kSlot = (PD ? 4u : 2u) * kBox;   // psi block, psi mirrored block(, tgt block, tgt mirrored block)
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, Sh = a.Sh;
  const unsigned smem0 = (unsigned)__cvta_generic_to_shared(smem_raw);
  // image rows actually read: the ragged last stage only uses its first 4 kk_last rows (that trims 4 KB at n = 120, which
  // is what lets a tenth warp's ring fit)
  const unsigned img_rows = a.kk_last ? 16u * (Sh - 1) + 4u * a.kk_last : 16u * Sh;
  const unsigned img_bytes = 8u * img_rows * LDV;
  for (unsigned i = 2 * tid; i < img_rows * LDV; i += 2 * 32 * WARPS)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem0 + 8u * i), "l"(a.V + i) : "memory");
  asm volatile("cp.async.commit_group;\n" ::: "memory");
  const unsigned ring0 = (smem0 + img_bytes + 1023u) & ~1023u;
  const unsigned my_ring = ring0 + warp * (kDepth * kSlot);
  const unsigned my_bar = ring0 + WARPS * (kDepth * kSlot) + warp * (kDepth * 8u);
  const unsigned ctr_addr = ring0 + WARPS * (kDepth * kSlot) + WARPS * (kDepth * 8u);
  if (tid == 0) asm volatile("st.shared.u32 [%0], %1;\n" ::"r"(ctr_addr), "r"((unsigned)WARPS) : "memory");
  if (lane == 0) {
#pragma unroll
    for (int d = 0; d < kDepth; ++d) mbar_init(my_bar + 8u * d, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  asm volatile("griddepcontrol.wait;\n" ::: "memory");

  const unsigned tfirst = blockIdx.x + gridDim.x * warp;
  auto claim_tile = [&]() -> unsigned {
    unsigned i = 0;
    if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;\n" : "=r"(i) : "r"(ctr_addr) : "memory");
    i = __shfl_sync(0xffffffffu, i, 0);
    const unsigned long long t = (unsigned long long)blockIdx.x + (unsigned long long)gridDim.x * i;
    return t < a.n_tiles ? (unsigned)t : 0xffffffffu;
  };
  unsigned fifo[kDepth + 1];
  int fifo_n = 0;
  unsigned t_p = tfirst;
  int s_p = 0;
  int pr0 = 0, pr1 = 0;
  auto split_tile = [&](unsigned t, int& rhs, int& rb, int& jj, int& kq) {
    if (PD) {
      rb = (int)fast_div(t, a.div_nb);
      const int r = (int)t - rb * a.nb_rhs;
      jj = (int)fast_div((unsigned)r, a.div_nkq);
      kq = r - jj * a.nkq;
      rhs = kq * a.bd.nj + jj;
    } else {
      rhs = (int)fast_div(t, a.div_tiles);
      rb = (int)t - rhs * a.tiles_per_rhs;
      jj = kq = 0;
    }
  };
  auto tile_coords = [&](unsigned t) {
    int rhs, rb, jj, kq;
    split_tile(t, rhs, rb, jj, kq);
    if (PD) {
      pr0 = (a.bd.j0 + jj) * a.rows_per_rhs + rb * (8 * NT);
      pr1 = (a.bd.k0 + kq) * a.rows_per_rhs + rb * (8 * NT);
    } else {
      pr0 = rhs * a.rows_per_rhs + rb * (8 * NT);
    }
  };
  auto produce = [&](int slot) {
    if (t_p >= a.n_tiles) return;
    const unsigned bar = my_bar + 8u * slot;
    const unsigned dst = my_ring + slot * kSlot;
    if (elect_one()) {
      mbar_expect_tx(bar, kSlot);
      tma_load_2d(dst, &tm0, 16 * s_p, pr0, bar);
      tma_load_2d(dst + kBox, &tm0, a.mir0 - 16 * s_p, pr0, bar);
      if (PD) {
        tma_load_2d(dst + 2 * kBox, &tm1, 16 * s_p, pr1, bar);
        tma_load_2d(dst + 3 * kBox, &tm1, a.mir0 - 16 * s_p, pr1, bar);
      }
    }
    if (++s_p == Sh) {
      s_p = 0;
      t_p = claim_tile();
#pragma unroll
      for (int i = 0; i < kDepth + 1; ++i)
        if (i == fifo_n) fifo[i] = t_p;
      ++fifo_n;
      if (t_p < a.n_tiles) tile_coords(t_p);
    }
  };
  if (t_p < a.n_tiles) tile_coords(t_p);
#pragma unroll
  for (int d = 0; d < kDepth; ++d) produce(d);
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();

  unsigned a_lane_v = smem0 + 8u * (q * LDV + g);
  // k-step kk reads x = (q&1) + 8(q>>1) + 2kk of the block and 15 - x of the mirrored block
  unsigned xo[4], xm[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const unsigned x = (q & 1) + 8u * (q >> 1) + 2u * i;
    xo[i] = offx(x, g);
    xm[i] = kBox + offx(15u - x, g);
  }

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  while (t < a.n_tiles) {
    double acc[MT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;
    auto do_stage = [&](int s, auto rag_c) {  // `ragged` at compile time, as in k_mode_lf_sym
      constexpr bool ragged = decltype(rag_c)::value;
      asm volatile("" : "+r"(a_lane_v), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
      mbar_wait(my_bar + 8u * slot, parity);
      const unsigned sb = my_ring + slot * kSlot;
      const unsigned aa = a_lane_v + (unsigned)s * (16u * LDV * 8u);
      const int zf = a.zfix - 16 * s;
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
        if (!ragged || kk < a.kk_last) {
          double be[NT], bo[NT];
          const int xl = ragged ? 4 * kk + q : (q & 1) + 8 * (q >> 1) + 2 * kk;
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            const unsigned oa = sb + 1024u * nt + (ragged ? offx((unsigned)xl, g) : xo[kk]);
            const unsigned ob = sb + 1024u * nt + (ragged ? kBox + offx(15u - (unsigned)xl, g) : xm[kk]);
            const double va = PD ? lds64(oa) * lds64(oa + 2 * kBox) : lds64(oa);
            double vb = PD ? lds64(ob) * lds64(ob + 2 * kBox) : lds64(ob);
            if (xl == zf) vb = 0.0;
            be[nt] = va + vb;
            bo[nt] = va - vb;
          }
          double af[MT];
#pragma unroll
          for (int mt = 0; mt < MT; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
          for (int mt = 0; mt < MT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], mt < MS ? be[nt] : bo[nt]);
        }
      }
      __syncwarp();
      produce(slot);
      if (++slot == kDepth) {
        slot = 0;
        parity ^= 1u;
      }
    };
    {
      const int s_full = a.kk_last ? Sh - 1 : Sh;
      for (int s = 0; s < s_full; ++s) do_stage(s, std::false_type{});
      if (a.kk_last) do_stage(Sh - 1, std::true_type{});
    }
    // epilogue: C[mode 8 (mt % MS) + g of block mt / MS][row 8nt + 2q + e]; positions: even modes 0.., odd modes nh..
    {
      int rhs, rb, jj_, kq_;
      split_tile(t, rhs, rb, jj_, kq_);
      const int row0 = rhs * a.rows_per_rhs + rb * (8 * NT);
      const int limit = (rhs + 1) * a.rows_per_rhs;
      double* base = a.out + (long long)(row0 + 2 * q) * n;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          if (row0 + 8 * nt + 2 * q + e < limit) {
            double* dst = base + (long long)(8 * nt + e) * n;
#pragma unroll
            for (int mt = 0; mt < MT; ++mt) {
              const int blk = mt >= MS ? 1 : 0;
              const int ml = 8 * (mt - blk * MS) + g;
              if (ml < (blk ? n - a.nh : a.nh)) dst[blk * a.nh + ml] = acc[mt][nt][e];
            }
          }
        }
    }
    t = fifo[0];
#pragma unroll
    for (int i = 0; i < kDepth; ++i) fifo[i] = fifo[i + 1];
    --fifo_n;
  }
}

// GEN: items with individual loop ranges and general strides (the pair-symmetric apply); without it every item loops over
// all L = nj orbitals of the batch with i = target (the full apply).
template <int MS, int NT, int WARPS, bool GEN>
__global__ void __launch_bounds__(32 * WARPS, 1)
    k_mode_xacc_sym(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1, const XSArgs a) {
  constexpr int LDV = 8 * MS + 4;
  constexpr unsigned kBox = 1024u * NT;
  // A ring slot holds BPS boxes: a data stage is ALL boxes of one parity block of the modes (at most 4 for NT = 1, at most
  // 2 for NT = 2, where the image is small enough for the larger ring), a psi stage PP = BPS / 2 pairs (block, mirrored block) of 16 half-range points.  Per step (one j) that
  // is 2 data stages + ceil(SP / PP) psi stages = 4 barrier waits instead of one per box (12 at n = 120).
  constexpr int BPS = 4;
  constexpr int PP = BPS / 2;
  constexpr unsigned kSlot = BPS * kBox;
  constexpr int SPMAX = (MS + 1) / 2;
  constexpr int PSMAX = (SPMAX + PP - 1) / PP;
  static_assert((MS + 1) / 2 <= BPS, "a parity block of the modes must fit one ring slot");
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, SE = a.Sh, ST = a.Sh + a.So, SP = a.Sp;
  const unsigned smem0 = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned img_bytes = 8u * (16u * ST) * LDV;
  for (unsigned i = 2 * tid; i < 16u * ST * LDV; i += 2 * 32 * WARPS)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem0 + 8u * i), "l"(a.V + i) : "memory");
  asm volatile("cp.async.commit_group;\n" ::: "memory");
  const unsigned ring0 = (smem0 + img_bytes + 1023u) & ~1023u;
  const unsigned my_ring = ring0 + warp * (kDepth * kSlot);
  const unsigned my_bar = ring0 + WARPS * (kDepth * kSlot) + warp * (kDepth * 8u);
  const unsigned ctr_addr = ring0 + WARPS * (kDepth * kSlot) + WARPS * (kDepth * 8u);
  if (tid == 0) asm volatile("st.shared.u32 [%0], %1;\n" ::"r"(ctr_addr), "r"((unsigned)WARPS) : "memory");
  if (lane == 0) {
#pragma unroll
    for (int d = 0; d < kDepth; ++d) mbar_init(my_bar + 8u * d, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  asm volatile("griddepcontrol.wait;\n" ::: "memory");

  unsigned tfirst = blockIdx.x + gridDim.x * warp;
  auto claim_tile = [&]() -> unsigned {
    unsigned i = 0;
    if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;\n" : "=r"(i) : "r"(ctr_addr) : "memory");
    i = __shfl_sync(0xffffffffu, i, 0);
    const unsigned long long t = (unsigned long long)blockIdx.x + (unsigned long long)gridDim.x * i;
    return t < a.n_tiles ? (unsigned)t : 0xffffffffu;
  };
  unsigned fifo[kDepth + 1];
  int fifo_n = 0;

  // producer: item (row tile, i) = hi - lo steps of 2 data stages (even modes, odd modes) + PS psi stages
  const int PS = (SP + PP - 1) / PP;
  const int stages_per_step = 2 + PS;
  auto item_range = [&](unsigned t, int& rb, int& i, int& lo, int& hi) {
    rb = (int)fast_div(t, a.div_items);
    i = (int)t - rb * a.n_items;
    lo = 0;
    hi = a.L;
    if (GEN) {
      lo = i + a.c_lo;
      if (lo < 0) lo = 0;
      hi = i + a.c_hi;
      if (hi > a.L) hi = a.L;
    }
  };
  auto next_tile = [&]() -> unsigned {  // the next claimed item whose loop is not empty
    for (;;) {
      const unsigned tn = claim_tile();
      if (!GEN || tn >= a.n_tiles) return tn;
      int rb, i, lo, hi;
      item_range(tn, rb, i, lo, hi);
      if (lo < hi) return tn;
    }
  };
  if (GEN) {
    int rb, i, lo = 0, hi = 0;
    if (tfirst < a.n_tiles) item_range(tfirst, rb, i, lo, hi);
    if (lo >= hi) tfirst = next_tile();
  }
  unsigned t_p = tfirst;
  int s_p = 0, rem_p = 0;  // rem_p: steps of the current item still to be produced
  int prow_d = 0, prow_p = 0;
  auto tile_coords = [&](unsigned t) {
    int rb, i, lo, hi;
    item_range(t, rb, i, lo, hi);
    rem_p = hi - lo;
    prow_d = (GEN ? i * a.stride_i + lo * a.stride_l : a.L * i) * a.rows_per_rhs + rb * (8 * NT);
    prow_p = (a.p0 + lo) * a.rows_per_rhs + rb * (8 * NT);
  };
  auto produce = [&](int slot) {
    if (t_p >= a.n_tiles) return;
    const unsigned bar = my_bar + 8u * slot;
    const unsigned dst = my_ring + slot * kSlot;
    if (elect_one()) {
      if (s_p < 2) {
        const int cnt = s_p ? ST - SE : SE, col0 = s_p ? a.nh : 0;
        mbar_expect_tx(bar, kBox * (unsigned)cnt);
#pragma unroll
        for (int b = 0; b < BPS; ++b)
          if (b < cnt) tma_load_2d(dst + kBox * b, &tm0, col0 + 16 * b, prow_d, bar);
      } else {
        const int sp0 = (s_p - 2) * PP;
        const int np = SP - sp0 < PP ? SP - sp0 : PP;
        mbar_expect_tx(bar, 2u * kBox * (unsigned)np);
#pragma unroll
        for (int pp = 0; pp < PP; ++pp)
          if (pp < np) {
            tma_load_2d(dst + 2u * kBox * pp, &tm1, 16 * (sp0 + pp), prow_p, bar);
            tma_load_2d(dst + 2u * kBox * pp + kBox, &tm1, a.mir0 - 16 * (sp0 + pp), prow_p, bar);
          }
      }
    }
    if (++s_p == stages_per_step) {
      s_p = 0;
      if (--rem_p == 0) {
        t_p = next_tile();
#pragma unroll
        for (int i = 0; i < kDepth + 1; ++i)
          if (i == fifo_n) fifo[i] = t_p;
        ++fifo_n;
        if (t_p < a.n_tiles) tile_coords(t_p);
      } else {
        prow_d += GEN ? a.stride_l * a.rows_per_rhs : a.rows_per_rhs;
        prow_p += a.rows_per_rhs;
      }
    }
  };
  if (t_p < a.n_tiles) tile_coords(t_p);
#pragma unroll
  for (int d = 0; d < kDepth; ++d) produce(d);
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();

  unsigned a_lane_v = smem0 + 8u * (q * LDV + g);
  unsigned xo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) xo[i] = offx((q & 1) + 8u * (q >> 1) + 2u * i, g);
  // psi fragments in accumulator layout: box row 2q + e, x = 8h + g of the block / 15 - (8h + g) of the mirrored block
  unsigned pq[2][2], pm[2][2];
#pragma unroll
  for (int e = 0; e < 2; ++e)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const unsigned row = 2u * q + e, x = 8u * h + g, xb = 15u - x;
      pq[e][h] = 128u * row + 16u * ((x >> 1) ^ row) + 8u * (x & 1);
      pm[e][h] = kBox + 128u * row + 16u * ((xb >> 1) ^ row) + 8u * (xb & 1);
    }

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  while (t < a.n_tiles) {
    int rb, it, l_lo, l_hi;
    item_range(t, rb, it, l_lo, l_hi);
    const int row0 = rb * (8 * NT);
    double* vbase = a.vx + ((long long)it * a.rows_per_rhs + row0 + 2 * q) * n;
    // vx_k's tile: lo[mt][nt][e] at row 8nt + 2q + e, x = 8mt + g; hi[mt][nt][e] at mir(x)
    double lo[MS][NT][2], hi[MS][NT][2];
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const bool rok = !a.first && row0 + 8 * nt + 2 * q + e < a.rows_per_rhs;
        const double* src = vbase + (long long)(8 * nt + e) * n;
#pragma unroll
        for (int mt = 0; mt < MS; ++mt) {
          const int x = 8 * mt + g, xb = a.mirc - x;
          lo[mt][nt][e] = (rok && x < a.nh) ? src[x] : 0.0;
          hi[mt][nt][e] = (rok && x < a.nh && xb != x && xb < n) ? src[xb] : 0.0;
        }
      }
    for (int jj = l_lo; jj < l_hi; ++jj) {
      const double oc = __ldg(a.occ + jj);
      double pa[MS][NT][2], pb[MS][NT][2];
#pragma unroll
      for (int mt = 0; mt < MS; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) pa[mt][nt][0] = pa[mt][nt][1] = pb[mt][nt][0] = pb[mt][nt][1] = 0.0;
      // one box of 16 modes (`ragged`, a compile-time flag: the last box of a block when its size is not a multiple of 16)
      auto box = [&](auto& acc, unsigned sb, int s, auto rag_c, int kk_last) {
        constexpr bool ragged = decltype(rag_c)::value;
        asm volatile("" : "+r"(a_lane_v), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
        const unsigned aa = a_lane_v + (unsigned)s * (16u * LDV * 8u);
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          if (!ragged || kk < kk_last) {
            double bf[NT];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) bf[nt] = lds64(sb + 1024u * nt + (ragged ? offx(4u * kk + q, g) : xo[kk]));
            double af[MS];
#pragma unroll
            for (int mt = 0; mt < MS; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
            for (int mt = 0; mt < MS; ++mt)
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], bf[nt]);
          }
        }
      };
      // a data stage: every box of one parity block (image stages s0 .. s0 + cnt - 1) behind a single barrier wait
      auto data_stage = [&](auto& acc, int s0, int cnt, int kk_last) {
        mbar_wait(my_bar + 8u * slot, parity);
        const unsigned sb = my_ring + slot * kSlot;
        for (int b = 0; b < cnt - 1; ++b) box(acc, sb + kBox * b, s0 + b, std::false_type{}, 0);
        if (kk_last) box(acc, sb + kBox * (cnt - 1), s0 + cnt - 1, std::true_type{}, kk_last);
        else box(acc, sb + kBox * (cnt - 1), s0 + cnt - 1, std::false_type{}, 0);
        __syncwarp();
        produce(slot);
        if (++slot == kDepth) {
          slot = 0;
          parity ^= 1u;
        }
      };
      data_stage(pa, 0, SE, a.kk_last);
      data_stage(pb, SE, ST - SE, a.kk_last_o);
      // a5: vx_k[x] -= occ_j psi_j[x] (a + b), vx_k[mir x] -= occ_j psi_j[mir x] (a - b)
#pragma unroll
      for (int ps = 0; ps < PSMAX; ++ps) {
        if (ps < PS) {
          mbar_wait(my_bar + 8u * slot, parity);
          const unsigned sb0 = my_ring + slot * kSlot;
#pragma unroll
          for (int pp = 0; pp < PP; ++pp) {
            const int sp = ps * PP + pp;  // compile-time after unrolling
            if (sp < SPMAX && sp < SP) {
              const unsigned sb = sb0 + 2u * kBox * pp;
#pragma unroll
              for (int h = 0; h < 2; ++h) {
                constexpr int kZ = 0;
                const int mt = 2 * sp + h < MS ? 2 * sp + h : kZ;
                if (2 * sp + h < MS) {
#pragma unroll
                  for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                    for (int e = 0; e < 2; ++e) {
                      const double p0 = lds64(sb + 1024u * nt + pq[e][h]), p1 = lds64(sb + 1024u * nt + pm[e][h]);
                      lo[mt][nt][e] -= oc * p0 * (pa[mt][nt][e] + pb[mt][nt][e]);
                      hi[mt][nt][e] -= oc * p1 * (pa[mt][nt][e] - pb[mt][nt][e]);
                    }
                }
              }
            }
          }
          __syncwarp();
          produce(slot);
          if (++slot == kDepth) {
            slot = 0;
            parity ^= 1u;
          }
        }
      }
    }
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        if (row0 + 8 * nt + 2 * q + e < a.rows_per_rhs) {
          double* dst = vbase + (long long)(8 * nt + e) * n;
#pragma unroll
          for (int mt = 0; mt < MS; ++mt) {
            const int x = 8 * mt + g, xb = a.mirc - x;
            if (x < a.nh) {
              dst[x] = lo[mt][nt][e];
              if (xb != x && xb < n) dst[xb] = hi[mt][nt][e];
            }
          }
        }
      }
    t = fifo[0];
#pragma unroll
    for (int i = 0; i < kDepth; ++i) fifo[i] = fifo[i + 1];
    --fifo_n;
  }
}

// k_mode_xb_sym: the x-backward product alone (the bare solver): a = E t_even, b = O t_odd over the half range,
// out[x] = a + b, out[mir x] = a - b, in place over the rows of a tile.  Data stages as in k_mode_xacc_sym.
template <int MS, int NT, int WARPS>
__global__ void __launch_bounds__(32 * WARPS, 1) k_mode_xb_sym(const __grid_constant__ CUtensorMap tm0, const XSArgs a) {
  constexpr int LDV = 8 * MS + 4;
  constexpr unsigned kBox = 1024u * NT;
  constexpr int SETS = MS <= 3 ? 1 : 2;  // boxes of 16 modes per ring slot (as k_mode_lb_sym)
  constexpr unsigned kSlot = SETS * kBox;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, SE = a.Sh, ST = a.Sh + a.So;
  const int SE2 = (SE + SETS - 1) / SETS, ST2 = SE2 + (ST - SE + SETS - 1) / SETS;
  const unsigned smem0 = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned img_bytes = 8u * (16u * ST) * LDV;
  for (unsigned i = 2 * tid; i < 16u * ST * LDV; i += 2 * 32 * WARPS)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem0 + 8u * i), "l"(a.V + i) : "memory");
  asm volatile("cp.async.commit_group;\n" ::: "memory");
  const unsigned ring0 = (smem0 + img_bytes + 1023u) & ~1023u;
  const unsigned my_ring = ring0 + warp * (kDepth * kSlot);
  const unsigned my_bar = ring0 + WARPS * (kDepth * kSlot) + warp * (kDepth * 8u);
  const unsigned ctr_addr = ring0 + WARPS * (kDepth * kSlot) + WARPS * (kDepth * 8u);
  if (tid == 0) asm volatile("st.shared.u32 [%0], %1;\n" ::"r"(ctr_addr), "r"((unsigned)WARPS) : "memory");
  if (lane == 0) {
#pragma unroll
    for (int d = 0; d < kDepth; ++d) mbar_init(my_bar + 8u * d, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  asm volatile("griddepcontrol.wait;\n" ::: "memory");

  const unsigned tfirst = blockIdx.x + gridDim.x * warp;
  auto claim_tile = [&]() -> unsigned {
    unsigned i = 0;
    if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;\n" : "=r"(i) : "r"(ctr_addr) : "memory");
    i = __shfl_sync(0xffffffffu, i, 0);
    const unsigned long long t = (unsigned long long)blockIdx.x + (unsigned long long)gridDim.x * i;
    return t < a.n_tiles ? (unsigned)t : 0xffffffffu;
  };
  unsigned fifo[kDepth + 1];
  int fifo_n = 0;
  unsigned t_p = tfirst;
  int s_p = 0;
  int prow = 0;
  auto tile_coords = [&](unsigned t) {
    const int rhs = (int)fast_div(t, a.div_tiles);
    const int rb = (int)t - rhs * a.tiles_per_rhs;
    prow = rhs * a.rows_per_rhs + rb * (8 * NT);
  };
  auto produce = [&](int slot) {
    if (t_p >= a.n_tiles) return;
    const unsigned bar = my_bar + 8u * slot;
    const unsigned dst = my_ring + slot * kSlot;
    if (elect_one()) {
      const int blk = s_p < SE2 ? 0 : 1, b0 = SETS * (s_p - blk * SE2), cnt = blk ? ST - SE : SE;
      const int nbx = cnt - b0 < SETS ? cnt - b0 : SETS;
      mbar_expect_tx(bar, kBox * (unsigned)nbx);
#pragma unroll
      for (int hh = 0; hh < SETS; ++hh)
        if (hh < nbx) tma_load_2d(dst + kBox * hh, &tm0, (blk ? a.nh : 0) + 16 * (b0 + hh), prow, bar);
    }
    if (++s_p == ST2) {
      s_p = 0;
      t_p = claim_tile();
#pragma unroll
      for (int i = 0; i < kDepth + 1; ++i)
        if (i == fifo_n) fifo[i] = t_p;
      ++fifo_n;
      if (t_p < a.n_tiles) tile_coords(t_p);
    }
  };
  if (t_p < a.n_tiles) tile_coords(t_p);
#pragma unroll
  for (int d = 0; d < kDepth; ++d) produce(d);
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();

  unsigned a_lane_v = smem0 + 8u * (q * LDV + g);
  unsigned xo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) xo[i] = offx((q & 1) + 8u * (q >> 1) + 2u * i, g);

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  while (t < a.n_tiles) {
    double pa[MS][NT][2], pb[MS][NT][2];
#pragma unroll
    for (int mt = 0; mt < MS; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) pa[mt][nt][0] = pa[mt][nt][1] = pb[mt][nt][0] = pb[mt][nt][1] = 0.0;
    auto box = [&](auto& acc, unsigned sb, int s, auto rag_c, int kk_last) {
      constexpr bool ragged = decltype(rag_c)::value;
      asm volatile("" : "+r"(a_lane_v), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
      const unsigned aa = a_lane_v + (unsigned)s * (16u * LDV * 8u);
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
        if (!ragged || kk < kk_last) {
          double bf[NT];
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) bf[nt] = lds64(sb + 1024u * nt + (ragged ? offx(4u * kk + q, g) : xo[kk]));
          double af[MS];
#pragma unroll
          for (int mt = 0; mt < MS; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
          for (int mt = 0; mt < MS; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], bf[nt]);
        }
      }
    };
    auto block = [&](auto& acc, int s0, int cnt, int kk_last) {
      for (int b0 = 0; b0 < cnt; b0 += SETS) {
        const int nbx = cnt - b0 < SETS ? cnt - b0 : SETS;
        mbar_wait(my_bar + 8u * slot, parity);
        const unsigned sb = my_ring + slot * kSlot;
        if (SETS == 2 && nbx == 2) box(acc, sb, s0 + b0, std::false_type{}, 0);
        const unsigned sl = sb + kBox * (unsigned)(nbx - 1);
        if (kk_last && b0 + nbx == cnt) box(acc, sl, s0 + b0 + nbx - 1, std::true_type{}, kk_last);
        else box(acc, sl, s0 + b0 + nbx - 1, std::false_type{}, 0);
        __syncwarp();
        produce(slot);
        if (++slot == kDepth) {
          slot = 0;
          parity ^= 1u;
        }
      }
    };
    block(pa, 0, SE, a.kk_last);
    block(pb, SE, ST - SE, a.kk_last_o);
    // epilogue: C[x = 8mt + g][row 8nt + 2q + e]: out[x] = a + b, out[mir x] = a - b
    {
      const int rhs = (int)fast_div(t, a.div_tiles);
      const int rb = (int)t - rhs * a.tiles_per_rhs;
      const int row0 = rhs * a.rows_per_rhs + rb * (8 * NT);
      const int limit = (rhs + 1) * a.rows_per_rhs;
      double* base = a.out + (long long)(row0 + 2 * q) * n;
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          if (row0 + 8 * nt + 2 * q + e < limit) {
            double* dst = base + (long long)(8 * nt + e) * n;
#pragma unroll
            for (int mt = 0; mt < MS; ++mt) {
              const int x = 8 * mt + g, xb = a.mirc - x;
              if (x < a.nh) {
                dst[x] = pa[mt][nt][e] + pb[mt][nt][e];
                if (xb != x && xb < n) dst[xb] = pa[mt][nt][e] - pb[mt][nt][e];
              }
            }
          }
        }
    }
    t = fifo[0];
#pragma unroll
    for (int i = 0; i < kDepth; ++i) fifo[i] = fifo[i + 1];
    --fifo_n;
  }
}

// ---- host side ------------------------------------------------------------------------------------------------

template <typename Kern>
cudaError_t launch_sym(Kern kern, SmemOptIn& opt, size_t smem, int warps, const exx_plan* p, const CUtensorMap& m0,
                       const SArgs& a, cudaStream_t s) {
  const size_t floor_bytes = 117 * 1024;  // exactly one CTA per SM
  if (smem < floor_bytes) smem = floor_bytes;
  if (smem > (size_t)p->smem_optin) return cudaErrorNotSupported;
  cudaError_t e = opt.ensure(kern, p->device, smem, true);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  const unsigned grid = a.n_tiles < (unsigned)p->sm_count ? a.n_tiles : (unsigned)p->sm_count;
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(32 * warps);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, m0, a);
}

template <int MS, bool HC>
cudaError_t launch_lf(const exx_plan* p, const CUtensorMap& m0, const SArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  constexpr int W = 12, NT = MS <= 4 ? 4 : 2;
  const size_t smem = sizeof(double) * 16 * (size_t)a.Sh * (16 * MS + 4) + 1024 + (size_t)W * kDepth * 2 * 1024 * NT +
                      (size_t)W * kDepth * 8 + 16;
  return launch_sym(k_mode_lf_sym<MS, NT, W, HC>, opt, smem, W, p, m0, a, s);
}
template <int MS, bool HC>
cudaError_t launch_lb(const exx_plan* p, const CUtensorMap& m0, const SArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  constexpr int W = 12, NT = MS <= 4 ? 4 : 2;
  constexpr int SETS = MS <= 3 ? 1 : 2;  // sets of 16 modes per ring slot, as in the kernel
  const size_t smem = sizeof(double) * 16 * (size_t)(a.Sh + a.So) * (8 * MS + 4) + 1024 + (size_t)W * kDepth * SETS * 1024 * NT +
                      (size_t)W * kDepth * 8 + 16;
  return launch_sym(k_mode_lb_sym<MS, NT, W, HC>, opt, smem, W, p, m0, a, s);
}

template <typename Kern>
cudaError_t launch_sym2(Kern kern, SmemOptIn& opt, size_t smem, int warps, const exx_plan* p, const CUtensorMap& m0,
                        const CUtensorMap& m1, const XSArgs& a, cudaStream_t s) {
  const size_t floor_bytes = 117 * 1024;
  if (smem < floor_bytes) smem = floor_bytes;
  if (smem > (size_t)p->smem_optin) return cudaErrorNotSupported;
  cudaError_t e = opt.ensure(kern, p->device, smem, true);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  const unsigned grid = a.n_tiles < (unsigned)p->sm_count ? a.n_tiles : (unsigned)p->sm_count;
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(32 * warps);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, m0, m1, a);
}

template <int MS>
cudaError_t launch_xf(const exx_plan* p, const CUtensorMap& m0, const CUtensorMap& m1, const XSArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  // twelve warps where the image leaves room for twelve four-box rings (up to 80 points per axis), ten up to 112, else eight
  constexpr int NT = 2;
  const size_t rows = a.kk_last ? 16 * (size_t)(a.Sh - 1) + 4 * a.kk_last : 16 * (size_t)a.Sh;  // image rows the kernel stages
  const size_t img = (sizeof(double) * rows * (16 * MS + 4) + 1023) / 1024 * 1024;
  auto need = [&](int w) { return img + 1024 + (size_t)w * kDepth * 4 * 1024 * NT + (size_t)w * kDepth * 8 + 16; };
  if (MS >= 8) {  // 120-128 points: ten warps if the (trimmed) image leaves room, else eight
    if (need(10) <= (size_t)p->smem_optin) {
      static SmemOptIn opt10;
      return launch_sym2(k_mode_xf_sym<MS, NT, 10, true>, opt10, need(10), 10, p, m0, m1, a, s);
    }
    return launch_sym2(k_mode_xf_sym<MS, NT, 8, true>, opt, need(8), 8, p, m0, m1, a, s);
  }
  constexpr int W = MS <= 5 ? 12 : 10;
  const size_t smem = need(W);
  return launch_sym2(k_mode_xf_sym<MS, NT, W, true>, opt, smem, W, p, m0, m1, a, s);
}
// bare solver: one stream, two boxes per stage, twelve warps
template <int MS>
cudaError_t launch_xf_plain(const exx_plan* p, const CUtensorMap& m0, const XSArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  constexpr int W = 12, NT = 2;
  const size_t smem = sizeof(double) * 16 * (size_t)a.Sh * (16 * MS + 4) + 1024 + (size_t)W * kDepth * 2 * 1024 * NT +
                      (size_t)W * kDepth * 8 + 16;
  return launch_sym2(k_mode_xf_sym<MS, NT, W, false>, opt, smem, W, p, m0, m0, a, s);
}
template <typename Kern>
cudaError_t launch_sym1x(Kern kern, SmemOptIn& opt, size_t smem, int warps, const exx_plan* p, const CUtensorMap& m0,
                         const XSArgs& a, cudaStream_t s) {
  const size_t floor_bytes = 117 * 1024;
  if (smem < floor_bytes) smem = floor_bytes;
  if (smem > (size_t)p->smem_optin) return cudaErrorNotSupported;
  cudaError_t e = opt.ensure(kern, p->device, smem, true);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  const unsigned grid = a.n_tiles < (unsigned)p->sm_count ? a.n_tiles : (unsigned)p->sm_count;
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(32 * warps);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kern, m0, a);
}
template <int MS>
cudaError_t launch_xb(const exx_plan* p, const CUtensorMap& m0, const XSArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  constexpr int W = 12, NT = 2, SETS = MS <= 3 ? 1 : 2;
  const size_t smem = sizeof(double) * 16 * (size_t)(a.Sh + a.So) * (8 * MS + 4) + 1024 + (size_t)W * kDepth * SETS * 1024 * NT +
                      (size_t)W * kDepth * 8 + 16;
  return launch_sym1x(k_mode_xb_sym<MS, NT, W>, opt, smem, W, p, m0, a, s);
}
template <int MS, bool GEN>
cudaError_t launch_xacc_sym(const exx_plan* p, const CUtensorMap& m0, const CUtensorMap& m1, const XSArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  constexpr int W = 12, NT = MS <= 4 ? 2 : 1, BPS = 4;  // boxes per ring slot, as in the kernel
  const size_t smem = sizeof(double) * 16 * (size_t)(a.Sh + a.So) * (8 * MS + 4) + 1024 + (size_t)W * kDepth * BPS * 1024 * NT +
                      (size_t)W * kDepth * 8 + 16;
  return launch_sym2(k_mode_xacc_sym<MS, NT, W, GEN>, opt, smem, W, p, m0, m1, a, s);
}

}  // namespace

// Images of the y axis on the reflection-adapted basis; `hc`: row order of the half-chunk tiles.  Forward: rows = half
// range (k_mode_t's L-mode stage order), columns = even modes | 8 MS + odd modes.  Backward: rows = even modes in stages
// of 16, then odd modes in stages of 16, columns = half-range points.
static cudaError_t sym_init_y(exx_plan* p);
static cudaError_t sym_init_x(exx_plan* p);

cudaError_t sym_init(exx_plan* p) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st) return cudaSuccess;
  st->d_img_yf = st->d_img_yb = st->d_img_xf = st->d_img_xb = st->d_mult_symx = nullptr;
  st->ys_nh = st->xs_nh = 0;
  if (p->bloch || !p->h_Vi[0].empty() || !p->h_Vi[1].empty() || !p->h_Vi[2].empty()) return cudaSuccess;
  cudaError_t e = sym_init_y(p);
  if (e == cudaSuccess) e = sym_init_x(p);
  return e;
}

// x axis: forward image = rows over the half range in X-mode stage order, columns even modes | 8 MS + odd modes;
// backward image = rows over the even modes in stages of 16 then the odd modes, columns over the half range.
static cudaError_t sym_init_x(exx_plan* p) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  const int n = p->n[0];
  // x is the contiguous index: the boxes of the mirrored block and of the odd modes must start at an even element (TMA
  // wants 16-byte aligned starts along the innermost dimension), hence the reflection x -> n - 1 - x on either kind of
  // axis (mirrored block of stage s starts at n - 16 - 16 s) and nx a multiple of 4 (odd modes start at n / 2)
  if (n > 128 || (n & 3)) return cudaSuccess;
  int nh = 0;
  if (!symmetrize_axis(n, p->bc[0], p->h_lam[0], p->h_V[0], st->lam_xs, st->V_xs, &nh, true)) return cudaSuccess;
  const int ms = (nh + 7) / 8;
  if (ms < 3 || ms > 8) return cudaSuccess;
  const int no = n - nh, Sh = (nh + 15) / 16, So = (no + 15) / 16;
  const std::vector<double>& Vs = st->V_xs;
  {
    const int ld = 16 * ms + 4;
    std::vector<double> img((size_t)16 * Sh * ld, 0.0);
    for (int s = 0; s < Sh; ++s)
      for (int kk = 0; kk < 4; ++kk)
        for (int q = 0; q < 4; ++q) {
          const int x = 16 * s + within_stage(true, nh, s, kk, q);
          if (x >= nh) continue;
          double* row = &img[(size_t)(16 * s + 4 * kk + q) * ld];
          for (int m = 0; m < n; ++m) row[m < nh ? m : 8 * ms + (m - nh)] = Vs[(size_t)x * n + m];
        }
    cudaError_t e = cudaMalloc(&st->d_img_xf, sizeof(double) * img.size());
    if (e == cudaSuccess) e = cudaMemcpy(st->d_img_xf, img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
  }
  {
    const int ld = 8 * ms + 4;
    std::vector<double> img((size_t)16 * (Sh + So) * ld, 0.0);
    for (int blk = 0; blk < 2; ++blk) {
      const int cnt = blk ? no : nh, S = blk ? So : Sh, row0 = blk ? 16 * Sh : 0;
      for (int s = 0; s < S; ++s)
        for (int kk = 0; kk < 4; ++kk)
          for (int q = 0; q < 4; ++q) {
            const int m = 16 * s + within_stage(true, cnt, s, kk, q);
            if (m >= cnt) continue;
            double* row = &img[(size_t)(row0 + 16 * s + 4 * kk + q) * ld];
            for (int x = 0; x < nh; ++x) row[x] = Vs[(size_t)x * n + (blk ? nh + m : m)];
          }
    }
    cudaError_t e = cudaMalloc(&st->d_img_xb, sizeof(double) * img.size());
    if (e == cudaSuccess) e = cudaMemcpy(st->d_img_xb, img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
  }
  st->xs_nh = nh;
  return cudaSuccess;
}

static cudaError_t sym_init_y(exx_plan* p) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  const int n = p->n[1];
  if (n > 128 || (p->n[0] & 1)) return cudaSuccess;
  int nh = 0;
  if (!symmetrize_axis(n, p->bc[1], p->h_lam[1], p->h_V[1], st->lam_ys, st->V_ys, &nh, true)) return cudaSuccess;
  const int ms = (nh + 7) / 8;
  if (ms < 3 || ms > 8) return cudaSuccess;
  const bool hc = p->n[0] % 16 == 8;
  const int no = n - nh, Sh = (nh + 15) / 16, So = (no + 15) / 16;
  const std::vector<double>& Vs = st->V_ys;
  {
    const int ld = 16 * ms + 4;
    std::vector<double> img((size_t)16 * Sh * ld, 0.0);
    for (int s = 0; s < Sh; ++s)
      for (int kk = 0; kk < 4; ++kk)
        for (int q = 0; q < 4; ++q) {
          const int y = 16 * s + within_stage(false, nh, s, kk, q, hc);
          if (y >= nh) continue;
          double* row = &img[(size_t)(16 * s + 4 * kk + q) * ld];
          for (int m = 0; m < n; ++m) row[m < nh ? m : 8 * ms + (m - nh)] = Vs[(size_t)y * n + m];
        }
    cudaError_t e = cudaMalloc(&st->d_img_yf, sizeof(double) * img.size());
    if (e == cudaSuccess) e = cudaMemcpy(st->d_img_yf, img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
  }
  {
    const int ld = 8 * ms + 4;
    std::vector<double> img((size_t)16 * (Sh + So) * ld, 0.0);
    for (int blk = 0; blk < 2; ++blk) {
      const int cnt = blk ? no : nh, S = blk ? So : Sh, row0 = blk ? 16 * Sh : 0;
      for (int s = 0; s < S; ++s)
        for (int kk = 0; kk < 4; ++kk)
          for (int q = 0; q < 4; ++q) {
            const int m = 16 * s + within_stage(false, cnt, s, kk, q, hc);
            if (m >= cnt) continue;
            double* row = &img[(size_t)(row0 + 16 * s + 4 * kk + q) * ld];
            for (int y = 0; y < nh; ++y) row[y] = Vs[(size_t)y * n + (blk ? nh + m : m)];
          }
    }
    cudaError_t e = cudaMalloc(&st->d_img_yb, sizeof(double) * img.size());
    if (e == cudaSuccess) e = cudaMemcpy(st->d_img_yb, img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) return e;
  }
  st->ys_nh = nh;
  st->ys_hc = hc;
  return cudaSuccess;
}

void sym_destroy(exx_plan* p) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st) return;
  if (st->d_img_yf) cudaFree(st->d_img_yf);
  if (st->d_img_yb) cudaFree(st->d_img_yb);
  if (st->d_img_xf) cudaFree(st->d_img_xf);
  if (st->d_img_xb) cudaFree(st->d_img_xb);
  if (st->d_mult_symx) cudaFree(st->d_mult_symx);
  st->d_img_yf = st->d_img_yb = st->d_img_xf = st->d_img_xb = st->d_mult_symx = nullptr;
}

// y product of nb right-hand sides on the reflection-adapted basis, in place.  The caller has established that the whole
// batch runs in "symmetric" mode (sym_axis_capable(p, 1) and TMA-addressable buffers).
cudaError_t sym_mode_product_y(exx_plan* p, bool forward, double* buf, int nb, cudaStream_t s) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  // NotSupported means exactly one thing to the caller: the plan has no symmetric y axis (the table then keeps y in
  // ascending order and the dense product serves).  Past that point the table is in (even | odd) y order, so a kernel
  // that cannot run is a hard error, never a reason to fall back to the dense product.
  if (!st || !st->ys_nh) return cudaErrorNotSupported;
  if (!aligned16(buf)) return cudaErrorUnknown;
  const int n = p->n[1], nh = st->ys_nh, no = n - nh, ms = (nh + 7) / 8;
  const bool per = false, hc = st->ys_hc;  // centred reflection y -> n - 1 - y on either kind of axis (sym_init_y)
  const long long inner = p->n[0], outer = (long long)p->n[2] * nb;
  SArgs a{};
  a.out = buf;
  a.V = forward ? st->d_img_yf : st->d_img_yb;
  a.n = n;
  a.nh = nh;
  a.Sh = (nh + 15) / 16;
  a.So = (no + 15) / 16;
  a.kk_last = tail_ksteps(nh);
  a.kk_last_o = tail_ksteps(no);
  a.mir0 = per ? n - 15 : n - 16;
  a.mirc = per ? n : n - 1;
  a.zfix = per ? ((n % 2 == 0 && n >= 2) ? n / 2 : -1) : ((n % 2) ? (n - 1) / 2 : -1);
  const int cw = hc ? 8 : 16;
  a.inner = (int)inner;
  a.cpo = (int)((inner + cw - 1) / cw);
  const long long chunks = (long long)a.cpo * outer;
  if (chunks >= (1LL << 31) - 64) return cudaErrorUnknown;
  a.total_chunks = (unsigned)chunks;
  a.outer = (int)outer;
  a.div_cpo = make_fastdiv((unsigned)a.cpo);
  const int NT = ms <= 4 ? 4 : 2, CH = hc ? NT : NT / 2;
  a.n_tiles = (unsigned)((chunks + CH - 1) / CH);
  if (a.n_tiles == 0) return cudaSuccess;
  CUtensorMap m0;
  cudaError_t e;
  if ((e = get_map(st, buf, inner, n, outer, 16, &m0, cw)) != cudaSuccess) return e;
  auto launch = [&]() -> cudaError_t {
#define EXX_SYM_CASE(MSV)                                                                       \
  case MSV:                                                                                     \
    if (forward) return hc ? launch_lf<MSV, true>(p, m0, a, s) : launch_lf<MSV, false>(p, m0, a, s); \
    return hc ? launch_lb<MSV, true>(p, m0, a, s) : launch_lb<MSV, false>(p, m0, a, s);
    switch (ms) {
      EXX_SYM_CASE(3)
      EXX_SYM_CASE(4)
      EXX_SYM_CASE(5)
      EXX_SYM_CASE(6)
      EXX_SYM_CASE(7)
      default:
        if (forward) return hc ? launch_lf<8, true>(p, m0, a, s) : launch_lf<8, false>(p, m0, a, s);
        return hc ? launch_lb<8, true>(p, m0, a, s) : launch_lb<8, false>(p, m0, a, s);
    }
#undef EXX_SYM_CASE
  };
  e = launch();
  if (e == cudaSuccess) ++p->tma_launches;
  return e == cudaErrorNotSupported ? cudaErrorUnknown : e;
}

// Whether the exchange-apply batch `fa` can run its x passes on the reflection-adapted basis: the plan has the images and
// the symmetric table with x, the fused accumulate is on, and every buffer the two kernels touch is TMA-addressable.
bool sym_x_usable(const exx_plan* p, const double* work, const FastArgs* fa) {
  const TmaState* st = static_cast<const TmaState*>(p->tma_state);
  if (!st || !st->xs_nh || !st->d_mult_symx || !fa || !(p->fusion & 2)) return false;
  if (!aligned16(work) || !aligned16(fa->psi) || !aligned16(fa->tgt) || !aligned16(fa->vx)) return false;
  const long long rpr = p->N / p->n[0];
  return rpr * fa->n_occ < (1LL << 31) - 64 && rpr * fa->n_tgt < (1LL << 31) - 64;
}

// rows of a work item of k_mode_xacc_sym (0: the plan has no symmetric x axis)
int sym_xacc_tile_rows(const exx_plan* p) {
  const TmaState* st = static_cast<const TmaState*>(p->tma_state);
  if (!st || !st->xs_nh) return 0;
  return (st->xs_nh + 7) / 8 <= 4 ? 16 : 8;
}

static void fill_x(const exx_plan* p, const TmaState* st, XSArgs& a) {
  const int n = p->n[0], nh = st->xs_nh, no = n - nh;
  const bool per = false;  // the x axis always uses the centred reflection x -> n - 1 - x (sym_init_x)
  a.n = n;
  a.nh = nh;
  a.Sh = (nh + 15) / 16;
  a.So = (no + 15) / 16;
  a.Sp = (nh + 15) / 16;
  a.kk_last = tail_ksteps(nh);
  a.kk_last_o = tail_ksteps(no);
  a.kk_last_p = tail_ksteps(nh);
  a.mir0 = per ? n - 15 : n - 16;
  a.mirc = per ? n : n - 1;
  a.zfix = per ? ((n % 2 == 0 && n >= 2) ? n / 2 : -1) : ((n % 2) ? (n - 1) / 2 : -1);
  a.rows_per_rhs = (int)(p->N / n);
}

// x-forward product with the pair density formed on the fly, modes stored even block first.
cudaError_t sym_xf(exx_plan* p, double* out, int nb, const FastArgs* fa, cudaStream_t s) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!sym_x_usable(p, out, fa)) return cudaErrorNotSupported;
  constexpr int NT = 2;
  XSArgs a{};
  fill_x(p, st, a);
  a.out = out;
  a.V = st->d_img_xf;
  a.bd = fa->bd;
  a.tiles_per_rhs = (a.rows_per_rhs + 8 * NT - 1) / (8 * NT);
  a.div_tiles = make_fastdiv((unsigned)a.tiles_per_rhs);
  a.div_nj = make_fastdiv((unsigned)fa->bd.nj);
  a.nb_rhs = nb;
  a.nkq = fa->bd.nk;
  a.div_nb = make_fastdiv((unsigned)nb);
  a.div_nkq = make_fastdiv((unsigned)fa->bd.nk);
  if ((long long)a.rows_per_rhs * nb >= (1LL << 31) - 64) return cudaErrorNotSupported;
  a.n_tiles = (unsigned)a.tiles_per_rhs * (unsigned)nb;
  if (a.n_tiles == 0) return cudaSuccess;
  CUtensorMap m0, m1;
  cudaError_t e;
  if ((e = get_map(st, fa->psi, a.n, (long long)a.rows_per_rhs * fa->n_occ, 0, 8 * NT, &m0)) != cudaSuccess) return e;
  if ((e = get_map(st, fa->tgt, a.n, (long long)a.rows_per_rhs * fa->n_tgt, 0, 8 * NT, &m1)) != cudaSuccess) return e;
  switch ((a.nh + 7) / 8) {
    case 3: e = launch_xf<3>(p, m0, m1, a, s); break;
    case 4: e = launch_xf<4>(p, m0, m1, a, s); break;
    case 5: e = launch_xf<5>(p, m0, m1, a, s); break;
    case 6: e = launch_xf<6>(p, m0, m1, a, s); break;
    case 7: e = launch_xf<7>(p, m0, m1, a, s); break;
    default: e = launch_xf<8>(p, m0, m1, a, s); break;
  }
  // counted only once the kernel is enqueued: NotSupported here (shared memory) sends the caller to the dense x-forward
  // pass, and the batch's symmetric-mode decision reads this counter
  if (e == cudaSuccess) ++p->tma_launches;
  return e;
}

// Bare solver (exx_poisson_solve): whether its x passes can run on the reflection-adapted basis.
bool sym_x_usable_plain(const exx_plan* p, const double* src, const double* work, int nb) {
  const TmaState* st = static_cast<const TmaState*>(p->tma_state);
  if (!st || !st->xs_nh || !st->d_mult_symx || !(p->fusion & 2)) return false;
  if (!aligned16(src) || !aligned16(work)) return false;
  return (p->N / p->n[0]) * (long long)nb < (1LL << 31) - 64;
}

// x-forward product of nb right-hand sides in `in` (modes stored even block first in `out`; in == out allowed) and the
// x-backward product in place over `buf`, both on the reflection-adapted basis.
cudaError_t sym_xf_plain(exx_plan* p, const double* in, double* out, int nb, cudaStream_t s) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!sym_x_usable_plain(p, in, out, nb)) return cudaErrorNotSupported;
  constexpr int NT = 2;
  XSArgs a{};
  fill_x(p, st, a);
  a.out = out;
  a.V = st->d_img_xf;
  a.tiles_per_rhs = (a.rows_per_rhs + 8 * NT - 1) / (8 * NT);
  a.div_tiles = make_fastdiv((unsigned)a.tiles_per_rhs);
  a.div_nj = make_fastdiv(1u);
  a.n_tiles = (unsigned)a.tiles_per_rhs * (unsigned)nb;
  if (a.n_tiles == 0) return cudaSuccess;
  CUtensorMap m0;
  cudaError_t e;
  if ((e = get_map(st, in, a.n, (long long)a.rows_per_rhs * nb, 0, 8 * NT, &m0)) != cudaSuccess) return e;
  switch ((a.nh + 7) / 8) {
    case 3: e = launch_xf_plain<3>(p, m0, a, s); break;
    case 4: e = launch_xf_plain<4>(p, m0, a, s); break;
    case 5: e = launch_xf_plain<5>(p, m0, a, s); break;
    case 6: e = launch_xf_plain<6>(p, m0, a, s); break;
    case 7: e = launch_xf_plain<7>(p, m0, a, s); break;
    default: e = launch_xf_plain<8>(p, m0, a, s); break;
  }
  if (e == cudaSuccess) ++p->tma_launches;  // as in sym_xf: counted once enqueued
  return e;
}

cudaError_t sym_xb_plain(exx_plan* p, double* buf, int nb, cudaStream_t s) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!sym_x_usable_plain(p, buf, buf, nb)) return cudaErrorNotSupported;
  constexpr int NT = 2;
  XSArgs a{};
  fill_x(p, st, a);
  a.out = buf;
  a.V = st->d_img_xb;
  a.tiles_per_rhs = (a.rows_per_rhs + 8 * NT - 1) / (8 * NT);
  a.div_tiles = make_fastdiv((unsigned)a.tiles_per_rhs);
  a.n_tiles = (unsigned)a.tiles_per_rhs * (unsigned)nb;
  if (a.n_tiles == 0) return cudaSuccess;
  CUtensorMap m0;
  cudaError_t e;
  if ((e = get_map(st, buf, a.n, (long long)a.rows_per_rhs * nb, 0, 8 * NT, &m0)) != cudaSuccess) return e;
  ++p->tma_launches;
  switch ((a.nh + 7) / 8) {
    case 3: return launch_xb<3>(p, m0, a, s);
    case 4: return launch_xb<4>(p, m0, a, s);
    case 5: return launch_xb<5>(p, m0, a, s);
    case 6: return launch_xb<6>(p, m0, a, s);
    case 7: return launch_xb<7>(p, m0, a, s);
    default: return launch_xb<8>(p, m0, a, s);
  }
}

// x-backward product fused with the accumulate; `in` holds the batch with the x modes even block first.  side 0: the
// work items are the batch's targets (vx_k -= sum_j occ_j psi_j phi_jk; pair-symmetric apply: only j <= k).  side 1
// (pair-symmetric apply only): the items are the batch's orbitals, vx_j -= sum_{k > j} occ_k psi_k phi_jk -- the same
// product over the same batch with the roles of the two indices exchanged, so phi never exists in memory either way.
cudaError_t sym_xacc(exx_plan* p, const double* in, int nb, const FastArgs* fa, cudaStream_t s, int side) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!sym_x_usable(p, in, fa)) return cudaErrorNotSupported;
  if (nb != fa->bd.nj * fa->bd.nk || (side && !fa->sym)) return cudaErrorInvalidValue;
  constexpr int kBig = 1 << 28;
  XSArgs a{};
  fill_x(p, st, a);
  a.V = st->d_img_xb;
  if (!side) {
    a.n_items = fa->bd.nk;
    a.L = fa->bd.nj;
    a.stride_i = fa->bd.nj;
    a.stride_l = 1;
    a.p0 = fa->bd.j0;
    a.c_lo = -kBig;
    a.c_hi = fa->sym ? fa->bd.k0 - fa->bd.j0 + 1 : kBig;
    a.vx = fa->vx + (size_t)fa->bd.k0 * (size_t)p->N;
  } else {
    a.n_items = fa->bd.nj;
    a.L = fa->bd.nk;
    a.stride_i = 1;
    a.stride_l = fa->bd.nj;
    a.p0 = fa->bd.k0;
    a.c_lo = fa->bd.j0 - fa->bd.k0 + 1;
    a.c_hi = kBig;
    a.vx = fa->vx + (size_t)fa->bd.j0 * (size_t)p->N;
  }
  a.occ = fa->occ + a.p0;
  a.first = fa->first ? 1 : 0;
  a.div_items = make_fastdiv((unsigned)a.n_items);
  const long long rows_total = (long long)a.rows_per_rhs * nb, rows_psi = (long long)a.rows_per_rhs * fa->n_occ;
  if (rows_total >= (1LL << 31) - 64) return cudaErrorNotSupported;
  const int ms = (a.nh + 7) / 8, NT = ms <= 4 ? 2 : 1;
  const long long tiles_per_rhs = (a.rows_per_rhs + 8 * NT - 1) / (8 * NT);
  if (tiles_per_rhs * a.n_items >= (1LL << 31) - 64) return cudaErrorNotSupported;
  a.n_tiles = (unsigned)(tiles_per_rhs * a.n_items);
  if (a.n_tiles == 0) return cudaSuccess;
  CUtensorMap m0, m1;
  cudaError_t e;
  if ((e = get_map(st, in, a.n, rows_total, 0, 8 * NT, &m0)) != cudaSuccess) return e;
  if ((e = get_map(st, fa->psi, a.n, rows_psi, 0, 8 * NT, &m1)) != cudaSuccess) return e;
  ++p->tma_launches;
  const bool gen = fa->sym;
#define EXX_XACC_CASE(MSV) \
  case MSV: return gen ? launch_xacc_sym<MSV, true>(p, m0, m1, a, s) : launch_xacc_sym<MSV, false>(p, m0, m1, a, s);
  switch (ms) {
    EXX_XACC_CASE(3)
    EXX_XACC_CASE(4)
    EXX_XACC_CASE(5)
    EXX_XACC_CASE(6)
    EXX_XACC_CASE(7)
    default: return gen ? launch_xacc_sym<8, true>(p, m0, m1, a, s) : launch_xacc_sym<8, false>(p, m0, m1, a, s);
  }
#undef EXX_XACC_CASE
}

}  // namespace exx
