// Fused passes of the default variant: fewer trips of a batch through HBM than the six in-place products of
// kernels_tma.cu.  Same machinery as k_mode_t -- FP64 tensor cores (DMMA.8x8x4),
// operands staged by TMA into per-warp mbarrier rings, persistent CTAs, programmatic dependent launch -- plus two
// things k_mode_t does not have:
//
//   * k_mode_zz: z-forward product, eigen-space multiply and z-backward product in ONE pass (Eq. 11's third and
//     fourth GEMM and the Hadamard product of Eq. 16).  The forward product is issued with
//     the MMA operands swapped, C^T = B^T A^T, so that its accumulator fragment (lane (g,q): T[m = 8mt+2q+e][column
//     8nt+g]) IS the A fragment of the backward product written as Y^T = T'^T Vz^T: the intermediate T never leaves
//     the registers, no shuffle, no shared-memory bounce.  The multiplier tile follows the data tile through the same
//     TMA ring and is read in accumulator layout.  One shared-memory image of Vz serves both products (its columns are
//     permuted so that both access patterns are bank-conflict free).
//   * k_mode_xacc: x-backward product and accumulate (a5) in one pass.  A work item is (row tile, target k); the
//     warp loops over the occupied orbitals j of the batch, keeps vx_k's tile in a second set of accumulators and
//     reads the psi_j tile, which follows the data tile through the TMA ring, in accumulator layout:
//     vx_k -= occ_j psi_j phi_jk with j ascending, exactly the order of k_accumulate (bitwise run-to-run
//     reproducible, independent of the batch shape).  phi is never written to memory.
#include <type_traits>

#include "tma_common.cuh"

namespace exx {
namespace {

// ---------------------------------------------------------------------------------------------------------------
// k_mode_zz
// ---------------------------------------------------------------------------------------------------------------
struct ZArgs {
  double* out;
  const double* V;  // image [16*S][8*MTOT+4]: row 16s+4kk+q = z index read by lane q in k-step kk, column sigma(m)
  int n;
  int S;        // stages of 16 contraction indices per product
  int kk_last;  // 0: n % 16 == 0; else k-steps of the ragged last stage
  unsigned n_tiles;
  int inner;              // nx*ny
  int cpo;                // chunks of 16 columns per right-hand side
  unsigned total_chunks;  // cpo * nb
  int outer;              // nb
  FastDiv div_cpo;
};

// CPLX (Bloch plans, complex z axis with n <= 64): a function is a (re, im) pair of planes and V the real embedding
// E = [[Vr, -Vi], [Vi, Vr]] of the complex eigenvector matrix (forward product with E^T = embedding of V^H, backward
// with E): the same kernel with 2 S stages and 2 MH row tiles, the second half of each belonging to the im plane; the
// (real) multiplier tile is fetched once per plane.
template <int MTOT, int NT, int WARPS, int IC, bool CPLX = false>
__global__ void __launch_bounds__(32 * WARPS, 1)
    k_mode_zz(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1, const ZArgs a) {
  static_assert(NT == 2 || NT == 4, "a tile is one or two 16-column chunks");
  static_assert(MTOT % IC == 0, "output row tiles are processed IC at a time");
  static_assert(!CPLX || MTOT % 2 == 0, "row tiles of the re plane, then of the im plane");
  constexpr int MH = CPLX ? MTOT / 2 : MTOT;
  constexpr int LDV = 8 * MTOT + 4;
  constexpr unsigned kStage = 1024u * NT;
  constexpr int CH = NT / 2;
  constexpr int SMAX = (MTOT + 1) / 2;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, S = a.S;
  const int S2 = CPLX ? 2 * S : S;  // stages per product
  const unsigned smem0 = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned img_bytes = 8u * (16u * S2) * LDV;

  for (unsigned i = 2 * tid; i < 16u * S2 * LDV; i += 2 * 32 * WARPS)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem0 + 8u * i), "l"(a.V + i) : "memory");
  asm volatile("cp.async.commit_group;\n" ::: "memory");

  const unsigned ring0 = (smem0 + img_bytes + 1023u) & ~1023u;
  const unsigned my_ring = ring0 + warp * (kDepth * kStage);
  const unsigned my_bar = ring0 + WARPS * (kDepth * kStage) + warp * (kDepth * 8u);
  const unsigned ctr_addr = ring0 + WARPS * (kDepth * kStage) + WARPS * (kDepth * 8u);
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

  // ---- producer: a tile is S2 data stages (tm0) followed by S2 multiplier stages (tm1, same columns) -----------
  unsigned t_p = tfirst;
  int s_p = 0;
  int pc0[CH], pc2[CH];
  auto tile_coords = [&](unsigned t) {
#pragma unroll
    for (int ch = 0; ch < CH; ++ch) {
      const unsigned cc = t * CH + ch;
      if (cc < a.total_chunks) {
        const unsigned o = fast_div(cc, a.div_cpo);
        pc2[ch] = CPLX ? 2 * (int)o : (int)o;  // CPLX: o counts complex functions, plane 2o is the re plane
        pc0[ch] = 16 * (int)(cc - o * (unsigned)a.cpo);
      } else {  // past the end: an all-out-of-bounds data box (zeros), never stored
        pc2[ch] = a.outer;
        pc0[ch] = 0;
      }
    }
  };
  auto produce = [&](int slot) {
    if (t_p >= a.n_tiles) return;
    const unsigned bar = my_bar + 8u * slot;
    const unsigned dst = my_ring + slot * kStage;
    if (elect_one()) {
      mbar_expect_tx(bar, kStage);
#pragma unroll
      for (int ch = 0; ch < CH; ++ch) {
        if (s_p < S2) {
          const bool im = CPLX && s_p >= S;
          tma_load_3d(dst + 2048u * ch, &tm0, pc0[ch], 16 * (im ? s_p - S : s_p), pc2[ch] + (im ? 1 : 0), bar);
        } else {
          const int tl = s_p - S2;
          tma_load_3d(dst + 2048u * ch, &tm1, pc0[ch], 16 * (CPLX && tl >= S ? tl - S : tl), 0, bar);
        }
      }
    }
    if (++s_p == 2 * S2) {
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

  // ---- per-lane fragment addresses --------------------------------------------------------------------------
  const unsigned b1 = (unsigned)(q >> 1);
  // forward product, Vz fragment: image row 16s + 4kk + q, column sigma(8mt + g), sigma(c) = c ^ ((c >> 2) & 1)
  unsigned v1_lane = smem0 + 8u * (q * LDV + (g ^ ((g >> 2) & 1)));
  // data fragment inside a stage (as k_mode_t's L-mode): box row 2q + (kk&1) + 8(kk>>1), column 8(nt&1)+g
  unsigned xo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const unsigned row = 2u * q + (i & 1);
    xo[i] = 128u * row + 16u * ((4u * (i >> 1) + (g >> 1)) ^ row) + 8u * (g & 1);
  }
  // multiplier fragment in accumulator layout: box row 8h + 2q + e (the eigen index m within its 16), column 8(nt&1)+g
  unsigned tq[2][2];
#pragma unroll
  for (int e = 0; e < 2; ++e)
#pragma unroll
    for (int np = 0; np < 2; ++np) {
      const unsigned row = 2u * q + e;
      tq[e][np] = 128u * row + 16u * ((4u * np + (g >> 1)) ^ row) + 8u * (g & 1);
    }
  // backward product, Vz fragment: image row 8it + g (an output index), column sigma(8mt + 2q + e) = 8mt + 2q + (e ^ b1)
  unsigned v2_lane[2];
  v2_lane[0] = smem0 + 8u * (g * LDV + 2u * q + b1);
  v2_lane[1] = smem0 + 8u * (g * LDV + 2u * q + (1u ^ b1));
  // z index of output row 8it + 2q + e: the index image row 8it + 2q + e holds (standard stage / ragged last stage)
  const int zo_std[2] = {4 * (q & 1) + (q >> 1), 4 * (q & 1) + 2 + (q >> 1)};
  const int zo_lin[2] = {2 * q, 2 * q + 1};

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  while (t < a.n_tiles) {
    double acc[MTOT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    // ---- forward product, operands swapped: acc[mt][nt][e] = T[m = 8mt + 2q + e][column 8nt + g] -------------
    for (int s = 0; s < S2; ++s) {
      asm volatile("" : "+r"(v1_lane), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
      mbar_wait(my_bar + 8u * slot, parity);
      const unsigned sb = my_ring + slot * kStage;
      const unsigned aa = v1_lane + (unsigned)s * (16u * LDV * 8u);
      const bool ragged = a.kk_last && (s == S - 1 || (CPLX && s == S2 - 1));
      if (!ragged) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          double bf[NT];
#pragma unroll
          for (int nt = 0; nt < NT; ++nt)
            bf[nt] = lds64(sb + xo[2 * (nt & 1) + (kk & 1)] + 2048u * (nt >> 1) + 1024u * (kk >> 1));
          double af[MTOT];
#pragma unroll
          for (int mt = 0; mt < MTOT; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
          for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], bf[nt], af[mt]);
        }
      } else {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          if (kk < a.kk_last) {
            double bf[NT];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              const unsigned row = 4u * kk + q;
              bf[nt] = lds64(sb + 2048u * (nt >> 1) + 128u * row + 16u * ((4u * (nt & 1) + (g >> 1)) ^ (row & 7u)) +
                             8u * (g & 1));
            }
            double af[MTOT];
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], bf[nt], af[mt]);
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

    // ---- eigen-space multiply (a3): the multiplier tile arrives in S more stages, read in accumulator layout ---
#pragma unroll
    for (int sp = 0; sp < SMAX; ++sp) {
      if (sp < S2) {
        mbar_wait(my_bar + 8u * slot, parity);
        const unsigned sb = my_ring + slot * kStage;
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          if (2 * sp + h < MTOT) {
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
              for (int e = 0; e < 2; ++e)
                acc[2 * sp + h < MTOT ? 2 * sp + h : 0][nt][e] *=
                    lds64(sb + 2048u * (nt >> 1) + 1024u * h + tq[e][nt & 1]);
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

    // ---- backward product Y^T = T'^T Vz^T, IC output row tiles at a time; A fragments are the accumulators ------
    int o_ch[CH], col_ch[CH];
#pragma unroll
    for (int ch = 0; ch < CH; ++ch) {
      const unsigned cc = t * CH + ch;
      if (cc < a.total_chunks) {
        const unsigned o = fast_div(cc, a.div_cpo);
        o_ch[ch] = CPLX ? 2 * (int)o : (int)o;
        col_ch[ch] = 16 * (int)(cc - o * (unsigned)a.cpo) + g;
      } else {
        o_ch[ch] = 0;
        col_ch[ch] = a.inner;  // nothing stored
      }
    }
#pragma unroll 1
    for (int it0 = 0; it0 < MTOT; it0 += IC) {
      double acc2[IC][NT][2];
#pragma unroll
      for (int ic = 0; ic < IC; ++ic)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) acc2[ic][nt][0] = acc2[ic][nt][1] = 0.0;
      const unsigned wrow = (unsigned)it0 * (8u * LDV * 8u);
#pragma unroll
      for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          double w[IC];
#pragma unroll
          for (int ic = 0; ic < IC; ++ic) w[ic] = lds64(v2_lane[e] + wrow + (8u * ic * LDV + 8u * mt) * 8u);
#pragma unroll
          for (int ic = 0; ic < IC; ++ic)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(acc2[ic][nt], acc[mt][nt][e], w[ic]);
        }
      // store: lane (g,q) holds Y[z(8it + 2q + e)][column 8nt + g]
#pragma unroll
      for (int ic = 0; ic < IC; ++ic) {
        const int it = it0 + ic;
        const int im = (CPLX && it >= MH) ? 1 : 0;  // row tiles MH.. belong to the im plane
        const int itp = it - im * MH;
        const bool lin = a.kk_last && (itp >> 1) == S - 1;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int z = 8 * itp + (lin ? zo_lin[e] : zo_std[e]);
          if (z < n) {
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              const int col = col_ch[nt >> 1] + 8 * (nt & 1);
              if (col < a.inner)
                a.out[((long long)(o_ch[nt >> 1] + im) * n + z) * a.inner + col] = acc2[ic][nt][e];
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
// k_mode_zz_sym: k_mode_zz on the reflection-adapted eigenbasis of a real z axis (plan_host.cpp symmetrize_axis).
// Every eigenvector of the periodic or Dirichlet 1-D matrix can be taken even or odd under z -> mir(z), so
//     forward:   T[m] = sum_{z <= mir z} V[z][m] (f[z] +- f[mir z])        (+ for an even mode, - for an odd one)
//     backward:  a[z] = sum_{m even} V[z][m] t[m],  b[z] = sum_{m odd} V[z][m] t[m],  y[z] = a + b,  y[mir z] = a - b
// i.e. both products contract over HALF the range with two blocks of the matrix: about 55 % of the DMMAs of the dense
// kernel (n = 120: 2 x 512 against 2 x 900 per 16 columns).  A stage is two TMA boxes, rows [16 s, 16 s + 16) and the
// mirrored rows (row 15 - r of the second box is mir(16 s + r)); the butterfly f +- f[mir] happens on the fragments,
// the a +- b one on the accumulators.  Row tiles 0..MS-1 of the first accumulator set belong to the even modes, MS..2MS-1
// to the odd ones; the multiplier table is the plan's table with its z index in the same (even | odd) order.
// Everything else (operand swap, register chaining, image column permutation, multiplier tile through the ring) is
// k_mode_zz's.
// ---------------------------------------------------------------------------------------------------------------
struct ZSArgs {
  double* out;
  const double* V;  // image [16*Sh][16*MS+4]: row = half-range z (k_mode_t's L-mode order), columns sigma(even m) | 8 MS + sigma(odd m)
  int n;
  int nh;       // half range: number of z with z <= mir(z) = number of even modes
  int Sh;       // stages of 16 half-range indices
  int kk_last;  // ragged last stage (nh % 16 != 0): its k-steps
  int mir0;     // first row of the mirrored box of stage 0 (stage s: mir0 - 16 s)
  int mirc;     // mir(z) = mirc - z (periodic: n, with mir(0) = n read as "none"; Dirichlet: n - 1)
  int zfix;     // z == mir(z) inside the array (its mirrored read is replaced by zero), or -1
  unsigned n_tiles;
  int inner, cpo, outer;
  unsigned total_chunks;
  FastDiv div_cpo;
};

template <int MS, int NT, int WARPS, int IC>
__global__ void __launch_bounds__(32 * WARPS, 1)
    k_mode_zz_sym(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1, const ZSArgs a) {
  static_assert(NT == 2 || NT == 4, "a tile is one or two 16-column chunks");
  static_assert(MS % IC == 0, "output row tiles are processed IC at a time");
  constexpr int MT = 2 * MS;
  constexpr int LDV = 8 * MT + 4;
  constexpr unsigned kS1 = 1024u * NT;  // one box set (all chunks of a tile)
  constexpr unsigned kSlot = 2u * kS1;  // a data stage: the rows and the mirrored rows
  constexpr int CH = NT / 2;
  constexpr int TS = (MS + 1) / 2;      // multiplier boxes (16 modes = two row tiles) per block
  constexpr int TS2 = (TS + 1) / 2;     // multiplier stages per block: a slot (rows + mirrored rows of a data stage) holds two boxes
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

  // ---- producer: Sh data stages (rows + mirrored rows), TS2 multiplier stages for the even modes, TS2 for the odd ----
  const int stages_per_tile = Sh + 2 * TS2;
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
        pc0[ch] = 16 * (int)(cc - o * (unsigned)a.cpo);
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
      if (s_p < Sh) {
        mbar_expect_tx(bar, kSlot);
#pragma unroll
        for (int ch = 0; ch < CH; ++ch) {
          tma_load_3d(dst + 2048u * ch, &tm0, pc0[ch], 16 * s_p, pc2[ch], bar);
          tma_load_3d(dst + kS1 + 2048u * ch, &tm0, pc0[ch], a.mir0 - 16 * s_p, pc2[ch], bar);
        }
      } else {
        const int ts2 = s_p - Sh;
        const int blk = ts2 < TS2 ? 0 : 1, t0 = 2 * (ts2 - blk * TS2);  // first box of this stage within its block
        const int nbx = TS - t0 < 2 ? TS - t0 : 2;
        mbar_expect_tx(bar, kS1 * (unsigned)nbx);
#pragma unroll
        for (int hh = 0; hh < 2; ++hh)
          if (hh < nbx) {
            const int row = (blk ? a.nh : 0) + 16 * (t0 + hh);  // even modes: table rows 0.., odd modes: rows nh..
#pragma unroll
            for (int ch = 0; ch < CH; ++ch) tma_load_3d(dst + kS1 * hh + 2048u * ch, &tm1, pc0[ch], row, 0, bar);
          }
      }
    }
    if (++s_p == stages_per_tile) {
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

  // ---- per-lane fragment addresses --------------------------------------------------------------------------
  const unsigned b1 = (unsigned)(q >> 1);
  unsigned v1_lane = smem0 + 8u * (q * LDV + (g ^ ((g >> 2) & 1)));
  // data fragment of k-step kk, column tile nt: box row 2q + (kk&1) + 8(kk>>1); its mirror image is row 15 - that of
  // the second box
  unsigned xo[4], xm[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const unsigned row = 2u * q + (i & 1), rowm = 7u - row;
    xo[i] = 128u * row + 16u * ((4u * (i >> 1) + (g >> 1)) ^ row) + 8u * (g & 1);
    xm[i] = kS1 + 128u * rowm + 16u * ((4u * (i >> 1) + (g >> 1)) ^ rowm) + 8u * (g & 1);
  }
  unsigned tq[2][2];
#pragma unroll
  for (int e = 0; e < 2; ++e)
#pragma unroll
    for (int np = 0; np < 2; ++np) {
      const unsigned row = 2u * q + e;
      tq[e][np] = 128u * row + 16u * ((4u * np + (g >> 1)) ^ row) + 8u * (g & 1);
    }
  unsigned v2_lane[2];
  v2_lane[0] = smem0 + 8u * (g * LDV + 2u * q + b1);
  v2_lane[1] = smem0 + 8u * (g * LDV + 2u * q + (1u ^ b1));
  const int zo_std[2] = {4 * (q & 1) + (q >> 1), 4 * (q & 1) + 2 + (q >> 1)};
  const int zo_lin[2] = {2 * q, 2 * q + 1};

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  while (t < a.n_tiles) {
    double acc[MT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MT; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    // ---- forward: acc[mt][nt][e] = T[mode 8(mt % MS) + 2q + e of block mt / MS][column 8nt + g] -----------------
    auto do_stage = [&](int s, auto rag_c) {  // `ragged` at compile time: standard stages carry none of its address math
      constexpr bool ragged = decltype(rag_c)::value;
      asm volatile("" : "+r"(v1_lane), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
      mbar_wait(my_bar + 8u * slot, parity);
      const unsigned sb = my_ring + slot * kSlot;
      const unsigned aa = v1_lane + (unsigned)s * (16u * LDV * 8u);
      const int zf = a.zfix - 16 * s;  // local row whose mirror image is itself (its second read counts as zero)
#pragma unroll
      for (int kk = 0; kk < 4; ++kk) {
        if (!ragged || kk < a.kk_last) {
          double be[NT], bo[NT];
          const int rowl = ragged ? 4 * kk + q : 2 * q + (kk & 1) + 8 * (kk >> 1);
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            unsigned oa, ob;
            if (!ragged) {
              oa = sb + xo[2 * (nt & 1) + (kk & 1)] + 2048u * (nt >> 1) + 1024u * (kk >> 1);
              ob = sb + xm[2 * (nt & 1) + (kk & 1)] + 2048u * (nt >> 1) + 1024u * (1 - (kk >> 1));
            } else {
              const unsigned row = 4u * kk + q, rowm = 15u - row;
              oa = sb + 2048u * (nt >> 1) + 128u * row + 16u * ((4u * (nt & 1) + (g >> 1)) ^ (row & 7u)) + 8u * (g & 1);
              ob = sb + kS1 + 2048u * (nt >> 1) + 128u * rowm + 16u * ((4u * (nt & 1) + (g >> 1)) ^ (rowm & 7u)) + 8u * (g & 1);
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
            for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], mt < MS ? be[nt] : bo[nt], af[mt]);
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

    // ---- eigen-space multiply: TS2 stages for the even block, TS2 for the odd block, two boxes of 16 modes per stage ------
#pragma unroll
    for (int sp = 0; sp < 2 * TS2; ++sp) {
      mbar_wait(my_bar + 8u * slot, parity);
      const unsigned sb = my_ring + slot * kSlot;
#pragma unroll
      for (int hh = 0; hh < 2; ++hh)
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          constexpr int kZ = 0;
          const int blk = sp < TS2 ? 0 : 1, ts = 2 * (sp < TS2 ? sp : sp - TS2) + hh, mtl = 2 * ts + h;  // compile-time
          if (ts < TS && mtl < MS) {
            const int mt = blk * MS + mtl;
#pragma unroll
            for (int nt = 0; nt < NT; ++nt)
#pragma unroll
              for (int e = 0; e < 2; ++e)
                acc[mt < MT ? mt : kZ][nt][e] *= lds64(sb + kS1 * hh + 2048u * (nt >> 1) + 1024u * h + tq[e][nt & 1]);
          }
        }
      __syncwarp();
      produce(slot);
      if (++slot == kDepth) {
        slot = 0;
        parity ^= 1u;
      }
    }

    // ---- backward: a = E t_even, b = O t_odd over the half range, IC row tiles at a time; y = a + b, y[mir] = a - b ---
    int o_ch[CH], col_ch[CH];
#pragma unroll
    for (int ch = 0; ch < CH; ++ch) {
      const unsigned cc = t * CH + ch;
      if (cc < a.total_chunks) {
        const unsigned o = fast_div(cc, a.div_cpo);
        o_ch[ch] = (int)o;
        col_ch[ch] = 16 * (int)(cc - o * (unsigned)a.cpo) + g;
      } else {
        o_ch[ch] = 0;
        col_ch[ch] = a.inner;
      }
    }
#pragma unroll 1
    for (int it0 = 0; it0 < MS; it0 += IC) {
      double pa[IC][NT][2], pb[IC][NT][2];
#pragma unroll
      for (int ic = 0; ic < IC; ++ic)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) pa[ic][nt][0] = pa[ic][nt][1] = pb[ic][nt][0] = pb[ic][nt][1] = 0.0;
      const unsigned wrow = (unsigned)it0 * (8u * LDV * 8u);
#pragma unroll
      for (int mt = 0; mt < MT; ++mt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          double w[IC];
#pragma unroll
          for (int ic = 0; ic < IC; ++ic) w[ic] = lds64(v2_lane[e] + wrow + (8u * ic * LDV + 8u * mt) * 8u);
#pragma unroll
          for (int ic = 0; ic < IC; ++ic)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(mt < MS ? pa[ic][nt] : pb[ic][nt], acc[mt][nt][e], w[ic]);
        }
#pragma unroll
      for (int ic = 0; ic < IC; ++ic) {
        const int it = it0 + ic;
        const bool lin = a.kk_last && (it >> 1) == Sh - 1;
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const int z = 8 * it + (lin ? zo_lin[e] : zo_std[e]);
          if (z < a.nh) {
            const int zb = a.mirc - z;
            const bool two = zb != z && zb < n;
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              const int col = col_ch[nt >> 1] + 8 * (nt & 1);
              if (col < a.inner) {
                double* base = a.out + ((long long)o_ch[nt >> 1] * n) * a.inner + col;
                base[(long long)z * a.inner] = pa[ic][nt][e] + pb[ic][nt][e];
                if (two) base[(long long)zb * a.inner] = pa[ic][nt][e] - pb[ic][nt][e];
              }
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
// k_mode_xacc
// ---------------------------------------------------------------------------------------------------------------
struct XArgs {
  const double* V;    // X-mode image of Vx (backward), as k_mode_t stages it
  const double* occ;  // occ + j0
  double* vx;         // vx + k0 * N
  int n;
  int S;
  int kk_last;
  unsigned n_tiles;  // work items: tiles_per_rhs * nk
  int rows_per_rhs;  // N / nx
  int nj, nk, j0;
  int first;  // vx_k is overwritten (first batch of these targets), not accumulated into
  FastDiv div_nk;
};

template <int MTOT, int NT, int WARPS>
__global__ void __launch_bounds__(32 * WARPS, 1)
    k_mode_xacc(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1, const XArgs a) {
  static_assert(NT == 1 || NT == 2 || NT == 4, "a tile is 8, 16 or 32 rows");
  constexpr int LDV = 8 * MTOT + 4;
  constexpr unsigned kStage = 1024u * NT;  // a {16 x, 8 NT rows} box
  constexpr int SMAX = (MTOT + 1) / 2;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, S = a.S;
  const unsigned smem0 = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned img_bytes = 8u * (16u * S) * LDV;

  for (unsigned i = 2 * tid; i < 16u * S * LDV; i += 2 * 32 * WARPS)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem0 + 8u * i), "l"(a.V + i) : "memory");
  asm volatile("cp.async.commit_group;\n" ::: "memory");

  const unsigned ring0 = (smem0 + img_bytes + 1023u) & ~1023u;
  const unsigned my_ring = ring0 + warp * (kDepth * kStage);
  const unsigned my_bar = ring0 + WARPS * (kDepth * kStage) + warp * (kDepth * 8u);
  const unsigned ctr_addr = ring0 + WARPS * (kDepth * kStage) + WARPS * (kDepth * 8u);
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

  // ---- producer: item (row tile rb, target kq) = nj steps; a step is S stages of the batch's right-hand side
  //      (jj, kq) from tm0 followed by S stages of psi_{j0+jj} from tm1, same rows -----------------------------
  unsigned t_p = tfirst;
  int s_p = 0, jj_p = 0;
  int prow_d = 0, prow_p = 0;
  auto tile_coords = [&](unsigned t) {
    const int rb = (int)fast_div(t, a.div_nk);
    const int kq = (int)t - rb * a.nk;
    prow_d = (a.nj * kq) * a.rows_per_rhs + rb * (8 * NT);
    prow_p = a.j0 * a.rows_per_rhs + rb * (8 * NT);
  };
  auto produce = [&](int slot) {
    if (t_p >= a.n_tiles) return;
    const unsigned bar = my_bar + 8u * slot;
    const unsigned dst = my_ring + slot * kStage;
    if (elect_one()) {
      mbar_expect_tx(bar, kStage);
      if (s_p < S) tma_load_2d(dst, &tm0, 16 * s_p, prow_d, bar);
      else tma_load_2d(dst, &tm1, 16 * (s_p - S), prow_p, bar);
    }
    if (++s_p == 2 * S) {
      s_p = 0;
      if (++jj_p == a.nj) {
        jj_p = 0;
        t_p = claim_tile();
#pragma unroll
        for (int i = 0; i < kDepth + 1; ++i)
          if (i == fifo_n) fifo[i] = t_p;
        ++fifo_n;
        if (t_p < a.n_tiles) tile_coords(t_p);
      } else {
        prow_d += a.rows_per_rhs;
        prow_p += a.rows_per_rhs;
      }
    }
  };
  if (t_p < a.n_tiles) tile_coords(t_p);
#pragma unroll
  for (int d = 0; d < kDepth; ++d) produce(d);
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();

  // ---- per-lane fragment addresses --------------------------------------------------------------------------
  unsigned a_lane_v = smem0 + 8u * (q * LDV + g);
  unsigned xo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) xo[i] = 128u * g + 16u * ((4u * (q >> 1) + i) ^ (unsigned)g) + 8u * (q & 1);
  // psi fragment in accumulator layout: box row 8nt + 2q + e (a data row), x = 8h + g within the stage's 16
  unsigned pq[2][2];
#pragma unroll
  for (int e = 0; e < 2; ++e)
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const unsigned row = 2u * q + e;
      pq[e][h] = 128u * row + 16u * ((4u * h + (g >> 1)) ^ row) + 8u * (g & 1);
    }

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  const int s_std = a.kk_last ? S - 1 : S;
  while (t < a.n_tiles) {
    const int rb = (int)fast_div(t, a.div_nk);
    const int kq = (int)t - rb * a.nk;
    const int row0 = rb * (8 * NT);  // within the target's rows
    double* vbase = a.vx + ((long long)kq * a.rows_per_rhs + row0 + 2 * q) * n + g;
    double vacc[MTOT][NT][2];
    if (a.first) {
#pragma unroll
      for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) vacc[mt][nt][0] = vacc[mt][nt][1] = 0.0;
    } else {
#pragma unroll
      for (int nt = 0; nt < NT; ++nt)
#pragma unroll
        for (int e = 0; e < 2; ++e) {
          const bool rok = row0 + 8 * nt + 2 * q + e < a.rows_per_rhs;
          const double* src = vbase + (long long)(8 * nt + e) * n;
#pragma unroll
          for (int mt = 0; mt < MTOT; ++mt) vacc[mt][nt][e] = (rok && 8 * mt + g < n) ? src[8 * mt] : 0.0;
        }
    }

    for (int jj = 0; jj < a.nj; ++jj) {
      const double oc = __ldg(a.occ + jj);
      double acc[MTOT][NT][2];
#pragma unroll
      for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
        for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

      // phi_jk tile: acc[mt][nt][e] = phi[row 8nt + 2q + e][x = 8mt + g]
      for (int s = 0; s < S; ++s) {
        asm volatile("" : "+r"(a_lane_v), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
        mbar_wait(my_bar + 8u * slot, parity);
        const unsigned sb = my_ring + slot * kStage;
        const unsigned aa = a_lane_v + (unsigned)s * (16u * LDV * 8u);
        if (s < s_std) {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) {
            double bf[NT];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) bf[nt] = lds64(sb + xo[kk] + 1024u * nt);
            double af[MTOT];
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
              for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], bf[nt]);
          }
        } else {
#pragma unroll
          for (int kk = 0; kk < 4; ++kk) {
            if (kk < a.kk_last) {
              double bf[NT];
#pragma unroll
              for (int nt = 0; nt < NT; ++nt)
                bf[nt] = lds64(sb + 1024u * nt + 128u * g + 16u * ((2u * kk + (q >> 1)) ^ (unsigned)g) + 8u * (q & 1));
              double af[MTOT];
#pragma unroll
              for (int mt = 0; mt < MTOT; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
              for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
                for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], bf[nt]);
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

      // a5: vx_k -= occ_j psi_j phi_jk; the psi_j tile arrives in S more stages, read in accumulator layout
#pragma unroll
      for (int sp = 0; sp < SMAX; ++sp) {
        if (sp < S) {
          mbar_wait(my_bar + 8u * slot, parity);
          const unsigned sb = my_ring + slot * kStage;
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            if (2 * sp + h < MTOT) {
              constexpr int kZero = 0;
              const int mt = 2 * sp + h < MTOT ? 2 * sp + h : kZero;
#pragma unroll
              for (int nt = 0; nt < NT; ++nt)
#pragma unroll
                for (int e = 0; e < 2; ++e) {
                  const double ps = lds64(sb + 1024u * nt + pq[e][h]);
                  vacc[mt][nt][e] -= oc * ps * acc[mt][nt][e];
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

    // vx_k tile back to memory
#pragma unroll
    for (int nt = 0; nt < NT; ++nt)
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        if (row0 + 8 * nt + 2 * q + e < a.rows_per_rhs) {
          double* dst = vbase + (long long)(8 * nt + e) * n;
#pragma unroll
          for (int mt = 0; mt < MTOT; ++mt)
            if (8 * mt + g < n) dst[8 * mt] = vacc[mt][nt][e];
        }
      }

    t = fifo[0];
#pragma unroll
    for (int i = 0; i < kDepth; ++i) fifo[i] = fifo[i + 1];
    --fifo_n;
  }
}

// ---- host side ------------------------------------------------------------------------------------------------

template <typename Kern, typename Args>
cudaError_t launch_persistent(Kern kern, SmemOptIn& opt, size_t smem, int warps, unsigned n_tiles, const exx_plan* p,
                              const CUtensorMap& m0, const CUtensorMap& m1, const Args& a, cudaStream_t s) {
  // padded above half an SM's shared memory: exactly one CTA per SM (the tile split assumes it)
  const size_t floor_bytes = 117 * 1024;
  if (smem < floor_bytes) smem = floor_bytes;
  if (smem > (size_t)p->smem_optin) return cudaErrorNotSupported;
  cudaError_t e = opt.ensure(kern, p->device, smem, true);
  if (e != cudaSuccess) return e;
  cudaLaunchConfig_t cfg = {};
  const unsigned grid = n_tiles < (unsigned)p->sm_count ? n_tiles : (unsigned)p->sm_count;
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

template <int MTOT, int NT, int WARPS, int IC>
cudaError_t launch_zz_c(const exx_plan* p, const CUtensorMap& m0, const CUtensorMap& m1, const ZArgs& a, cudaStream_t s);

inline size_t smem_need(int S, int mtot, int warps, int nt) {
  const size_t img = sizeof(double) * 16 * (size_t)S * (8 * mtot + 4);
  return img + 1024 + (size_t)warps * kDepth * 1024 * nt + (size_t)warps * kDepth * 8 + 16;
}

template <int MTOT, int NT, int WARPS, int IC>
cudaError_t launch_zz(const exx_plan* p, const CUtensorMap& m0, const CUtensorMap& m1, const ZArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  return launch_persistent(k_mode_zz<MTOT, NT, WARPS, IC>, opt, smem_need(a.S, MTOT, WARPS, NT), WARPS, a.n_tiles, p, m0,
                           m1, a, s);
}

template <int MTOT, int NT, int WARPS, int IC>
cudaError_t launch_zz_c(const exx_plan* p, const CUtensorMap& m0, const CUtensorMap& m1, const ZArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  return launch_persistent(k_mode_zz<MTOT, NT, WARPS, IC, true>, opt, smem_need(2 * a.S, MTOT, WARPS, NT), WARPS, a.n_tiles,
                           p, m0, m1, a, s);
}

template <int MS, int NT, int WARPS, int IC>
cudaError_t launch_zz_sym(const exx_plan* p, const CUtensorMap& m0, const CUtensorMap& m1, const ZSArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  const size_t img = sizeof(double) * 16 * (size_t)a.Sh * (16 * MS + 4);
  const size_t smem = img + 1024 + (size_t)WARPS * kDepth * 2 * 1024 * NT + (size_t)WARPS * kDepth * 8 + 16;
  return launch_persistent(k_mode_zz_sym<MS, NT, WARPS, IC>, opt, smem, WARPS, a.n_tiles, p, m0, m1, a, s);
}

template <int MTOT, int NT, int WARPS>
cudaError_t launch_xacc(const exx_plan* p, const CUtensorMap& m0, const CUtensorMap& m1, const XArgs& a, cudaStream_t s) {
  static SmemOptIn opt;
  return launch_persistent(k_mode_xacc<MTOT, NT, WARPS>, opt, smem_need(a.S, MTOT, WARPS, NT), WARPS, a.n_tiles, p, m0, m1,
                           a, s);
}

// class of ceil(n/8), as kernels_tma.cu's pick_class (the images are shared with it)
inline int mtot_class(int n) {
  const int need = (n + 7) / 8;
  if (need > 16) return 0;
  return need <= 2 ? 2 : need <= 4 ? 4 : need <= 6 ? 6 : need <= 8 ? 8 : need <= 12 ? 12 : need <= 15 ? 15 : 16;
}

// rows per warp tile (in units of 8) of k_mode_xacc: two accumulator sets have to fit the register file.  (Sharing a
// 16-row tile between two warps above n = 64 -- one ring per pair, a named barrier per stage -- was built and measured
// in round 2: 1 % SLOWER at 96^3 and 120^3 than 8-row tiles.)
inline int xacc_nt(int mtot) { return mtot <= 8 ? 2 : 1; }

}  // namespace

// Rows of a k_mode_xacc work item (exx_apply sizes its batches with it).
int fused_xacc_tile_rows(const exx_plan* p) {
  const int mtot = mtot_class(p->n[0]);
  return mtot ? 8 * xacc_nt(mtot) : 0;
}

// The image k_mode_zz stages: row 16s + 4kk + q holds the z index the lane with that q reads in k-step kk of stage
// s (k_mode_t's L-mode order), column sigma(m) = m ^ ((m >> 2) & 1) holds eigenvector m: image[row(z)][sigma(m)] =
// Vz[z][m].  The forward product reads it as V^T (lane (g,q): row by q, column by g), the backward product as V (row
// by g, column by q); the column permutation makes both patterns bank-conflict free.
cudaError_t fused_init(exx_plan* p) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st) return cudaSuccess;
  st->d_img_zz = nullptr;
  st->d_img_zz_c = nullptr;
  st->d_img_zzs = nullptr;
  st->d_mult_sym = nullptr;
  st->zs_nh = 0;
  const int n = p->n[2], mtot = mtot_class(n);
  if (!p->bloch && p->h_Vi[2].empty() && p->h_Vi[0].empty() && p->h_Vi[1].empty()) {
    // reflection-adapted basis of the z axis: image over the half range; three to eight row tiles per block (nz = 34
    // .. 128; below, the padding of the two blocks to whole row tiles eats the saving)
    std::vector<double> lam_s, Vs;
    int nh = 0;
    const bool zcap = mtot && symmetrize_axis(n, p->bc[2], p->h_lam[2], p->h_V[2], lam_s, Vs, &nh, true) && (nh + 7) / 8 >= 3 &&
                      (nh + 7) / 8 <= 8;
    if (zcap) {
      const int ms = (nh + 7) / 8, Sh = (nh + 15) / 16, lds = 16 * ms + 4;
      std::vector<double> img((size_t)16 * Sh * lds, 0.0);
      for (int s = 0; s < Sh; ++s)
        for (int kk = 0; kk < 4; ++kk)
          for (int q = 0; q < 4; ++q) {
            const int z = 16 * s + within_stage(false, nh, s, kk, q);
            if (z >= nh) continue;
            double* row = &img[(size_t)(16 * s + 4 * kk + q) * lds];
            for (int m = 0; m < n; ++m) {
              const int mm = m < nh ? m : m - nh;
              row[(m < nh ? 0 : 8 * ms) + (mm ^ ((mm >> 2) & 1))] = Vs[(size_t)z * n + m];
            }
          }
      cudaError_t e = cudaMalloc(&st->d_img_zzs, sizeof(double) * img.size());
      if (e == cudaSuccess) e = cudaMemcpy(st->d_img_zzs, img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
      if (e != cudaSuccess) return e;
      st->zs_nh = nh;
    }
    if (zcap || st->ys_nh || st->xs_nh) {  // the tables in the mode order of the symmetric pipeline, without and with x
      for (int withx = 0; withx < (st->xs_nh ? 2 : 1); ++withx) {
        const std::vector<double> tab = multiplier_table(withx ? st->lam_xs : p->h_lam[0], st->ys_nh ? st->lam_ys : p->h_lam[1],
                                                         zcap ? lam_s : p->h_lam[2], p->omega, p->zero_tol);
        double** dst = withx ? &st->d_mult_symx : &st->d_mult_sym;
        cudaError_t e = cudaMalloc(dst, sizeof(double) * tab.size());
        if (e == cudaSuccess) e = cudaMemcpy(*dst, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice);
        if (e != cudaSuccess) return e;
      }
    }
  }
  if (!mtot) return cudaSuccess;
  const int S = (n + 15) / 16, ldv = 8 * mtot + 4;
  if (!p->h_Vi[2].empty()) {
    // complex z axis: E = [[Vr, -Vi], [Vi, Vr]], rows (plane, z) and columns (plane, m), same permutations per block
    if (mtot > 8) return cudaSuccess;
    const int ldc = 16 * mtot + 4;
    std::vector<double> img((size_t)32 * S * ldc, 0.0);
    for (int s = 0; s < S; ++s)
      for (int kk = 0; kk < 4; ++kk)
        for (int q = 0; q < 4; ++q) {
          const int z = 16 * s + within_stage(false, n, s, kk, q);
          if (z >= n) continue;
          double* row_re = &img[(size_t)(16 * s + 4 * kk + q) * ldc];
          double* row_im = &img[(size_t)(16 * S + 16 * s + 4 * kk + q) * ldc];
          for (int m = 0; m < n; ++m) {
            const int c = m ^ ((m >> 2) & 1);
            const double vr = p->h_V[2][(size_t)z * n + m], vi = p->h_Vi[2][(size_t)z * n + m];
            row_re[c] = vr;
            row_re[8 * mtot + c] = -vi;
            row_im[c] = vi;
            row_im[8 * mtot + c] = vr;
          }
        }
    cudaError_t e = cudaMalloc(&st->d_img_zz_c, sizeof(double) * img.size());
    if (e != cudaSuccess) return e;
    return cudaMemcpy(st->d_img_zz_c, img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
  }
  std::vector<double> img((size_t)16 * S * ldv, 0.0);
  for (int s = 0; s < S; ++s)
    for (int kk = 0; kk < 4; ++kk)
      for (int q = 0; q < 4; ++q) {
        const int z = 16 * s + within_stage(false, n, s, kk, q);
        if (z >= n) continue;
        double* row = &img[(size_t)(16 * s + 4 * kk + q) * ldv];
        for (int m = 0; m < n; ++m) row[m ^ ((m >> 2) & 1)] = p->h_V[2][(size_t)z * n + m];
      }
  cudaError_t e = cudaMalloc(&st->d_img_zz, sizeof(double) * img.size());
  if (e != cudaSuccess) return e;
  return cudaMemcpy(st->d_img_zz, img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
}

void fused_destroy(exx_plan* p) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st) return;
  if (st->d_img_zz) cudaFree(st->d_img_zz);
  if (st->d_img_zz_c) cudaFree(st->d_img_zz_c);
  if (st->d_img_zzs) cudaFree(st->d_img_zzs);
  if (st->d_mult_sym) cudaFree(st->d_mult_sym);
  st->d_img_zzs = st->d_mult_sym = nullptr;
  st->d_img_zz = nullptr;
  st->d_img_zz_c = nullptr;
}

// z-forward product, multiplier and z-backward product of nb right-hand sides in one pass, in place or out of place.
// cudaErrorNotSupported: the caller runs the two k_mode_t passes instead.
cudaError_t fused_zz(exx_plan* p, const double* in, double* out, int nb, cudaStream_t s, int sym) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st || !st->d_img_zz || !(p->fusion & 1)) return cudaErrorNotSupported;
  const int n = p->n[2], mtot = mtot_class(n);
  if (!mtot) return cudaErrorNotSupported;
  if ((p->n[0] & 1) || !aligned16(out) || !aligned16(in) || !aligned16(p->d_mult)) return cudaErrorNotSupported;
  const long long inner = (long long)p->n[0] * p->n[1];
  // symmetric mode (the caller decides it for the whole batch): the z axis on its reflection-adapted basis where the plan
  // has one, and in any case the table in the symmetric pipeline's mode order
  const double* table = sym == 2 ? st->d_mult_symx : sym ? st->d_mult_sym : p->d_mult;
  if (sym && !table) return cudaErrorInvalidValue;
  if (sym && st->d_img_zzs) {
    const int nh = st->zs_nh, ms = (nh + 7) / 8;
    const bool per = false;  // centred reflection z -> n - 1 - z on either kind of axis (fused_init)
    ZSArgs z{};
    z.out = out;
    z.V = st->d_img_zzs;
    z.n = n;
    z.nh = nh;
    z.Sh = (nh + 15) / 16;
    z.kk_last = tail_ksteps(nh);
    z.mir0 = per ? n - 15 : n - 16;
    z.mirc = per ? n : n - 1;
    z.zfix = per ? ((n % 2 == 0 && n >= 2) ? n / 2 : -1) : ((n % 2) ? (n - 1) / 2 : -1);
    z.inner = (int)inner;
    z.cpo = (int)((inner + 15) / 16);
    const long long chunks = (long long)z.cpo * nb;
    if (chunks >= (1LL << 31) - 64) return cudaErrorUnknown;  // see below: no fallback from here
    z.total_chunks = (unsigned)chunks;
    z.outer = nb;
    z.div_cpo = make_fastdiv((unsigned)z.cpo);
    CUtensorMap m0, m1;
    cudaError_t e;
    if ((e = get_map(st, in, inner, n, nb, 16, &m0)) != cudaSuccess) return e;
    if ((e = get_map(st, table, inner, n, 1, 16, &m1)) != cudaSuccess) return e;
    const int NT = ms <= 4 ? 4 : 2;
    const int CH = NT / 2;
    z.n_tiles = (unsigned)((chunks + CH - 1) / CH);
    if (z.n_tiles == 0) return cudaSuccess;
    switch (ms) {
      case 3: e = launch_zz_sym<3, 4, 8, 1>(p, m0, m1, z, s); break;
      case 4: e = launch_zz_sym<4, 4, 8, 1>(p, m0, m1, z, s); break;
      case 5: e = launch_zz_sym<5, 2, 12, 1>(p, m0, m1, z, s); break;
      case 6: e = launch_zz_sym<6, 2, 12, 1>(p, m0, m1, z, s); break;
      case 7: e = launch_zz_sym<7, 2, 12, 1>(p, m0, m1, z, s); break;
      default: e = launch_zz_sym<8, 2, 12, 1>(p, m0, m1, z, s); break;
    }
    if (e == cudaSuccess) ++p->tma_launches;
    // The table is in (even | odd) z-mode order (lam_s), the dense kernel below contracts with the ascending basis in
    // d_img_zz: a symmetric kernel that cannot run is a hard error, not a fallback.
    return e == cudaErrorNotSupported ? cudaErrorUnknown : e;
  }
  ZArgs a{};
  a.out = out;
  a.V = st->d_img_zz;
  a.n = n;
  a.S = (n + 15) / 16;
  a.kk_last = tail_ksteps(n);
  a.inner = (int)inner;
  a.cpo = (int)((inner + 15) / 16);
  const long long chunks = (long long)a.cpo * nb;
  if (chunks >= (1LL << 31) - 64) return cudaErrorNotSupported;
  a.total_chunks = (unsigned)chunks;
  a.outer = nb;
  a.div_cpo = make_fastdiv((unsigned)a.cpo);
  CUtensorMap m0, m1;
  cudaError_t e;
  if ((e = get_map(st, in, inner, n, nb, 16, &m0)) != cudaSuccess) return e;
  if ((e = get_map(st, table, inner, n, 1, 16, &m1)) != cudaSuccess) return e;
  const int NT = mtot <= 8 ? 4 : 2;
  const int CH = NT / 2;
  a.n_tiles = (unsigned)((chunks + CH - 1) / CH);
  if (a.n_tiles == 0) return cudaSuccess;
  ++p->tma_launches;
  switch (mtot) {
    case 2: return launch_zz<2, 4, 16, 2>(p, m0, m1, a, s);
    case 4: return launch_zz<4, 4, 16, 1>(p, m0, m1, a, s);
    case 6: return launch_zz<6, 4, 12, 1>(p, m0, m1, a, s);
    case 8: return launch_zz<8, 4, 8, 2>(p, m0, m1, a, s);
    case 12: return launch_zz<12, 2, 12, 3>(p, m0, m1, a, s);
    case 15: return launch_zz<15, 2, 12, 1>(p, m0, m1, a, s);
    default: return launch_zz<16, 2, 12, 1>(p, m0, m1, a, s);
  }
}

// FP64 operations one pair solve executes in the mode products when every buffer is TMA-addressable: 4 N n per dense
// axis (two products, a multiply-add = 2, padding not counted); a z axis on the reflection-adapted basis contracts
// nh even modes over nh points and n - nh odd modes over n - nh points per column and product, plus n butterfly
// additions per column and product.
// FP64 operations of ONE product along axis ax per pair solve with the plan's current settings.
double fused_executed_flops_axis(const exx_plan* p, int ax) {
  const TmaState* st = static_cast<const TmaState*>(p->tma_state);
  const bool sym = fused_sym_mode(p);
  const double n = p->n[ax];
  const int nh_ax = !sym ? 0 : ax == 2 ? st->zs_nh : ax == 1 ? st->ys_nh : ((p->fusion & 2) && st->d_mult_symx ? st->xs_nh : 0);
  if (!nh_ax) return 2.0 * (double)p->N * n;
  const double nh = nh_ax, no = n - nh;
  return 2.0 * (nh * nh + no * no) * (double)p->N / n + (double)p->N;
}

// pair_symmetric: one executed solve of exx_apply_symmetric, whose x-backward product runs twice (once per side of the
// two-sided accumulate) when the x axis is on the reflection-adapted basis.
double fused_executed_flops_per_solve(const exx_plan* p, bool pair_symmetric) {
  const TmaState* st = static_cast<const TmaState*>(p->tma_state);
  const bool sym = fused_sym_mode(p);
  double f = 0.0;
  for (int ax = 0; ax < 3; ++ax) {
    const double n = p->n[ax];
    const int nh_ax = !sym ? 0 : ax == 2 ? st->zs_nh : ax == 1 ? st->ys_nh : ((p->fusion & 2) && st->d_mult_symx ? st->xs_nh : 0);
    if (nh_ax) {
      const double nh = nh_ax, no = n - nh;
      const double one = 2.0 * (nh * nh + no * no) * (double)p->N / n + (double)p->N;
      f += (ax == 0 && pair_symmetric ? 3.0 : 2.0) * one;
    } else {
      f += 4.0 * (double)p->N * n;
    }
  }
  return f;
}

// Whether a batch whose buffers TMA can address runs in symmetric mode: the fused z pass on, bit 3 on, a capable axis,
// and (where the y images are in half-chunk row order) the half-chunk tiles on.
bool fused_sym_mode(const exx_plan* p) {
  const TmaState* st = static_cast<const TmaState*>(p->tma_state);
  if (!st || p->variant != EXX_VARIANT_FUSED_DMMA || (p->fusion & 9) != 9 || !st->d_mult_sym || !st->d_img_zz) return false;
  if (st->ys_nh && st->ys_hc && !(p->fusion & 4)) return false;
  return st->zs_nh || st->ys_nh || st->xs_nh;
}

// The same for nb complex functions ([nb][2][N] planes) of a Bloch plan whose z axis is complex with n <= 64, in place.
cudaError_t fused_zz_c(exx_plan* p, double* buf, int nb, cudaStream_t s) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st || !st->d_img_zz_c || !(p->fusion & 1)) return cudaErrorNotSupported;
  const int n = p->n[2], mh = mtot_class(n);
  if (!mh || mh > 8) return cudaErrorNotSupported;
  if ((p->n[0] & 1) || !aligned16(buf) || !aligned16(p->d_mult)) return cudaErrorNotSupported;
  const long long inner = (long long)p->n[0] * p->n[1];
  ZArgs a{};
  a.out = buf;
  a.V = st->d_img_zz_c;
  a.n = n;
  a.S = (n + 15) / 16;
  a.kk_last = tail_ksteps(n);
  a.inner = (int)inner;
  a.cpo = (int)((inner + 15) / 16);
  const long long chunks = (long long)a.cpo * nb;
  if (chunks >= (1LL << 31) - 64) return cudaErrorNotSupported;
  a.total_chunks = (unsigned)chunks;
  a.outer = 2 * nb;
  a.div_cpo = make_fastdiv((unsigned)a.cpo);
  CUtensorMap m0, m1;
  cudaError_t e;
  if ((e = get_map(st, buf, inner, n, 2LL * nb, 16, &m0)) != cudaSuccess) return e;
  if ((e = get_map(st, p->d_mult, inner, n, 1, 16, &m1)) != cudaSuccess) return e;
  const int NT = mh <= 4 ? 4 : 2;
  const int CH = NT / 2;
  a.n_tiles = (unsigned)((chunks + CH - 1) / CH);
  if (a.n_tiles == 0) return cudaSuccess;
  ++p->tma_launches;
  switch (mh) {
    case 2: return launch_zz_c<4, 4, 16, 1>(p, m0, m1, a, s);
    case 4: return launch_zz_c<8, 4, 8, 2>(p, m0, m1, a, s);
    case 6: return launch_zz_c<12, 2, 12, 3>(p, m0, m1, a, s);
    default: return launch_zz_c<16, 2, 12, 1>(p, m0, m1, a, s);
  }
}

// x-backward product of the batch in `in` (nb = nj*nk right-hand sides, pair (j0 + b % nj, k0 + b / nj)) fused with the
// accumulate into vx.  cudaErrorNotSupported: the caller runs k_mode_t and k_accumulate instead.
cudaError_t fused_xacc(exx_plan* p, const double* in, int nb, const FastArgs* fa, cudaStream_t s) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st || !(p->fusion & 2) || !fa || fa->sym) return cudaErrorNotSupported;
  const int n = p->n[0], mtot = mtot_class(n);
  if (!mtot || !st->d_img[0][1]) return cudaErrorNotSupported;
  if ((n & 1) || !aligned16(in) || !aligned16(fa->psi) || !aligned16(fa->vx)) return cudaErrorNotSupported;
  if (nb != fa->bd.nj * fa->bd.nk) return cudaErrorInvalidValue;
  const int NT = xacc_nt(mtot);
  XArgs a{};
  a.V = st->d_img[0][1];
  a.occ = fa->occ + fa->bd.j0;
  a.vx = fa->vx + (size_t)fa->bd.k0 * (size_t)p->N;
  a.n = n;
  a.S = (n + 15) / 16;
  a.kk_last = tail_ksteps(n);
  a.rows_per_rhs = (int)(p->N / n);
  a.nj = fa->bd.nj;
  a.nk = fa->bd.nk;
  a.j0 = fa->bd.j0;
  a.first = fa->first ? 1 : 0;
  a.div_nk = make_fastdiv((unsigned)a.nk);
  const long long rows_total = (long long)a.rows_per_rhs * nb, rows_psi = (long long)a.rows_per_rhs * fa->n_occ;
  if (rows_total >= (1LL << 31) - 64 || rows_psi >= (1LL << 31) - 64) return cudaErrorNotSupported;
  const long long tiles_per_rhs = (a.rows_per_rhs + 8 * NT - 1) / (8 * NT);
  if (tiles_per_rhs * a.nk >= (1LL << 31) - 64) return cudaErrorNotSupported;
  a.n_tiles = (unsigned)(tiles_per_rhs * a.nk);
  if (a.n_tiles == 0) return cudaSuccess;
  CUtensorMap m0, m1;
  cudaError_t e;
  if ((e = get_map(st, in, n, rows_total, 0, 8 * NT, &m0)) != cudaSuccess) return e;
  if ((e = get_map(st, fa->psi, n, rows_psi, 0, 8 * NT, &m1)) != cudaSuccess) return e;
  ++p->tma_launches;
  switch (mtot) {
    case 2: return launch_xacc<2, 2, 16>(p, m0, m1, a, s);
    case 4: return launch_xacc<4, 2, 16>(p, m0, m1, a, s);
    case 6: return launch_xacc<6, 2, 12>(p, m0, m1, a, s);
    case 8: return launch_xacc<8, 2, 12>(p, m0, m1, a, s);
    case 12: return launch_xacc<12, 1, 12>(p, m0, m1, a, s);
    case 15: return launch_xacc<15, 1, 12>(p, m0, m1, a, s);
    default: return launch_xacc<16, 1, 12>(p, m0, m1, a, s);
  }
}

}  // namespace exx
