// Default variant (EXX_VARIANT_FUSED_DMMA): mode products on the FP64 tensor pipe, operands staged by TMA.
//
// Every mode product of Eq. 11 is "a small stationary matrix times a very wide one":
// out[:, c] = M in[:, c], M = V^T (forward) or V (backward), n x n with n <= 128, c running over N*n_c/n
// columns.  What the measurements of the first-generation kernel (kernels_dmma.cu, profiles/
// r1_cfg2_cpasync_ncu.md) say bounds it: not the DMMA pipe but everything around it -- per-lane 8-byte
// LDGSTS copies (8 L1 wavefronts per 256 B), their 64-bit address arithmetic (5 other instructions per
// DMMA), and only two warps per scheduler to hide it.  This kernel removes that work from the SM's issue
// slots instead of tuning it:
//   * The streamed operand arrives by TMA (cp.async.bulk.tensor, SASS UTMALDG): one elected lane per warp
//     issues one or two box copies per 16 contraction indices; hardware computes the addresses, clips
//     ragged edges (out-of-bounds elements arrive as zeros) and signals an mbarrier.  No LSU wavefronts,
//     no per-lane pointers, no predicates.
//   * Boxes are 16 doubles (128 B) wide and land with the hardware 128-byte swizzle, so the B-fragment
//     reads are bank-conflict free without padding.  The order of the contraction index inside a block of
//     16 is free (it is a sum), so the k <-> lane assignment is chosen to fit the swizzle and the rows of the
//     plan's shared-memory image of V are permuted to match (tma_init).  Forward/backward and the axis only
//     change that image: the kernel has no FWD/BWD variants.
//   * Warps stay fully independent (a warp owns 8*NT columns for all n output rows; its accumulators never
//     leave registers): each warp runs its own two-stage mbarrier pipeline, there is no block barrier in
//     the steady state.  With the address work gone the kernel fits 12-16 warps per SM (3-4 per scheduler)
//     instead of 8, which is what keeps the DMMA pipe fed while a warp waits, stores or sets up a tile.
//   * Fused into the passes as before: the pair density psi_j*tgt_k (a1) as a second TMA stream of the first
//     product, the multiplier f(Lambda~) (a3) as a second stream of the z-backward product.
//
// L-mode (axis y or z; contracted index strided by `inner`): the operand is the 3-D tensor
// [outer][n][inner]; a warp tile is NT/2 chunks of 16 consecutive inner-columns, a stage is a
// {16 cols, 16 rows} box per chunk.  X-mode (axis x; contracted index contiguous): the transposed product
// out^T = M in^T, the operand is the 2-D tensor [rows][n]; a warp tile is 8*NT rows, a stage is a
// {16 x, 8*NT rows} box.
//
// The paper's four data reorganisations (Eqs. 12-15) do not exist here: they are
// artefacts of calling a 2-D GEMM library and are replaced by tensor-map strides.
#include "tma_common.cuh"

namespace exx {
namespace {

struct TArgs {
  double* out;
  const double* V;  // permuted, zero-padded image [16*S][8*MTOT+4] (tma_init)
  int n;
  int S;        // stages per tile = ceil(n/16); CPLX: per plane (a tile is 2 S stages, re plane then im plane)
  int kk_last;  // 0: n is a multiple of 16; else ceil((n % 16) / 4), the k-steps of the ragged last stage
  unsigned n_tiles;
  // L-mode
  int inner;              // contiguous run below the contracted axis
  int cpo;                // chunks of 16 columns per outer index = ceil(inner/16)
  unsigned total_chunks;  // cpo * outer
  int outer;
  FastDiv div_cpo;
  // X-mode
  int rows_per_rhs;   // N / nx
  int tiles_per_rhs;  // pair density only: ceil(rows_per_rhs / (8*NT))
  int rows_total;     // rows of the output tensor
  FastDiv div_tiles;
  FastDiv div_nj;  // pair density only
  int exact;       // no ragged edge in this launch: the epilogue stores without predicates
  BatchDesc bd;    // pair density only
  // Complex (Bloch) products, second launch: the result Q = Mi [in_re | in_im] is not stored but added into the first
  // launch's output P with the planes swapped, out_re = P_re - Q_im, out_im = P_im + Q_re (planes alternate re, im;
  // plane_stride = N doubles).  per_plane: rows (X-mode) / outer indices (L-mode) of one plane.
  // Complex (Bloch) products, single launch (CPLX): a function is a (re, im) pair of planes and the product is the real
  // embedding [[Mr, -Mi], [Mi, Mr]] of M: contraction over 2 S stages, output row tiles 0..MTOT/2-1 go to the re plane,
  // the rest to the im plane.  plane_rows: rows (X-mode) / plane_outer: outer indices (L-mode) between the two planes.
  int plane_rows;
  int plane_outer;
  int hc;  // L-mode plain pass on 8-column half-chunks (template flag HC): cpo / total_chunks count half-chunks
  int rmw;
  long long plane_stride;
  FastDiv div_plane;
};

// MTOT = ceil(n/8) rounded up to a supported class, NT = column tiles (of 8) per warp.
// HC (L-mode, plain pass only): a tile is NT half-chunks of 8 columns (boxes of 8 x 16, 64-byte rows) instead of NT/2
// chunks of 16, for an inner extent that is 8 (mod 16): the y pass at nx = 120 then runs 15 half-chunks per row
// instead of 8 chunks, the last of them half empty (6.7 % of the pass).
template <int MTOT, int NT, bool XMODE, bool TWO, int WARPS, int MINB, bool RMW = false, bool CPLX = false, bool HC = false>
__global__ void __launch_bounds__(32 * WARPS, MINB)
    k_mode_t(const __grid_constant__ CUtensorMap tm0, const __grid_constant__ CUtensorMap tm1, const TArgs a) {
  static_assert(NT == 2 || NT == 4, "a tile is one or two 16-column chunks");
  static_assert(!CPLX || (!TWO && !RMW && MTOT % 2 == 0), "the embedded complex product is a plain one-stream pass");
  static_assert(!HC || (!XMODE && !TWO && !RMW && !CPLX), "half-chunk tiles: plain real L-mode pass only");
  constexpr int MH = CPLX ? MTOT / 2 : MTOT;  // row tiles per plane
  constexpr int LDV = 8 * MTOT + 4;  // == 4 (mod 8): the A-fragment reads are bank-conflict free
  constexpr int NS = TWO ? 2 : 1;    // two streams are staged separately and multiplied on consumption
  constexpr unsigned kStage = 1024u * NT;  // bytes per stage and stream: 16 x (8*NT) doubles
  constexpr int CH = HC ? NT : NT / 2;     // L-mode: 16-column chunks (HC: 8-column half-chunks) per tile
  constexpr int CW = HC ? 8 : 16;          // columns per chunk
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  const int tid = threadIdx.x, lane = tid & 31;
  // warp index through a shuffle: the compiler then knows it is warp-uniform and keeps everything derived
  // from it (ring and barrier addresses, tile counters) in uniform registers
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int g = lane >> 2, q = lane & 3;
  const int n = a.n, S = a.S;
  const int S2 = CPLX ? 2 * S : S;  // stages per tile
  const unsigned smem0 = (unsigned)__cvta_generic_to_shared(smem_raw);
  const unsigned img_bytes = 8u * (16u * S2) * LDV;

  // ---- stage the V image once per CTA (one burst of 16-byte asynchronous copies) -------------------------
  for (unsigned i = 2 * tid; i < 16u * S2 * LDV; i += 2 * 32 * WARPS)
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(smem0 + 8u * i), "l"(a.V + i) : "memory");
  asm volatile("cp.async.commit_group;\n" ::: "memory");

  const unsigned ring0 = (smem0 + img_bytes + 1023u) & ~1023u;  // swizzled boxes need 1024-byte alignment
  const unsigned my_ring = ring0 + warp * (kDepth * NS * kStage);
  const unsigned my_bar = ring0 + WARPS * (kDepth * NS * kStage) + warp * (kDepth * 8u);
  // CTA-wide tile counter (dynamic tile claiming, below): local tile indices 0..WARPS-1 are pre-assigned
  const unsigned ctr_addr = ring0 + WARPS * (kDepth * NS * kStage) + WARPS * (kDepth * 8u);
  if (tid == 0) asm volatile("st.shared.u32 [%0], %1;\n" ::"r"(ctr_addr), "r"((unsigned)WARPS) : "memory");
  if (lane == 0) {
#pragma unroll
    for (int d = 0; d < kDepth; ++d) mbar_init(my_bar + 8u * d, 1u);
    asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory");
  }
  __syncthreads();  // barriers and tile counter initialised (the V image is still in flight)
  // Programmatic dependent launch: everything above touched only plan constants, so it overlaps the tail
  // of the previous pass; from here on we read that pass's output.
  asm volatile("griddepcontrol.launch_dependents;\n" ::: "memory");
  asm volatile("griddepcontrol.wait;\n" ::: "memory");

  // Tiles b, b + grid, b + 2 grid, ... belong to CTA b (static, equal shares); inside the CTA the warps claim
  // them one at a time from a shared counter, so no warp idles while the CTA still has tiles, however unevenly
  // the schedulers share the DMMA pipe (measured: neutral against a static split on the five configs).
  const unsigned tfirst = blockIdx.x + gridDim.x * warp;
  auto claim_tile = [&]() -> unsigned {  // whole warp; returns the same tile id in every lane
    unsigned i = 0;
    if (lane == 0) asm volatile("atom.shared.add.u32 %0, [%1], 1;\n" : "=r"(i) : "r"(ctr_addr) : "memory");
    i = __shfl_sync(0xffffffffu, i, 0);
    const unsigned long long t = (unsigned long long)blockIdx.x + (unsigned long long)gridDim.x * i;
    return t < a.n_tiles ? (unsigned)t : 0xffffffffu;
  };
  // tiles the producer has claimed and the consumer has not started yet (the producer runs at most kDepth
  // stages, i.e. at most kDepth tiles, ahead)
  unsigned fifo[kDepth + 1];
  int fifo_n = 0;

  // ---- producer: warp-uniform bookkeeping, one elected lane issues the copies; runs kDepth stages ahead,
  //      straight across tile boundaries ----------------------------------------------------------------
  unsigned t_p = tfirst;
  int s_p = 0;
  int pc0[CH], pc2[CH];  // L-mode: column and outer coordinate of each chunk
  int pr0 = 0, pr1 = 0;  // X-mode: first row in tm0 / tm1
  auto tile_coords = [&](unsigned t) {
    if (XMODE) {
      if (TWO) {
        const int rhs = (int)fast_div(t, a.div_tiles);
        const int rb = (int)t - rhs * a.tiles_per_rhs;
        const int kq = (int)fast_div((unsigned)rhs, a.div_nj);
        const int j = a.bd.j0 + (rhs - kq * a.bd.nj), k = a.bd.k0 + kq;
        pr0 = j * a.rows_per_rhs + rb * (8 * NT);
        pr1 = k * a.rows_per_rhs + rb * (8 * NT);
      } else if (CPLX) {
        const int fn = (int)fast_div(t, a.div_tiles);
        const int rb = (int)t - fn * a.tiles_per_rhs;
        pr0 = 2 * fn * a.rows_per_rhs + rb * (8 * NT);
      } else {
        pr0 = (int)t * (8 * NT);
      }
    } else {
#pragma unroll
      for (int ch = 0; ch < CH; ++ch) {
        const unsigned cc = t * CH + ch;
        if (cc < a.total_chunks) {
          const unsigned o = fast_div(cc, a.div_cpo);
          // CPLX: o counts the outer indices of the re planes only; the re plane of function b starts 2 b planes in
          pc2[ch] = CPLX ? (int)(o + fast_div(o, a.div_plane) * (unsigned)a.plane_outer) : (int)o;
          pc0[ch] = CW * (int)(cc - o * (unsigned)a.cpo);
        } else {  // past the end: an all-out-of-bounds box (zeros), never stored
          pc2[ch] = a.outer;
          pc0[ch] = 0;
        }
      }
    }
  };
  auto produce = [&](int slot) {  // called by the whole (converged) warp
    if (t_p >= a.n_tiles) return;
    const unsigned bar = my_bar + 8u * slot;
    const unsigned dst = my_ring + slot * (NS * kStage);
    if (elect_one()) {
      mbar_expect_tx(bar, NS * kStage);
      const bool im = CPLX && s_p >= S;  // second half of a complex tile: the im plane
      const int sl = im ? s_p - S : s_p;
      if (XMODE) {
        tma_load_2d(dst, &tm0, 16 * sl, pr0 + (im ? a.plane_rows : 0), bar);
        if (TWO) tma_load_2d(dst + kStage, &tm1, 16 * sl, pr1, bar);
      } else {
#pragma unroll
        for (int ch = 0; ch < CH; ++ch) {
          tma_load_3d(dst + (HC ? 1024u : 2048u) * ch, &tm0, pc0[ch], 16 * sl, pc2[ch] + (im ? a.plane_outer : 0), bar);
          if (TWO) tma_load_3d(dst + kStage + 2048u * ch, &tm1, pc0[ch], 16 * sl, 0, bar);
        }
      }
    }
    if (++s_p == S2) {
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
  // the V image has been landing behind the dependency wait and the first data copies
  asm volatile("cp.async.wait_group 0;\n" ::: "memory");
  __syncthreads();

  // ---- per-lane fragment addresses --------------------------------------------------------------------
  // A fragment (M[m][k]) of (stage s, k-step kk, row tile mt): image row 16s + 4kk + q, column 8mt + g.
  unsigned a_lane_v = smem0 + 8u * (q * LDV + g);
  // B fragment of (k-step kk, column tile nt) inside a stage, 128-byte swizzle (16-byte chunk index XOR row%8):
  //   X-mode: box row 8nt+g (a data row), x = (q&1) + 8(q>>1) + 2kk      -> xo[kk] + 1024 nt
  //   L-mode: box row 2q + (kk&1) + 8(kk>>1) (a contraction index), column 8(nt&1)+g of chunk nt>>1
  //                                                                       -> xo[2(nt&1) + (kk&1)] + 2048 (nt>>1) + 1024 (kk>>1)
  unsigned xo[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    if (XMODE) {
      xo[i] = 128u * g + 16u * ((4u * (q >> 1) + i) ^ (unsigned)g) + 8u * (q & 1);
    } else if (HC) {
      // box of 8 columns x 16 rows, 64-byte rows, 64-byte swizzle (16-byte chunk index XOR (row >> 1) & 3): k-step i
      // reads box row r = (q&1) + 4(q>>1) + 2(i&1) + 8(i>>1), column g (conflict-free: the 16-byte positions
      // 4 (r&1) + ((g>>1) ^ ((r>>1)&3)) of a half-warp are all distinct for rows {0,1,4,5} + 2(i&1))
      const unsigned r = (q & 1) + 4u * (q >> 1) + 2u * (i & 1) + 8u * (i >> 1);
      xo[i] = 64u * r + 16u * ((g >> 1) ^ ((r >> 1) & 3u)) + 8u * (g & 1);
    } else {
      const unsigned row = 2u * q + (i & 1);
      xo[i] = 128u * row + 16u * ((4u * (i >> 1) + (g >> 1)) ^ row) + 8u * (g & 1);
    }
  }

  int slot = 0;
  unsigned parity = 0;
  unsigned t = tfirst;
  while (t < a.n_tiles) {
    double acc[MTOT][NT][2];
#pragma unroll
    for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
      for (int nt = 0; nt < NT; ++nt) acc[mt][nt][0] = acc[mt][nt][1] = 0.0;

    for (int s = 0; s < S2; ++s) {
      // opaque uses: keep the per-lane fragment offsets in registers (at the register cap the compiler
      // otherwise rebuilds them from %tid in every k-step, ~20 instructions ahead of the first LDS)
      asm volatile("" : "+r"(a_lane_v), "+r"(xo[0]), "+r"(xo[1]), "+r"(xo[2]), "+r"(xo[3]));
      mbar_wait(my_bar + 8u * slot, parity);
      const unsigned sb = my_ring + slot * (NS * kStage);
      const unsigned aa = a_lane_v + (unsigned)s * (16u * LDV * 8u);
      const bool ragged = a.kk_last && (s == S - 1 || (CPLX && s == S2 - 1));  // last stage of a plane, n % 16 != 0
      if (!ragged) {
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          double bf[NT];
#pragma unroll
          for (int nt = 0; nt < NT; ++nt) {
            const unsigned off = (XMODE || HC) ? (sb + xo[kk] + 1024u * nt)
                                               : (sb + xo[2 * (nt & 1) + (kk & 1)] + 2048u * (nt >> 1) + 1024u * (kk >> 1));
            bf[nt] = lds64(off);
            if (TWO) bf[nt] *= lds64(off + kStage);
          }
          double af[MTOT];
#pragma unroll
          for (int mt = 0; mt < MTOT; ++mt) af[mt] = lds64(aa + (4u * kk * LDV + 8u * mt) * 8u);
#pragma unroll
          for (int mt = 0; mt < MTOT; ++mt)
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) dmma884(acc[mt][nt], af[mt], bf[nt]);
        }
      } else {
        // ragged last stage (n % 16 != 0): contraction index 4 kk + q in k-step kk, so that ceil(rem / 4) k-steps
        // cover the rem valid indices (60 -> 3 instead of 4, X-mode 120 -> 2 instead of 4); tma_init lays the
        // image rows of this stage out in the same order
#pragma unroll
        for (int kk = 0; kk < 4; ++kk) {
          if (kk < a.kk_last) {
            double bf[NT];
#pragma unroll
            for (int nt = 0; nt < NT; ++nt) {
              unsigned off;
              if (XMODE) {
                off = sb + 1024u * nt + 128u * g + 16u * ((2u * kk + (q >> 1)) ^ (unsigned)g) + 8u * (q & 1);
              } else if (HC) {
                const unsigned r = 4u * kk + q;
                off = sb + 1024u * nt + 64u * r + 16u * ((g >> 1) ^ ((r >> 1) & 3u)) + 8u * (g & 1);
              } else {
                const unsigned row = 4u * kk + q;
                off = sb + 2048u * (nt >> 1) + 128u * row + 16u * ((4u * (nt & 1) + (g >> 1)) ^ (row & 7u)) + 8u * (g & 1);
              }
              bf[nt] = lds64(off);
              if (TWO) bf[nt] *= lds64(off + kStage);
            }
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
      // every lane's reads of this stage have completed (their values fed the DMMAs above): refill it
      __syncwarp();
      produce(slot);
      if (++slot == kDepth) {
        slot = 0;
        parity ^= 1u;
      }
    }

    // ---- epilogue: C[m = 8mt+g][column 8nt + 2q + e] straight from the fragments (every pass is in place).
    //      a.exact: no ragged edge anywhere in this launch -> no per-store predicates ------------------------
    if (XMODE) {
      int row0, limit;
      if (TWO) {
        const int rhs = (int)fast_div(t, a.div_tiles);
        const int rb = (int)t - rhs * a.tiles_per_rhs;
        row0 = rhs * a.rows_per_rhs + rb * (8 * NT);
        limit = (rhs + 1) * a.rows_per_rhs;
      } else if (CPLX) {  // rows of the re plane of function fn; the im plane lies plane_rows rows further
        const int fn = (int)fast_div(t, a.div_tiles);
        const int rb = (int)t - fn * a.tiles_per_rhs;
        row0 = 2 * fn * a.rows_per_rhs + rb * (8 * NT);
        limit = (2 * fn + 1) * a.rows_per_rhs;
      } else {
        row0 = (int)t * (8 * NT);
        limit = a.rows_total;
      }
      double* base = a.out + ((long long)(row0 + 2 * q) * n + g);
      // CPLX: row tile mt >= MH is row tile mt - MH of the im plane
      const long long xim = CPLX ? (long long)a.plane_rows * n - 8 * MH : 0;
      if (RMW) {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            const int r = row0 + 8 * nt + 2 * q + e;
            if (r < limit) {
              const bool odd = fast_div((unsigned)r, a.div_plane) & 1u;  // this row belongs to an imaginary plane
              const double sgn = odd ? -1.0 : 1.0;
              double* dst = base + (long long)(8 * nt + e) * n + (odd ? -a.plane_stride : a.plane_stride);
#pragma unroll
              for (int m0 = 0; m0 < MTOT; m0 += 4) {
                double old[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                  if (m0 + u < MTOT && 8 * (m0 + u) + g < n) old[u] = dst[8 * (m0 + u)];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                  if (m0 + u < MTOT && 8 * (m0 + u) + g < n) dst[8 * (m0 + u)] = fma(sgn, acc[m0 + u][nt][e], old[u]);
              }
            }
          }
      } else if (a.exact) {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            double* dst = base + (long long)(8 * nt + e) * n;
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt) dst[8 * mt + (mt >= MH ? xim : 0)] = acc[mt][nt][e];
          }
      } else {
#pragma unroll
        for (int nt = 0; nt < NT; ++nt)
#pragma unroll
          for (int e = 0; e < 2; ++e) {
            if (row0 + 8 * nt + 2 * q + e < limit) {
              double* dst = base + (long long)(8 * nt + e) * n;
#pragma unroll
              for (int mt = 0; mt < MTOT; ++mt)
                if (8 * (mt >= MH ? mt - MH : mt) + g < n) dst[8 * mt + (mt >= MH ? xim : 0)] = acc[mt][nt][e];
            }
          }
      }
    } else if (HC) {
      const long long mstep = 8LL * a.inner;
#pragma unroll
      for (int ch = 0; ch < NT; ++ch) {  // column tile nt = half-chunk ch
        const unsigned cc = t * NT + ch;
        if (cc < a.total_chunks) {
          const unsigned o = fast_div(cc, a.div_cpo);
          const int col0 = 8 * (int)(cc - o * (unsigned)a.cpo) + 2 * q;
          double* ptr = a.out + ((long long)o * n + g) * a.inner + col0;
          const bool in0 = col0 < a.inner;  // inner is even: the pair (c, c+1) is inside or outside together
#pragma unroll
          for (int mt = 0; mt < MTOT; ++mt) {
            if (in0 && 8 * mt + g < n) stg_v2(ptr, acc[mt][ch][0], acc[mt][ch][1]);
            ptr += mstep;
          }
        }
      }
    } else {
      const long long mstep = 8LL * a.inner;  // doubles between consecutive row tiles
#pragma unroll
      for (int ch = 0; ch < CH; ++ch) {
        const unsigned cc = t * CH + ch;
        if (cc < a.total_chunks) {
          const unsigned o_t = fast_div(cc, a.div_cpo);
          const int col0 = 16 * (int)(cc - o_t * (unsigned)a.cpo) + 2 * q;
          const unsigned o = CPLX ? o_t + fast_div(o_t, a.div_plane) * (unsigned)a.plane_outer : o_t;
          double* ptr = a.out + ((long long)o * n + g) * a.inner + col0;
          // CPLX: row tile mt >= MH is row tile mt - MH of the im plane, plane_outer outer indices further
          const long long lim = CPLX ? ((long long)a.plane_outer * n - 8 * MH) * a.inner : 0;
          if (RMW) {
            const bool odd = fast_div(o, a.div_plane) & 1u;
            const double sgn = odd ? -1.0 : 1.0;
            double* pr = ptr + (odd ? -a.plane_stride : a.plane_stride);
            const bool in0 = col0 < a.inner, in1 = col0 + 8 < a.inner;
#pragma unroll
            for (int m0 = 0; m0 < MTOT; m0 += 2) {
              double2 o0[2], o1[2];
#pragma unroll
              for (int u = 0; u < 2; ++u)
                if (m0 + u < MTOT && 8 * (m0 + u) + g < n) {
                  if (in0) o0[u] = *reinterpret_cast<const double2*>(pr + u * mstep);
                  if (in1) o1[u] = *reinterpret_cast<const double2*>(pr + u * mstep + 8);
                }
#pragma unroll
              for (int u = 0; u < 2; ++u)
                if (m0 + u < MTOT && 8 * (m0 + u) + g < n) {
                  if (in0) stg_v2(pr + u * mstep, fma(sgn, acc[m0 + u][2 * ch][0], o0[u].x), fma(sgn, acc[m0 + u][2 * ch][1], o0[u].y));
                  if (in1) stg_v2(pr + u * mstep + 8, fma(sgn, acc[m0 + u][2 * ch + 1][0], o1[u].x), fma(sgn, acc[m0 + u][2 * ch + 1][1], o1[u].y));
                }
              pr += 2 * mstep;
            }
          } else if (a.exact) {
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt) {
              if (CPLX && mt == MH) ptr += lim;
              stg_v2(ptr, acc[mt][2 * ch][0], acc[mt][2 * ch][1]);
              stg_v2(ptr + 8, acc[mt][2 * ch + 1][0], acc[mt][2 * ch + 1][1]);
              ptr += mstep;
            }
          } else {
            // inner is even, so the pair (c, c+1) is inside or outside together
            const bool in0 = col0 < a.inner, in1 = col0 + 8 < a.inner;
#pragma unroll
            for (int mt = 0; mt < MTOT; ++mt) {
              if (CPLX && mt == MH) ptr += lim;
              if (8 * (mt >= MH ? mt - MH : mt) + g < n) {
                if (in0) stg_v2(ptr, acc[mt][2 * ch][0], acc[mt][2 * ch][1]);
                if (in1) stg_v2(ptr + 8, acc[mt][2 * ch + 1][0], acc[mt][2 * ch + 1][1]);
              }
              ptr += mstep;
            }
          }
        }
      }
    }
    // next tile: the oldest one the producer has claimed (it always has: it claimed the successor when it
    // issued this tile's last stage)
    t = fifo[0];
#pragma unroll
    for (int i = 0; i < kDepth; ++i) fifo[i] = fifo[i + 1];
    --fifo_n;
  }
}

// ---- host side ----------------------------------------------------------------------------------------

// supported classes of ceil(n/8); per class the columns-per-warp choice (NT), the warps per CTA and the CTAs
// per SM, for the plain and for the two-stream (TWO) kernels.
//   lanes == 1: one persistent CTA per SM, as many warps as the register file allows.
//   lanes == 2 (exx_apply runs two batches at a time on two streams): where the V image is small enough
//     (n <= 64) a CTA takes half an SM (8 warps, <= 128 registers, <= 113 KB) so that kernels of the two lanes
//     are co-resident and each fills the other's launch gaps, ramps, tails and epilogues; larger axes keep
//     one CTA per SM and leave a few thousand registers free for the other lane's accumulate kernel.
struct ClassCfg {
  int mtot;
  int nt, warps, minb;
  int nt_two, warps_two, minb_two;
};
inline bool pick_class(int n, int lanes, ClassCfg* c) {
  const int need = (n + 7) / 8;
  if (need > 16) return false;
  if (lanes == 2 && need <= 8) {
    const int m = need <= 2 ? 2 : need <= 4 ? 4 : need <= 6 ? 6 : 8;
    if (m == 8) *c = {8, 2, 8, 2, 2, 8, 2};
    else *c = {m, 4, 8, 2, 2, 8, 2};
    return true;
  }
  if (need <= 2) *c = {2, 4, 16, 1, 4, 12, 1};
  else if (need <= 4) *c = {4, 4, 16, 1, 4, 12, 1};
  else if (need <= 6) *c = {6, 4, 16, 1, 4, 12, 1};
  else if (need <= 8) *c = {8, 4, 12, 1, 4, 8, 1};
  else if (need <= 12) *c = {12, 2, 12, 1, 2, 12, 1};
  else if (need <= 15) *c = {15, 2, 12, 1, 2, 12, 1};
  else *c = {16, 2, 12, 1, 2, 8, 1};
  return true;
}

template <int MTOT, int NT, bool XMODE, bool TWO, int WARPS, int MINB, bool RMW = false, bool CPLX = false, bool HC = false>
cudaError_t launch_one(const CUtensorMap& m0, const CUtensorMap& m1, const TArgs& a, int sm_count, int device,
                       cudaStream_t s) {
  constexpr int LDV = 8 * MTOT + 4;
  const size_t img = sizeof(double) * 16 * (size_t)a.S * (CPLX ? 2 : 1) * LDV;
  // image | (alignment slack) | rings | mbarriers.  The request is padded so that exactly MINB CTAs fit an SM
  // (above 1/(MINB+1) of its shared memory): the tile split assumes one CTA of this launch per SM.
  size_t smem = img + 1024 + (size_t)WARPS * kDepth * (TWO ? 2 : 1) * 1024 * NT + (size_t)WARPS * kDepth * 8 + 16;
  const size_t floor_bytes = MINB == 1 ? 117 * 1024 : 77 * 1024;
  if (MINB == 2 && smem > 113 * 1024) return cudaErrorInvalidConfiguration;
  if (smem < floor_bytes) smem = floor_bytes;
  auto kern = k_mode_t<MTOT, NT, XMODE, TWO, WARPS, MINB, RMW, CPLX, HC>;
  // always the largest shared-memory carveout: kernels of the two lanes must agree on the SM's L1/shared
  // split to be resident together (and a switch between launches drains the SM)
  static SmemOptIn opt;  // per instantiation and device
  {
    cudaError_t e = opt.ensure(kern, device, smem, true);
    if (e != cudaSuccess) return e;
  }
  cudaLaunchConfig_t cfg = {};
  const unsigned grid = a.n_tiles < (unsigned)sm_count ? a.n_tiles : (unsigned)sm_count;
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(32 * WARPS);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  // Half-SM kernels (MINB == 2) are launched without programmatic serialization: an early-launched successor
  // would sit in griddepcontrol.wait in the very slot the other lane's kernel is meant to use.
  cfg.numAttrs = MINB == 1 ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, m0, m1, a);
}

template <int MTOT, int NT, int WARPS, int MINB, int NT2, int WARPS2, int MINB2>
cudaError_t launch_class(bool xmode, bool two, const CUtensorMap& m0, const CUtensorMap& m1, const TArgs& a,
                         int sm_count, int device, cudaStream_t s) {
  if (xmode) {
    if (two) return launch_one<MTOT, NT2, true, true, WARPS2, MINB2>(m0, m1, a, sm_count, device, s);
    if (a.rmw) return launch_one<MTOT, NT, true, false, WARPS, MINB, true>(m0, m1, a, sm_count, device, s);
    return launch_one<MTOT, NT, true, false, WARPS, MINB>(m0, m1, a, sm_count, device, s);
  }
  if (two) return launch_one<MTOT, NT2, false, true, WARPS2, MINB2>(m0, m1, a, sm_count, device, s);
  if (a.rmw) return launch_one<MTOT, NT, false, false, WARPS, MINB, true>(m0, m1, a, sm_count, device, s);
  if (a.hc) return launch_one<MTOT, NT, false, false, WARPS, MINB, false, false, true>(m0, m1, a, sm_count, device, s);
  return launch_one<MTOT, NT, false, false, WARPS, MINB>(m0, m1, a, sm_count, device, s);
}

}  // namespace

// One mode product along `axis` for nb right-hand sides; in == out is allowed (and is the normal case).
// pd != nullptr (axis 0, forward only): the input is psi_j .* tgt_k formed on the fly (a1).
// apply_mult (axis 2, backward only): the input is multiplied by f(Lambda~) while it is consumed (a3).
// cudaErrorNotSupported: sizes or alignment outside what TMA can address (odd nx, n > 128, unaligned
// buffers, no driver entry point); the caller then uses the cp.async kernels of kernels_dmma.cu.
cudaError_t tma_mode_product(exx_plan* p, int axis, bool forward, const double* in, double* out, int nb,
                             bool apply_mult, const FastArgs* pd, cudaStream_t s, int part, bool rmw) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st) return cudaErrorNotSupported;
  const int n = p->n[axis];
  ClassCfg cc;
  if (!pick_class(n, p->lanes, &cc)) return cudaErrorNotSupported;
  const double* img = part ? st->d_img_im[axis][forward ? 0 : 1] : st->d_img[axis][forward ? 0 : 1];
  if (!img) return cudaErrorNotSupported;
  if ((p->n[0] & 1) || !aligned16(out) || (in && !aligned16(in))) return cudaErrorNotSupported;
  const bool xmode = axis == 0;
  if (pd && !(xmode && forward)) return cudaErrorInvalidValue;
  if (apply_mult && !(axis == 2 && !forward)) return cudaErrorInvalidValue;
  if (pd && (!aligned16(pd->psi) || !aligned16(pd->tgt))) return cudaErrorNotSupported;
  const bool two = pd != nullptr || apply_mult;
  const int NT = two ? cc.nt_two : cc.nt;

  TArgs a{};
  a.out = out;
  a.V = img;
  a.n = n;
  a.S = (n + 15) / 16;
  CUtensorMap m0, m1;
  cudaError_t e;
  if (xmode) {
    a.kk_last = tail_ksteps(n);
    a.rows_per_rhs = (int)(p->N / n);
    const long long rows_total = (long long)a.rows_per_rhs * nb;
    if (rows_total >= (1LL << 31) - 64) return cudaErrorNotSupported;
    a.rows_total = (int)rows_total;
    a.tiles_per_rhs = (a.rows_per_rhs + 8 * NT - 1) / (8 * NT);
    a.div_tiles = make_fastdiv((unsigned)a.tiles_per_rhs);
    a.exact = (n == 8 * cc.mtot) && ((pd ? a.rows_per_rhs : rows_total) % (8 * NT) == 0);
    if (pd) {
      a.bd = pd->bd;
      a.div_nj = make_fastdiv((unsigned)pd->bd.nj);
      a.n_tiles = (unsigned)a.tiles_per_rhs * (unsigned)nb;
      const long long rp = (long long)a.rows_per_rhs * pd->n_occ, rt = (long long)a.rows_per_rhs * pd->n_tgt;
      if (rp >= (1LL << 31) - 64 || rt >= (1LL << 31) - 64) return cudaErrorNotSupported;
      if ((e = get_map(st, pd->psi, n, rp, 0, 8 * NT, &m0)) != cudaSuccess) return e;
      if ((e = get_map(st, pd->tgt, n, rt, 0, 8 * NT, &m1)) != cudaSuccess) return e;
    } else {
      a.n_tiles = (unsigned)((rows_total + 8 * NT - 1) / (8 * NT));
      if ((e = get_map(st, in, n, rows_total, 0, 8 * NT, &m0)) != cudaSuccess) return e;
      m1 = m0;
    }
  } else {
    const long long inner = axis == 1 ? p->n[0] : (long long)p->n[0] * p->n[1];
    const long long outer = p->N / (n * inner) * nb;
    // half-chunk tiles where 16-column chunks would leave the last chunk of every row half empty
    const double* img_hc = st->d_img_hc[forward ? 0 : 1];
    const bool hc = axis == 1 && !two && !rmw && part == 0 && img_hc && inner % 16 == 8 && (p->fusion & 4);
    if (hc) {
      a.hc = 1;
      a.V = img_hc;
    }
    const int cw = hc ? 8 : 16;
    a.kk_last = tail_ksteps(n);
    a.inner = (int)inner;
    a.cpo = (int)((inner + cw - 1) / cw);
    const long long chunks = (long long)a.cpo * outer;
    if (chunks >= (1LL << 31) - 64) return cudaErrorNotSupported;
    a.total_chunks = (unsigned)chunks;
    a.outer = (int)outer;
    a.div_cpo = make_fastdiv((unsigned)a.cpo);
    a.exact = (n == 8 * cc.mtot) && (inner % 16 == 0);
    const int CH = hc ? NT : NT / 2;
    a.n_tiles = (unsigned)((chunks + CH - 1) / CH);
    if ((e = get_map(st, in, inner, n, outer, 16, &m0, cw)) != cudaSuccess) return e;
    if (apply_mult) {
      if ((e = get_map(st, p->d_mult, inner, n, 1, 16, &m1)) != cudaSuccess) return e;
    } else {
      m1 = m0;
    }
  }
  if (rmw) {  // only the plain (one-stream) kernels have the read-modify-write epilogue; planes come in (re, im) pairs
    if (two || (nb & 1)) return cudaErrorInvalidValue;
    a.rmw = 1;
    a.plane_stride = p->N;
    a.div_plane = make_fastdiv((unsigned)(xmode ? a.rows_per_rhs : (int)(p->N / ((long long)n * a.inner))));
  }
  if (a.n_tiles == 0) return cudaSuccess;
  ++p->tma_launches;
  if (cc.minb == 2) {
    switch (cc.mtot) {
      case 2: return launch_class<2, 4, 8, 2, 2, 8, 2>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
      case 4: return launch_class<4, 4, 8, 2, 2, 8, 2>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
      case 6: return launch_class<6, 4, 8, 2, 2, 8, 2>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
      default: return launch_class<8, 2, 8, 2, 2, 8, 2>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
    }
  }
  switch (cc.mtot) {
    case 2: return launch_class<2, 4, 16, 1, 4, 12, 1>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
    case 4: return launch_class<4, 4, 16, 1, 4, 12, 1>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
    case 6: return launch_class<6, 4, 16, 1, 4, 12, 1>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
    case 8: return launch_class<8, 4, 12, 1, 4, 8, 1>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
    case 12: return launch_class<12, 2, 12, 1, 2, 12, 1>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
    case 15: return launch_class<15, 2, 12, 1, 2, 12, 1>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
    default: return launch_class<16, 2, 12, 1, 2, 8, 1>(xmode, two, m0, m1, a, p->sm_count, p->device, s);
  }
}

// Complex (Bloch) mode product in ONE launch, in place: nb complex functions = 2 nb planes (re, im) in `buf`, the product
// with M = V^H (forward) or V (backward) taken as the real embedding [[Mr, -Mi], [Mi, Mr]] (contraction over both
// planes, output rows for both planes; 4x the real flops, the same as a Zgemm).  Needs 2 ceil(n/8) <= 16, i.e. n <= 64;
// cudaErrorNotSupported otherwise (the caller then runs the two-launch read-modify-write path).
cudaError_t tma_mode_product_c(exx_plan* p, int axis, bool forward, double* buf, int nb, cudaStream_t s) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st) return cudaErrorNotSupported;
  const int n = p->n[axis];
  const double* img = st->d_img_c[axis][forward ? 0 : 1];
  if (!img || (p->n[0] & 1) || !aligned16(buf)) return cudaErrorNotSupported;
  const int need = (n + 7) / 8;
  const int mh = need <= 2 ? 2 : need <= 4 ? 4 : need <= 6 ? 6 : 8;
  const bool xmode = axis == 0;
  const int NT = mh <= 4 ? 4 : 2;
  TArgs a{};
  a.out = buf;
  a.V = img;
  a.n = n;
  a.S = (n + 15) / 16;
  a.kk_last = tail_ksteps(n);
  CUtensorMap m0;
  cudaError_t e;
  if (xmode) {
    a.rows_per_rhs = (int)(p->N / n);
    a.plane_rows = a.rows_per_rhs;
    const long long rows_total = 2LL * a.rows_per_rhs * nb;
    if (rows_total >= (1LL << 31) - 64) return cudaErrorNotSupported;
    a.rows_total = (int)rows_total;
    a.tiles_per_rhs = (a.rows_per_rhs + 8 * NT - 1) / (8 * NT);
    a.div_tiles = make_fastdiv((unsigned)a.tiles_per_rhs);
    a.exact = (n == 8 * mh) && (a.rows_per_rhs % (8 * NT) == 0);
    a.n_tiles = (unsigned)a.tiles_per_rhs * (unsigned)nb;
    if ((e = get_map(st, buf, n, rows_total, 0, 8 * NT, &m0)) != cudaSuccess) return e;
  } else {
    const long long inner = axis == 1 ? p->n[0] : (long long)p->n[0] * p->n[1];
    const long long P = p->N / (n * inner);  // outer indices per plane
    a.inner = (int)inner;
    a.cpo = (int)((inner + 15) / 16);
    const long long chunks = (long long)a.cpo * P * nb;
    if (chunks >= (1LL << 31) - 64) return cudaErrorNotSupported;
    a.total_chunks = (unsigned)chunks;
    a.outer = (int)(2 * P * nb);
    a.plane_outer = (int)P;
    a.div_plane = make_fastdiv((unsigned)P);
    a.div_cpo = make_fastdiv((unsigned)a.cpo);
    a.exact = (n == 8 * mh) && (inner % 16 == 0);
    const int CH = NT / 2;
    a.n_tiles = (unsigned)((chunks + CH - 1) / CH);
    if ((e = get_map(st, buf, inner, n, 2 * P * nb, 16, &m0)) != cudaSuccess) return e;
  }
  if (a.n_tiles == 0) return cudaSuccess;
  ++p->tma_launches;
#define EXX_LAUNCH_C(MT, NTT, W)                                                                            \
  (xmode ? launch_one<MT, NTT, true, false, W, 1, false, true>(m0, m0, a, p->sm_count, p->device, s)       \
         : launch_one<MT, NTT, false, false, W, 1, false, true>(m0, m0, a, p->sm_count, p->device, s))
  switch (mh) {
    case 2: return EXX_LAUNCH_C(4, 4, 16);
    case 4: return EXX_LAUNCH_C(8, 4, 12);
    case 6: return EXX_LAUNCH_C(12, 2, 12);
    default: return EXX_LAUNCH_C(16, 2, 12);
  }
#undef EXX_LAUNCH_C
}

// Upload, per axis and direction, the shared-memory image of M (M[m][k] = V[k][m] forward, V[m][k] backward)
// that k_mode_t stages verbatim: row 16s + 4kk + q holds the contraction index the lane with that q reads in
// k-step kk of stage s (see the fragment-address comment in the kernel), zero beyond n.
cudaError_t tma_init(exx_plan* p) {
  p->tma_state = nullptr;
  if (!encode_fn()) return cudaSuccess;  // no driver entry point: the cp.async kernels serve every pass
  TmaState* st = new (std::nothrow) TmaState();
  if (!st) return cudaErrorMemoryAllocation;
  for (int ax = 0; ax < 3; ++ax)
    for (int d = 0; d < 2; ++d) {
      st->d_img[ax][d] = nullptr;
      st->img_owned[ax][d] = false;
      st->d_img_im[ax][d] = nullptr;
      st->d_img_c[ax][d] = nullptr;
    }
  st->d_img_hc[0] = st->d_img_hc[1] = nullptr;
  p->tma_state = st;
  for (int ax = 0; ax < 3; ++ax) {
    ClassCfg cc;
    if (!pick_class(p->n[ax], 1, &cc)) continue;  // this axis runs on the plain kernel (mtot does not depend on lanes)
    const bool xmode = ax == 0;
    // axes 1 and 2 are both L-mode: identical matrices share the images
    if (ax == 2 && p->d_V[2] == p->d_V[1] && st->d_img[1][0]) {
      st->d_img[2][0] = st->d_img[1][0];
      st->d_img[2][1] = st->d_img[1][1];
      st->d_img_im[2][0] = st->d_img_im[1][0];
      st->d_img_im[2][1] = st->d_img_im[1][1];
      st->d_img_c[2][0] = st->d_img_c[1][0];
      st->d_img_c[2][1] = st->d_img_c[1][1];
      continue;
    }
    const int n = p->n[ax], S = (n + 15) / 16, ldv = 8 * cc.mtot + 4;
    // Bloch axis with n <= 64: the real embedding [[Mr, -Mi], [Mi, Mr]] for the single-launch complex product; rows:
    // contraction index over the re plane (16 S rows) then the im plane, columns: output index, re rows then im rows
    for (int d = 0; d < 2 && !p->h_Vi[ax].empty() && (p->n[ax] + 7) / 8 <= 8; ++d) {
      const int need = (n + 7) / 8, mh = need <= 2 ? 2 : need <= 4 ? 4 : need <= 6 ? 6 : 8, ldc = 16 * mh + 4;
      std::vector<double> img((size_t)32 * S * ldc, 0.0);
      for (int s = 0; s < S; ++s)
        for (int kk = 0; kk < 4; ++kk)
          for (int q = 0; q < 4; ++q) {
            const int k = 16 * s + within_stage(xmode, n, s, kk, q);
            if (k >= n) continue;
            double* row_re = &img[(size_t)(16 * s + 4 * kk + q) * ldc];
            double* row_im = &img[(size_t)(16 * S + 16 * s + 4 * kk + q) * ldc];
            for (int m = 0; m < n; ++m) {
              const double mr = d == 0 ? p->h_V[ax][(size_t)k * n + m] : p->h_V[ax][(size_t)m * n + k];
              const double mi = d == 0 ? -p->h_Vi[ax][(size_t)k * n + m] : p->h_Vi[ax][(size_t)m * n + k];
              row_re[m] = mr;            // out_re += Mr in_re
              row_re[8 * mh + m] = mi;   // out_im += Mi in_re
              row_im[m] = -mi;           // out_re -= Mi in_im
              row_im[8 * mh + m] = mr;   // out_im += Mr in_im
            }
          }
      cudaError_t e = cudaMalloc(&st->d_img_c[ax][d], sizeof(double) * img.size());
      if (e != cudaSuccess) return e;
      e = cudaMemcpy(st->d_img_c[ax][d], img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
      if (e != cudaSuccess) return e;
    }
    for (int d = 0; d < 2 && !p->h_Vi[ax].empty(); ++d) {  // Bloch axis: forward M = V^H, Im = -Vi^T; backward Im = Vi
      std::vector<double> img((size_t)16 * S * ldv, 0.0);
      for (int s = 0; s < S; ++s)
        for (int kk = 0; kk < 4; ++kk)
          for (int q = 0; q < 4; ++q) {
            const int within = within_stage(xmode, n, s, kk, q);
            const int k = 16 * s + within;
            if (k >= n) continue;
            double* row = &img[(size_t)(16 * s + 4 * kk + q) * ldv];
            for (int m = 0; m < n; ++m)
              row[m] = d == 0 ? -p->h_Vi[ax][(size_t)k * n + m] : p->h_Vi[ax][(size_t)m * n + k];
          }
      cudaError_t e = cudaMalloc(&st->d_img_im[ax][d], sizeof(double) * img.size());
      if (e != cudaSuccess) return e;
      e = cudaMemcpy(st->d_img_im[ax][d], img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
      if (e != cudaSuccess) return e;
    }
    // y axis of a real plan with nx == 8 (mod 16): the same images in the row order of the half-chunk tiles
    for (int d = 0; d < 2 && ax == 1 && p->h_Vi[ax].empty() && p->n[0] % 16 == 8; ++d) {
      std::vector<double> img((size_t)16 * S * ldv, 0.0);
      for (int s = 0; s < S; ++s)
        for (int kk = 0; kk < 4; ++kk)
          for (int q = 0; q < 4; ++q) {
            const int k = 16 * s + within_stage(false, n, s, kk, q, true);
            if (k >= n) continue;
            double* row = &img[(size_t)(16 * s + 4 * kk + q) * ldv];
            for (int m = 0; m < n; ++m)
              row[m] = d == 0 ? p->h_V[ax][(size_t)k * n + m] : p->h_V[ax][(size_t)m * n + k];
          }
      cudaError_t e = cudaMalloc(&st->d_img_hc[d], sizeof(double) * img.size());
      if (e != cudaSuccess) return e;
      e = cudaMemcpy(st->d_img_hc[d], img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
      if (e != cudaSuccess) return e;
    }
    for (int d = 0; d < 2; ++d) {
      std::vector<double> img((size_t)16 * S * ldv, 0.0);
      for (int s = 0; s < S; ++s)
        for (int kk = 0; kk < 4; ++kk)
          for (int q = 0; q < 4; ++q) {
            const int within = within_stage(xmode, n, s, kk, q);
            const int k = 16 * s + within;
            if (k >= n) continue;
            double* row = &img[(size_t)(16 * s + 4 * kk + q) * ldv];
            for (int m = 0; m < n; ++m)
              row[m] = d == 0 ? p->h_V[ax][(size_t)k * n + m] : p->h_V[ax][(size_t)m * n + k];
          }
      cudaError_t e = cudaMalloc(&st->d_img[ax][d], sizeof(double) * img.size());
      if (e != cudaSuccess) return e;
      st->img_owned[ax][d] = true;
      e = cudaMemcpy(st->d_img[ax][d], img.data(), sizeof(double) * img.size(), cudaMemcpyHostToDevice);
      if (e != cudaSuccess) return e;
    }
  }
  return cudaSuccess;
}

void tma_destroy(exx_plan* p) {
  TmaState* st = static_cast<TmaState*>(p->tma_state);
  if (!st) return;
  for (int ax = 0; ax < 3; ++ax)
    for (int d = 0; d < 2; ++d)
    {
      if (st->img_owned[ax][d] && st->d_img[ax][d]) cudaFree(st->d_img[ax][d]);
      if (st->d_img_im[ax][d] && !(ax == 2 && st->d_img_im[2][d] == st->d_img_im[1][d])) cudaFree(st->d_img_im[ax][d]);
      if (st->d_img_c[ax][d] && !(ax == 2 && st->d_img_c[2][d] == st->d_img_c[1][d])) cudaFree(st->d_img_c[ax][d]);
    }
  for (int d = 0; d < 2; ++d)
    if (st->d_img_hc[d]) cudaFree(st->d_img_hc[d]);
  delete st;
  p->tma_state = nullptr;
}

}  // namespace exx
