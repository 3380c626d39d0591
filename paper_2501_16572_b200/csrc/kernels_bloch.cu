// Bloch-periodic (k-point) variant of the exchange apply (Eqs. 1-3 with
// complex orbitals, :159 "complex-valued computations", :218 cublasZgemm; R18-R20).
//
// A complex grid function is two real planes [2][N] (real part, imaginary part), so a batch of nb complex
// right-hand sides is 2 nb real ones and a complex mode product out = M in, M = Mr + i Mi (V^H forward, V backward),
// is two launches of the REAL tensor-core kernel k_mode_t over those 2 nb planes,
//     P = Mr [in_re | in_im],   Q = Mi [in_re | in_im],
// combined as out_re = P_re - Q_im, out_im = P_im + Q_re: the Q launch adds its result straight into P's planes in its
// epilogue (read-modify-write, k_mode_t `rmw`); only the z-backward product, whose launches carry the multiplier as a
// second TMA stream, writes Q out and runs the streaming k_combine.
// That is the 4x real flops of a Zgemm on the FP64 tensor pipe with no new MMA kernel.  An axis whose matrix is
// real (Dirichlet, or theta = 0) needs neither Q nor the combine: one in-place launch.  The eigen-space multiplier
// is real and rides as the second TMA stream of the z-backward launches, exactly as in the real path.
//
// The cross-check variant (EXX_VARIANT_REFERENCE, and the fallback for sizes TMA cannot address) is one plain DFMA
// kernel per complex mode product (k_mode_product_c).
#include <cstdint>

#include "exx_internal.h"

namespace exx {
namespace {

inline int grid_for(long long work, int threads, int sm_count) {
  long long g = (work + threads - 1) / threads;
  const long long cap = (long long)sm_count * 16;
  if (g > cap) g = cap;
  if (g < 1) g = 1;
  return (int)g;
}

// rho_b = conj(psi_j) .* tgt_k (Eq. 2), b = kk * nj + jj; planes [2][N].  grid.y = nb.  VEC = 2: 16-byte
// accesses (N even, 16-byte aligned buffers).
template <int VEC>
__global__ void __launch_bounds__(256) k_pair_density_c(const double* __restrict__ psi, const double* __restrict__ tgt,
                                                        BatchDesc bd, long long N, double* __restrict__ out) {
  const int b = blockIdx.y;
  const int j = bd.j0 + b % bd.nj, k = bd.k0 + b / bd.nj;
  const double* ar = psi + (size_t)j * 2 * N;
  const double* br = tgt + (size_t)k * 2 * N;
  double* o = out + (size_t)b * 2 * N;
  for (long long i = (blockIdx.x * (long long)blockDim.x + threadIdx.x) * VEC; i < N;
       i += (long long)gridDim.x * blockDim.x * VEC) {
    if (VEC == 2) {
      const double2 a_re = *reinterpret_cast<const double2*>(ar + i), a_im = *reinterpret_cast<const double2*>(ar + N + i);
      const double2 b_re = *reinterpret_cast<const double2*>(br + i), b_im = *reinterpret_cast<const double2*>(br + N + i);
      *reinterpret_cast<double2*>(o + i) = make_double2(a_re.x * b_re.x + a_im.x * b_im.x, a_re.y * b_re.y + a_im.y * b_im.y);
      *reinterpret_cast<double2*>(o + N + i) =
          make_double2(a_re.x * b_im.x - a_im.x * b_re.x, a_re.y * b_im.y - a_im.y * b_re.y);
    } else {
      const double a_re = ar[i], a_im = ar[N + i], b_re = br[i], b_im = br[N + i];
      o[i] = a_re * b_re + a_im * b_im;
      o[N + i] = a_re * b_im - a_im * b_re;
    }
  }
}

// out = P + i Q for planar data: P_re -= Q_im, P_im += Q_re, in place over P.  grid.y = nb.
__global__ void k_combine(double* __restrict__ P, const double* __restrict__ Q, long long N) {
  double* p = P + (size_t)blockIdx.y * 2 * N;
  const double* q = Q + (size_t)blockIdx.y * 2 * N;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < N; i += (long long)gridDim.x * blockDim.x) {
    p[i] -= q[N + i];
    p[N + i] += q[i];
  }
}

// vx_k (-)= sum_j occ_j psi_j .* phi_jk (complex product, no conjugate; Eq. 1), j ascending.  grid.y = nk.
// VEC = 2: 16-byte accesses; the arithmetic per element is the same for both instantiations.
template <int VEC>
__global__ void __launch_bounds__(256) k_accumulate_c(const double* __restrict__ psi, const double* __restrict__ occ,
                                                      const double* __restrict__ phi, BatchDesc bd, bool first,
                                                      long long N, double* __restrict__ vx) {
  const int kk = blockIdx.y;
  double* v = vx + (size_t)(bd.k0 + kk) * 2 * N;
  for (long long i = (blockIdx.x * (long long)blockDim.x + threadIdx.x) * VEC; i < N;
       i += (long long)gridDim.x * blockDim.x * VEC) {
    double v_re[VEC], v_im[VEC];
#pragma unroll
    for (int e = 0; e < VEC; ++e) {
      v_re[e] = first ? 0.0 : v[i + e];
      v_im[e] = first ? 0.0 : v[N + i + e];
    }
    const double* a = psi + (size_t)bd.j0 * 2 * N + i;
    const double* f = phi + (size_t)kk * bd.nj * 2 * N + i;
#pragma unroll 2
    for (int jj = 0; jj < bd.nj; ++jj) {
      const double o = occ[bd.j0 + jj];
      double a_re[VEC], a_im[VEC], f_re[VEC], f_im[VEC];
      if (VEC == 2) {
        const double2 t0 = *reinterpret_cast<const double2*>(a), t1 = *reinterpret_cast<const double2*>(a + N);
        const double2 t2 = *reinterpret_cast<const double2*>(f), t3 = *reinterpret_cast<const double2*>(f + N);
        a_re[0] = t0.x; a_re[VEC - 1] = t0.y; a_im[0] = t1.x; a_im[VEC - 1] = t1.y;
        f_re[0] = t2.x; f_re[VEC - 1] = t2.y; f_im[0] = t3.x; f_im[VEC - 1] = t3.y;
      } else {
        a_re[0] = a[0]; a_im[0] = a[N]; f_re[0] = f[0]; f_im[0] = f[N];
      }
#pragma unroll
      for (int e = 0; e < VEC; ++e) {
        v_re[e] -= o * (a_re[e] * f_re[e] - a_im[e] * f_im[e]);
        v_im[e] -= o * (a_re[e] * f_im[e] + a_im[e] * f_re[e]);
      }
      a += 2 * N;
      f += 2 * N;
    }
#pragma unroll
    for (int e = 0; e < VEC; ++e) {
      v[i + e] = v_re[e];
      v[N + i + e] = v_im[e];
    }
  }
}

// Plain complex mode product, one thread per output point: out[m] = sum_i M[m][i] in[i] along `axis`,
// forward M = V^H (M[m][i] = conj(V[i][m])), backward M = V.  Vi == nullptr: real matrix.  mult (optional) is applied
// to the output.  total = nb * N complex points.
__global__ void k_mode_product_c(const double* __restrict__ in, double* __restrict__ out, const double* __restrict__ Vr,
                                 const double* __restrict__ Vi, int n, long long inner, long long N, long long total,
                                 bool forward, const double* __restrict__ mult) {
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const long long b = t / N, r = t - b * N;
    const int m = (int)((r / inner) % n);
    const double* src = in + (size_t)b * 2 * N + (r - (long long)m * inner);
    double s_re = 0.0, s_im = 0.0;
    for (int i = 0; i < n; ++i) {
      const double x_re = src[(long long)i * inner], x_im = src[N + (long long)i * inner];
      double m_re, m_im;
      if (forward) {
        m_re = Vr[(long long)i * n + m];
        m_im = Vi ? -Vi[(long long)i * n + m] : 0.0;
      } else {
        m_re = Vr[(long long)m * n + i];
        m_im = Vi ? Vi[(long long)m * n + i] : 0.0;
      }
      s_re += m_re * x_re - m_im * x_im;
      s_im += m_re * x_im + m_im * x_re;
    }
    if (mult) {
      s_re *= mult[r];
      s_im *= mult[r];
    }
    out[(size_t)b * 2 * N + r] = s_re;
    out[(size_t)b * 2 * N + N + r] = s_im;
  }
}

}  // namespace

cudaError_t bloch_pair_density(const exx_plan* p, const double* psi, const double* tgt, BatchDesc bd, double* out,
                               cudaStream_t s) {
  const bool vec2 = (p->N % 2 == 0) && ((((uintptr_t)psi | (uintptr_t)tgt | (uintptr_t)out) & 15) == 0);
  if (vec2) {
    dim3 grid(grid_for(p->N / 2, 256, p->sm_count), bd.nj * bd.nk);
    k_pair_density_c<2><<<grid, 256, 0, s>>>(psi, tgt, bd, p->N, out);
  } else {
    dim3 grid(grid_for(p->N, 256, p->sm_count), bd.nj * bd.nk);
    k_pair_density_c<1><<<grid, 256, 0, s>>>(psi, tgt, bd, p->N, out);
  }
  return cudaGetLastError();
}

cudaError_t bloch_accumulate(const exx_plan* p, const double* psi, const double* occ, const double* phi, BatchDesc bd,
                             bool first, double* vx, cudaStream_t s) {
  const bool vec2 = (p->N % 2 == 0) && ((((uintptr_t)psi | (uintptr_t)phi | (uintptr_t)vx) & 15) == 0);
  if (vec2) {
    dim3 grid(grid_for(p->N / 2, 256, p->sm_count), bd.nk);
    k_accumulate_c<2><<<grid, 256, 0, s>>>(psi, occ, phi, bd, first, p->N, vx);
  } else {
    dim3 grid(grid_for(p->N, 256, p->sm_count), bd.nk);
    k_accumulate_c<1><<<grid, 256, 0, s>>>(psi, occ, phi, bd, first, p->N, vx);
  }
  return cudaGetLastError();
}

// nb complex right-hand sides in buf[0] ([nb][2][N]) -> f(L_theta) of them, returned in *result (one of the three
// buffers).  Six complex mode products; buf[0..2] each hold 2 nb N doubles.
cudaError_t bloch_solve_batch(exx_plan* p, double* const buf[3], int nb, cudaStream_t s, long long* launches,
                              double** result) {
  static const int axis[6] = {0, 1, 2, 2, 1, 0};
  double *cur = buf[0], *other = buf[1], *q = buf[2];
  const long long N = p->N;
  cudaError_t e;
  for (int i = 0; i < 6; ++i) {
    const int ax = axis[i];
    const bool fwd = i < 3, mult = i == 3, cplx = p->d_Vi[ax] != nullptr;
    bool done = false;
    if (i == 2 && p->variant != EXX_VARIANT_REFERENCE) {
      // z-forward + multiplier + z-backward in one pass (kernels_fused.cu): the real kernel over the 2 nb planes for a
      // real z axis, the embedded complex one for a complex z axis with n <= 64
      ProfScope ps(p, KC_MODE_PRODUCT, s);
      e = cplx ? fused_zz_c(p, cur, nb, s) : fused_zz(p, cur, cur, 2 * nb, s);
      if (e == cudaSuccess) {
        ++*launches;
        ++i;  // the z-backward product is done too
        continue;
      }
      ps.cancel();
      if (e != cudaErrorNotSupported) return e;
    }
    if (p->variant != EXX_VARIANT_REFERENCE) {
      ProfScope ps(p, KC_MODE_PRODUCT, s);
      if (!cplx) {
        e = tma_mode_product(p, ax, fwd, cur, cur, 2 * nb, mult, nullptr, s, 0);
        if (e == cudaSuccess) { ++*launches; done = true; }
        else if (e != cudaErrorNotSupported) return e;
      } else if (!mult && (e = tma_mode_product_c(p, ax, fwd, cur, nb, s)) != cudaErrorNotSupported) {
        // n <= 64: one in-place launch on the real embedding [[Mr, -Mi], [Mi, Mr]] (kernels_tma.cu, CPLX)
        if (e != cudaSuccess) return e;
        ++*launches;
        done = true;
      } else {
        e = tma_mode_product(p, ax, fwd, cur, other, 2 * nb, mult, nullptr, s, 0);
        if (e == cudaSuccess) {
          if (!mult) {
            // second launch adds Q into P's planes in its epilogue (read-modify-write): no Q buffer, no combine pass
            if ((e = tma_mode_product(p, ax, fwd, cur, other, 2 * nb, false, nullptr, s, 1, true)) != cudaSuccess) return e;
            *launches += 2;
          } else {
            // the two-stream (multiplier) kernel has no read-modify-write epilogue: separate Q, then the combine
            if ((e = tma_mode_product(p, ax, fwd, cur, q, 2 * nb, mult, nullptr, s, 1)) != cudaSuccess) return e;
            dim3 grid(grid_for(N, 256, p->sm_count), nb);
            k_combine<<<grid, 256, 0, s>>>(other, q, N);
            if ((e = cudaGetLastError()) != cudaSuccess) return e;
            *launches += 3;
          }
          double* t = cur; cur = other; other = t;
          done = true;
        } else if (e != cudaErrorNotSupported) {
          return e;
        }
      }
    }
    if (!done) {  // plain complex kernel: cross-check variant, and sizes TMA cannot address
      ProfScope ps(p, KC_MODE_PRODUCT, s);
      const long long inner = ax == 0 ? 1 : (ax == 1 ? p->n[0] : (long long)p->n[0] * p->n[1]);
      const long long total = N * nb;
      // the multiplier belongs to the INPUT of the z-backward product = the output of the z-forward one
      k_mode_product_c<<<grid_for(total, 256, p->sm_count), 256, 0, s>>>(cur, other, p->d_V[ax], p->d_Vi[ax], p->n[ax],
                                                                        inner, N, total, fwd, i == 2 ? p->d_mult : nullptr);
      if ((e = cudaGetLastError()) != cudaSuccess) return e;
      ++*launches;
      double* t = cur; cur = other; other = t;
    }
  }
  *result = cur;
  return cudaSuccess;
}

}  // namespace exx
