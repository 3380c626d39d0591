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

// ---- axes held in their real form (plan_host.cpp bloch_eigh_real_form): the butterfly U^H / U -----------------------------
// For an axis with a Bloch phase the plan holds the REAL orthogonal W of K' = U^H K U; a complex mode product V^H f is
// g = U^H f followed by the real product W^T on both planes, and V t = U (W t).  U only couples a point x with its mirror
// image Rx = n - 1 - x:
//     forward  g[x] = (f[x] + f[Rx])/sqrt 2,        g[Rx] = -i (f[x] - f[Rx])/sqrt 2      (x < Rx; a self-paired point is kept)
//     inverse  f[x] = (g[x] + i g[Rx])/sqrt 2,      f[Rx] = (g[x] - i g[Rx])/sqrt 2
// and the butterflies of different axes commute with the products of the other axes, so all of them are applied at once,
// on the orbit of a point under the reflections of the butterfly axes (up to 8 points), in the kernels that stream the
// data anyway: the pair density (forward) and the accumulate (inverse); k_bfly_c serves the bare solver.
struct BflyDims {
  int n[3];     // nx, ny, nz
  int half[3];  // points per axis a thread block enumerates: ceil(n/2) on a butterfly axis, n otherwise
  int on[3];
};

// Orbit of a half-domain point under the reflections of the butterfly axes: point c (bit 0: x, bit 1: y, bit 2: z mirrored)
// sits at base + (c & 1 ? dx : 0) + (c & 2 ? dy : 0) + (c & 4 ? dz : 0); a zero offset means the axis does not pair here
// (no butterfly on it, or a self-paired point).  N < 2^31 (exx_plan_create), so 32-bit offsets suffice.
struct Orbit {
  int base, dx, dy, dz;
  int px, py, pz;  // 1: the axis pairs two distinct points
  __device__ __forceinline__ int idx(int c) const { return base + ((c & 1) ? dx : 0) + ((c & 2) ? dy : 0) + ((c & 4) ? dz : 0); }
};

__device__ __forceinline__ Orbit orbit_of(const BflyDims& d, unsigned t) {
  const unsigned hx = t % (unsigned)d.half[0], u = t / (unsigned)d.half[0];
  const unsigned hy = u % (unsigned)d.half[1], hz = u / (unsigned)d.half[1];
  Orbit o;
  o.base = (int)(hx + (unsigned)d.n[0] * (hy + (unsigned)d.n[1] * hz));
  o.dx = d.on[0] ? d.n[0] - 1 - 2 * (int)hx : 0;
  o.dy = d.on[1] ? (d.n[1] - 1 - 2 * (int)hy) * d.n[0] : 0;
  o.dz = d.on[2] ? (d.n[2] - 1 - 2 * (int)hz) * d.n[0] * d.n[1] : 0;
  o.px = o.dx != 0;
  o.py = o.dy != 0;
  o.pz = o.dz != 0;
  return o;
}
// point c of the orbit is distinct from the points before it
__device__ __forceinline__ bool orbit_has(const Orbit& o, int c) {
  return (!(c & 1) || o.px) && (!(c & 2) || o.py) && (!(c & 4) || o.pz);
}

template <bool INVERSE>
__device__ __forceinline__ void bfly_pair(double& ar, double& ai, double& br, double& bi) {
  const double r = 0.70710678118654752440;
  if (!INVERSE) {  // a' = (a + b) r, b' = -i (a - b) r
    const double sr = (ar + br) * r, si = (ai + bi) * r, dr = (ar - br) * r, di = (ai - bi) * r;
    ar = sr; ai = si; br = di; bi = -dr;
  } else {         // a' = (a + i b) r, b' = (a - i b) r
    const double pr = (ar - bi) * r, pi = (ai + br) * r, mr = (ar + bi) * r, mi = (ai - br) * r;
    ar = pr; ai = pi; br = mr; bi = mi;
  }
}
// all butterfly axes of one orbit, values v[c] = (vr[c], vi[c]) at orbit point c (bit 0: x, bit 1: y, bit 2: z)
template <bool INVERSE>
__device__ __forceinline__ void bfly_orbit(const Orbit& o, double (&vr)[8], double (&vi)[8]) {
  if (o.px) {
#pragma unroll
    for (int c = 0; c < 8; c += 2) bfly_pair<INVERSE>(vr[c], vi[c], vr[c + 1], vi[c + 1]);
  }
  if (o.py) {
#pragma unroll
    for (int c = 0; c < 8; ++c)
      if (!(c & 2)) bfly_pair<INVERSE>(vr[c], vi[c], vr[c + 2], vi[c + 2]);
  }
  if (o.pz) {
#pragma unroll
    for (int c = 0; c < 4; ++c) bfly_pair<INVERSE>(vr[c], vi[c], vr[c + 4], vi[c + 4]);
  }
}

// rho_b = conj(psi_j) .* tgt_k followed by the forward butterflies; grid.y = nb, a thread per orbit
__global__ void __launch_bounds__(256, 4) k_pair_density_c_bfly(const double* __restrict__ psi, const double* __restrict__ tgt,
                                                             BatchDesc bd, long long N, BflyDims d, long long orbits,
                                                             double* __restrict__ out) {
  // blocks in (orbital, target) order with the target fastest: the nk right-hand sides that share psi_j are formed back to
  // back and find it in L2 (with the right-hand-side order b = kk nj + jj a batch of 64 orbitals cycles through more
  // than the L2 holds between two uses of the same psi_j)
  const int jj = blockIdx.y / bd.nk, kk = blockIdx.y - jj * bd.nk;
  const int b = kk * bd.nj + jj;
  const int j = bd.j0 + jj, k = bd.k0 + kk;
  const double* ar = psi + (size_t)j * 2 * N;
  const double* br = tgt + (size_t)k * 2 * N;
  double* o = out + (size_t)b * 2 * N;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < orbits; t += (long long)gridDim.x * blockDim.x) {
    const Orbit ob = orbit_of(d, (unsigned)t);
    double vr[8], vi[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      vr[c] = vi[c] = 0.0;
      if (orbit_has(ob, c)) {
        const int i = ob.idx(c);
        const double a_re = ar[i], a_im = ar[N + i], b_re = br[i], b_im = br[N + i];
        vr[c] = a_re * b_re + a_im * b_im;
        vi[c] = a_re * b_im - a_im * b_re;
      }
    }
    bfly_orbit<false>(ob, vr, vi);
#pragma unroll
    for (int c = 0; c < 8; ++c)
      if (orbit_has(ob, c)) {
        o[ob.idx(c)] = vr[c];
        o[N + ob.idx(c)] = vi[c];
      }
  }
}

// in-place butterflies of nb complex functions (the bare solver): forward before the products, inverse after them
template <bool INVERSE>
__global__ void __launch_bounds__(256, 4) k_bfly_c(double* __restrict__ buf, long long N, BflyDims d, long long orbits) {
  double* o = buf + (size_t)blockIdx.y * 2 * N;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < orbits; t += (long long)gridDim.x * blockDim.x) {
    const Orbit ob = orbit_of(d, (unsigned)t);
    double vr[8], vi[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      vr[c] = vi[c] = 0.0;
      if (orbit_has(ob, c)) {
        vr[c] = o[ob.idx(c)];
        vi[c] = o[N + ob.idx(c)];
      }
    }
    bfly_orbit<INVERSE>(ob, vr, vi);
#pragma unroll
    for (int c = 0; c < 8; ++c)
      if (orbit_has(ob, c)) {
        o[ob.idx(c)] = vr[c];
        o[N + ob.idx(c)] = vi[c];
      }
  }
}

// vx_k (-)= sum_j occ_j psi_j .* (U phi~_jk): inverse butterflies of the solver's output, then the complex product, j
// ascending; grid.y = nk, a thread per orbit
__global__ void __launch_bounds__(256, 3) k_accumulate_c_bfly(const double* __restrict__ psi, const double* __restrict__ occ,
                                                           const double* __restrict__ phi, BatchDesc bd, bool first,
                                                           long long N, BflyDims d, long long orbits,
                                                           double* __restrict__ vx) {
  const int kk = blockIdx.y;
  double* v = vx + (size_t)(bd.k0 + kk) * 2 * N;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < orbits; t += (long long)gridDim.x * blockDim.x) {
    const Orbit ob = orbit_of(d, (unsigned)t);
    double ar[8], ai[8];
#pragma unroll
    for (int c = 0; c < 8; ++c) {
      ar[c] = ai[c] = 0.0;
      if (!first && orbit_has(ob, c)) {
        ar[c] = v[ob.idx(c)];
        ai[c] = v[N + ob.idx(c)];
      }
    }
    const double* a = psi + (size_t)bd.j0 * 2 * N;
    const double* f = phi + (size_t)kk * bd.nj * 2 * N;
    for (int jj = 0; jj < bd.nj; ++jj) {
      const double oc = occ[bd.j0 + jj];
      double fr[8], fi[8];
#pragma unroll
      for (int c = 0; c < 8; ++c) {
        fr[c] = fi[c] = 0.0;
        if (orbit_has(ob, c)) {
          fr[c] = f[ob.idx(c)];
          fi[c] = f[N + ob.idx(c)];
        }
      }
      bfly_orbit<true>(ob, fr, fi);
#pragma unroll
      for (int c = 0; c < 8; ++c)
        if (orbit_has(ob, c)) {
          const double p_re = a[ob.idx(c)], p_im = a[N + ob.idx(c)];
          ar[c] -= oc * (p_re * fr[c] - p_im * fi[c]);
          ai[c] -= oc * (p_re * fi[c] + p_im * fr[c]);
        }
      a += 2 * N;
      f += 2 * N;
    }
#pragma unroll
    for (int c = 0; c < 8; ++c)
      if (orbit_has(ob, c)) {
        v[ob.idx(c)] = ar[c];
        v[N + ob.idx(c)] = ai[c];
      }
  }
}

inline bool any_bfly(const exx_plan* p) { return p->bfly[0] || p->bfly[1] || p->bfly[2]; }
inline BflyDims bfly_dims(const exx_plan* p, long long* orbits) {
  BflyDims d;
  *orbits = 1;
  for (int a = 0; a < 3; ++a) {
    d.n[a] = p->n[a];
    d.on[a] = p->bfly[a] ? 1 : 0;
    d.half[a] = p->bfly[a] ? (p->n[a] + 1) / 2 : p->n[a];
    *orbits *= d.half[a];
  }
  return d;
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
  if (any_bfly(p)) {  // axes held in their real form: the forward butterflies ride on the pair density
    long long orbits;
    const BflyDims d = bfly_dims(p, &orbits);
    dim3 grid(grid_for(orbits, 256, p->sm_count), bd.nj * bd.nk);
    k_pair_density_c_bfly<<<grid, 256, 0, s>>>(psi, tgt, bd, p->N, d, orbits, out);
    return cudaGetLastError();
  }
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
  if (any_bfly(p)) {  // the inverse butterflies ride on the accumulate
    long long orbits;
    const BflyDims d = bfly_dims(p, &orbits);
    dim3 grid(grid_for(orbits, 256, p->sm_count), bd.nk);
    k_accumulate_c_bfly<<<grid, 256, 0, s>>>(psi, occ, phi, bd, first, p->N, d, orbits, vx);
    return cudaGetLastError();
  }
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

// In-place butterflies of nb complex functions for the bare solver (no-op for a plan without real-form axes).
cudaError_t bloch_butterfly(const exx_plan* p, double* buf, int nb, bool inverse, cudaStream_t s, long long* launches) {
  if (!any_bfly(p) || nb <= 0) return cudaSuccess;
  long long orbits;
  const BflyDims d = bfly_dims(p, &orbits);
  dim3 grid(grid_for(orbits, 256, p->sm_count), nb);
  if (inverse) k_bfly_c<true><<<grid, 256, 0, s>>>(buf, p->N, d, orbits);
  else k_bfly_c<false><<<grid, 256, 0, s>>>(buf, p->N, d, orbits);
  ++*launches;
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
