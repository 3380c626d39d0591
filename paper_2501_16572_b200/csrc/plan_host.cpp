// Host-side planner of libexx.so: FD second-derivative matrices, a cyclic Jacobi eigensolver and the
// multiplier table.  Runs once per plan (Eqs. 6-7: "eigenvectors of the discrete second
// derivative operators"); not on the timed path.  No LAPACK dependency, no code shared with oracle/.
#include <algorithm>
#include <cmath>
#include <numeric>

#include "exx_internal.h"

namespace exx {

// w_q = (1/q^2) * prod_{m != q} m^2 / (m^2 - q^2), q = 1..n0 (Lagrange form of the centred stencil),
// w_0 = -2 sum_q w_q; all divided by h^2.  DESIGN.md R4.
std::vector<double> fd_weights(int order, double h) {
  const int n0 = order / 2;
  std::vector<double> w(n0 + 1, 0.0);
  for (int q = 1; q <= n0; ++q) {
    long double prod = 1.0L;
    for (int m = 1; m <= n0; ++m) {
      if (m == q) continue;
      prod *= (long double)(m * m) / (long double)(m * m - q * q);
    }
    w[q] = (double)(prod / (long double)(q * q));
  }
  long double s = 0.0L;
  for (int q = n0; q >= 1; --q) s += (long double)w[q];
  w[0] = (double)(-2.0L * s);
  for (auto& x : w) x /= (h * h);
  return w;
}

std::vector<double> second_derivative_matrix(int n, double h, int bc, int order) {
  const std::vector<double> w = fd_weights(order, h);
  const int n0 = order / 2;
  std::vector<double> K((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i) {
    for (int q = -n0; q <= n0; ++q) {
      int j = i + q;
      if (bc == EXX_BC_PERIODIC) {
        j %= n;
        if (j < 0) j += n;
        K[(size_t)i * n + j] += w[std::abs(q)];  // accumulate: the stencil may wrap more than once
      } else if (j >= 0 && j < n) {
        K[(size_t)i * n + j] = w[std::abs(q)];   // truncated at the Dirichlet boundary
      }
    }
  }
  return K;
}

// Cyclic-by-row Jacobi with the standard stable rotation (Golub & Van Loan, Alg. 8.5.x restated).
bool jacobi_eigh(int n, std::vector<double>& A, std::vector<double>& lam, std::vector<double>& V) {
  V.assign((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i) V[(size_t)i * n + i] = 1.0;
  lam.assign(n, 0.0);
  if (n == 1) {
    lam[0] = A[0];
    return true;
  }
  double fro = 0.0;
  for (double a : A) fro += a * a;
  fro = std::sqrt(fro);
  if (fro == 0.0) return true;
  const int max_sweeps = 60;
  bool converged = false;
  for (int sweep = 0; sweep < max_sweeps && !converged; ++sweep) {
    double off = 0.0;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) off += A[(size_t)p * n + q] * A[(size_t)p * n + q];
    if (std::sqrt(2.0 * off) <= 1e-17 * fro) {
      converged = true;
      break;
    }
    for (int p = 0; p < n - 1; ++p) {
      for (int q = p + 1; q < n; ++q) {
        const double apq = A[(size_t)p * n + q];
        if (apq == 0.0) continue;
        const double app = A[(size_t)p * n + p], aqq = A[(size_t)q * n + q];
        if (std::fabs(apq) < 1e-300) continue;
        const double tau = (aqq - app) / (2.0 * apq);
        const double t = (tau >= 0.0 ? 1.0 : -1.0) / (std::fabs(tau) + std::sqrt(1.0 + tau * tau));
        const double c = 1.0 / std::sqrt(1.0 + t * t), s = t * c;
        // A <- J^T A J on rows/columns p, q
        for (int k = 0; k < n; ++k) {
          const double akp = A[(size_t)k * n + p], akq = A[(size_t)k * n + q];
          A[(size_t)k * n + p] = c * akp - s * akq;
          A[(size_t)k * n + q] = s * akp + c * akq;
        }
        for (int k = 0; k < n; ++k) {
          const double apk = A[(size_t)p * n + k], aqk = A[(size_t)q * n + k];
          A[(size_t)p * n + k] = c * apk - s * aqk;
          A[(size_t)q * n + k] = s * apk + c * aqk;
        }
        A[(size_t)p * n + q] = 0.0;
        A[(size_t)q * n + p] = 0.0;
        for (int k = 0; k < n; ++k) {
          const double vkp = V[(size_t)k * n + p], vkq = V[(size_t)k * n + q];
          V[(size_t)k * n + p] = c * vkp - s * vkq;
          V[(size_t)k * n + q] = s * vkp + c * vkq;
        }
      }
    }
  }
  if (!converged) {
    double off = 0.0;
    for (int p = 0; p < n; ++p)
      for (int q = p + 1; q < n; ++q) off += A[(size_t)p * n + q] * A[(size_t)p * n + q];
    if (std::sqrt(2.0 * off) > 1e-14 * fro) return false;
  }
  // sort ascending
  std::vector<int> idx(n);
  std::iota(idx.begin(), idx.end(), 0);
  std::sort(idx.begin(), idx.end(),
            [&](int a, int b) { return A[(size_t)a * n + a] < A[(size_t)b * n + b]; });
  std::vector<double> Vs((size_t)n * n);
  for (int m = 0; m < n; ++m) {
    lam[m] = A[(size_t)idx[m] * n + idx[m]];
    for (int i = 0; i < n; ++i) Vs[(size_t)i * n + m] = V[(size_t)i * n + idx[m]];
  }
  V.swap(Vs);
  return true;
}

// Bloch-periodic axis (R18): K = A + iB Hermitian, A symmetric, B antisymmetric; every wrapped stencil
// entry carries exp(i theta wraps).  Solved through the real symmetric embedding S = [[A, -B], [B, A]] (2n x 2n):
// each complex eigenvector u + iv appears twice, as (u; v) and as (-v; u) = i (u + iv).  Going through the 2n
// real eigenvectors in ascending order and keeping those that survive a complex modified Gram-Schmidt against
// the ones already kept leaves exactly n orthonormal complex eigenvectors (any orthonormal basis of a
// degenerate eigenspace serves: f(L) does not depend on it).
bool bloch_eigh(int n, double h, int order, double theta, std::vector<double>& lam, std::vector<double>& Vr,
                std::vector<double>& Vi) {
  const std::vector<double> w = fd_weights(order, h);
  const int n0 = order / 2, m2 = 2 * n;
  std::vector<double> S((size_t)m2 * m2, 0.0);
  for (int i = 0; i < n; ++i)
    for (int q = -n0; q <= n0; ++q) {
      int j = i + q, wraps = 0;
      while (j < 0) { j += n; --wraps; }
      while (j >= n) { j -= n; ++wraps; }
      const double a = w[std::abs(q)] * std::cos(theta * wraps), b = w[std::abs(q)] * std::sin(theta * wraps);
      S[(size_t)i * m2 + j] += a;              // A
      S[(size_t)(n + i) * m2 + n + j] += a;    // A
      S[(size_t)i * m2 + n + j] -= b;          // -B
      S[(size_t)(n + i) * m2 + j] += b;        // B
    }
  for (int i = 0; i < m2; ++i)                 // remove the rounding-level asymmetry of cos/sin sums
    for (int j = i + 1; j < m2; ++j) {
      const double v = 0.5 * (S[(size_t)i * m2 + j] + S[(size_t)j * m2 + i]);
      S[(size_t)i * m2 + j] = S[(size_t)j * m2 + i] = v;
    }
  std::vector<double> l2, V2;
  if (!jacobi_eigh(m2, S, l2, V2)) return false;
  lam.assign(n, 0.0);
  Vr.assign((size_t)n * n, 0.0);
  Vi.assign((size_t)n * n, 0.0);
  int kept = 0;
  std::vector<double> zr(n), zi(n);
  for (int c = 0; c < m2 && kept < n; ++c) {
    for (int i = 0; i < n; ++i) {
      zr[i] = V2[(size_t)i * m2 + c];
      zi[i] = V2[(size_t)(n + i) * m2 + c];
    }
    for (int pass = 0; pass < 2; ++pass)       // MGS twice
      for (int m = 0; m < kept; ++m) {
        double pr = 0.0, pi = 0.0;             // <v_m, z> = sum conj(v_m) z
        for (int i = 0; i < n; ++i) {
          const double vr = Vr[(size_t)i * n + m], vi = Vi[(size_t)i * n + m];
          pr += vr * zr[i] + vi * zi[i];
          pi += vr * zi[i] - vi * zr[i];
        }
        for (int i = 0; i < n; ++i) {
          const double vr = Vr[(size_t)i * n + m], vi = Vi[(size_t)i * n + m];
          zr[i] -= pr * vr - pi * vi;
          zi[i] -= pr * vi + pi * vr;
        }
      }
    double nrm = 0.0;
    for (int i = 0; i < n; ++i) nrm += zr[i] * zr[i] + zi[i] * zi[i];
    if (nrm < 0.25) continue;                  // the partner i*(u+iv) of a vector already kept
    nrm = std::sqrt(nrm);
    for (int i = 0; i < n; ++i) {
      Vr[(size_t)i * n + kept] = zr[i] / nrm;
      Vi[(size_t)i * n + kept] = zi[i] / nrm;
    }
    lam[kept++] = l2[c];
  }
  return kept == n;
}

// Bloch axis through its REAL form (round 2).  K(theta) is Hermitian and, with the phase carried by the
// wrapped stencil entries, satisfies R K R = conj(K) for the centred reflection R: x -> n - 1 - x, i.e. it commutes with
// the antiunitary T = R o conj (T^2 = 1).  In a basis of T-invariant vectors a T-symmetric Hermitian matrix is REAL
// symmetric.  Such a basis is the fixed, sparse unitary U whose columns are, for every pair x < Rx,
//     (e_x + e_Rx)/sqrt 2   (stored at index x)    and    i (e_x - e_Rx)/sqrt 2   (stored at index Rx),
// and e_x for a self-paired point.  K' = U^H K U is real symmetric, K' = W diag(lam) W^T with W real orthogonal (Jacobi),
// and K = (U W) diag(lam) (U W)^H.  A complex mode product V^H f then is the butterfly g = U^H f (a +- b on pairs of
// points, mixing the real and imaginary planes) followed by the REAL product W^T on the two planes: half the real
// operations of a complex matrix product.  Outputs: lam ascending, W row-major [i][m], and V = U W as (Vr, Vi) for the
// test hook.
bool bloch_eigh_real_form(int n, double h, int order, double theta, std::vector<double>& lam, std::vector<double>& W,
                          std::vector<double>& Vr, std::vector<double>& Vi) {
  const std::vector<double> w = fd_weights(order, h);
  const int n0 = order / 2;
  std::vector<double> Kr((size_t)n * n, 0.0), Ki((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i)
    for (int q = -n0; q <= n0; ++q) {
      int j = i + q, wraps = 0;
      while (j < 0) { j += n; --wraps; }
      while (j >= n) { j -= n; ++wraps; }
      Kr[(size_t)i * n + j] += w[std::abs(q)] * std::cos(theta * wraps);
      Ki[(size_t)i * n + j] += w[std::abs(q)] * std::sin(theta * wraps);
    }
  // U as dense complex columns (n <= a few hundred: the n^3 products below are trivial)
  const double r = 1.0 / std::sqrt(2.0);
  std::vector<double> Ur((size_t)n * n, 0.0), Ui((size_t)n * n, 0.0);
  for (int x = 0; x < n; ++x) {
    const int xb = n - 1 - x;
    if (x < xb) {
      Ur[(size_t)x * n + x] = r;  Ur[(size_t)xb * n + x] = r;      // column x: (e_x + e_Rx)/sqrt 2
      Ui[(size_t)x * n + xb] = r; Ui[(size_t)xb * n + xb] = -r;    // column Rx: i (e_x - e_Rx)/sqrt 2
    } else if (x == xb) {
      Ur[(size_t)x * n + x] = 1.0;
    }
  }
  // T = K U (complex), K' = U^H T; keep the real part, symmetrise (the imaginary part is rounding)
  std::vector<double> Tr((size_t)n * n, 0.0), Ti((size_t)n * n, 0.0), Kp((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i)
    for (int k = 0; k < n; ++k) {
      const double kr = Kr[(size_t)i * n + k], ki = Ki[(size_t)i * n + k];
      if (kr == 0.0 && ki == 0.0) continue;
      for (int b = 0; b < n; ++b) {
        const double ur = Ur[(size_t)k * n + b], ui = Ui[(size_t)k * n + b];
        Tr[(size_t)i * n + b] += kr * ur - ki * ui;
        Ti[(size_t)i * n + b] += kr * ui + ki * ur;
      }
    }
  double im_max = 0.0, re_max = 0.0;
  for (int a = 0; a < n; ++a)
    for (int b = 0; b < n; ++b) {
      double sr = 0.0, si = 0.0;  // sum_i conj(U[i][a]) T[i][b]
      for (int i = 0; i < n; ++i) {
        const double ur = Ur[(size_t)i * n + a], ui = Ui[(size_t)i * n + a];
        sr += ur * Tr[(size_t)i * n + b] + ui * Ti[(size_t)i * n + b];
        si += ur * Ti[(size_t)i * n + b] - ui * Tr[(size_t)i * n + b];
      }
      Kp[(size_t)a * n + b] = sr;
      im_max = std::fmax(im_max, std::fabs(si));
      re_max = std::fmax(re_max, std::fabs(sr));
    }
  if (im_max > 1e-10 * (re_max > 0.0 ? re_max : 1.0)) return false;  // not T-symmetric: cannot happen for this stencil
  for (int a = 0; a < n; ++a)
    for (int b = a + 1; b < n; ++b) {
      const double v = 0.5 * (Kp[(size_t)a * n + b] + Kp[(size_t)b * n + a]);
      Kp[(size_t)a * n + b] = Kp[(size_t)b * n + a] = v;
    }
  if (!jacobi_eigh(n, Kp, lam, W)) return false;
  Vr.assign((size_t)n * n, 0.0);
  Vi.assign((size_t)n * n, 0.0);
  for (int i = 0; i < n; ++i)
    for (int k = 0; k < n; ++k) {
      const double ur = Ur[(size_t)i * n + k], ui = Ui[(size_t)i * n + k];
      if (ur == 0.0 && ui == 0.0) continue;
      for (int m = 0; m < n; ++m) {
        Vr[(size_t)i * n + m] += ur * W[(size_t)k * n + m];
        Vi[(size_t)i * n + m] += ui * W[(size_t)k * n + m];
      }
    }
  return true;
}

// Reflection-adapted eigenbasis of a REAL axis (R13: f(L) does not depend on the basis chosen inside a
// degenerate eigenspace).  The periodic matrix is circulant and symmetric, the Dirichlet one symmetric Toeplitz: both
// commute with the reflection z -> mir(z) (periodic: (n - z) mod n, Dirichlet: n - 1 - z), so every eigenspace splits
// into vectors that are even (v[mir z] = v[z]) or odd (v[mir z] = -v[z]) under it.  Output: the same eigenpairs
// re-expressed in such a basis, EVEN vectors first (n_even of them = number of z with z <= mir z), each block in
// ascending eigenvalue order; Vs row-major [z][m'].  A contraction with an even (odd) vector only needs the half range
// z <= mir(z) of the symmetrised (antisymmetrised) data: half the multiply-adds of the dense product.
// `centered`: use z -> n - 1 - z on a periodic axis too (a symmetric circulant matrix commutes with every reflection);
// the x-axis kernels want it because their mirrored TMA boxes then start at an even, i.e. 16-byte aligned, element.
bool symmetrize_axis(int n, int bc, const std::vector<double>& lam, const std::vector<double>& V, std::vector<double>& lam_s,
                     std::vector<double>& Vs, int* n_even, bool centered) {
  auto mir = [&](int z) { return (bc == EXX_BC_PERIODIC && !centered) ? (n - z) % n : n - 1 - z; };
  int nh = 0;
  for (int z = 0; z < n; ++z) nh += z <= mir(z) ? 1 : 0;
  double scale = 0.0;
  for (int m = 0; m < n; ++m) scale = std::fmax(scale, std::fabs(lam[m]));
  const double tol = 1e-9 * (scale > 0.0 ? scale : 1.0);
  std::vector<std::vector<double>> ev, od;  // kept vectors
  std::vector<double> ev_l, od_l;
  int m0 = 0;
  while (m0 < n) {  // clusters of (numerically) equal eigenvalues, lam ascending
    int m1 = m0 + 1;
    while (m1 < n && std::fabs(lam[m1] - lam[m0]) < tol) ++m1;
    size_t ne0 = ev.size(), no0 = od.size();
    for (int parity = 0; parity < 2; ++parity) {
      auto& keep = parity ? od : ev;
      auto& keep_l = parity ? od_l : ev_l;
      const size_t first = parity ? no0 : ne0;
      // parity parts of the cluster's vectors; keep them by decreasing norm (pivoted Gram-Schmidt): the parts of a
      // vector that is nearly of the other parity are rounding noise and must not be normalised
      std::vector<std::vector<double>> cand;
      for (int m = m0; m < m1; ++m) {
        std::vector<double> v(n);
        for (int z = 0; z < n; ++z) {
          const double a = V[(size_t)z * n + m], b = V[(size_t)mir(z) * n + m];
          v[z] = 0.5 * (parity ? a - b : a + b);
        }
        cand.push_back(v);
      }
      while (!cand.empty()) {
        size_t best = 0;
        double best_n = -1.0;
        for (size_t c = 0; c < cand.size(); ++c) {
          std::vector<double>& v = cand[c];
          for (int pass = 0; pass < 2; ++pass)
            for (size_t k = first; k < keep.size(); ++k) {
              double d = 0.0;
              for (int z = 0; z < n; ++z) d += v[z] * keep[k][z];
              for (int z = 0; z < n; ++z) v[z] -= d * keep[k][z];
            }
          double nrm = 0.0;
          for (int z = 0; z < n; ++z) nrm += v[z] * v[z];
          if (nrm > best_n) { best_n = nrm; best = c; }
        }
        if (best_n < 1e-3) break;  // what is left has no component of this parity (the squared norms sum to the dimension)
        std::vector<double> v = cand[best];
        cand.erase(cand.begin() + (long)best);
        const double nrm = std::sqrt(best_n);
        for (int z = 0; z < n; ++z) v[z] /= nrm;
        for (int z = 0; z < n; ++z) {  // make the parity exact
          const int zb = mir(z);
          if (zb == z) { if (parity) v[z] = 0.0; }
          else if (z < zb) { const double a = 0.5 * (v[z] + (parity ? -v[zb] : v[zb])); v[z] = a; v[zb] = parity ? -a : a; }
        }
        keep.push_back(v);
        keep_l.push_back(lam[m0]);
      }
    }
    if ((int)(ev.size() - ne0 + od.size() - no0) != m1 - m0) return false;  // the cluster did not split cleanly
    m0 = m1;
  }
  if ((int)ev.size() != nh || (int)(ev.size() + od.size()) != n) return false;
  lam_s.assign(n, 0.0);
  Vs.assign((size_t)n * n, 0.0);
  for (int m = 0; m < n; ++m) {
    const bool is_ev = m < nh;
    const std::vector<double>& v = is_ev ? ev[m] : od[m - nh];
    lam_s[m] = is_ev ? ev_l[m] : od_l[m - nh];
    for (int z = 0; z < n; ++z) Vs[(size_t)z * n + m] = v[z];
  }
  *n_even = nh;
  return true;
}

std::vector<double> multiplier_table(const std::vector<double>& lx, const std::vector<double>& ly,
                                     const std::vector<double>& lz, double omega, double zero_tol) {
  const size_t nx = lx.size(), ny = ly.size(), nz = lz.size();
  std::vector<double> m(nx * ny * nz);
  const double four_pi = 4.0 * M_PI;
  for (size_t c = 0; c < nz; ++c)
    for (size_t b = 0; b < ny; ++b)
      for (size_t a = 0; a < nx; ++a) {
        const double ls = lz[c] + ly[b] + lx[a];
        const double mu = -ls;
        double v;
        if (std::fabs(ls) < zero_tol) {
          v = omega > 0.0 ? M_PI / (omega * omega) : 0.0;  // R3: keep the limit (HSE) / drop (PBE0)
        } else if (omega > 0.0) {
          v = -four_pi * std::expm1(-mu / (4.0 * omega * omega)) / mu;  // R1
        } else {
          v = four_pi / mu;  // R2
        }
        m[a + nx * (b + ny * c)] = v;
      }
  return m;
}

}  // namespace exx
