// C-ABI layer of libexx.so (include/exx.h): argument validation, batching of the (j,k) pair space,
// dispatch to the kernel variants.  No host synchronisation in exx_apply / exx_poisson_solve.
#include <cmath>
#include <cstdint>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "exx_internal.h"

namespace {

#ifndef EXX_ITEMS_PER_WARP
#define EXX_ITEMS_PER_WARP 24
#endif
constexpr int kItemsPerWarp = EXX_ITEMS_PER_WARP;

using exx::DeviceScope;

thread_local cudaError_t g_last_cuda = cudaSuccess;
thread_local char g_msg[256];

constexpr int kDefaultBatch = 32;
constexpr int kEnergyChunk = 1024;  // targets per energy launch (bounds the plan-owned scratch)
constexpr int kEnergyBlocks = 64;   // must match kernels_ref.cu

constexpr int kHostChunks = 4;  // exx_apply_host: target chunks whose download overlaps the next chunk's compute
struct HostApiBuffers {
  double* base = nullptr;
  size_t bytes = 0;
  cudaStream_t stream = nullptr;
  cudaStream_t copy_stream = nullptr;
  cudaEvent_t done[kHostChunks] = {nullptr, nullptr, nullptr, nullptr};
  cudaEvent_t up[2] = {nullptr, nullptr};    // orbital block b uploaded into ring buffer b % 2
  cudaEvent_t used[2] = {nullptr, nullptr};  // the compute that read ring buffer b % 2 has finished
};

inline exx_status cuda_fail(cudaError_t e) {
  g_last_cuda = e;
  return EXX_ERR_CUDA;
}

#define EXX_CUDA(call)                              \
  do {                                              \
    cudaError_t e__ = (call);                       \
    if (e__ != cudaSuccess) return cuda_fail(e__);  \
  } while (0)

inline bool overlaps(const void* a, size_t na, const void* b, size_t nb) {
  if (!a || !b || na == 0 || nb == 0) return false;
  const uintptr_t a0 = (uintptr_t)a, a1 = a0 + na, b0 = (uintptr_t)b, b1 = b0 + nb;
  return a0 < b1 && b0 < a1;
}

// the DMMA kernels serve every axis (n <= 128): no pass needs the second workspace half as scratch
inline bool all_axes_fast(const exx_plan* p) { return p->d_Vpad[0] && p->d_Vpad[1] && p->d_Vpad[2]; }

// a plan with a nonzero Bloch phase has complex eigenvectors: only the *_bloch entry points may use it
inline bool is_complex_plan(const exx_plan* p) { return p->bloch || p->d_Vi[0] || p->d_Vi[1] || p->d_Vi[2] ||
                                                         !p->h_Vi[0].empty() || !p->h_Vi[1].empty() || !p->h_Vi[2].empty(); }

// n_c == 0: about 4 GB of right-hand sides per batch (measured: larger batches only amortise launch ramps and tails,
// DESIGN.md section 9), at least kDefaultBatch, at most max_batch
inline int resolve_nc(const exx_plan* p, int n_c) {
  if (n_c == 0) {
    long long want = (4LL << 30) / (8 * p->N);  // about 4 GB of right-hand sides per batch
    if (want < kDefaultBatch) want = kDefaultBatch;
    n_c = want < p->max_batch ? (int)want : p->max_batch;
  }
  return n_c;
}

}  // namespace

namespace exx {
// for entry points that live in other files (energy_static.cu): the error exx_status_string shows for EXX_ERR_CUDA
void note_cuda_error(cudaError_t e) { g_last_cuda = e; }
}  // namespace exx

// plan-owned extras that are not part of the struct shared with the kernels
struct PlanExtras {
  double* d_energy_scratch = nullptr;  // kEnergyChunk * kEnergyBlocks doubles
  HostApiBuffers hb;
};
static PlanExtras* extras_of(const exx_plan* p);

struct exx_plan_full : exx_plan {
  PlanExtras ex;
};
static PlanExtras* extras_of(const exx_plan* p) {
  return &const_cast<exx_plan_full*>(static_cast<const exx_plan_full*>(p))->ex;
}

extern "C" {

const char* exx_version(void) { return "exx-b200 0.1 (sm_100a)"; }

const char* exx_status_string(exx_status s) {
  switch (s) {
    case EXX_OK: return "EXX_OK";
    case EXX_ERR_INVALID_ARG: return "EXX_ERR_INVALID_ARG: invalid argument";
    case EXX_ERR_ALLOC: return "EXX_ERR_ALLOC: allocation failed";
    case EXX_ERR_CUDA:
      snprintf(g_msg, sizeof(g_msg), "EXX_ERR_CUDA: %s (%s)", cudaGetErrorName(g_last_cuda),
               cudaGetErrorString(g_last_cuda));
      return g_msg;
    case EXX_ERR_EIGENSOLVE: return "EXX_ERR_EIGENSOLVE: Jacobi eigensolver did not converge";
    case EXX_ERR_WORKSPACE: return "EXX_ERR_WORKSPACE: workspace too small or missing";
    case EXX_ERR_ALIAS: return "EXX_ERR_ALIAS: output overlaps an input or the workspace";
    case EXX_ERR_LIMIT:
      return "EXX_ERR_LIMIT: size exceeds a capacity fixed at build time (exx_energy_static: at most "
             "EXX_ENERGY_STATIC_MAX_TGT = 4096 targets per call)";
  }
  return "unknown exx_status";
}

}  // extern "C"

// exx_plan_create / exx_plan_create_bloch (theta == nullptr: real plan)
static exx_status create_plan(exx_plan** out, int nx, int ny, int nz, double h, const int bc[3], int fd_order,
                              double omega, const double* theta, int max_batch, int device, int bloch_form = 0) {
  if (!out) return EXX_ERR_INVALID_ARG;
  *out = nullptr;
  if (nx < 1 || ny < 1 || nz < 1 || !(h > 0.0) || !std::isfinite(h) || !bc || fd_order < 2 ||
      (fd_order & 1) || fd_order > 64 || max_batch < 1 || max_batch > 65535 || !std::isfinite(omega))
    return EXX_ERR_INVALID_ARG;
  if ((long long)nx * ny * nz > (1LL << 31)) return EXX_ERR_INVALID_ARG;
  for (int a = 0; a < 3; ++a)
    if (bc[a] != EXX_BC_PERIODIC && bc[a] != EXX_BC_DIRICHLET) return EXX_ERR_INVALID_ARG;

  exx_plan_full* p = new (std::nothrow) exx_plan_full();
  if (!p) return EXX_ERR_ALLOC;
  p->n[0] = nx; p->n[1] = ny; p->n[2] = nz;
  p->h = h; p->order = fd_order; p->omega = omega; p->max_batch = max_batch; p->device = device;
  p->variant = EXX_VARIANT_FUSED_DMMA;
  p->N = (long long)nx * ny * nz;
  p->d_mult = nullptr; p->tma_state = nullptr; p->sm_count = 148; p->smem_optin = 0; p->last_launches = 0; p->last_solves = 0; p->tma_launches = 0;
  p->prof_on = false; p->accumulate = false;
  for (int c = 0; c < exx::PASS_COUNT; ++c) { p->prof_pass_ms[c] = 0.0; p->prof_pass_count[c] = 0; }
  p->fusion = 15;
  p->bloch = false;
  p->lanes = 1; p->lane_stream = nullptr; p->ev_fork = nullptr; p->ev_join = nullptr;
  for (int a = 0; a < 3; ++a) {
    p->bc[a] = bc[a]; p->d_V[a] = nullptr; p->d_Vpad[a] = nullptr; p->d_Vi[a] = nullptr; p->bfly[a] = false;
    // a Bloch phase only exists on a periodic axis; theta == 0 there is the real periodic matrix
    p->theta[a] = (theta && bc[a] == EXX_BC_PERIODIC) ? theta[a] : 0.0;
    if (theta && !std::isfinite(theta[a])) { delete p; return EXX_ERR_INVALID_ARG; }
  }

  try {
    for (int a = 0; a < 3; ++a) {
      // identical axes share the eigendecomposition (and, on the device, the matrix)
      int same = -1;
      for (int b = 0; b < a; ++b)
        if (p->n[b] == p->n[a] && p->bc[b] == p->bc[a] && p->theta[b] == p->theta[a]) same = b;
      if (same >= 0) {
        p->h_lam[a] = p->h_lam[same];
        p->h_V[a] = p->h_V[same];
        p->h_Vi[a] = p->h_Vi[same];
        p->h_Vc_re[a] = p->h_Vc_re[same];
        p->h_Vc_im[a] = p->h_Vc_im[same];
        p->bfly[a] = p->bfly[same];
        continue;
      }
      if (p->theta[a] != 0.0 && bloch_form == EXX_BLOCH_FORM_EMBEDDED) {
        // cross-check form: complex eigenvectors, products on the real embedding [[Mr, -Mi], [Mi, Mr]]
        if (!exx::bloch_eigh(p->n[a], h, fd_order, p->theta[a], p->h_lam[a], p->h_V[a], p->h_Vi[a])) {
          delete p;
          return EXX_ERR_EIGENSOLVE;
        }
        p->bloch = true;
        continue;
      }
      if (p->theta[a] != 0.0) {
        // the axis in its real form: h_V = W (real orthogonal), the kernels apply the butterfly U around the real products
        if (!exx::bloch_eigh_real_form(p->n[a], h, fd_order, p->theta[a], p->h_lam[a], p->h_V[a], p->h_Vc_re[a],
                                       p->h_Vc_im[a])) {
          delete p;
          return EXX_ERR_EIGENSOLVE;
        }
        p->bfly[a] = true;
        p->bloch = true;
        continue;
      }
      std::vector<double> K = exx::second_derivative_matrix(p->n[a], h, bc[a], fd_order);
      if (!exx::jacobi_eigh(p->n[a], K, p->h_lam[a], p->h_V[a])) {
        delete p;
        return EXX_ERR_EIGENSOLVE;
      }
    }
    const double w0 = std::fabs(exx::fd_weights(fd_order, h)[0]);
    p->zero_tol = 1e-8 * 3.0 * w0;
    p->h_mult = exx::multiplier_table(p->h_lam[0], p->h_lam[1], p->h_lam[2], omega, p->zero_tol);
  } catch (const std::bad_alloc&) {
    delete p;
    return EXX_ERR_ALLOC;
  }

  if (device >= 0) {  // device < 0: host-only plan (planner tests); compute calls return EXX_ERR_CUDA
    DeviceScope dev_scope(device);  // the caller's current device is restored on return
    cudaError_t e = dev_scope.err;
    if (e == cudaSuccess) e = cudaDeviceGetAttribute(&p->sm_count, cudaDevAttrMultiProcessorCount, device);
    if (e == cudaSuccess)
      e = cudaDeviceGetAttribute(&p->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, device);
    for (int a = 0; a < 3 && e == cudaSuccess; ++a) {
      int same = -1;
      for (int b = 0; b < a; ++b)
        if (p->n[b] == p->n[a] && p->bc[b] == p->bc[a] && p->theta[b] == p->theta[a]) same = b;
      if (same >= 0) { p->d_V[a] = p->d_V[same]; p->d_Vi[a] = p->d_Vi[same]; continue; }
      const size_t bytes = sizeof(double) * p->h_V[a].size();
      e = cudaMalloc(&p->d_V[a], bytes);
      if (e == cudaSuccess) e = cudaMemcpy(p->d_V[a], p->h_V[a].data(), bytes, cudaMemcpyHostToDevice);
      if (e == cudaSuccess && !p->h_Vi[a].empty()) {
        e = cudaMalloc(&p->d_Vi[a], bytes);
        if (e == cudaSuccess) e = cudaMemcpy(p->d_Vi[a], p->h_Vi[a].data(), bytes, cudaMemcpyHostToDevice);
      }
    }
    if (e == cudaSuccess) e = cudaMalloc(&p->d_mult, sizeof(double) * p->N);
    if (e == cudaSuccess)
      e = cudaMemcpy(p->d_mult, p->h_mult.data(), sizeof(double) * p->N, cudaMemcpyHostToDevice);
    if (e == cudaSuccess)
      e = cudaMalloc(&p->ex.d_energy_scratch, sizeof(double) * kEnergyChunk * kEnergyBlocks);
    if (e == cudaSuccess) e = exx::fast_init(p);
    if (e == cudaSuccess) e = exx::tma_init(p);
    if (e == cudaSuccess) e = exx::sym_init(p);
    if (e == cudaSuccess) e = exx::fused_init(p);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&p->lane_stream, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_fork, cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&p->ev_join, cudaEventDisableTiming);
    if (e != cudaSuccess) {
      exx_plan_destroy(p);
      return e == cudaErrorMemoryAllocation ? EXX_ERR_ALLOC : cuda_fail(e);
    }
  }
  *out = p;
  return EXX_OK;
}

extern "C" {

exx_status exx_plan_create(exx_plan** out, int nx, int ny, int nz, double h, const int bc[3],
                           int fd_order, double omega, int max_batch, int device) {
  return create_plan(out, nx, ny, nz, h, bc, fd_order, omega, nullptr, max_batch, device);
}

exx_status exx_plan_create_bloch(exx_plan** out, int nx, int ny, int nz, double h, const int bc[3], int fd_order,
                                 double omega, const double theta[3], int max_batch, int device) {
  if (!theta) return EXX_ERR_INVALID_ARG;
  return create_plan(out, nx, ny, nz, h, bc, fd_order, omega, theta, max_batch, device);
}

exx_status exx_plan_create_bloch_form(exx_plan** out, int nx, int ny, int nz, double h, const int bc[3], int fd_order,
                                      double omega, const double theta[3], int max_batch, int device, int form) {
  if (!theta || (form != EXX_BLOCH_FORM_REAL && form != EXX_BLOCH_FORM_EMBEDDED)) return EXX_ERR_INVALID_ARG;
  return create_plan(out, nx, ny, nz, h, bc, fd_order, omega, theta, max_batch, device, form);
}

exx_status exx_plan_destroy(exx_plan* plan) {
  if (!plan) return EXX_OK;
  exx_plan_full* p = static_cast<exx_plan_full*>(plan);
  if (p->device >= 0) {
    DeviceScope dev_scope(p->device);
    exx::fast_destroy(p);
    exx::fused_destroy(p);
    exx::sym_destroy(p);
    exx::tma_destroy(p);
    if (p->lane_stream) cudaStreamDestroy(p->lane_stream);
    if (p->ev_fork) cudaEventDestroy(p->ev_fork);
    if (p->ev_join) cudaEventDestroy(p->ev_join);
    for (int a = 0; a < 3; ++a) {
      bool shared = false;
      for (int b = 0; b < a; ++b) shared |= (p->d_V[b] == p->d_V[a]);
      if (!shared && p->d_V[a]) cudaFree(p->d_V[a]);
      if (!shared && p->d_Vi[a]) cudaFree(p->d_Vi[a]);
    }
    if (p->d_mult) cudaFree(p->d_mult);
    if (p->ex.d_energy_scratch) cudaFree(p->ex.d_energy_scratch);
    if (p->ex.hb.base) cudaFree(p->ex.hb.base);
    if (p->ex.hb.stream) cudaStreamDestroy(p->ex.hb.stream);
    if (p->ex.hb.copy_stream) cudaStreamDestroy(p->ex.hb.copy_stream);
    for (int c = 0; c < kHostChunks; ++c)
      if (p->ex.hb.done[c]) cudaEventDestroy(p->ex.hb.done[c]);
    for (int c = 0; c < 2; ++c) {
      if (p->ex.hb.up[c]) cudaEventDestroy(p->ex.hb.up[c]);
      if (p->ex.hb.used[c]) cudaEventDestroy(p->ex.hb.used[c]);
    }
  }
  delete p;
  return EXX_OK;
}

exx_status exx_plan_set_variant(exx_plan* plan, int variant) {
  if (!plan || (variant != EXX_VARIANT_FUSED_DMMA && variant != EXX_VARIANT_REFERENCE && variant != EXX_VARIANT_CPASYNC))
    return EXX_ERR_INVALID_ARG;
  plan->variant = variant;
  return EXX_OK;
}

exx_status exx_plan_set_lanes(exx_plan* plan, int lanes) {
  if (!plan || (lanes != 1 && lanes != 2)) return EXX_ERR_INVALID_ARG;
  if (lanes == 2 && (plan->device < 0 || !all_axes_fast(plan))) return EXX_ERR_INVALID_ARG;
  plan->lanes = lanes;
  return EXX_OK;
}

int exx_plan_get_lanes(const exx_plan* plan) { return plan ? plan->lanes : 0; }

exx_status exx_plan_set_fusion(exx_plan* plan, int mask) {
  if (!plan || mask < 0 || mask > 15) return EXX_ERR_INVALID_ARG;
  plan->fusion = mask;
  return EXX_OK;
}

int exx_plan_get_fusion(const exx_plan* plan) { return plan ? plan->fusion : 0; }

exx_status exx_plan_set_accumulate(exx_plan* plan, int on) {
  if (!plan) return EXX_ERR_INVALID_ARG;
  plan->accumulate = on != 0;
  return EXX_OK;
}

size_t exx_plan_workspace_bytes(const exx_plan* plan, int n_c) {
  if (!plan) return 0;
  n_c = resolve_nc(plan, n_c);
  if (n_c < 1 || n_c > plan->max_batch) return 0;
  return 2 * sizeof(double) * (size_t)plan->N * (size_t)n_c;
}

exx_status exx_plan_get_axis(const exx_plan* plan, int axis, double* h_lambda, double* h_V) {
  if (!plan || axis < 0 || axis > 2) return EXX_ERR_INVALID_ARG;
  const int n = plan->n[axis];
  if (h_lambda) std::memcpy(h_lambda, plan->h_lam[axis].data(), sizeof(double) * n);
  if (h_V)
    for (int i = 0; i < n; ++i)
      for (int m = 0; m < n; ++m) h_V[i + (size_t)n * m] = plan->h_V[axis][(size_t)i * n + m];
  return EXX_OK;
}

exx_status exx_plan_get_axis_symmetric(const exx_plan* plan, int axis, double* h_lambda, double* h_V, int* n_even) {
  // a Bloch axis has no reflection-adapted real basis: in the embedded form its eigenvectors are complex (h_Vi), in the
  // real form (bfly) h_V holds W of K' = U^H K U, which the periodic reflection does not act on
  if (!plan || axis < 0 || axis > 2 || !plan->h_Vi[axis].empty() || plan->bfly[axis]) return EXX_ERR_INVALID_ARG;
  const int n = plan->n[axis];
  std::vector<double> lam_s, Vs;
  int nh = 0;
  if (!exx::symmetrize_axis(n, plan->bc[axis], plan->h_lam[axis], plan->h_V[axis], lam_s, Vs, &nh, true)) return EXX_ERR_EIGENSOLVE;
  if (h_lambda) std::memcpy(h_lambda, lam_s.data(), sizeof(double) * n);
  if (h_V)
    for (int i = 0; i < n; ++i)
      for (int m = 0; m < n; ++m) h_V[i + (size_t)n * m] = Vs[(size_t)i * n + m];
  if (n_even) *n_even = nh;
  return EXX_OK;
}

exx_status exx_plan_get_multiplier(const exx_plan* plan, double* h_mult) {
  if (!plan || !h_mult) return EXX_ERR_INVALID_ARG;
  std::memcpy(h_mult, plan->h_mult.data(), sizeof(double) * plan->N);
  return EXX_OK;
}

double exx_plan_executed_flops_per_solve(const exx_plan* plan) {
  if (!plan) return 0.0;
  if (plan->device < 0 || is_complex_plan(plan)) return 4.0 * (double)plan->N * (plan->n[0] + plan->n[1] + plan->n[2]);
  return exx::fused_executed_flops_per_solve(plan);
}

double exx_plan_executed_flops_per_symmetric_solve(const exx_plan* plan) {
  if (!plan) return 0.0;
  if (plan->device < 0 || is_complex_plan(plan)) return 4.0 * (double)plan->N * (plan->n[0] + plan->n[1] + plan->n[2]);
  return exx::fused_executed_flops_per_solve(plan, true);
}

long long exx_plan_last_launch_count(const exx_plan* plan) { return plan ? plan->last_launches : 0; }

long long exx_plan_last_solve_count(const exx_plan* plan) { return plan ? plan->last_solves : 0; }

long long exx_plan_tma_launch_count(const exx_plan* plan) { return plan ? plan->tma_launches : 0; }

exx_status exx_plan_set_profiling(exx_plan* plan, int on) {
  if (!plan) return EXX_ERR_INVALID_ARG;
  plan->prof_on = on != 0;
  return EXX_OK;
}

exx_status exx_plan_get_profile(exx_plan* plan, double* h_ms, long long* h_count) {
  if (!plan || !h_ms || !h_count) return EXX_ERR_INVALID_ARG;
  for (int c = 0; c < exx::KC_COUNT; ++c) { h_ms[c] = 0.0; h_count[c] = 0; }
  for (int c = 0; c < exx::PASS_COUNT; ++c) { plan->prof_pass_ms[c] = 0.0; plan->prof_pass_count[c] = 0; }
  cudaError_t err = cudaSuccess;
  for (auto& r : plan->prof) {
    float ms = 0.f;
    cudaError_t e = cudaEventSynchronize(r.e1);
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, r.e0, r.e1);
    if (e != cudaSuccess) err = e;
    else {
      h_ms[r.cls] += ms;
      h_count[r.cls] += 1;
      if (r.pass >= 0 && r.pass < exx::PASS_COUNT) { plan->prof_pass_ms[r.pass] += ms; plan->prof_pass_count[r.pass] += 1; }
    }
    cudaEventDestroy(r.e0);
    cudaEventDestroy(r.e1);
  }
  plan->prof.clear();
  return err == cudaSuccess ? EXX_OK : cuda_fail(err);
}

exx_status exx_plan_get_profile_passes(const exx_plan* plan, double* h_ms, long long* h_count, double* h_flops_per_solve) {
  if (!plan || !h_ms || !h_count) return EXX_ERR_INVALID_ARG;
  for (int c = 0; c < exx::PASS_COUNT; ++c) {
    h_ms[c] = plan->prof_pass_ms[c];
    h_count[c] = plan->prof_pass_count[c];
    if (h_flops_per_solve) h_flops_per_solve[c] = 0.0;
  }
  if (h_flops_per_solve && plan->device >= 0 && !is_complex_plan(plan)) {
    // executed operations of one product per axis (exx_plan_executed_flops_per_solve counts two per axis)
    const int ax_of[exx::PASS_COUNT] = {0, 1, 2, 2, 1, 0, 0, -1};
    for (int c = 0; c < exx::PASS_COUNT; ++c)
      if (ax_of[c] >= 0) h_flops_per_solve[c] = exx::fused_executed_flops_axis(plan, ax_of[c]);
    if (plan->prof_pass_count[exx::PASS_ZB] == 0) {  // fused z pass: both z products in PASS_Z
      h_flops_per_solve[exx::PASS_Z] *= 2.0;
      h_flops_per_solve[exx::PASS_ZB] = 0.0;
    }
  }
  return EXX_OK;
}

}  // extern "C"

namespace {

// One batch of the reference variant: buf0 holds the right-hand sides on entry, phi on exit.
cudaError_t ref_solve_batch(exx_plan* p, double* buf0, double* buf1, int nb, cudaStream_t s,
                            long long* launches) {
  cudaError_t e;
  const int axis[6] = {0, 1, 2, 2, 1, 0};
  double *src = buf0, *dst = buf1;
  for (int i = 0; i < 6; ++i) {
    {
      exx::ProfScope ps(p, exx::KC_MODE_PRODUCT, s);
      e = exx::ref_mode_product(p, axis[i], i < 3, src, dst, nb, i == 2, s);
    }
    if (e != cudaSuccess) return e;
    double* t = src; src = dst; dst = t;
  }
  *launches += 6;
  return cudaSuccess;
}

}  // namespace

// a6 for n_tgt targets: e_k = h^3 <tgt_k, vx_k>, *d_ex = 1/2 sum_k occ_tgt_k e_k (chunked: bounded plan-owned scratch)
static exx_status run_energy(exx_plan* plan, const double* d_tgt, const double* d_vx, const double* d_occ_tgt, int n_tgt,
                             double* d_ex, double* d_ex_k, cudaStream_t s, long long* launches) {
  PlanExtras* ex = extras_of(plan);
  const size_t N = (size_t)plan->N;
  for (int k0 = 0; k0 < n_tgt; k0 += kEnergyChunk) {
    const int nk = n_tgt - k0 < kEnergyChunk ? n_tgt - k0 : kEnergyChunk;
    if (k0 == 0 && d_ex) { EXX_CUDA(exx::zero_fill(plan, d_ex, 1, s)); ++*launches; }   // the first chunk overwrites *d_ex
    {
      exx::ProfScope ps(plan, exx::KC_OTHER, s);
      EXX_CUDA(exx::energy(plan, d_tgt + N * (size_t)k0, d_vx + N * (size_t)k0, d_occ_tgt ? d_occ_tgt + k0 : nullptr,
                           nk, ex->d_energy_scratch, d_ex_k ? d_ex_k + k0 : nullptr, d_ex, s));
    }
    *launches += 2;
  }
  return EXX_OK;
}

extern "C" {

exx_status exx_poisson_solve(exx_plan* plan, const double* d_rhs, double* d_phi, int n_rhs, int n_c,
                             void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_rhs < 0 || (n_rhs > 0 && (!d_rhs || !d_phi))) return EXX_ERR_INVALID_ARG;
  if (is_complex_plan(plan)) return EXX_ERR_INVALID_ARG;
  n_c = resolve_nc(plan, n_c);
  if (n_c < 1 || n_c > plan->max_batch) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  if (n_rhs == 0) { plan->last_launches = 0; return EXX_OK; }
  const size_t need = exx_plan_workspace_bytes(plan, n_c);
  if (!d_workspace || workspace_bytes < need) return EXX_ERR_WORKSPACE;
  const size_t N = (size_t)plan->N, fn = sizeof(double) * N;
  if (d_rhs != d_phi && overlaps(d_rhs, fn * n_rhs, d_phi, fn * n_rhs)) return EXX_ERR_ALIAS;
  if (overlaps(d_workspace, need, d_phi, fn * n_rhs) || overlaps(d_workspace, need, d_rhs, fn * n_rhs))
    return EXX_ERR_ALIAS;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  double* buf0 = (double*)d_workspace;
  double* buf1 = buf0 + N * (size_t)n_c;
  long long launches = 0;
  for (int b0 = 0; b0 < n_rhs; b0 += n_c) {
    const int nb = n_rhs - b0 < n_c ? n_rhs - b0 : n_c;
    if (plan->variant == EXX_VARIANT_REFERENCE) {
      EXX_CUDA(cudaMemcpyAsync(buf0, d_rhs + N * (size_t)b0, fn * nb, cudaMemcpyDeviceToDevice, s));
      EXX_CUDA(ref_solve_batch(plan, buf0, buf1, nb, s, &launches));
      EXX_CUDA(cudaMemcpyAsync(d_phi + N * (size_t)b0, buf0, fn * nb, cudaMemcpyDeviceToDevice, s));
    } else {
      // first product reads the right-hand sides where they are and writes phi's storage; the other five
      // run in place there (no staging copies)
      EXX_CUDA(exx::fast_solve_batch(plan, d_rhs + N * (size_t)b0, d_phi + N * (size_t)b0, buf0, nb, nullptr, s,
                                     &launches));
    }
  }
  plan->last_launches = launches;
  return EXX_OK;
}

exx_status exx_poisson_solve_nonbatch(exx_plan* plan, const double* d_rhs, double* d_phi, int n_rhs, void* d_workspace,
                                      size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_rhs < 0 || (n_rhs > 0 && (!d_rhs || !d_phi))) return EXX_ERR_INVALID_ARG;
  if (is_complex_plan(plan)) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  if (n_rhs == 0) { plan->last_launches = 0; return EXX_OK; }
  const size_t N = (size_t)plan->N, fn = sizeof(double) * N;
  const size_t need = 2 * fn;
  if (!d_workspace || workspace_bytes < need) return EXX_ERR_WORKSPACE;
  if (d_rhs != d_phi && overlaps(d_rhs, fn * n_rhs, d_phi, fn * n_rhs)) return EXX_ERR_ALIAS;
  if (overlaps(d_workspace, need, d_phi, fn * n_rhs) || overlaps(d_workspace, need, d_rhs, fn * n_rhs))
    return EXX_ERR_ALIAS;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  double* buf0 = (double*)d_workspace;
  long long launches = 0;
  for (int b = 0; b < n_rhs; ++b)
    EXX_CUDA(exx::nonbatch_solve_one(plan, d_rhs + N * (size_t)b, d_phi + N * (size_t)b, buf0, buf0 + N, s, &launches));
  plan->last_launches = launches;
  return EXX_OK;
}

exx_status exx_apply(exx_plan* plan, const double* d_psi, const double* d_occ, int n_occ,
                     const double* d_tgt, const double* d_occ_tgt, int n_tgt, double* d_vx,
                     double* d_ex, double* d_ex_k, int n_c, void* d_workspace,
                     size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_occ < 0 || n_tgt < 0) return EXX_ERR_INVALID_ARG;
  if (is_complex_plan(plan)) return EXX_ERR_INVALID_ARG;
  if (n_occ > 0 && (!d_psi || !d_occ)) return EXX_ERR_INVALID_ARG;
  if (n_tgt > 0 && (!d_tgt || !d_vx)) return EXX_ERR_INVALID_ARG;
  if (d_ex && !d_occ_tgt && n_tgt > 0) return EXX_ERR_INVALID_ARG;
  n_c = resolve_nc(plan, n_c);
  if (n_c < 1 || n_c > plan->max_batch) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  const size_t N = (size_t)plan->N, fn = sizeof(double) * N;
  const size_t need = exx_plan_workspace_bytes(plan, n_c);
  if (n_occ > 0 && n_tgt > 0 && (!d_workspace || workspace_bytes < need)) return EXX_ERR_WORKSPACE;
  if (overlaps(d_vx, fn * n_tgt, d_psi, fn * n_occ) || overlaps(d_vx, fn * n_tgt, d_tgt, fn * n_tgt) ||
      overlaps(d_vx, fn * n_tgt, d_workspace, need) || overlaps(d_workspace, need, d_psi, fn * n_occ) ||
      overlaps(d_workspace, need, d_tgt, fn * n_tgt))
    return EXX_ERR_ALIAS;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  long long launches = 0;
  PlanExtras* ex = extras_of(plan);

  if (n_tgt > 0 && n_occ == 0) {
    if (!plan->accumulate) {
      EXX_CUDA(exx::zero_fill(plan, d_vx, (long long)N * n_tgt, s));
      ++launches;
    }
  } else if (n_tgt > 0) {
    double* buf0 = (double*)d_workspace;
    double* buf1 = buf0 + N * (size_t)n_c;
    // Batch = nk targets x nj occupied orbitals, nj*nk <= n_c.  With n_occ >= n_c one target per batch.
    int nj_max = n_occ < n_c ? n_occ : n_c;
    // Fused x-backward + accumulate (k_mode_xacc): a work item is (row tile, target) and loops over the batch's j, so a
    // batch needs enough targets to give every warp several items; nj only has to amortise the read-modify-write of
    // vx_k (16/nj bytes per point and pair).  The sum over j is ascending whatever the shape.
    const int xacc_rows = plan->variant == EXX_VARIANT_FUSED_DMMA && (plan->fusion & 2) ? exx::fused_xacc_tile_rows(plan) : 0;
    if (xacc_rows > 0 && !(plan->n[0] & 1)) {
      const long long tiles_per_rhs = (N / plan->n[0] + xacc_rows - 1) / xacc_rows;
      // about kItemsPerWarp items for each of the 12 warps of an SM: the items of a launch are uniform, so the last round
      // of an uneven split idles (items/warps)/ceil(items/warps) of the machine
      long long nk_want = ((long long)kItemsPerWarp * 12 * plan->sm_count + tiles_per_rhs - 1) / tiles_per_rhs;
      if (nk_want > n_tgt) nk_want = n_tgt;
      if (nk_want > n_c) nk_want = n_c;
      int nj = (int)(n_c / nk_want);
      const int nj_floor = n_occ < 8 ? n_occ : 8;
      if (nj < nj_floor) nj = nj_floor < n_c ? nj_floor : n_c;
      if (nj < nj_max) nj_max = nj;
    }
    const int nk_max = n_c / nj_max;
    // Two lanes: target block kb runs on lane kb % 2 (all its j-batches in order, so vx_k is accumulated in
    // the same order as with one lane and no vx_k is touched by both lanes); lane 1 works in the second half
    // of the workspace on the plan's own stream, forked from and joined back into the caller's stream.
    const int n_kblocks = (n_tgt + nk_max - 1) / nk_max;
    const bool two_lanes = plan->variant != EXX_VARIANT_REFERENCE && plan->lanes == 2 && n_kblocks > 1 &&
                           all_axes_fast(plan);
    if (two_lanes) {
      EXX_CUDA(cudaEventRecord(plan->ev_fork, s));
      EXX_CUDA(cudaStreamWaitEvent(plan->lane_stream, plan->ev_fork, 0));
    }
    int kb = 0;
    for (int k0 = 0; k0 < n_tgt; k0 += nk_max, ++kb) {
      const int nk = n_tgt - k0 < nk_max ? n_tgt - k0 : nk_max;
      const bool lane1 = two_lanes && (kb & 1);
      cudaStream_t ls = lane1 ? plan->lane_stream : s;
      for (int j0 = 0; j0 < n_occ; j0 += nj_max) {
        const int nj = n_occ - j0 < nj_max ? n_occ - j0 : nj_max;
        const exx::BatchDesc bd{j0, nj, k0, nk};
        const int nb = nj * nk;
        if (plan->variant == EXX_VARIANT_REFERENCE) {
          {
            exx::ProfScope ps(plan, exx::KC_PAIR_DENSITY, s);
            EXX_CUDA(exx::ref_pair_density(plan, d_psi, d_tgt, bd, buf0, s));
          }
          EXX_CUDA(ref_solve_batch(plan, buf0, buf1, nb, s, &launches));
          {
            exx::ProfScope ps(plan, exx::KC_ACCUMULATE, s);
            EXX_CUDA(exx::ref_accumulate(plan, d_psi, d_occ, buf0, bd, j0 == 0 && !plan->accumulate, d_vx, s));
          }
          launches += 2;
        } else {
          const exx::FastArgs fa{d_psi, d_tgt, d_occ, d_vx, bd, n_occ, n_tgt, j0 == 0 && !plan->accumulate, false};
          EXX_CUDA(exx::fast_solve_batch(plan, nullptr, lane1 ? buf1 : buf0, two_lanes ? nullptr : buf1, nb, &fa, ls,
                                         &launches));
        }
      }
    }
    if (two_lanes) {
      EXX_CUDA(cudaEventRecord(plan->ev_join, plan->lane_stream));
      EXX_CUDA(cudaStreamWaitEvent(s, plan->ev_join, 0));
    }
  }
  if (d_ex && n_tgt == 0) {
    EXX_CUDA(exx::zero_fill(plan, d_ex, 1, s));
    ++launches;
  }
  if ((d_ex || d_ex_k) && n_tgt > 0) {
    exx_status st = run_energy(plan, d_tgt, d_vx, d_occ_tgt, n_tgt, d_ex, d_ex_k, s, &launches);
    if (st != EXX_OK) return st;
  }
  plan->last_launches = launches;
  plan->last_solves = (long long)n_occ * n_tgt;
  return EXX_OK;
}

exx_status exx_apply_symmetric(exx_plan* plan, const double* d_psi, const double* d_occ, int n_orb, double* d_vx,
                               double* d_ex, double* d_ex_k, int n_c, void* d_workspace, size_t workspace_bytes,
                               void* cuda_stream) {
  if (!plan || n_orb < 0 || is_complex_plan(plan)) return EXX_ERR_INVALID_ARG;
  if (n_orb > 0 && (!d_psi || !d_occ || !d_vx)) return EXX_ERR_INVALID_ARG;
  n_c = resolve_nc(plan, n_c);
  if (n_c < 1 || n_c > plan->max_batch) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  const size_t N = (size_t)plan->N, fn = sizeof(double) * N;
  const size_t need = exx_plan_workspace_bytes(plan, n_c);
  if (n_orb > 0 && (!d_workspace || workspace_bytes < need)) return EXX_ERR_WORKSPACE;
  if (overlaps(d_vx, fn * n_orb, d_psi, fn * n_orb) || overlaps(d_vx, fn * n_orb, d_workspace, need) ||
      overlaps(d_workspace, need, d_psi, fn * n_orb))
    return EXX_ERR_ALIAS;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  long long launches = 0, solves = 0;
  PlanExtras* ex = extras_of(plan);
  double* buf0 = (double*)d_workspace;
  double* buf1 = buf0 + N * (size_t)n_c;
  if (n_orb > 0) {
    // contributions are scattered to vx_k and vx_j: start from zero, every batch accumulates
    EXX_CUDA(exx::zero_fill(plan, d_vx, (long long)N * n_orb, s));
    ++launches;
  }
  auto run_batch = [&](int j0, int nj, int k0, int nk) -> exx_status {
    const exx::BatchDesc bd{j0, nj, k0, nk};
    const int nb = nj * nk;
    solves += nb;
    if (plan->variant == EXX_VARIANT_REFERENCE) {
      {
        exx::ProfScope ps(plan, exx::KC_PAIR_DENSITY, s);
        EXX_CUDA(exx::ref_pair_density(plan, d_psi, d_psi, bd, buf0, s));
      }
      EXX_CUDA(ref_solve_batch(plan, buf0, buf1, nb, s, &launches));
      {
        exx::ProfScope ps(plan, exx::KC_ACCUMULATE, s);
        EXX_CUDA(exx::ref_accumulate(plan, d_psi, d_occ, buf0, bd, false, d_vx, s, true));
        EXX_CUDA(exx::sym_accumulate_transposed(plan, d_psi, d_occ, buf0, bd, d_vx, s));
      }
      launches += 3;
    } else {
      const exx::FastArgs fa{d_psi, d_psi, d_occ, d_vx, bd, n_orb, n_orb, false, true};
      EXX_CUDA(exx::fast_solve_batch(plan, nullptr, buf0, buf1, nb, &fa, s, &launches));
    }
    return EXX_OK;
  };
  // Batches are rectangles of the (j,k) plane that cover the triangle j <= k: a block of nk consecutive targets
  // against the orbitals 0 .. k0+nk-1 (the nk(nk-1)/2 pairs with j > k inside the diagonal block are solved and
  // ignored), nk as large as n_c allows; a block with more than n_c pairs is cut into j-chunks.  Where both sides of
  // the accumulate run fused with the x-backward product (k_mode_xacc_sym, twice), a block has enough targets (at most
  // 8) to give every warp of the target-side pass a work item.
  int nk_min = 1;
  if (plan->variant == EXX_VARIANT_FUSED_DMMA && n_orb > 0) {
    const exx::FastArgs probe{d_psi, d_psi, d_occ, d_vx, exx::BatchDesc{0, 1, 0, 1}, n_orb, n_orb, false, true};
    const int rows = exx::sym_xacc_tile_rows(plan);
    if (rows > 0 && exx::fused_sym_mode(plan) && exx::sym_x_usable(plan, buf0, &probe)) {
      const long long tiles = ((long long)(N / plan->n[0]) + rows - 1) / rows;
      const long long want = (12LL * plan->sm_count + tiles - 1) / tiles;
      nk_min = (int)(want < 1 ? 1 : want > 8 ? 8 : want);
    }
  }
  for (int k0 = 0; k0 < n_orb;) {
    int nk = 1;
    while (k0 + nk + 1 <= n_orb && (long long)(nk + 1) * (k0 + nk + 1) <= n_c) ++nk;
    if (nk < nk_min) nk = nk_min;
    if (nk > n_orb - k0) nk = n_orb - k0;
    if (nk > n_c) nk = n_c;
    const int nj_max = n_c / nk;
    for (int j0 = 0; j0 < k0 + nk; j0 += nj_max) {
      const int nj = k0 + nk - j0 < nj_max ? k0 + nk - j0 : nj_max;
      exx_status st = run_batch(j0, nj, k0, nk);
      if (st != EXX_OK) return st;
    }
    k0 += nk;
  }
  if (d_ex && n_orb == 0) {
    EXX_CUDA(exx::zero_fill(plan, d_ex, 1, s));
    ++launches;
  }
  if ((d_ex || d_ex_k) && n_orb > 0) {
    for (int k0 = 0; k0 < n_orb; k0 += kEnergyChunk) {
      const int nk = n_orb - k0 < kEnergyChunk ? n_orb - k0 : kEnergyChunk;
      if (k0 == 0 && d_ex) { EXX_CUDA(exx::zero_fill(plan, d_ex, 1, s)); ++launches; }
      {
        exx::ProfScope ps(plan, exx::KC_OTHER, s);
        EXX_CUDA(exx::energy(plan, d_psi + N * (size_t)k0, d_vx + N * (size_t)k0, d_occ + k0, nk,
                             ex->d_energy_scratch, d_ex_k ? d_ex_k + k0 : nullptr, d_ex, s));
      }
      launches += 2;
    }
  }
  plan->last_launches = launches;
  plan->last_solves = solves;
  return EXX_OK;
}

exx_status exx_apply_host(exx_plan* plan, const double* h_psi, const double* h_occ, int n_occ,
                          const double* h_tgt, int tgt_start, const double* h_occ_tgt, int n_tgt,
                          double* h_vx, double* h_ex, double* h_ex_k, int n_c) {
  if (!plan || n_occ < 0 || n_tgt < 0 || (n_occ > 0 && (!h_psi || !h_occ))) return EXX_ERR_INVALID_ARG;
  const bool tgt_in_psi = tgt_start >= 0;
  if (tgt_in_psi && tgt_start + n_tgt > n_occ) return EXX_ERR_INVALID_ARG;
  if (!tgt_in_psi && n_tgt > 0 && !h_tgt) return EXX_ERR_INVALID_ARG;
  if (h_ex && !h_occ_tgt && n_tgt > 0) return EXX_ERR_INVALID_ARG;
  if (is_complex_plan(plan)) return EXX_ERR_INVALID_ARG;
  n_c = resolve_nc(plan, n_c);
  if (n_c < 1 || n_c > plan->max_batch) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  PlanExtras* ex = extras_of(plan);
  const size_t N = (size_t)plan->N;
  const size_t ws = exx_plan_workspace_bytes(plan, n_c);
  // Orbital blocks (Eq. 1's sum over j split with the plan's accumulate mode): with more orbitals than a batch holds,
  // a block is one batch's worth of orbitals (n_c); otherwise the set is cut into kHostChunks blocks so that the
  // upload of block b+1 still overlaps the compute of block b.  Only two blocks are resident at a time.
  int blk = n_occ > n_c ? n_c : (n_occ + kHostChunks - 1) / kHostChunks;
  if (blk < 1) blk = 1;
  const int n_blocks = n_occ > 0 ? (n_occ + blk - 1) / blk : 0;
  const int n_buf = n_blocks > 1 ? 2 : 1;
  // carve: tgt | vx | psi block ring | occ | occ_tgt | ex_k | ex | workspace
  size_t n_dbl = 2 * N * n_tgt + (size_t)n_buf * N * blk + n_occ + 2 * (size_t)n_tgt + 8;
  size_t bytes = sizeof(double) * n_dbl + ws + 512;
  if (ex->hb.bytes < bytes) {
    if (ex->hb.base) cudaFree(ex->hb.base);
    ex->hb.base = nullptr; ex->hb.bytes = 0;
    cudaError_t e = cudaMalloc(&ex->hb.base, bytes);
    if (e != cudaSuccess) { g_last_cuda = e; return EXX_ERR_ALLOC; }
    ex->hb.bytes = bytes;
  }
  if (!ex->hb.stream) EXX_CUDA(cudaStreamCreateWithFlags(&ex->hb.stream, cudaStreamNonBlocking));
  if (!ex->hb.copy_stream) {
    EXX_CUDA(cudaStreamCreateWithFlags(&ex->hb.copy_stream, cudaStreamNonBlocking));
    for (int c = 0; c < kHostChunks; ++c) EXX_CUDA(cudaEventCreateWithFlags(&ex->hb.done[c], cudaEventDisableTiming));
    for (int c = 0; c < 2; ++c) {
      EXX_CUDA(cudaEventCreateWithFlags(&ex->hb.up[c], cudaEventDisableTiming));
      EXX_CUDA(cudaEventCreateWithFlags(&ex->hb.used[c], cudaEventDisableTiming));
    }
  }
  cudaStream_t s = ex->hb.stream, cs = ex->hb.copy_stream;
  double* q = ex->hb.base;
  double* d_tgt = q; q += N * n_tgt;
  double* d_vx = q; q += N * n_tgt;
  double* d_blk[2] = {q, q + (n_buf > 1 ? N * (size_t)blk : 0)}; q += (size_t)n_buf * N * blk;
  double* d_occ = q; q += n_occ;
  double* d_occ_tgt = q; q += n_tgt;
  double* d_ex_k = q; q += n_tgt;
  double* d_ex = q; q += 8;
  void* d_ws = (void*)(((uintptr_t)q + 255) & ~(uintptr_t)255);

  auto upload_block = [&](int b) -> exx_status {  // on the copy stream, once the buffer's previous user is done
    const int j0 = b * blk, nj = n_occ - j0 < blk ? n_occ - j0 : blk;
    if (b >= 2) EXX_CUDA(cudaStreamWaitEvent(cs, ex->hb.used[b & 1], 0));
    EXX_CUDA(cudaMemcpyAsync(d_blk[b & 1], h_psi + N * (size_t)j0, sizeof(double) * N * nj, cudaMemcpyHostToDevice, cs));
    EXX_CUDA(cudaEventRecord(ex->hb.up[b & 1], cs));
    return EXX_OK;
  };
  if (n_blocks > 0) { exx_status st = upload_block(0); if (st != EXX_OK) return st; }
  if (n_tgt > 0)
    EXX_CUDA(cudaMemcpyAsync(d_tgt, tgt_in_psi ? h_psi + N * (size_t)tgt_start : h_tgt, sizeof(double) * N * n_tgt,
                             cudaMemcpyHostToDevice, s));
  if (n_occ > 0) EXX_CUDA(cudaMemcpyAsync(d_occ, h_occ, sizeof(double) * n_occ, cudaMemcpyHostToDevice, s));
  if (h_occ_tgt && n_tgt > 0)
    EXX_CUDA(cudaMemcpyAsync(d_occ_tgt, h_occ_tgt, sizeof(double) * n_tgt, cudaMemcpyHostToDevice, s));

  // the call owns d_vx: the plan's accumulate mode (meant for exx_apply on caller buffers) is overridden per block
  const bool saved_accumulate = plan->accumulate;
  long long launches = 0, solves = 0;
  exx_status result = EXX_OK;
  auto apply_block = [&](int b, int k0, int nk) -> exx_status {
    const int j0 = b * blk, nj = n_occ - j0 < blk ? n_occ - j0 : blk;
    plan->accumulate = b > 0;
    exx_status st = exx_apply(plan, d_blk[b & 1], d_occ + j0, nj, d_tgt + N * (size_t)k0, nullptr, nk,
                              d_vx + N * (size_t)k0, nullptr, nullptr, n_c, d_ws, ws, s);
    launches += plan->last_launches;
    solves += plan->last_solves;
    return st;
  };
  if (n_blocks == 0 && n_tgt > 0) {
    plan->accumulate = false;
    result = exx_apply(plan, nullptr, nullptr, 0, d_tgt, nullptr, n_tgt, d_vx, nullptr, nullptr, n_c, d_ws, ws, s);
    launches += plan->last_launches;
    if (result == EXX_OK && h_vx)
      result = cudaMemcpyAsync(h_vx, d_vx, sizeof(double) * N * n_tgt, cudaMemcpyDeviceToHost, s) == cudaSuccess
                   ? EXX_OK : cuda_fail(cudaGetLastError());
  }
  for (int b = 0; b < n_blocks && result == EXX_OK && n_tgt > 0; ++b) {
    cudaError_t ce = cudaStreamWaitEvent(s, ex->hb.up[b & 1], 0);
    if (ce != cudaSuccess) { result = cuda_fail(ce); break; }
    if (b + 1 < n_blocks) {
      if ((result = apply_block(b, 0, n_tgt)) != EXX_OK) break;
      if ((ce = cudaEventRecord(ex->hb.used[b & 1], s)) != cudaSuccess) { result = cuda_fail(ce); break; }
      // enqueued after this block's kernels: a pageable h_psi makes the copy call block the host, and the GPU then
      // already has its work (with pinned memory the order does not matter)
      if ((result = upload_block(b + 1)) != EXX_OK) break;
    } else {
      // last block: the targets go in up to kHostChunks chunks and a finished chunk's vx is downloaded on the copy
      // stream (idle by now) while the next chunk computes
      int chunk = (n_tgt + kHostChunks - 1) / kHostChunks;
      if (chunk < 1) chunk = 1;
      int c = 0;
      for (int k0 = 0; k0 < n_tgt && result == EXX_OK; k0 += chunk, ++c) {
        const int nk = n_tgt - k0 < chunk ? n_tgt - k0 : chunk;
        if ((result = apply_block(b, k0, nk)) != EXX_OK) break;
        if (h_vx) {
          if ((ce = cudaEventRecord(ex->hb.done[c], s)) == cudaSuccess) ce = cudaStreamWaitEvent(cs, ex->hb.done[c], 0);
          if (ce == cudaSuccess)
            ce = cudaMemcpyAsync(h_vx + N * (size_t)k0, d_vx + N * (size_t)k0, sizeof(double) * N * nk,
                                 cudaMemcpyDeviceToHost, cs);
          if (ce != cudaSuccess) result = cuda_fail(ce);
        }
      }
    }
  }
  plan->accumulate = saved_accumulate;
  if (result != EXX_OK) {
    cudaStreamSynchronize(s);
    cudaStreamSynchronize(cs);
    return result;
  }
  if (n_tgt == 0 && h_ex) { EXX_CUDA(exx::zero_fill(plan, d_ex, 1, s)); ++launches; }
  if ((h_ex || h_ex_k) && n_tgt > 0) {
    exx_status st = run_energy(plan, d_tgt, d_vx, h_occ_tgt ? d_occ_tgt : nullptr, n_tgt, h_ex ? d_ex : nullptr,
                               h_ex_k ? d_ex_k : nullptr, s, &launches);
    if (st != EXX_OK) return st;
  }
  plan->last_launches = launches;
  plan->last_solves = solves;
  if (h_ex_k && n_tgt > 0)
    EXX_CUDA(cudaMemcpyAsync(h_ex_k, d_ex_k, sizeof(double) * n_tgt, cudaMemcpyDeviceToHost, s));
  if (h_ex) EXX_CUDA(cudaMemcpyAsync(h_ex, d_ex, sizeof(double), cudaMemcpyDeviceToHost, s));
  EXX_CUDA(cudaStreamSynchronize(s));
  EXX_CUDA(cudaStreamSynchronize(cs));
  return EXX_OK;
}

size_t exx_ace_workspace_bytes(const exx_plan* plan, int n_orb, int n_trial) {
  if (!plan || n_orb < 1 || n_trial < 0) return 0;
  const size_t b = exx::ace_build_workspace_doubles(plan, n_orb);
  const size_t a = n_trial > 0 ? exx::ace_apply_workspace_doubles(plan, n_orb, n_trial) : 0;
  return sizeof(double) * (a > b ? a : b);
}

exx_status exx_ace_build(exx_plan* plan, const double* d_psi, const double* d_w, int n_orb, double* d_xi,
                         double* d_M, int* d_info, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_orb < 1 || n_orb > 32768 || !d_psi || !d_w || !d_xi || is_complex_plan(plan)) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  const size_t need = sizeof(double) * exx::ace_build_workspace_doubles(plan, n_orb);
  if (!d_workspace || workspace_bytes < need) return EXX_ERR_WORKSPACE;
  if (((uintptr_t)d_workspace) & 15) return EXX_ERR_INVALID_ARG;
  const size_t fn = sizeof(double) * (size_t)plan->N * (size_t)n_orb;
  const size_t mm = sizeof(double) * (size_t)n_orb * n_orb;
  if ((d_xi != d_w && overlaps(d_xi, fn, d_w, fn)) || overlaps(d_xi, fn, d_psi, fn) ||
      overlaps(d_xi, fn, d_workspace, need) || overlaps(d_workspace, need, d_psi, fn) ||
      overlaps(d_workspace, need, d_w, fn) || overlaps(d_M, mm, d_workspace, need) || overlaps(d_M, mm, d_xi, fn) ||
      overlaps(d_info, sizeof(int), d_workspace, need) || overlaps(d_info, sizeof(int), d_xi, fn))
    return EXX_ERR_ALIAS;
  long long launches = 0;
  EXX_CUDA(exx::ace_build(plan, d_psi, d_w, n_orb, d_xi, d_M, d_info, (double*)d_workspace,
                          (cudaStream_t)cuda_stream, &launches));
  plan->last_launches = launches;
  return EXX_OK;
}

exx_status exx_ace_apply(exx_plan* plan, const double* d_xi, int n_orb, const double* d_phi, int n_trial,
                         double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_orb < 1 || n_orb > 32768 || n_trial < 0 || n_trial > 32768 || !d_xi || is_complex_plan(plan))
    return EXX_ERR_INVALID_ARG;
  if (n_trial > 0 && (!d_phi || !d_out)) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  if (n_trial == 0) { plan->last_launches = 0; return EXX_OK; }
  const size_t need = sizeof(double) * exx::ace_apply_workspace_doubles(plan, n_orb, n_trial);
  if (!d_workspace || workspace_bytes < need) return EXX_ERR_WORKSPACE;
  if (((uintptr_t)d_workspace) & 15) return EXX_ERR_INVALID_ARG;
  const size_t fx = sizeof(double) * (size_t)plan->N * (size_t)n_orb;
  const size_t fp = sizeof(double) * (size_t)plan->N * (size_t)n_trial;
  if (overlaps(d_out, fp, d_xi, fx) || overlaps(d_out, fp, d_phi, fp) || overlaps(d_out, fp, d_workspace, need) ||
      overlaps(d_workspace, need, d_xi, fx) || overlaps(d_workspace, need, d_phi, fp))
    return EXX_ERR_ALIAS;
  long long launches = 0;
  EXX_CUDA(exx::ace_apply(plan, d_xi, n_orb, d_phi, n_trial, d_out, (double*)d_workspace,
                          (cudaStream_t)cuda_stream, &launches));
  plan->last_launches = launches;
  return EXX_OK;
}

size_t exx_ace_workspace_bytes_bloch(const exx_plan* plan, int n_orb, int n_trial) {
  if (!plan || n_orb < 1 || n_trial < 0) return 0;
  const size_t b = exx::ace_build_c_workspace_doubles(plan, n_orb);
  const size_t a = n_trial > 0 ? exx::ace_apply_c_workspace_doubles(plan, n_orb, n_trial) : 0;
  return sizeof(double) * (a > b ? a : b);
}

exx_status exx_ace_build_bloch(exx_plan* plan, const double* d_psi, const double* d_w, int n_orb, double* d_xi,
                               double* d_M, int* d_info, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_orb < 1 || n_orb > 16384 || !d_psi || !d_w || !d_xi) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  const size_t need = sizeof(double) * exx::ace_build_c_workspace_doubles(plan, n_orb);
  if (!d_workspace || workspace_bytes < need) return EXX_ERR_WORKSPACE;
  if ((((uintptr_t)d_workspace) & 15) || (((uintptr_t)d_M) & 15)) return EXX_ERR_INVALID_ARG;
  const size_t fn = 2 * sizeof(double) * (size_t)plan->N * (size_t)n_orb;
  const size_t mm = 2 * sizeof(double) * (size_t)n_orb * n_orb;
  if ((d_xi != d_w && overlaps(d_xi, fn, d_w, fn)) || overlaps(d_xi, fn, d_psi, fn) ||
      overlaps(d_xi, fn, d_workspace, need) || overlaps(d_workspace, need, d_psi, fn) ||
      overlaps(d_workspace, need, d_w, fn) || overlaps(d_M, mm, d_workspace, need) || overlaps(d_M, mm, d_xi, fn) ||
      overlaps(d_info, sizeof(int), d_workspace, need) || overlaps(d_info, sizeof(int), d_xi, fn))
    return EXX_ERR_ALIAS;
  long long launches = 0;
  EXX_CUDA(exx::ace_build_c(plan, d_psi, d_w, n_orb, d_xi, d_M, d_info, (double*)d_workspace,
                            (cudaStream_t)cuda_stream, &launches));
  plan->last_launches = launches;
  return EXX_OK;
}

exx_status exx_ace_apply_bloch(exx_plan* plan, const double* d_xi, int n_orb, const double* d_phi, int n_trial,
                               double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_orb < 1 || n_orb > 16384 || n_trial < 0 || n_trial > 16384 || !d_xi) return EXX_ERR_INVALID_ARG;
  if (n_trial > 0 && (!d_phi || !d_out)) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  if (n_trial == 0) { plan->last_launches = 0; return EXX_OK; }
  const size_t need = sizeof(double) * exx::ace_apply_c_workspace_doubles(plan, n_orb, n_trial);
  if (!d_workspace || workspace_bytes < need) return EXX_ERR_WORKSPACE;
  if (((uintptr_t)d_workspace) & 15) return EXX_ERR_INVALID_ARG;
  const size_t fx = 2 * sizeof(double) * (size_t)plan->N * (size_t)n_orb;
  const size_t fp = 2 * sizeof(double) * (size_t)plan->N * (size_t)n_trial;
  if (overlaps(d_out, fp, d_xi, fx) || overlaps(d_out, fp, d_phi, fp) || overlaps(d_out, fp, d_workspace, need) ||
      overlaps(d_workspace, need, d_xi, fx) || overlaps(d_workspace, need, d_phi, fp))
    return EXX_ERR_ALIAS;
  long long launches = 0;
  EXX_CUDA(exx::ace_apply_c(plan, d_xi, n_orb, d_phi, n_trial, d_out, (double*)d_workspace,
                            (cudaStream_t)cuda_stream, &launches));
  plan->last_launches = launches;
  return EXX_OK;
}

size_t exx_plan_workspace_bytes_bloch(const exx_plan* plan, int n_c) {
  if (!plan) return 0;
  n_c = resolve_nc(plan, n_c);
  if (n_c < 1 || n_c > plan->max_batch) return 0;
  return 6 * sizeof(double) * (size_t)plan->N * (size_t)n_c;  // three buffers of n_c complex functions
}

exx_status exx_plan_get_axis_bloch(const exx_plan* plan, int axis, double* h_lambda, double* h_V_re, double* h_V_im) {
  if (!plan || axis < 0 || axis > 2) return EXX_ERR_INVALID_ARG;
  const int n = plan->n[axis];
  if (h_lambda) std::memcpy(h_lambda, plan->h_lam[axis].data(), sizeof(double) * n);
  for (int i = 0; i < n; ++i)
    for (int m = 0; m < n; ++m) {
      const bool cplx = plan->bfly[axis] && !plan->h_Vc_re[axis].empty();  // V = U W of an axis held in its real form
      if (h_V_re) h_V_re[i + (size_t)n * m] = cplx ? plan->h_Vc_re[axis][(size_t)i * n + m] : plan->h_V[axis][(size_t)i * n + m];
      if (h_V_im)
        h_V_im[i + (size_t)n * m] = cplx ? plan->h_Vc_im[axis][(size_t)i * n + m]
                                         : plan->h_Vi[axis].empty() ? 0.0 : plan->h_Vi[axis][(size_t)i * n + m];
    }
  return EXX_OK;
}

exx_status exx_poisson_solve_bloch(exx_plan* plan, const double* d_rhs, double* d_phi, int n_rhs, int n_c,
                                   void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_rhs < 0 || (n_rhs > 0 && (!d_rhs || !d_phi))) return EXX_ERR_INVALID_ARG;
  n_c = resolve_nc(plan, n_c);
  if (n_c < 1 || n_c > plan->max_batch) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  if (n_rhs == 0) { plan->last_launches = 0; return EXX_OK; }
  const size_t need = exx_plan_workspace_bytes_bloch(plan, n_c);
  if (!d_workspace || workspace_bytes < need) return EXX_ERR_WORKSPACE;
  if (((uintptr_t)d_workspace) & 15) return EXX_ERR_INVALID_ARG;
  const size_t N = (size_t)plan->N, fn = 2 * sizeof(double) * N;
  if (d_rhs != d_phi && overlaps(d_rhs, fn * n_rhs, d_phi, fn * n_rhs)) return EXX_ERR_ALIAS;
  if (overlaps(d_workspace, need, d_phi, fn * n_rhs) || overlaps(d_workspace, need, d_rhs, fn * n_rhs))
    return EXX_ERR_ALIAS;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  double* b0 = (double*)d_workspace;
  double* const buf[3] = {b0, b0 + 2 * N * (size_t)n_c, b0 + 4 * N * (size_t)n_c};
  long long launches = 0;
  for (int r0 = 0; r0 < n_rhs; r0 += n_c) {
    const int nb = n_rhs - r0 < n_c ? n_rhs - r0 : n_c;
    EXX_CUDA(cudaMemcpyAsync(buf[0], d_rhs + 2 * N * (size_t)r0, fn * nb, cudaMemcpyDeviceToDevice, s));
    double* res = nullptr;
    EXX_CUDA(exx::bloch_butterfly(plan, buf[0], nb, false, s, &launches));  // axes held in their real form: g = U^H f
    EXX_CUDA(exx::bloch_solve_batch(plan, buf, nb, s, &launches, &res));
    EXX_CUDA(exx::bloch_butterfly(plan, res, nb, true, s, &launches));      // phi = U (W ...)
    EXX_CUDA(cudaMemcpyAsync(d_phi + 2 * N * (size_t)r0, res, fn * nb, cudaMemcpyDeviceToDevice, s));
  }
  plan->last_launches = launches;
  return EXX_OK;
}

exx_status exx_apply_bloch(exx_plan* plan, const double* d_psi, const double* d_occ, int n_occ, const double* d_tgt,
                           int n_tgt, double* d_vx, int accumulate, double* d_ex_k, int n_c, void* d_workspace,
                           size_t workspace_bytes, void* cuda_stream) {
  if (!plan || n_occ < 0 || n_tgt < 0) return EXX_ERR_INVALID_ARG;
  if (n_occ > 0 && (!d_psi || !d_occ)) return EXX_ERR_INVALID_ARG;
  if (n_tgt > 0 && (!d_tgt || !d_vx)) return EXX_ERR_INVALID_ARG;
  n_c = resolve_nc(plan, n_c);
  if (n_c < 1 || n_c > plan->max_batch) return EXX_ERR_INVALID_ARG;
  if (plan->device < 0) return cuda_fail(cudaErrorNoDevice);
  DeviceScope dev_scope(plan->device);
  if (!dev_scope.ok()) return cuda_fail(dev_scope.err);
  const size_t N = (size_t)plan->N, fn = 2 * sizeof(double) * N;
  const size_t need = exx_plan_workspace_bytes_bloch(plan, n_c);
  if (n_occ > 0 && n_tgt > 0 && (!d_workspace || workspace_bytes < need)) return EXX_ERR_WORKSPACE;
  if (d_workspace && (((uintptr_t)d_workspace) & 15)) return EXX_ERR_INVALID_ARG;
  if (overlaps(d_vx, fn * n_tgt, d_psi, fn * n_occ) || overlaps(d_vx, fn * n_tgt, d_tgt, fn * n_tgt) ||
      overlaps(d_vx, fn * n_tgt, d_workspace, need) || overlaps(d_workspace, need, d_psi, fn * n_occ) ||
      overlaps(d_workspace, need, d_tgt, fn * n_tgt))
    return EXX_ERR_ALIAS;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  long long launches = 0;
  PlanExtras* ex = extras_of(plan);
  if (n_tgt > 0 && n_occ == 0) {
    if (!accumulate) { EXX_CUDA(exx::zero_fill(plan, d_vx, 2 * (long long)N * n_tgt, s)); ++launches; }
  } else if (n_tgt > 0) {
    double* b0 = (double*)d_workspace;
    double* const buf[3] = {b0, b0 + 2 * N * (size_t)n_c, b0 + 4 * N * (size_t)n_c};
    const int nj_max = n_occ < n_c ? n_occ : n_c;
    const int nk_max = n_c / nj_max;
    for (int k0 = 0; k0 < n_tgt; k0 += nk_max) {
      const int nk = n_tgt - k0 < nk_max ? n_tgt - k0 : nk_max;
      for (int j0 = 0; j0 < n_occ; j0 += nj_max) {
        const int nj = n_occ - j0 < nj_max ? n_occ - j0 : nj_max;
        const exx::BatchDesc bd{j0, nj, k0, nk};
        {
          exx::ProfScope ps(plan, exx::KC_PAIR_DENSITY, s);
          EXX_CUDA(exx::bloch_pair_density(plan, d_psi, d_tgt, bd, buf[0], s));
        }
        double* res = nullptr;
        EXX_CUDA(exx::bloch_solve_batch(plan, buf, nj * nk, s, &launches, &res));
        {
          exx::ProfScope ps(plan, exx::KC_ACCUMULATE, s);
          EXX_CUDA(exx::bloch_accumulate(plan, d_psi, d_occ, res, bd, j0 == 0 && !accumulate, d_vx, s));
        }
        launches += 2;
      }
    }
  }
  if (d_ex_k && n_tgt > 0) {
    // e_k = h^3 Re <tgt_k, vx_k> = h^3 times the real dot product of the two planar arrays of length 2N (R20)
    for (int k0 = 0; k0 < n_tgt; k0 += kEnergyChunk) {
      const int nk = n_tgt - k0 < kEnergyChunk ? n_tgt - k0 : kEnergyChunk;
      exx::ProfScope ps(plan, exx::KC_OTHER, s);
      EXX_CUDA(exx::energy(plan, d_tgt + 2 * N * (size_t)k0, d_vx + 2 * N * (size_t)k0, nullptr, nk,
                           ex->d_energy_scratch, d_ex_k + k0, nullptr, s, 2 * (long long)N));
      launches += 2;
    }
  }
  plan->last_launches = launches;
  plan->last_solves = (long long)n_occ * n_tgt;
  return EXX_OK;
}

}  // extern "C"
