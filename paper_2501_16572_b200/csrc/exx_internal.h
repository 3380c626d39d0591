// Internal declarations shared by the host planner, the kernels and the C-ABI layer of libexx.so.
#pragma once
#include <nvtx3/nvToolsExt.h>
#include <cuda_runtime.h>

#include <atomic>
#include <vector>

#include "exx.h"

namespace exx {

// ---- host planner (plan_host.cpp) -------------------------------------------------------------
// Central second-derivative weights w[0..n0], order = 2*n0 (R4).
std::vector<double> fd_weights(int order, double h);
// Dense symmetric n x n matrix of +d^2/dx^2, row-major (R2, R6).
std::vector<double> second_derivative_matrix(int n, double h, int bc, int order);
// Cyclic Jacobi: A (row-major, symmetric, destroyed) -> eigenvalues ascending in lam, eigenvectors in
// V row-major V[i*n + m] = component i of eigenvector m.  Returns false if not converged.
bool jacobi_eigh(int n, std::vector<double>& A, std::vector<double>& lam, std::vector<double>& V);
// Hermitian Bloch-periodic axis (R18): K(theta) = V diag(lam) V^H, V = Vr + i Vi row-major [i][m].
bool bloch_eigh(int n, double h, int order, double theta, std::vector<double>& lam, std::vector<double>& Vr,
                std::vector<double>& Vi);
// The same axis through its real form K' = U^H K U = W diag(lam) W^T (U: the fixed butterfly of plan_host.cpp); V = U W.
bool bloch_eigh_real_form(int n, double h, int order, double theta, std::vector<double>& lam, std::vector<double>& W,
                          std::vector<double>& Vr, std::vector<double>& Vi);
// Reflection-adapted eigenbasis of a real axis: even vectors first, then odd (plan_host.cpp); false if it cannot be built.
bool symmetrize_axis(int n, int bc, const std::vector<double>& lam, const std::vector<double>& V, std::vector<double>& lam_s,
                     std::vector<double>& Vs, int* n_even, bool centered = false);
// f(Lambda~) table (PAPER.md:61 Eq. 5, :134 Eq. 16; R1-R3), entry [a + nx*(b + ny*c)].
std::vector<double> multiplier_table(const std::vector<double>& lx, const std::vector<double>& ly,
                                     const std::vector<double>& lz, double omega, double zero_tol);

}  // namespace exx

namespace exx {
enum KernelClass { KC_MODE_PRODUCT = 0, KC_PAIR_DENSITY = 1, KC_ACCUMULATE = 2, KC_OTHER = 3, KC_COUNT = 4 };
// Passes of a batch (exx_plan_get_profile_passes): x-forward (+ a1), y-forward, z (fused z-forward / a3 / z-backward, or
// the z-forward product alone), z-backward (unfused only), y-backward, x-backward (+ a5), x-backward of the orbital side
// of the pair-symmetric apply.
enum PassId { PASS_XF = 0, PASS_YF = 1, PASS_Z = 2, PASS_ZB = 3, PASS_YB = 4, PASS_XB = 5, PASS_XB2 = 6, PASS_COUNT = 8 };
struct ProfRec {
  cudaEvent_t e0, e1;
  int cls;
  int pass;  // PassId, or -1
};
}  // namespace exx

struct exx_plan {
  int n[3];  // nx, ny, nz
  double h;
  int bc[3];
  int order;
  double omega;
  int max_batch;
  int device;
  int variant;
  long long N;
  std::vector<double> h_lam[3];
  std::vector<double> h_V[3];  // row-major [i][m]
  // Bloch-periodic plans (exx_plan_create_bloch): imaginary parts of the eigenvectors; empty for an axis whose
  // matrix is real (Dirichlet, or theta == 0)
  double theta[3];
  std::vector<double> h_Vi[3];
  // Bloch plans, round 2: an axis with a phase is held in its REAL form (h_V = W, h_Vi empty) and the kernels apply the
  // butterfly U^H / U around the real products (bfly[a]); the complex eigenvectors V = U W are kept for the test hook
  bool bloch;
  bool bfly[3];
  std::vector<double> h_Vc_re[3], h_Vc_im[3];
  std::vector<double> h_mult;
  double zero_tol;  // R3 threshold on |lam_sum| the table was built with
  // device copies
  double* d_Vi[3];   // Bloch plans: imaginary parts, same layout; nullptr for a real axis
  double* d_V[3];    // row-major [i][m], n*n (axes with identical matrices share one allocation)
  double* d_Vpad[3]; // zero-padded shared-memory images of V for the DMMA kernels (kernels_dmma.cu)
  double* d_mult;    // N
  void* tma_state;   // TMA-staged kernels: permuted V images and the tensor-map cache (kernels_tma.cu)
  int sm_count;
  int smem_optin;
  long long last_launches;
  long long last_solves;   // pair solves the last exx_apply / exx_apply_symmetric call executed
  long long tma_launches;  // cumulative count of TMA-staged mode-product launches (test hook)
  // exx_apply runs `lanes` batches at a time (1 or 2): lane 0 on the caller's stream, lane 1 on lane_stream,
  // forked and joined with the two events
  int lanes;
  // bit 0: z-forward + multiplier + z-backward in one pass (k_mode_zz); bit 1: x-backward + accumulate in one pass
  // (k_mode_xacc); bit 2: y passes on 8-column half-chunk tiles where nx == 8 (mod 16); bit 3 (needs bit 0): the mode products
  // on the reflection-adapted eigenbases (symmetric mode).  Default 15 = all on; exx_plan_set_fusion
  // (test / measurement hook)
  int fusion;
  cudaStream_t lane_stream;
  cudaEvent_t ev_fork, ev_join;
  // optional per-kernel-class CUDA-event timing (exx_plan_set_profiling)
  bool accumulate;  // exx_plan_set_accumulate: exx_apply adds into d_vx instead of overwriting it
  bool prof_on;
  std::vector<exx::ProfRec> prof;
  double prof_pass_ms[exx::PASS_COUNT];        // filled by exx_plan_get_profile, read by exx_plan_get_profile_passes
  long long prof_pass_count[exx::PASS_COUNT];
};

namespace exx {

// Batch descriptor: right-hand side b of a batch is the pair (j0 + b % nj, k0 + b / nj).
struct BatchDesc {
  int j0, nj, k0, nk;
};

// ---- reference variant (kernels_ref.cu): one plain DFMA kernel per step ----------------------
cudaError_t ref_pair_density(const exx_plan* p, const double* psi, const double* tgt, BatchDesc bd,
                             double* out, cudaStream_t s);
cudaError_t ref_mode_product(const exx_plan* p, int axis, bool forward, const double* in, double* out,
                             int nb, bool apply_mult, cudaStream_t s);
cudaError_t ref_accumulate(const exx_plan* p, const double* psi, const double* occ, const double* phi,
                           BatchDesc bd, bool first, double* vx, cudaStream_t s, bool sym = false);
// pair-symmetric apply: vx_j -= sum_{k in batch, k > j} occ_k psi_k phi_jk for every j of the batch
cudaError_t sym_accumulate_transposed(const exx_plan* p, const double* psi, const double* occ, const double* phi,
                                      BatchDesc bd, double* vx, cudaStream_t s);
// shared by both variants: e_k = h^3 <tgt_k, vx_k>, then E_x
cudaError_t energy(const exx_plan* p, const double* tgt, const double* vx, const double* occ_tgt,
                   int n_tgt, double* ex_k_scratch, double* ex_k, double* ex, cudaStream_t s, long long len = 0);
cudaError_t zero_fill(const exx_plan* p, double* ptr, long long n, cudaStream_t s);

// Opt-in to more than 48 KB of dynamic shared memory, remembered per kernel instantiation AND per device
// (cudaFuncSetAttribute applies to the current device only; a plan may live on any device of the process).  One static
// instance per launch site.  Concurrent callers race benignly: the attribute call is idempotent.
struct SmemOptIn {
  static constexpr int kMaxDevices = 64;
  std::atomic<size_t> bytes[kMaxDevices];
  template <typename K>
  cudaError_t ensure(K kern, int device, size_t need, bool max_carveout = false) {
    const bool tracked = device >= 0 && device < kMaxDevices;
    if (tracked && bytes[device].load(std::memory_order_acquire) >= need) return cudaSuccess;
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)need);
    if (e != cudaSuccess) return e;
    if (max_carveout) {
      e = cudaFuncSetAttribute(kern, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
      if (e != cudaSuccess) return e;
    }
    if (tracked) bytes[device].store(need, std::memory_order_release);
    return cudaSuccess;
  }
};

// Makes the plan's device current for the duration of an entry point and restores the caller's device afterwards.
struct DeviceScope {
  int prev = -1;
  cudaError_t err = cudaSuccess;
  explicit DeviceScope(int device) {
    err = cudaGetDevice(&prev);
    if (err == cudaSuccess && prev != device) err = cudaSetDevice(device);
    else if (err == cudaSuccess) prev = -1;  // nothing to restore
  }
  ~DeviceScope() {
    if (prev >= 0) cudaSetDevice(prev);
  }
  bool ok() const { return err == cudaSuccess; }
};

// RAII event pair around one launch when profiling is on (no-op otherwise).
// Every scope is also an NVTX range on the host thread (a range per stage), named after the pass of a
// batch or the kernel class, so a tool that understands NVTX (ncu --nvtx --nvtx-include "exx:z/", a timeline viewer) can
// select or label the launches of one pass.  Header-only NVTX v3: without a tool attached a push/pop is a null-pointer test.
inline const char* prof_scope_name(int cls, int pass) {
  static const char* const kPassName[PASS_COUNT] = {"exx:x_forward", "exx:y_forward", "exx:z", "exx:z_backward",
                                                    "exx:y_backward", "exx:x_backward", "exx:x_backward_orbital_side",
                                                    "exx:mode_product"};
  static const char* const kClassName[KC_COUNT] = {"exx:mode_product", "exx:pair_density", "exx:accumulate", "exx:energy"};
  if (cls == KC_MODE_PRODUCT && pass >= 0 && pass < PASS_COUNT) return kPassName[pass];
  return cls >= 0 && cls < KC_COUNT ? kClassName[cls] : "exx";
}

struct ProfScope {
  exx_plan* p;
  cudaStream_t s;
  cudaEvent_t e1;
  ProfScope(exx_plan* plan, int cls, cudaStream_t stream, int pass = -1) : p(plan), s(stream), e1(nullptr) {
    nvtxRangePushA(prof_scope_name(cls, pass));
    if (!p->prof_on) return;
    cudaEvent_t e0;
    if (cudaEventCreate(&e0) != cudaSuccess) return;
    if (cudaEventCreate(&e1) != cudaSuccess) { cudaEventDestroy(e0); e1 = nullptr; return; }
    cudaEventRecord(e0, s);
    p->prof.push_back(ProfRec{e0, e1, cls, pass});
  }
  ~ProfScope() {
    if (e1) cudaEventRecord(e1, s);
    nvtxRangePop();
  }
  void cancel() {  // nothing was launched inside this scope: drop the record
    if (!e1) return;
    cudaEventDestroy(p->prof.back().e0);
    cudaEventDestroy(e1);
    p->prof.pop_back();
    e1 = nullptr;
  }
};

// ---- fast variant (kernels_dmma.cu) ----------------------------------------------------------
// Returns cudaErrorNotSupported if the plan's sizes are outside what the fast kernels handle
// (the caller then reports EXX_ERR_INVALID_ARG; there is no silent fallback).
cudaError_t fast_init(exx_plan* p);
void fast_destroy(exx_plan* p);
// One batch of solves; see kernels_dmma.cu.
struct FastArgs {
  const double* psi;
  const double* tgt;
  const double* occ;
  double* vx;
  BatchDesc bd;
  int n_occ, n_tgt;  // extents of psi / tgt (tensor maps cover the whole arrays)
  bool first;  // first batch for these targets: vx is overwritten, not accumulated into
  bool sym;    // pair-symmetric apply (tgt == psi): only j <= k contributes to vx_k, and phi_jk also feeds vx_j
};
// ---- TMA-staged mode products (kernels_tma.cu), the default; cudaErrorNotSupported -> cp.async kernels ----
cudaError_t tma_init(exx_plan* p);
void tma_destroy(exx_plan* p);
cudaError_t tma_mode_product(exx_plan* p, int axis, bool forward, const double* in, double* out, int nb,
                             bool apply_mult, const FastArgs* pd, cudaStream_t s, int part = 0, bool rmw = false);
cudaError_t tma_mode_product_c(exx_plan* p, int axis, bool forward, double* buf, int nb, cudaStream_t s);
// ---- fused passes (kernels_fused.cu); cudaErrorNotSupported -> the unfused passes above ----
cudaError_t fused_init(exx_plan* p);   // after tma_init
void fused_destroy(exx_plan* p);       // before tma_destroy
// sym: 0 = plain mode order and table, 1 = symmetric mode (y, z), 2 = symmetric mode with the x axis too
cudaError_t fused_zz(exx_plan* p, const double* in, double* out, int nb, cudaStream_t s, int sym = 0);
bool fused_sym_mode(const exx_plan* p);
// y products on the reflection-adapted basis (kernels_sym.cu); sym_init after tma_init and before fused_init
cudaError_t sym_init(exx_plan* p);
void sym_destroy(exx_plan* p);
cudaError_t sym_mode_product_y(exx_plan* p, bool forward, double* buf, int nb, cudaStream_t s);
bool sym_x_usable(const exx_plan* p, const double* work, const FastArgs* fa);
int sym_xacc_tile_rows(const exx_plan* p);
bool sym_x_usable_plain(const exx_plan* p, const double* src, const double* work, int nb);
cudaError_t sym_xf_plain(exx_plan* p, const double* in, double* out, int nb, cudaStream_t s);
cudaError_t sym_xb_plain(exx_plan* p, double* buf, int nb, cudaStream_t s);
cudaError_t sym_xf(exx_plan* p, double* out, int nb, const FastArgs* fa, cudaStream_t s);
cudaError_t sym_xacc(exx_plan* p, const double* in, int nb, const FastArgs* fa, cudaStream_t s, int side = 0);
cudaError_t fused_zz_c(exx_plan* p, double* buf, int nb, cudaStream_t s);  // Bloch plans, complex z axis, n <= 64
cudaError_t fused_xacc(exx_plan* p, const double* in, int nb, const FastArgs* fa, cudaStream_t s);
int fused_xacc_tile_rows(const exx_plan* p);
double fused_executed_flops_per_solve(const exx_plan* p, bool pair_symmetric = false);
double fused_executed_flops_axis(const exx_plan* p, int ax);
// ---- non-batch Eq. 8 solver, the Fig. 2 comparison line (kernels_nonbatch.cu) ----
cudaError_t nonbatch_solve_one(exx_plan* p, const double* rhs, double* phi, double* buf0, double* buf1, cudaStream_t s,
                               long long* launches);
// ---- ACE tail and application (kernels_ace.cu) ----
size_t ace_build_workspace_doubles(const exx_plan* p, int n);
size_t ace_apply_workspace_doubles(const exx_plan* p, int n, int m);
cudaError_t ace_build(exx_plan* p, const double* psi, const double* w, int n, double* xi, double* M_out, int* info,
                      double* ws, cudaStream_t s, long long* launches);
cudaError_t ace_apply(exx_plan* p, const double* xi, int n, const double* phi, int m, double* out, double* ws,
                      cudaStream_t s, long long* launches);
// complex (k-point) orbitals, [n][2][N] planes
size_t ace_build_c_workspace_doubles(const exx_plan* p, int n);
size_t ace_apply_c_workspace_doubles(const exx_plan* p, int n, int m);
cudaError_t ace_build_c(exx_plan* p, const double* psi, const double* w, int n, double* xi, double* M_out, int* info,
                        double* ws, cudaStream_t s, long long* launches);
cudaError_t ace_apply_c(exx_plan* p, const double* xi, int n, const double* phi, int m, double* out, double* ws,
                        cudaStream_t s, long long* launches);
// ---- Bloch-periodic complex variant (kernels_bloch.cu) ----
cudaError_t bloch_pair_density(const exx_plan* p, const double* psi, const double* tgt, BatchDesc bd, double* out,
                               cudaStream_t s);
cudaError_t bloch_accumulate(const exx_plan* p, const double* psi, const double* occ, const double* phi, BatchDesc bd,
                             bool first, double* vx, cudaStream_t s);
cudaError_t bloch_butterfly(const exx_plan* p, double* buf, int nb, bool inverse, cudaStream_t s, long long* launches);
cudaError_t bloch_solve_batch(exx_plan* p, double* const buf[3], int nb, cudaStream_t s, long long* launches,
                              double** result);
cudaError_t fast_solve_batch(exx_plan* p, const double* src, double* work, double* scratch, int nb,
                             const FastArgs* fa, cudaStream_t s, long long* launches);

}  // namespace exx
