/*
 * exx.h -- C ABI of libexx.so: the exact-exchange apply on a real-space finite-difference grid,
 * hand-written CUDA for sm_100a (NVIDIA B200).  One hot path of arxiv 2501.16572
 * ("GPU acceleration of hybrid functional calculations in the SPARC electronic structure code").
 * Citations are /root/reference/PAPER.md:<line> plus the equation; "R<n>" are the readings listed in
 * DESIGN.md (= SURVEY.md section 8(c) A<n>).
 *
 * What the library computes (all real FP64, "double-precision arithmetic"):
 *
 *   phi_jk = f(L) (psi_j .* tgt_k)                                   Eqs. 2-5
 *   vx_k   = - sum_j occ_j * psi_j .* phi_jk                          Eq. 1 / Eq. 19b
 *   e_k    = h^3 * <tgt_k, vx_k>,   E_x = 1/2 sum_k occ_tgt_k e_k     BASELINE.json north_star (R7)
 *   xi = W R^-T, V~ Phi = -xi (h^3 xi^T Phi)                          ACE, Eqs. 17-20, 26-29
 *
 * f(L) is evaluated with the batch Kronecker-product formalism (Eqs. 6-7, 9-11, 16; PAPER.md:66-70,
 * 86-98, 134): L = I(x)I(x)Kx + I(x)Ky(x)I + Kz(x)I(x)I, K_a = V_a diag(lam_a) V_a^T, three mode products
 * with V^T, a pointwise multiply by m(lam_x+lam_y+lam_z), three mode products with V.
 *   unscreened (omega <= 0):  m = 4 pi / mu, mu = -lam_sum; the zero mode is dropped (m := 0)
 *   screened   (omega  > 0):  m = 4 pi (1 - exp(-mu/(4 omega^2))) / mu, m(0) = pi/omega^2       (R1-R3)
 *
 * Layout: a grid function is N = nx*ny*nz contiguous doubles, x fastest: idx = ix + nx*(iy + ny*iz)
 * (the paper's vec of an n1 x n2 x n3 array).  A set of n functions is [n][N], each
 * function contiguous (the column blocks of Eq. 10).
 *
 * Conventions
 *  - Pointers named d_* are DEVICE pointers on the plan's device; h_* are HOST pointers.  The caller owns
 *    every buffer passed in, including the workspace; the plan owns V, lambda and the multiplier table.
 *  - All work is enqueued on `cuda_stream` (a cudaStream_t passed as void*, NULL = default stream).
 *    exx_apply / exx_poisson_solve never synchronise the host; results (including *d_ex) are valid once
 *    the caller has synchronised that stream.  The calls are CUDA-graph capturable.
 *  - Every entry point returns an exx_status; no host code throws, exits or aborts.  Arguments are validated
 *    before the first launch, so a call that returns EXX_ERR_INVALID_ARG / _WORKSPACE / _ALIAS has
 *    enqueued nothing.  One device-side exception: a TMA-pipeline kernel whose mbarrier wait has not completed
 *    after 2^30 polls (minutes; only a hardware fault or a corrupted tensor map can cause it) executes a trap
 *    rather than hang the stream, which the next synchronising CUDA call reports (EXX_ERR_CUDA from this library;
 *    the CUDA context is lost, as after any device-side fault).
 *  - occ is used exactly as passed: no mixing fraction, spin factor or Brillouin weight (R8), no
 *    thresholding of small occupations (R9).
 *  - There is no CPU fallback: without a CUDA device every compute call returns EXX_ERR_CUDA.
 */
#ifndef EXX_H
#define EXX_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct exx_plan exx_plan; /* opaque; created/destroyed by the library */

typedef enum {
  EXX_OK = 0,
  EXX_ERR_INVALID_ARG = 1,
  EXX_ERR_ALLOC = 2,
  EXX_ERR_CUDA = 3,
  EXX_ERR_EIGENSOLVE = 4,
  EXX_ERR_WORKSPACE = 5,
  EXX_ERR_ALIAS = 6,
  EXX_ERR_LIMIT = 7 /* a size exceeds a fixed capacity compiled into the library (exx_energy_static) */
} exx_status;

enum { EXX_BC_PERIODIC = 0, EXX_BC_DIRICHLET = 1 };

/* Kernel variants (test hook; the default is the fast path). */
enum {
  EXX_VARIANT_FUSED_DMMA = 0, /* tensor-core (mma.sync f64 -> DMMA) mode products, operands staged by TMA */
  EXX_VARIANT_REFERENCE = 1,  /* one plain DFMA kernel per mode product; slow, for cross-checks        */
  EXX_VARIANT_CPASYNC = 2     /* DMMA mode products with per-lane cp.async staging (first generation;  */
                              /* also what variant 0 uses for sizes TMA cannot address, e.g. odd nx)   */
};

/*
 * Build the plan: per-axis FD second-derivative matrices (central stencil of half-width fd_order/2,
 * periodic wrap or Dirichlet truncation, R4/R6), their eigendecompositions (Eqs. 6-7;
 * a cyclic Jacobi solver inside the library, host side, once) and the multiplier table f(Lambda~)
 * (Eq. 16), uploaded to `device`.
 *   nx,ny,nz >= 1; h > 0; bc[a] in {EXX_BC_PERIODIC, EXX_BC_DIRICHLET}; fd_order even >= 2;
 *   omega <= 0 selects the unscreened kernel; max_batch >= 1 bounds n_c; device = CUDA ordinal.
 * Errors: INVALID_ARG (nothing allocated), EIGENSOLVE (Jacobi did not converge), ALLOC, CUDA.
 */
exx_status exx_plan_create(exx_plan** out, int nx, int ny, int nz, double h, const int bc[3],
                           int fd_order, double omega, int max_batch, int device);
exx_status exx_plan_destroy(exx_plan* plan);

/* Select a kernel variant (EXX_VARIANT_*). INVALID_ARG for unknown values. */
exx_status exx_plan_set_variant(exx_plan* plan, int variant);

/*
 * How many batches exx_apply keeps in flight: 1 (default) = every kernel on the caller's stream; 2 (allowed
 * where the fast kernels serve all three axes) = consecutive target blocks alternate between the caller's stream and
 * a plan-owned second stream, forked from and joined back into the caller's stream with events inside the
 * call, so the call is still asynchronous, ordered with respect to the caller's stream and graph capturable.
 * Each lane uses one half of the workspace.  The two lanes never touch the same vx_k, and every vx_k is
 * accumulated in the same order as with one lane: results are bitwise identical.  INVALID_ARG otherwise.
 */
exx_status exx_plan_set_lanes(exx_plan* plan, int lanes);
int exx_plan_get_lanes(const exx_plan* plan);

/*
 * Pass fusion of the default variant (test and measurement hook; default 15 = all on).  Bit 0: the z-forward product,
 * the eigen-space multiply and the z-backward product of a batch (Eq. 11's third and fourth GEMM and Eq. 16,
 * PAPER.md:96-98, :134) run as ONE kernel, the intermediate staying in registers.  Bit 1: the x-backward product and
 * the accumulate of Eq. 1 run as one kernel; phi_jk is never written to memory and exx_apply shapes its
 * batches as nj occupied orbitals x nk targets with nk large enough to keep every SM busy.  Bit 2: where nx is 8
 * (mod 16) the y products tile their columns in half-chunks of 8 instead of chunks of 16, the last of which would be
 * half empty in every row.  Bit 3 (needs bit 0): the fused z pass contracts with the reflection-adapted eigenbasis of
 * the z axis -- every eigenvector even or odd under z -> mir(z), DESIGN.md 6.9 -- so both of its products run over half
 * the range with two half-size blocks: about 55 % of the multiply-adds of the dense products, same result to rounding
 * (f(L) does not depend on the basis chosen inside a degenerate eigenspace).  With a bit off (or where
 * TMA cannot address the buffers, or an axis has more than 128 points) the separate passes run.  The result does not
 * depend on the mask beyond rounding (the sum over j is taken in ascending order either way).
 */
exx_status exx_plan_set_fusion(exx_plan* plan, int mask);
int exx_plan_get_fusion(const exx_plan* plan);

/*
 * Accumulate mode (off by default): while on, exx_apply ADDS its result into d_vx instead of overwriting it, so the
 * sum over the occupied orbitals of Eq. 1 can be split over several calls -- the orbital ring of
 * SURVEY.md 8(e), where each rank holds one block of orbitals at a time (paper_2501_16572_b200/sharding.py).  d_ex /
 * d_ex_k are computed from the d_vx found after the call, so request them on the last call only.
 */
exx_status exx_plan_set_accumulate(exx_plan* plan, int on);

/* Bytes of device workspace exx_apply / exx_poisson_solve need for batches of n_c right-hand sides: two buffers of n_c
 * grid functions, 16 N n_c bytes (0 if plan is NULL or n_c is outside 1..max_batch).  n_c = 0 asks for the library's
 * default batch -- about 4 GB of right-hand sides, at least 32, at most max_batch -- so for a plan with a large
 * max_batch exx_plan_workspace_bytes(plan, 0) is about 8 GB (it was about 2 GB before the default grew from 1 GB to
 * 4 GB of right-hand sides); pass an explicit n_c to bound it. */
size_t exx_plan_workspace_bytes(const exx_plan* plan, int n_c);

/* Test hook: copy out one axis' eigenpairs. h_lambda: n doubles; h_V: n*n doubles, column-major
 * (h_V[i + n*m] = component i of eigenvector m).  Either may be NULL. axis: 0=x, 1=y, 2=z. */
exx_status exx_plan_get_axis(const exx_plan* plan, int axis, double* h_lambda, double* h_V);

/* Test hook: the reflection-adapted eigenbasis of a real axis that the fused z pass contracts with (even vectors under
 * z -> mir(z) first, *n_even of them, then the odd ones; each block in ascending eigenvalue order; same layout as
 * exx_plan_get_axis).  mir(z) = n - 1 - z on either kind of axis (a symmetric circulant matrix commutes with every
 * reflection, a symmetric Toeplitz one with this one).  Host only.
 * INVALID_ARG for a Bloch axis, EIGENSOLVE if the basis cannot be built. */
exx_status exx_plan_get_axis_symmetric(const exx_plan* plan, int axis, double* h_lambda, double* h_V, int* n_even);

/* Instrumentation: FP64 operations the mode products of ONE pair solve execute with the plan's current settings
 * (padding not counted).  4 N (nx + ny + nz) -- the algorithmic count of the dense products -- unless an axis runs on the
 * reflection-adapted basis (exx_plan_set_fusion bit 3), whose two products cost about half of that.  bench.py reports
 * the roofline fraction in these executed operations, so that it cannot exceed 1. */
double exx_plan_executed_flops_per_solve(const exx_plan* plan);
/* The same for one EXECUTED solve of exx_apply_symmetric: with the x axis on the reflection-adapted basis its x-backward
 * product runs twice (once for vx_k, once for vx_j: the two-sided accumulate never materialises phi_jk). */
double exx_plan_executed_flops_per_symmetric_solve(const exx_plan* plan);

/* Test hook: copy out the multiplier table, N doubles, entry [a + nx*(b + ny*c)] = m(lam_x[a]+lam_y[b]+lam_z[c]). */
exx_status exx_plan_get_multiplier(const exx_plan* plan, double* h_mult);

/*
 * Bare batched solver, Y = f(L) C (Eq. 9, 96-98 Eq. 11): d_phi[b] = f(L) d_rhs[b] for
 * b < n_rhs, processed in batches of at most n_c (0 = library default).  d_phi may equal d_rhs (in
 * place) but must not partially overlap it.  This is the unit of the "Poisson solves/s" metric.
 */
exx_status exx_poisson_solve(exx_plan* plan, const double* d_rhs, double* d_phi, int n_rhs, int n_c,
                             void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The NON-batch Kronecker solver of PAPER.md:74-78 (Eq. 8a/8b), the comparison line of the paper's Fig. 2 (not the
 * product path): the right-hand sides are solved one at a time; for each, every frontal slice B(:,:,k) is multiplied
 * by V1^T and V2, the stacked slices by V3, then by f(Lambda~), and the same back -- 4 nz + 2 small dense products,
 * one kernel launch each (exx_plan_last_launch_count reports them).  Same result as exx_poisson_solve.  Real plans
 * only.  d_workspace: at least 2 N doubles (exx_plan_workspace_bytes(plan, 1)); d_phi may equal d_rhs.  Errors as
 * exx_poisson_solve.
 */
exx_status exx_poisson_solve_nonbatch(exx_plan* plan, const double* d_rhs, double* d_phi, int n_rhs, void* d_workspace,
                                      size_t workspace_bytes, void* cuda_stream);

/*
 * Exchange apply (Eq. 1, 42 Eq. 2, 178 Eq. 19b):
 *   d_vx[k]  = - sum_{j<n_occ} d_occ[j] * d_psi[j] .* f(L)(d_psi[j] .* d_tgt[k])     [n_tgt][N], overwritten
 *   d_ex_k[k] = h^3 <d_tgt[k], d_vx[k]>                                            [n_tgt], optional (NULL)
 *   *d_ex    = 1/2 sum_k d_occ_tgt[k] d_ex_k[k]                                     optional (NULL); needs d_occ_tgt
 * d_psi [n_occ][N], d_occ [n_occ]; d_tgt [n_tgt][N] may alias a block of d_psi.  d_vx must not overlap
 * d_psi / d_tgt / the workspace (EXX_ERR_ALIAS).  n_c = right-hand sides per batch, 1..max_batch,
 * 0 = library default (about 4 GB of right-hand sides per
 * batch, at least 32, at most max_batch).  Every (j,k) pair is solved (no symmetry shortcut, R12).  n_occ == 0 gives vx = 0.
 */
exx_status exx_apply(exx_plan* plan, const double* d_psi, const double* d_occ, int n_occ,
                     const double* d_tgt, const double* d_occ_tgt, int n_tgt, double* d_vx,
                     double* d_ex, double* d_ex_k, int n_c, void* d_workspace,
                     size_t workspace_bytes, void* cuda_stream);

/*
 * Pair-symmetric exchange apply for the case targets == orbitals: phi_jk = phi_kj
 * (Eq. 2, is symmetric in the pair for real orbitals), so only the pairs j <= k are solved and each
 * solution feeds both vx_k (-= occ_j psi_j phi_jk) and, for j != k, vx_j (-= occ_k psi_k phi_jk).  Same result as
 * exx_apply(psi, occ, n, psi, occ, n, ...) up to the order of the sum over j (not bitwise: the terms arrive in a
 * different order), with about half the Poisson solves: exx_plan_last_solve_count reports how many were executed
 * (n(n+1)/2 plus the few j > k pairs inside the diagonal blocks of the rectangular batches).
 * d_vx [n_orb][N] is overwritten; d_ex / d_ex_k as in exx_apply with occ_tgt = occ.  Same workspace and errors.
 */
exx_status exx_apply_symmetric(exx_plan* plan, const double* d_psi, const double* d_occ, int n_orb, double* d_vx,
                               double* d_ex, double* d_ex_k, int n_c, void* d_workspace, size_t workspace_bytes,
                               void* cuda_stream);

/* Pair solves executed by the last exx_apply (n_occ*n_tgt) / exx_apply_symmetric call on this plan. */
long long exx_plan_last_solve_count(const exx_plan* plan);

/*
 * Convenience end-to-end call with HOST buffers (pageable or pinned): uploads psi/occ (and tgt unless
 * tgt_start >= 0 selects the block h_psi[tgt_start .. tgt_start+n_tgt) as targets), runs exx_apply on an
 * internal stream, downloads vx / e_k / E_x and synchronises.  The targets are applied in up to four blocks
 * (multiples of a batch's target block, so the result is bitwise that of one exx_apply) and a finished block's vx
 * is downloaded on a second stream while the next block computes.  The device buffers are owned by the plan, grown
 * on demand and released by exx_plan_destroy.  Any of h_vx, h_ex, h_ex_k may be NULL.  Not thread safe per plan.
 */
exx_status exx_apply_host(exx_plan* plan, const double* h_psi, const double* h_occ, int n_occ,
                          const double* h_tgt, int tgt_start, const double* h_occ_tgt, int n_tgt,
                          double* h_vx, double* h_ex, double* h_ex_k, int n_c);

/*
 * ACE tail (Section III.A, Eqs. 17-20 and 26), the step right after exx_apply with the
 * orbitals themselves as targets (then W^(n) = vx_n, Eq. 19):
 *   M  = h^3 Psi^T W                  [n_orb][n_orb]   Eq. 20 (grid inner product, R15)
 *   R R^T = -(M + M^T)/2              R lower triangular; the paper's "Cholesky factor of M": M is negative
 *                                     definite because Vx is, so -M is what is factored (R16, R17)
 *   xi = W R^-T                       [n_orb][N]       Eqs. 18, 26
 * d_psi, d_w [n_orb][N]; d_xi [n_orb][N] may equal d_w (in place) but must not partially overlap it, nor d_psi.
 * d_M (optional, NULL): receives M, n_orb*n_orb doubles, row-major.  d_info (optional, NULL): device int, set to
 * 0 on success or to the 1-based index of the first non-positive pivot (then xi holds NaNs); the call itself
 * never synchronises, so the caller reads d_info after synchronising the stream.
 * Workspace: exx_ace_workspace_bytes(plan, n_orb, n_trial) bytes (n_trial = 0 if only building).
 */
size_t exx_ace_workspace_bytes(const exx_plan* plan, int n_orb, int n_trial);
exx_status exx_ace_build(exx_plan* plan, const double* d_psi, const double* d_w, int n_orb, double* d_xi,
                         double* d_M, int* d_info, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * ACE application (Section III.B, Eqs. 27-29) to n_trial trial functions:
 *   chi = h^3 xi^T Phi  [n_orb][n_trial] (Eq. 28),   d_out = -xi chi  [n_trial][N] (Eqs. 27, 29; sign per R17).
 * d_out must not overlap d_xi or d_phi (EXX_ERR_ALIAS).  With Phi = Psi the result equals W.
 */
exx_status exx_ace_apply(exx_plan* plan, const double* d_xi, int n_orb, const double* d_phi, int n_trial,
                         double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * Bloch-periodic (k-point) variant, complex FP64 (Eqs. 1-3 "subject to Bloch
 * boundary conditions at the wavevector k-q in the directions that the system is extended"; :159, :218 complex
 * arithmetic).  Readings R18-R20:
 *   - theta[a] = (k-q)_a * n_a * h is the Bloch phase across the cell along periodic axis a (ignored on Dirichlet
 *     axes): u(x + n_a h) = exp(i theta[a]) u(x); the 1-D FD matrix is Hermitian, K = V diag(lam) V^H.
 *   - one call handles ONE (k,q) pair: every d_psi[j] carries the phase of q, every d_tgt[k] that of k, the plan is
 *     built for theta = theta_k - theta_q; the caller loops over q with `accumulate` != 0 and passes
 *     d_occ[j] = w_q * g_jq (used verbatim).
 *   - a complex grid function is two real planes [2][N] (real part, then imaginary part); a set is [n][2][N].
 *       d_vx[k] (+)= - sum_j d_occ[j] * d_psi[j] .* f(L_theta)( conj(d_psi[j]) .* d_tgt[k] )
 *       d_ex_k[k] = h^3 Re <d_tgt[k], d_vx[k]>            (optional, NULL; computed after the update)
 * exx_plan_create_bloch validates like exx_plan_create (theta must be finite).  Workspace:
 * exx_plan_workspace_bytes_bloch(plan, n_c) (three buffers of n_c complex functions).  An axis with a phase is held
 * in its real form: K(theta) commutes with (reflection x -> n-1-x) o (complex conjugation), so in the fixed butterfly basis
 * U it is real symmetric, K = (U W) diag(lam) (U W)^H with W real; a complex mode product is the butterfly U^H / U (fused
 * into the pair-density and accumulate kernels) and one real tensor-core launch over both planes, like a real axis
 * (Dirichlet, theta = 0).  exx_apply / exx_poisson_solve / exx_ace_* on a plan with a nonzero phase
 * return EXX_ERR_INVALID_ARG.  Errors and aliasing rules as for exx_apply.
 */
exx_status exx_plan_create_bloch(exx_plan** out, int nx, int ny, int nz, double h, const int bc[3], int fd_order,
                                 double omega, const double theta[3], int max_batch, int device);
/* Test / measurement hook: the same plan with the form of its phase axes chosen.  EXX_BLOCH_FORM_REAL (what
 * exx_plan_create_bloch builds) is the real form described above; EXX_BLOCH_FORM_EMBEDDED keeps complex eigenvectors
 * V = Vr + i Vi and runs every complex mode product on the real embedding [[Mr, -Mi], [Mi, Mr]] (one launch for axes of up
 * to 64 points, two read-modify-write launches above; twice the real operations) -- the cross-check the GPU tests
 * compare with the oracle as well. */
enum { EXX_BLOCH_FORM_REAL = 0, EXX_BLOCH_FORM_EMBEDDED = 1 };
exx_status exx_plan_create_bloch_form(exx_plan** out, int nx, int ny, int nz, double h, const int bc[3], int fd_order,
                                      double omega, const double theta[3], int max_batch, int device, int form);
size_t exx_plan_workspace_bytes_bloch(const exx_plan* plan, int n_c);
exx_status exx_poisson_solve_bloch(exx_plan* plan, const double* d_rhs, double* d_phi, int n_rhs, int n_c,
                                   void* d_workspace, size_t workspace_bytes, void* cuda_stream);
exx_status exx_apply_bloch(exx_plan* plan, const double* d_psi, const double* d_occ, int n_occ, const double* d_tgt,
                           int n_tgt, double* d_vx, int accumulate, double* d_ex_k, int n_c, void* d_workspace,
                           size_t workspace_bytes, void* cuda_stream);
/* Test hook: eigenpairs of one axis of a Bloch plan; h_V_re / h_V_im column-major like exx_plan_get_axis. */
exx_status exx_plan_get_axis_bloch(const exx_plan* plan, int axis, double* h_lambda, double* h_V_re, double* h_V_im);

/*
 * ACE tail and application for COMPLEX (k-point) orbitals ("cublasDgemm/cublasZgemm",
 * "cusolver_dpotrf/cusolver_zpotrf", "cublasDtrsm/cublasZtrsm ... in the case of real/complex-valued computations";
 * Eqs. 17-20, 26-29 with the transposes read as conjugate transposes, R21):
 *   M  = h^3 Psi^H W   [n_orb][n_orb] complex,   R R^H = -(M + M^H)/2 (R lower triangular, real positive diagonal),
 *   xi = W R^-H,       chi = h^3 xi^H Phi,       d_out = -xi chi.
 * Every function set is [n][2][N] (real plane, then imaginary plane, as in exx_apply_bloch); d_M (optional) receives
 * M row-major with interleaved (re, im) pairs, 2 n_orb^2 doubles, 16-byte aligned.  The operator does not depend on
 * the plan's phase (only on N and h), so any plan of the grid serves.  d_xi may equal d_w; d_info, aliasing rules,
 * workspace alignment and errors as for exx_ace_build / exx_ace_apply; n_orb, n_trial <= 16384.
 * Workspace: exx_ace_workspace_bytes_bloch(plan, n_orb, n_trial).
 */
size_t exx_ace_workspace_bytes_bloch(const exx_plan* plan, int n_orb, int n_trial);
exx_status exx_ace_build_bloch(exx_plan* plan, const double* d_psi, const double* d_w, int n_orb, double* d_xi,
                               double* d_M, int* d_info, void* d_workspace, size_t workspace_bytes, void* cuda_stream);
exx_status exx_ace_apply_bloch(exx_plan* plan, const double* d_xi, int n_orb, const double* d_phi, int n_trial,
                               double* d_out, void* d_workspace, size_t workspace_bytes, void* cuda_stream);

/*
 * The energy step on its own, for callers that cannot allocate device memory (BASELINE.json north_star: "together with
 * the exchange energy"; R7):
 *   d_ex_k[k] = dv * <d_tgt[k], d_vx[k]>   for k < n_tgt      (optional, NULL)      dv = h^3, the grid weight
 *   *d_ex     = 1/2 sum_k d_occ_tgt[k] d_ex_k[k]              (optional, NULL; overwritten; needs d_occ_tgt)
 * d_tgt, d_vx: [n_tgt][n_points] device doubles, e.g. the targets and the d_vx an exx_apply without d_ex / d_ex_k
 * produced; they may be real sets (n_points = N) or the two-plane complex sets of exx_apply_bloch (n_points = 2 N,
 * which gives Re <tgt, vx>).  The values equal those exx_apply returns for the same d_vx.
 *
 * Who needs it.  Some host programs give all of the GPU's memory to an arena of their own when they start (a
 * hybrid-functional code sizes its orbital arrays to fill the card), after which cudaMalloc fails; others call from a
 * loop that keeps several streams busy, where the device-wide synchronisation inside cudaMalloc / cudaFree would stall
 * every one of them.  Every other compute call here needs a plan (whose creation allocates) and a workspace.  This call
 * needs no plan and no workspace and calls no cudaMalloc, cudaFree or allocating library routine, on any call: the
 * block sums of its two-stage reduction go to a fixed array inside the library image, EXX_ENERGY_STATIC_MAX_TGT * 64
 * doubles = 2 MiB, which every GPU that loads libexx.so holds until the process exits.
 *
 * Limits and rules:
 *  - n_tgt > EXX_ENERGY_STATIC_MAX_TGT returns EXX_ERR_LIMIT and enqueues nothing (split the targets over several
 *    calls and sum *d_ex yourself, or use exx_apply's own energy outputs).
 *  - It runs on the CURRENT device (cudaSetDevice), which must be the one the buffers live on, on `cuda_stream`, and
 *    never synchronises the host.  The first call on each device looks up the array's address on that device
 *    (cudaGetSymbolAddress; thread safe) -- make that first call during set-up, outside any stream capture.
 *  - All calls on a device share the one array.  Nothing in it has to be zero beforehand (every slot a call reads it
 *    has written itself first), but two calls that run on the GPU at the same time -- different streams, or different
 *    host threads on different streams -- overwrite each other's block sums: order them on one stream or with events.
 *  - Errors: INVALID_ARG (n_tgt < 0, n_points < 1, dv <= 0, a missing input, d_ex without d_occ_tgt), LIMIT, CUDA.
 *    n_tgt == 0 writes *d_ex = 0.
 */
#define EXX_ENERGY_STATIC_MAX_TGT 4096
exx_status exx_energy_static(const double* d_tgt, const double* d_vx, const double* d_occ_tgt, int n_tgt,
                             long long n_points, double dv, double* d_ex_k, double* d_ex, void* cuda_stream);

/* Number of kernels the last exx_apply / exx_poisson_solve call on this plan enqueued. */
long long exx_plan_last_launch_count(const exx_plan* plan);

/* Test hook: how many mode-product launches of this plan, since it was created, went through the TMA-staged
 * kernels (the default path; sizes TMA cannot address -- odd nx, an axis longer than 128 points, buffers not
 * 16-byte aligned -- use the cp.async or plain kernels instead, still on the GPU). */
long long exx_plan_tma_launch_count(const exx_plan* plan);

/*
 * Per-kernel-class timing (bench instrumentation).  With profiling on, every kernel the library launches
 * is bracketed by a CUDA-event pair on the caller's stream (this perturbs the stream slightly: do not
 * report whole-call times taken with it on).  exx_plan_get_profile synchronises the recorded events, adds
 * the durations per class into h_ms[4] / h_count[4] and clears the records.  Classes: 0 = mode products
 * (a2-a4, with fused a1/a3/a5 where the variant fuses them), 1 = pair density (a1), 2 = accumulate (a5),
 * 3 = energy and housekeeping (a6).
 */
exx_status exx_plan_set_profiling(exx_plan* plan, int on);
exx_status exx_plan_get_profile(exx_plan* plan, double* h_ms, long long* h_count);
/* The mode-product launches of the records the last exx_plan_get_profile call consumed, per pass of a batch, h_ms[8] /
 * h_count[8]: 0 = x-forward (with a1), 1 = y-forward, 2 = z (the fused z-forward / a3 / z-backward pass, or the z-forward
 * product where it is not fused), 3 = z-backward (unfused only), 4 = y-backward, 5 = x-backward (with a5 where fused),
 * 6 = the second x-backward pass of exx_apply_symmetric (orbital side), 7 = unused.  h_flops_per_solve[8] (optional, NULL):
 * the FP64 operations one pair solve executes in that pass with the plan's current settings (as
 * exx_plan_executed_flops_per_solve counts them).  Host only, no synchronisation. */
exx_status exx_plan_get_profile_passes(const exx_plan* plan, double* h_ms, long long* h_count, double* h_flops_per_solve);

/*
 * Diagnostic: sustained FP64 throughput of this GPU in TFLOP/s over about `seconds` (0 < seconds <= 30) of
 * back-to-back launches of a register-resident issue loop.  kind 0 = DFMA (FP64 FMA pipe), kind 1 = DMMA
 * (mma.sync m8n8k4 f64).  Synchronises the device.  Used by bench.py for the roofline denominator
 * (MEASURED_PEAKS.json has no FP64 figure).
 */
exx_status exx_probe_fp64_peak(int kind, int device, double seconds, double* h_tflops);

/* Human-readable status; for EXX_ERR_CUDA includes the last cudaError_t seen by this thread. */
const char* exx_status_string(exx_status status);

/* Library version string. */
const char* exx_version(void);

#ifdef __cplusplus
}
#endif
#endif /* EXX_H */
