/* cclr.h — C ABI of the B200-native CC-LR hot path (arXiv:2307.14296; PAPER.md).
 *
 * The library evaluates the CCSD Jacobian transform  sigma = (A - (omega + i*gamma)) X  of relativistic
 * coupled-cluster linear response (Eq. 19, 183-187 Eq. 20-21; A = Hbar_N of PAPER.md:131 Eq. 14 and
 * Table 1; programmable form: supplementary S-Eq. 11-12 PAPER.md:885-893 with the intermediates
 * S-Eq. 15-28), solves the right response equations (A - z) t = -xi and
 * contracts t with a perturbation vector (Eq. 15, 203).  Every step runs in hand-written sm_100a
 * CUDA kernels of this library; there is no CPU fallback and no cuBLAS / cuTENSOR call.
 *
 * Conventions
 *   - complex128, interleaved (re, im); every pointer is a DEVICE pointer unless its comment says "host".
 *   - o occupied / v virtual spinors; i,j,m,n occupied, a,b,e,f virtual; n = o + v.
 *   - <pq||rs> antisymmetrised, upper index = bra: V[pq,rs] = conj(V[rs,pq]).
 *   - pair index P(p<q) = q(q-1)/2 + p; oo = o(o-1)/2, vv = v(v-1)/2.
 *   - amplitudes x1[a][i] ([v][o], row-major), x2[P(a<b)][P(i<j)] ([vv][oo], row-major); nvec vectors are stored
 *     vector-major ([nvec][v*o], [nvec][vv*oo]).  Antisymmetry is a property of the storage.
 *   - all dots / norms run over UNIQUE elements (singles + a<b,i<j).
 *   - every call returns 0 (CCLR_OK) or a negative error code; nothing aborts, throws or keeps global state.
 *     Calls on one context are not re-entrant.  Work is enqueued on the context's stream; calls that return host
 *     data (cclr_solve, cclr_property, *_host) synchronise that stream before returning.
 */
#ifndef CCLR_H
#define CCLR_H
#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct cclr_ctx cclr_ctx; /* opaque */
typedef struct { double re, im; } cclr_c128;

enum {
  CCLR_OK = 0,
  CCLR_EINVAL = -1,   /* bad argument (null pointer, o<2, v<2, nvec<1, ...) */
  CCLR_ENOMEM = -2,   /* device allocation failed */
  CCLR_ECUDA = -3,    /* a CUDA call or kernel failed; cclr_last_cuda_error() gives the CUDA code */
  CCLR_ENOTCONV = -4, /* cclr_solve hit maxiter; the best iterate is still written and info filled */
  CCLR_ENODEV = -5    /* no sm_100 device */
};

/* The six classes of MO integrals of PAPER.md:231, all <pq||rs>, packed over antisymmetric pairs. */
typedef struct {
  const cclr_c128 *oooo; /* [oo][oo]      <mn||ij>, m<n ; i<j   (Hermitian matrix)                     */
  const cclr_c128 *ooov; /* [oo][o][v]    <mn||ie>, m<n                                                */
  const cclr_c128 *oovv; /* [oo][vv]      <mn||ef>, m<n ; e<f                                          */
  const cclr_c128 *ovvo; /* [o][v][v][o]  <mb||ej>                                                     */
  const cclr_c128 *ovvv; /* [o][v][vv]    <mb||ef>, e<f                                                */
  const cclr_c128 *vvvv; /* [vv][vv]      <ab||ef>, a<b ; e<f   (Hermitian matrix)                     */
} cclr_eri_packed;

/* flags for cclr_create */
#define CCLR_ERI_INPLACE 1u /* the context adopts eri->vvvv and dresses it in place into W_vvvv (S-Eq. 22);
                               the caller must keep the buffer alive until cclr_destroy and not read it again */

#define CCLR_GEMM_4M 4u     /* every contraction of this context uses the 4M complex product (default: the large ones use 3M,
                               see cclr_zgemm); a per-context choice, nothing process-wide */

#define CCLR_NO_SUM_PLANES 16u /* do not keep / form the "sum planes" Re + Im that feed the 3M product from global memory (default:
                               a persistent plane of W_vvvv, 1/2 of its size, when memory allows, and per-call planes of operands
                               that are small next to the product); without them the sums are formed inside the kernel (~5 % slower) */
#define CCLR_NO_GRAPH 8u    /* never replay sigma as a CUDA graph (default: contexts with at most 2^21 unique amplitudes capture the sigma
                               plan once and replay it per trial vector -- they are launch bound; results are identical) */

#define CCLR_GEMM_DMMA 32u  /* keep EVERY contraction on the FP64 tensor cores (DMMA).  Default: the two contractions that are 91 % of
                               cclr_sigma -- the pp ladder T11 and the ring T8 -- run on the INT8 tensor path at FP64 accuracy when
                               their shapes allow (vv >= 512, oo >= 32 and at least 64 output tiles of 256 x 256 reals: configs 3, 4, 5): the context keeps 6 integer slices of 7 bits of W_vvvv and
                               W_ovvo (3/4 of their size) and slices the trial vector per call (cclr_zgemm_oz; csrc/zgemm_oz.cu;
                               DESIGN.md 6.1b).  The slice product holds north_star's 1e-10 on sigma (~1e-11 measured); every
                               other contraction, cclr_create and the left transform are DMMA either way.  CCLR_GEMM_4M implies
                               this flag.  cclr_set_gemm_path switches an existing context. */

#define CCLR_NO_LEFT_SLICES 128u /* do not keep the integer slices of W_vvvv's transpose (another 3/4 of W_vvvv) that put the transposed
                               ladder of cclr_sigma_left / cclr_f_transform on the INT8 tensor path as well (default: kept when
                               the free device memory allows); the left ladder then runs on the FP64 tensor cores */

#define CCLR_GEMM_INT8_ANY_SIZE 64u /* testing aid: ladder and ring take the INT8 tensor path at ANY size the kernel supports (default: only
                               where it pays, from 64 output tiles of 256 x 256 reals), so that small inputs can be compared with
                               the full-tensor oracle through that path */

#define CCLR_SMALL_CHUNKS 2u /* testing aid: run the chunked intermediate builds with chunks of 3 indices so that small
                               inputs exercise several chunks and a ragged last one (results are unchanged) */

/* Build the context: tau (S-Eq. 28), F_me/F_mi/F_ae (S-Eq. 15-17), W_oooo (S-Eq. 18
 * :913), W_vvvv (S-Eq. 22 :929), W_ovvo and Wbar (S-Eq. 19, 23 :916, 932), W_ooov / W_vovv (S-Eq. 24-25 :934-936),
 * W_ovoo (S-Eq. 20 :919) and W_vvvo (S-Eq. 21 :924) in the readings of DESIGN.md, and the orbital-energy
 * denominators D1, D2.  fock is [n][n] row-major <p|f|q>.  t1 is [v][o], t2 is [vv][oo]; they need
 * not be converged (sigma = dOmega/dt . x at any t).  Inputs are borrowed for the duration of the call (vvvv: see
 * CCLR_ERI_INPLACE).  cuda_stream is a cudaStream_t (NULL = default stream); all later work of the context runs on it. */
int cclr_create(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, const cclr_c128 *t1,
                const cclr_c128 *t2, unsigned flags, void *cuda_stream, cclr_ctx **out);

/* out = A x - (omega + i*gamma) x  for nvec trial vectors (S-Eq. 11-12; shift PAPER.md:163, 187).
 * out1/out2 must not alias x1/x2. */
int cclr_sigma(cclr_ctx *ctx, const cclr_c128 *x1, const cclr_c128 *x2, int nvec, double omega, double gamma,
               cclr_c128 *out1, cclr_c128 *out2);

/* out = l (A - (omega + i*gamma)) for nvec left vectors l1[a][i] = l^i_a, l2[(ab)][(ij)] = l^ij_ab (same layouts as amplitudes):
 * the left Jacobian transform of the Lambda equations and of left response equations (Eq. 13; S-Eq. 13,
 * PAPER.md:895-901 in the reading of DESIGN.md: the term-by-term adjoint of S-Eq. 11-12).  Same cost as cclr_sigma; the
 * pp ladder runs with W_vvvv as the [K][N] operand, so nothing is stored twice.  out must not alias l. */
int cclr_sigma_left(cclr_ctx *ctx, const cclr_c128 *l1, const cclr_c128 *l2, int nvec, double omega, double gamma,
                    cclr_c128 *out1, cclr_c128 *out2);

typedef struct {
  int iterations;       /* subspace expansions performed                                   */
  int sigma_calls;      /* number of single-vector A.b products evaluated                  */
  int subspace;         /* final subspace dimension                                        */
  int converged;        /* 1 if every system met tol                                       */
  double max_residual;  /* max over systems of ||(A-z)t+xi|| / ||xi|| (unique-element 2-norm) */
  double seconds;       /* wall time of the call                                           */
} cclr_solve_info;

/* Solve (A - z_k) t = -xi_r, z_k = omegas[k] + i*gamma, for every right-hand side r < nrhs and shift k < nomega with
 * one shared Krylov subspace (steps 1-5 of PAPER.md:952-967 in the readings of DESIGN.md; A is shift independent so
 * one sigma serves every frequency).  Convergence: ||(A - z)t + xi||_2 <= tol * ||xi||_2 over unique elements.
 * omegas (host) may be negative, gamma may be negative.  Outputs: t1_out [nrhs][nomega][v*o], t2_out
 * [nrhs][nomega][vv*oo].  info (host) may be NULL.
 * On a context whose ladder / ring run as integer-slice products (cclr_gemm_slices > 0, no CUDA-graph replay) the sigma vectors of
 * trial vectors that are added late use fewer slices -- they enter the solutions with coefficients of the size of the residual at
 * that time -- and a converged system is accepted only while the estimated effect of that on its TRUE residual stays below tol / 2;
 * otherwise the iteration falls back to all slices.  The environment variable
 * CCLR_SOLVER_ALL_SLICES=1 keeps every sigma vector at all slices.  The same holds for cclr_solve_left, cclr_lambda and the
 * response entry points built on them. */
int cclr_solve(cclr_ctx *ctx, const cclr_c128 *xi1, const cclr_c128 *xi2, int nrhs, const double *omegas,
               int nomega, double gamma, double tol, int maxiter, cclr_c128 *t1_out, cclr_c128 *t2_out,
               cclr_solve_info *info);

/* xi^X = <mu| exp(-T) X exp(T) |R>, the right-hand side of the response equations for the one-body perturbation X
 * (Eq. 19; S-Eq. 1-3): X is a DEVICE [n][n] row-major matrix <p|X|q>, n = o + v (all four
 * blocks are used); xi1 [v*o], xi2 [vv*oo] device outputs. */
int cclr_xi(cclr_ctx *ctx, const cclr_c128 *X, cclr_c128 *xi1, cclr_c128 *xi2);

/* eta^X = <Lambda| [Xbar, tau_nu] |R> (S-Eq. 4-6) for the one-body operator X (device [n][n]) and the
 * ground-state multipliers lam1 [v*o] (lambda^i_a at [a][i]), lam2 [vv*oo]; eom != 0 adds the EOM term of S-Eq. 7
 * (PAPER.md:853), giving the EOM-eta vector of the CC-CI response function Eq. 16.  eta1, eta2: device outputs. */
int cclr_eta(cclr_ctx *ctx, const cclr_c128 *X, const cclr_c128 *lam1, const cclr_c128 *lam2, int eom, cclr_c128 *eta1,
             cclr_c128 *eta2);

/* Left equations  l (A - z_k) = -eta_r  for every right-hand side and shift: the same shared-subspace method as cclr_solve on
 * the left transform (arguments as cclr_solve).  cclr_lambda solves the ground-state multiplier equations
 * lambda A = -eta0, eta0 = (F_me[i,a], <ij||ab>) (Eq. 13): lam1 [v*o], lam2 [vv*oo] device outputs; a converged
 * solution is also kept in the context, where cclr_response_ci / cclr_response_cc reuse it unless they ask for a tighter tol. */
int cclr_solve_left(cclr_ctx *ctx, const cclr_c128 *eta1, const cclr_c128 *eta2, int nrhs, const double *omegas, int nomega,
                    double gamma, double tol, int maxiter, cclr_c128 *l1_out, cclr_c128 *l2_out, cclr_solve_info *info);
int cclr_lambda(cclr_ctx *ctx, double tol, int maxiter, cclr_c128 *lam1, cclr_c128 *lam2, cclr_solve_info *info);

/* <<X;Y>>_z, z = omega + i*gamma, in the CC-CI (EOM-CC) form of PAPER.md:142 Eq. 16 with the symmetriser of Eq. 17
 * (readings 7-8 of DESIGN.md), computed end to end on the device: lambda (solved once per context and cached),
 * xi^X, xi^Y, EOM-eta^X, EOM-eta^Y, the response amplitudes t^Y(z), t^Y(-conj z), t^X(-z), t^X(conj z), and the dot products.
 * X, Y: device [n][n] one-body matrices; result: HOST, one complex number (alpha_XY = -<<X;Y>>, reading 9); info (host, may be
 * NULL) accumulates the solver statistics.  Returns CCLR_OK, or CCLR_ENOTCONV if a solve missed tol (result still written). */
int cclr_response_ci(cclr_ctx *ctx, const cclr_c128 *X, const cclr_c128 *Y, double omega, double gamma, double tol,
                     int maxiter, cclr_c128 *result, cclr_solve_info *info);

/* The whole CC-CI response tensor in one call -- steps 3 and 4 of the paper's workflow for a set of operators and
 * frequencies: result[k][r][s] = <<X_r; X_s>>_{omegas[k] + i gamma} (HOST, [nomega][nop][nop]) for the nop DEVICE matrices
 * X [nop][n][n].  All 2 nop nomega (4 nop nomega for gamma != 0) response systems of Eq. 16-17 share one trial space per sign of
 * gamma (cclr_solve with nop right-hand sides and the shifts +-omegas); lambda is solved once and cached; xi, EOM-eta and every dot
 * product run on the device.  alpha_rs(omega) = -result (reading 9); sigma_abs(omega) = 4 pi omega / c * Im mean_r alpha_rr (Eq. 22,
 * PAPER.md:191).  omegas: HOST.  Returns CCLR_OK, or CCLR_ENOTCONV if a solve missed tol (results still written). */
int cclr_response_ci_tensor(cclr_ctx *ctx, const cclr_c128 *X, int nop, const double *omegas, int nomega, double gamma, double tol,
                            int maxiter, cclr_c128 *result, cclr_solve_info *info);

/* out_k = F y_k for nvec amplitude-shaped device vectors y_k [nvec][v*o], [nvec][vv*oo] and the multipliers lam1, lam2:
 * (F y)_nu = <Lambda| [[Hbar, tau_nu], Y] |R>, F = the CC Hessian of Table 1 (S-Eq. 8).  F is never
 * formed, only its contraction with a vector.  The printed contraction formulas are
 * unrecoverable (reading 6); the routine evaluates the derivative of the left transform along y,
 * F y = d/db [eta0 + lambda A](t + b y)|_0, as one contraction plan over the context's dressed intermediates (csrc/plans.inc,
 * CCLR_PLAN_FY: one left ladder for all vectors of the call, then three ring-shaped GEMMs and o^3 v^3-class work per vector).
 * eri: the packed integrals the context was created from -- ooov, oovv, ovvo, ovvv are read (device, borrowed for the call);
 * oooo and vvvv are NOT (a CCLR_ERI_INPLACE context, whose vvvv block is overwritten, is fine).  out1 [nvec][v*o],
 * out2 [nvec][vv*oo]: device outputs, must not alias y.  x . F . y = the bilinear dot cclr_property(x, F y). */
int cclr_f_transform(cclr_ctx *ctx, const cclr_eri_packed *eri, const cclr_c128 *lam1, const cclr_c128 *lam2,
                     const cclr_c128 *y1, const cclr_c128 *y2, int nvec, cclr_c128 *out1, cclr_c128 *out2);

/* x . F . y by the stencil route, the independent cross-check of cclr_f_transform: the exact derivative
 * d/da [(eta0 + lambda A)(t + a x) . y] at a = 0 (a cubic in a, 4-point stencil), i.e. four cclr_create + cclr_sigma_left
 * evaluations at shifted amplitudes, without a context.  Needs the bare integrals (all six classes) and t (only read).
 * result: HOST. */
int cclr_xfy(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, const cclr_c128 *t1, const cclr_c128 *t2,
             const cclr_c128 *lam1, const cclr_c128 *lam2, const cclr_c128 *x1, const cclr_c128 *x2, const cclr_c128 *y1,
             const cclr_c128 *y2, void *cuda_stream, cclr_c128 *result);

/* <<X;Y>>_z in the symmetric CC-CC (LR-CC) form of PAPER.md:137 Eq. 15 with Eq. 17:
 * g(w) = eta^X . t^Y(w) + eta^Y . t^X(-w) + t^X(-w) . F . t^Y(w),  <<X;Y>>_z = 1/2 [g(z) + conj g(-conj z)].  Same arguments as
 * cclr_response_ci plus eri, the packed integrals the context was created from (read by cclr_f_transform as described there;
 * the context may have been created with CCLR_ERI_INPLACE). */
int cclr_response_cc(cclr_ctx *ctx, const cclr_eri_packed *eri, const cclr_c128 *X, const cclr_c128 *Y, double omega, double gamma,
                     double tol, int maxiter, cclr_c128 *result, cclr_solve_info *info);

/* result[k] = sum_ai eta1 x1_k + sum_{a<b,i<j} eta2 x2_k  (bilinear, no conjugation; PAPER.md:137 Eq. 15, :203) for
 * nvec vectors x_k; result is a HOST array of nvec complex numbers. */
int cclr_property(cclr_ctx *ctx, const cclr_c128 *eta1, const cclr_c128 *eta2, const cclr_c128 *x1,
                  const cclr_c128 *x2, int nvec, cclr_c128 *result);

typedef struct {
  int iterations;        /* residual evaluations that were followed by an amplitude update          */
  int converged;         /* 1 if ||Omega|| <= tol                                                    */
  int sigma_calls;       /* residual evaluations performed                                           */
  double residual;       /* final ||Omega||_2 over the FULL tensors (= sqrt(|O1|^2 + 4 |O2 unique|^2)) */
  double energy_re, energy_im; /* CCSD correlation energy  sum f[i,a] t1[a,i] + 1/4 sum <ij||ab> tau[ab,ij]  */
  double seconds;
} cclr_ccsd_info;

/* Ground-state CCSD amplitudes (paper step 1): solves Omega(t) = 0 by quasi-Newton steps
 * t -= Omega / D with DIIS on the direct residual plan (csrc/plans.inc CCLR_PLAN_OMEGA; the
 * quadrature of the Jacobian, cclr_ccsd_residual mode 1, is the independent cross-check).
 * t1 [v][o], t2 [vv][oo] are IN/OUT device arrays: the start amplitudes on entry (zeros are fine), the solution on exit.
 * The integrals are only read.  Returns CCLR_OK, or CCLR_ENOTCONV (best iterate written, info filled).
 * From the size where it pays (>= 64 output tiles) and when 7/8 of <ab||ef> + <ma||ef> fit twice into the free device memory, the
 * ladder, <ma||ef> tau and the ring-shaped contractions of the residual run as integer-slice products (csrc/zgemm_oz.cu) whose slice
 * count follows the residual: 2 slices far from convergence, one more than cclr_create would take near it; a residual that meets tol
 * with fewer than all slices is evaluated again with all of them before it is accepted. */
int cclr_ccsd(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, cclr_c128 *t1, cclr_c128 *t2, double tol,
              int maxiter, void *cuda_stream, cclr_ccsd_info *info);

typedef struct {
  int iterations;       /* subspace expansions performed                          */
  int sigma_calls;      /* single-vector A.b products evaluated                   */
  int subspace;         /* final trial-space dimension                            */
  int converged;        /* 1 if every root met tol                                */
  double max_residual;  /* max over roots of ||A x - theta x||_2, ||x||_2 = 1 (unique elements) */
  double seconds;
} cclr_eom_info;

/* The nroots EOM-EE excitation energies of lowest real part = eigenvalues of the Jacobian A = poles of the response function
 * and their right eigenvectors, by a block Davidson method on the same sigma routine
 * and orbital-energy preconditioner as cclr_solve.  eig: HOST array [nroots] (A is not Hermitian: eigenvalues are complex
 * in general, reading 17); r1_out [nroots][v*o], r2_out [nroots][vv*oo]: device, unit 2-norm over unique elements.
 * Returns CCLR_OK or CCLR_ENOTCONV (best Ritz pairs written, info filled). */
int cclr_eom(cclr_ctx *ctx, int nroots, double tol, int maxiter, cclr_c128 *eig, cclr_c128 *r1_out, cclr_c128 *r2_out,
             cclr_eom_info *info);

/* The CCSD residual Omega(t) = <mu| exp(-T) H exp(T) |R> at arbitrary amplitudes, by either of the library's two independent
 * routes: mode 0 = the direct residual plan cclr_ccsd iterates on, mode 1 = Omega(0) + 1/2 sum_k A(s_k t) . t through
 * cclr_create + cclr_sigma at the two Gauss points (the cross-check; ~6 times more work).  om1 [v*o], om2 [vv*oo]: device. */
int cclr_ccsd_residual(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, const cclr_c128 *t1, const cclr_c128 *t2,
                       int mode, void *cuda_stream, cclr_c128 *om1, cclr_c128 *om2);

/* Cap the trial-space dimension of cclr_solve (memory = 2 * dim * (v*o + vv*oo) * 16 bytes); 0 = sized from the free
 * device memory.  When the space is full it is collapsed onto the current solutions and the iteration continues. */
int cclr_set_max_subspace(cclr_ctx *ctx, int dim);

void cclr_destroy(cclr_ctx *ctx);
const char *cclr_strerror(int code);
int cclr_last_cuda_error(void); /* CUDA error code behind the last CCLR_ECUDA of the calling thread */
const char *cclr_last_error_message(void); /* text of the last failure of the calling thread ("" if none) */

/* The property contraction for callers that cannot allocate device memory (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc): result[k] = sum_i eta1[i] x1[k][i] + sum_i eta2[i] x2[k][i] (bilinear, as cclr_property) for
 * nvec <= CCLR_NOALLOC_MAX_VECS vectors, eta1 [n1], eta2 [n2], x1 [nvec][n1], x2 [nvec][n2] and result [nvec] all DEVICE arrays
 * (the caller owns inputs and outputs; the result stays on the device and the call does not synchronise).  No context, and no
 * cudaMalloc / cudaFree / allocating routine inside: the partial sums of the two-pass reduction live in a file-scope static
 * device array of 151,552 bytes (csrc/vecops.cu) that every GPU loading the library holds until exit.  Every call shares that array:
 * calls that overlap on the GPU (other streams or threads) race; calls on one stream are safe, and stale contents are harmless.
 * Returns CCLR_OK; CCLR_EINVAL with a message for null pointers, n1 < 1, n2 < 1, nvec < 1 or nvec > CCLR_NOALLOC_MAX_VECS;
 * CCLR_ECUDA if the device address of the array cannot be had or a launch fails. */
#define CCLR_NOALLOC_MAX_VECS 16
int cclr_property_noalloc(void *cuda_stream, const cclr_c128 *eta1, const cclr_c128 *eta2, const cclr_c128 *x1, const cclr_c128 *x2,
                          long n1, long n2, int nvec, cclr_c128 *result);

/* ---- host-buffer forms (end-to-end timing: host<->device copies are part of the call) ------------------------ */
/* Same as cclr_sigma with HOST x1, x2, out1, out2 (pinned or pageable). */
int cclr_sigma_host(cclr_ctx *ctx, const cclr_c128 *x1, const cclr_c128 *x2, int nvec, double omega, double gamma,
                    cclr_c128 *out1, cclr_c128 *out2);

/* ---- kernel-level entry points (unit tests, roofline measurement) ------------------------------------------------ */
/* C[M][N] = alpha * opA(A)[M][K] * opB(B) + beta * C, complex128, row-major with leading dimensions in elements.
 * A is always [M][K] (K contiguous).  b_is_kn = 0: B is [N][K] (K contiguous); 1: B is [K][N] (N contiguous).
 * conj_a / conj_b conjugate the operand elementwise.  batch > 1 repeats with element strides sa, sb, sc.
 * The complex product runs on the FP64 tensor cores (DMMA) from TMA-staged shared-memory tiles: 4M (four real products per
 * complex one), or, when three_m != 0 and the shape is large (M >= 512, N >= 24, K >= 64: ladder, ring, W builds), the 3M
 * product T1 = Ar Br, T2 = Ai Bi, T3 = (Ar+Ai)(Br+Bi), C = (T1 - T2) + i (T3 - T1 - T2) -- three real products instead of four.
 * Both hold the 1e-10 parity tolerance norm-wise; 3M loses relative accuracy in a component that is much smaller than its
 * partner (north_star: "3M only if it holds the tolerance").  N = 1 / M = 1 shapes go to
 * bandwidth-bound matrix-vector kernels.  alpha, beta are host pointers to one complex number. */
int cclr_zgemm(void *cuda_stream, int M, int N, int K, const cclr_c128 *alpha, const cclr_c128 *A, long lda,
               int conj_a, const cclr_c128 *B, long ldb, int b_is_kn, int conj_b, const cclr_c128 *beta,
               cclr_c128 *C, long ldc, int batch, long sa, long sb, long sc, int three_m);

/* The same product C = alpha opA(A) opB(B) + beta C (batch 1) at FP64 accuracy on the INT8 tensor path (tcgen05.mma.kind::i8, S32
 * accumulators in tensor memory) by integer slicing of the operands (csrc/zgemm_oz.cu): every row of A and every
 * column of B is scaled by a power of two and cut into `slices` (2..8) signed slices of 7 bits; the slices * (slices + 1) / 2
 * integer products with t + u < slices are exact, so the only error is the truncation of the operands 6 + 7 (slices - 1) bits below
 * their row / column maxima (slices = 6: norm-wise ~1e-11 for rows without outliers; it holds north_star's 1e-10 on sigma).
 * Shapes: M >= 512, N >= 32, 512 <= K < 2^17 and at least 64 output tiles, ceil(M / 256) * ceil(2 N / 256) >= 64 (else CCLR_EINVAL).  reps >= 1 repeats the product (timing); ms (HOST, may be NULL)
 * receives ms[0] = slicing A (done once), ms[1] = one product including the slicing of B, ms[2] = the slicing of B alone
 * (CUDA events on the stream).  slices + 100 (b_is_kn only): B is the constant operand -- its TRANSPOSE is sliced once and the
 * product runs as C^T = B^T A^T with a transposed store (the route of the left transform's ladder).  bn = 0 picks the tile width and cluster shape; else bn % 1000 forces the width (multiple of 16 in
 * [16, 256]) and (bn / 1000) % 10, bn / 10000 the CTAs of a cluster along N and M (tuning runs).  With beta != 0 use reps = 1. */
int cclr_zgemm_oz(void *cuda_stream, int M, int N, int K, const cclr_c128 *alpha, const cclr_c128 *A, long lda, int conj_a,
                  const cclr_c128 *B, long ldb, int b_is_kn, int conj_b, const cclr_c128 *beta, cclr_c128 *C, long ldc,
                  int slices, int bn, int reps, double *ms);

/* Switch the ladder / ring of an existing context between the integer-slice product (path = 1; only if the context holds the slices,
 * i.e. was created without CCLR_GEMM_DMMA / CCLR_GEMM_4M at an eligible size) and DMMA (path = 0).  Returns the path now in use. */
int cclr_set_gemm_path(cclr_ctx *ctx, int path);

/* Number of integer slices per operand the context's INT8 tensor path works with (6 for integrals without outliers inside their
 * rows; 7 or 8 when cclr_create found a wider range, from the rms over the rows of (power-of-two row scale / row rms) of W_vvvv and
 * W_ovvo, so that 2^(-7 s) rho^2 <= 3e-11), or 0 when ladder and ring run on the FP64 tensor cores. */
int cclr_gemm_slices(const cclr_ctx *ctx);

/* The particle-particle ladder alone (term T11 of S-Eq. 12):
 * out2[k][ab][ij] = sum_{e<f} W_vvvv[ab][ef] x2[k][ef][ij] for nvec vectors (no shift, no other term). */
int cclr_ladder(cclr_ctx *ctx, const cclr_c128 *x2, int nvec, cclr_c128 *out2);

/* The ring term alone (T8 of S-Eq. 12): out2[ab][ij] = P(ab)P(ij) sum_me W_mbej x2[ae][im], one vector. */
int cclr_ring(cclr_ctx *ctx, const cclr_c128 *x2, cclr_c128 *out2);

/* Copy a named intermediate to a device buffer of `capacity` elements (tests: block-by-block parity against the
 * oracle).  Names and layouts: see DESIGN.md "Data layout".  Returns the element count, or a negative error. */
long cclr_get_intermediate(cclr_ctx *ctx, const char *name, cclr_c128 *out, long capacity);
/* Same for `count` consecutive elements starting at element `offset` of the named intermediate (full-size parity tests: one
 * row of the 32 GB W_vvvv, one (b,j) slice of W_ovvo, ...).  Returns count, or CCLR_EINVAL if the range is outside the buffer. */
long cclr_get_intermediate_slice(cclr_ctx *ctx, const char *name, long offset, long count, cclr_c128 *out);

/* Number of CUDA kernels this library has launched in the calling process so far (every GEMM, layout and vector
 * kernel is counted at its launch site; memcpy / memset are not).  bench.py reports the difference over its timed
 * region as "gpu_launches". */
unsigned long long cclr_kernel_launches(void);

/* Device bytes currently owned by the context. */
size_t cclr_ctx_bytes(const cclr_ctx *ctx);

/* Milliseconds (CUDA events on the context's stream) spent in each phase of the last cclr_sigma call:
 * ms[0] total, ms[1] ladder GEMM, ms[2] ring GEMM, ms[3] other GEMMs, ms[4] layout / bandwidth kernels.
 * Only filled when profiling was enabled with cclr_set_profiling(ctx, 1) (which adds event records). */
int cclr_set_profiling(cclr_ctx *ctx, int on);
int cclr_last_sigma_ms(const cclr_ctx *ctx, double ms[5]);
/* Per operation of the sigma plan (csrc/plans.inc, CCLR_PLAN_SIGMA): the number of operations, the plan statement of
 * operation k (a string owned by the context), and the milliseconds each took in the last profiled cclr_sigma call
 * (summed over its nvec vectors); cclr_last_sigma_op_ms returns the count, or CCLR_EINVAL if capacity is too small. */
int cclr_sigma_op_count(const cclr_ctx *ctx);
const char *cclr_sigma_op_text(const cclr_ctx *ctx, int k);
int cclr_last_sigma_op_ms(const cclr_ctx *ctx, double *ms, int capacity);

/* The solver's multi-row update (steps 4-5 of PAPER.md:960-967): Y[r][i] = X[r][i] + sum_{j<m} coef[r][j] V[j][i] for R <= 8 rows
 * in ONE pass over the m vectors V (all DEVICE; leading dimensions in elements; X may be NULL = 0; ldx = 0 shares one X row),
 * optionally with nrm2[r] = ||Y[r]||_2^2 (DEVICE doubles, or NULL) and the preconditioned rows P[r][i] = Y[r][i] / (z[r] - D[i])
 * (D = the context's orbital-energy denominators, z DEVICE [R]; P NULL to skip; then n <= v*o + vv*oo). */
int cclr_vec_block_lincomb(cclr_ctx *ctx, int R, cclr_c128 *Y, long ldy, const cclr_c128 *X, long ldx, const cclr_c128 *coef,
                           const cclr_c128 *V, long ldv, int m, long n, double *nrm2, const cclr_c128 *z, cclr_c128 *P, long ldp);
/* Sesquilinear dot block out[ia*nb + ib] = sum_i conj(A[ia][i]) B[ib][i] (Eq. 29) through the path the solver
 * uses (one split-K DMMA GEMM for blocks, the chunked reduction kernel for single rows): A [na][n], B [nb][n] DEVICE dense rows
 * (ld must equal n), out HOST [na*nb]. */
int cclr_vec_dots(cclr_ctx *ctx, const cclr_c128 *A, int na, const cclr_c128 *B, int nb, long n, long ld, cclr_c128 *out);

/* HOST-only: the reduced-space step of cclr_solve: beta[k] = (G - z[k] I)^{-1} rhs for nz shifts sharing one
 * L x L row-major matrix G, through one Hessenberg reduction.  All pointers are host pointers; beta is [nz][L]. */
int cclr_host_shifted_solve(int L, const cclr_c128 *G, const cclr_c128 *rhs, int nz, const cclr_c128 *z, cclr_c128 *beta);

/* HOST-only: eigenvalues w [L] and right eigenvectors (columns of the row-major L x L matrix V, unit 2-norm) of a general
 * complex row-major L x L matrix G — the reduced eigenproblem of cclr_eom (Hessenberg reduction + complex QR). */
int cclr_host_eigen(int L, const cclr_c128 *G, cclr_c128 *w, cclr_c128 *V);

/* FP64 tensor-core (DMMA m8n8k4) issue-rate probe: runs `iters` dependent-chain-free DMMA per warp on every SM
 * and returns the measured TFLOP/s in *tflops (host).  This is the roofline denominator used by bench.py. */
int cclr_fp64_tensor_peak(void *cuda_stream, int iters, double *tflops);

/* FP64 datapath probe: mode 0 = DMMA only (same as cclr_fp64_tensor_peak), 1 = vector DFMA only, 2 = half the warps DMMA and
 * half DFMA.  On B200 all three give the same ~37 TFLOP/s: the tensor and vector FP64 paths share one datapath, so mixing
 * them cannot raise a contraction above the DMMA peak. */
int cclr_fp64_pipe_probe(void *cuda_stream, int mode, int iters, double *tflops);

/* Streaming-copy probe over `bytes` of device memory (read + write) -> GB/s in *gbs (host). */
int cclr_hbm_copy_peak(void *cuda_stream, size_t bytes, double *gbs);

#ifdef __cplusplus
}
#endif
#endif /* CCLR_H */
