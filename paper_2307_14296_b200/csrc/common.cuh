// common.cuh — shared declarations of the CC-LR library (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>
#include <stddef.h>
#include <vector>

typedef double2 c128;  // complex128, interleaved (re, im)
struct OzWorkspace;    // zgemm_oz.cu (below)

#define CCLR_HOST_DEVICE __host__ __device__ __forceinline__

CCLR_HOST_DEVICE c128 cmul(c128 a, c128 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
CCLR_HOST_DEVICE c128 cadd(c128 a, c128 b) { return make_double2(a.x + b.x, a.y + b.y); }
CCLR_HOST_DEVICE c128 csub(c128 a, c128 b) { return make_double2(a.x - b.x, a.y - b.y); }
CCLR_HOST_DEVICE c128 cneg(c128 a) { return make_double2(-a.x, -a.y); }
CCLR_HOST_DEVICE c128 cconj(c128 a) { return make_double2(a.x, -a.y); }
CCLR_HOST_DEVICE c128 cscale(double s, c128 a) { return make_double2(s * a.x, s * a.y); }
CCLR_HOST_DEVICE c128 czero() { return make_double2(0.0, 0.0); }
// a += b * c
CCLR_HOST_DEVICE void cfma(c128 &a, c128 b, c128 c) {
  a.x = fma(b.x, c.x, a.x); a.x = fma(-b.y, c.y, a.x);
  a.y = fma(b.x, c.y, a.y); a.y = fma(b.y, c.x, a.y);
}

// pair index P(p<q) = q(q-1)/2 + p   (include/cclr.h)
CCLR_HOST_DEVICE long pair_index(long p, long q) { return q * (q - 1) / 2 + p; }
CCLR_HOST_DEVICE long npair(long n) { return n * (n - 1) / 2; }

// process-wide count of kernels launched by the library (include/cclr.h: cclr_kernel_launches)
void cclr_count_launch(int n = 1);

// ---- zgemm.cu -------------------------------------------------------------------------------------------------
struct ZgemmWorkspace {
  c128 *buf = nullptr;   // split-K partial sums
  size_t elems = 0;      // capacity in complex elements
  int three_m = 1;       // complex product of the large contractions (M >= 512, N >= 24, K >= 64): 1 = 3M, 0 = 4M everywhere
  // sum planes of the 3M product (zgemm.cu): scratch for the per-call pre-pass over operands that are small next to the
  // product, and persistent planes registered for operands that are not (W_vvvv)
  double *plane = nullptr;
  size_t plane_elems = 0;
  const c128 *persist_key[2] = {nullptr, nullptr};     // operand base pointer (unconjugated use, full leading dimension)
  const double *persist_plane[2] = {nullptr, nullptr};
  long persist_ld[2] = {0, 0};                         // leading dimension of the operand (complex elements) ...
  long persist_pld[2] = {0, 0};                        // ... and of its plane (doubles, even)
  // integer-slice product on the INT8 tensor path (zgemm_oz.cu): when set and oz->slices > 0, eligible contractions go there
  OzWorkspace *oz = nullptr;
};
// C = alpha * opA(A) * opB(B) + beta * C; see include/cclr.h (cclr_zgemm).  ws may be null (no split-K then).
cudaError_t zgemm(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA,
                  const c128 *B, long ldb, bool b_is_kn, bool conjB, c128 beta, c128 *C, long ldc, int batch = 1,
                  long sa = 0, long sb = 0, long sc = 0, const ZgemmWorkspace *ws = nullptr);
int zgemm_num_sms();
// plane[r][c] = Re X[r][c] +- Im X[r][c] (the 3M product's sum operand; see ZgemmWorkspace)
cudaError_t zgemm_sum_plane(cudaStream_t st, const c128 *X, long ld, long rows, long cols, bool conj, double *plane, long ldp);

// ---- zgemm_oz.cu: the same product at FP64 accuracy from INT8 slices (tcgen05.mma.kind::i8, S32 accumulators in TMEM) --------
struct OzEntry {
  const c128 *key = nullptr;   // operand base pointer (A operand, [rows][K], K contiguous, leading dimension ld)
  long ld = 0, rows = 0, K = 0;
  int s = 0;
  bool transposed = false;     // slices of the operand's TRANSPOSE: key is stored [K][rows] (zgemm_oz_register_t)
  int8_t *slices = nullptr;    // [s][rows][ldp] with ldp = 2K rounded up to 16 bytes
  double *scale = nullptr;     // [rows] powers of two above the row maxima
  size_t bytes = 0;
};
struct OzWorkspace {
  int slices = 0;                             // 0 = off; 2..8 slices of 7 bits (6 + 7(s-1) bits below each row maximum are kept)
  int active = 0;                             // 0 = all slices; 2 .. slices - 1: the next products use only the leading `active` slices of every
                                              // operand (precision on demand: the response solver lowers it as its residual falls)
  bool any_size = false;                      // testing aid (CCLR_GEMM_INT8_ANY_SIZE): registered operands use the path at any supported size
  int force_bn = 0, force_cm = 0, force_cn = 0;   // tile width / cluster shape overrides (tuning runs); 0 = chosen per call
  cudaEvent_t ev_b[2] = {nullptr, nullptr};   // when set: recorded around the slicing of B (cclr_zgemm_oz timing)
  std::vector<OzEntry> persist;               // slices of constant A operands (W_vvvv, W_ovvo): made once, see zgemm_oz_register
  size_t persist_bytes = 0;
  int8_t *scratch[2] = {nullptr, nullptr};    // per-call slices of an unregistered A operand / of the B operand
  size_t scratch_bytes[2] = {0, 0};
  double *scale[2] = {nullptr, nullptr};
  size_t scale_bytes[2] = {0, 0};
};
bool zgemm_oz_supported(int M, int N, int K);   // the kernel can run the shape
bool zgemm_oz_eligible(int M, int N, int K);    // ... and it pays (what the dispatch in zgemm() uses)
cudaError_t zgemm_oz(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA, const c128 *B, long ldb,
                     bool b_is_kn, bool conjB, c128 beta, c128 *C, long ldc, OzWorkspace *ow);
// slice count (6..8) that holds ~3e-11 norm-wise for an operand with this range inside its rows, 0 if none does (zgemm_oz.cu)
cudaError_t zgemm_oz_suggest_slices(cudaStream_t st, const c128 *A, long lda, long rows, long K, int *slices, double *rho_out);
cudaError_t zgemm_oz_register(cudaStream_t st, OzWorkspace *ow, const c128 *A, long lda, long rows, long K);
// the same for a constant B operand stored [K][N]: slices of its transpose, used by zgemm_oz_bt (C^T = B^T A^T, transposed store)
cudaError_t zgemm_oz_register_t(cudaStream_t st, OzWorkspace *ow, const c128 *B, long ldb, long K, long N);
bool zgemm_oz_has_bt(const OzWorkspace *ow, const c128 *B, long ldb, int N, int K);
cudaError_t zgemm_oz_bt(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA, const c128 *B, long ldb,
                        bool conjB, c128 beta, c128 *C, long ldc, OzWorkspace *ow);
void zgemm_oz_release(OzWorkspace *ow);

// ---- permute.cu: generic index-permutation / pair (un)packing / antisymmetrising gather-scatter kernel ---------
// dst(iteration index) (+)= sum_k coef_k * sign_k * [conj] src_k(slots(letters)); see plans.inc for the semantics.
constexpr int PERM_MAX_AXES = 6, PERM_MAX_SLOTS = 5, PERM_MAX_SRC = 10, PERM_MAX_LETTERS = 12;
struct PermAxis {
  int kind;      // 0 = plain letter, 1 = packed pair (p<q), 2 = unit extent
  int ext;       // extent of the axis (pair axes: n(n-1)/2)
  int l0, l1;    // letter ids written by this axis (l1 for pairs)
  int off;       // global offset added to a plain letter (chunk loops)
};
struct PermSlot {
  int kind;      // 0 = plain, 1 = antisymmetric pair, 2 = unit
  int l0, l1;    // letter ids read by this slot
  int sub;       // subtracted from a plain letter's global value (buffer declared over a chunk)
  long stride;   // elements
};
struct PermOperand {
  const c128 *ptr;
  c128 coef;
  int conj, nslot;
  PermSlot slot[PERM_MAX_SLOTS];
};
struct PermArgs {
  int naxis, nsrc, accumulate, cond;   // cond: 0 = all, 1 = only dst-pair p<q, 2 = only p>q
  int cond_l0, cond_l1, dst_linear, ndslot;
  long total;
  c128 *dst;
  PermAxis axis[PERM_MAX_AXES];
  PermSlot dslot[PERM_MAX_SLOTS];
  PermOperand src[PERM_MAX_SRC];
};
cudaError_t permute(cudaStream_t st, const PermArgs &args);

// ---- layout.cu: the hot layout statements of sigma, specialised (semantics: see the kernels' comments) ----------------
cudaError_t layout_unpack_rows(cudaStream_t st, const c128 *src, c128 *dst, int n, long len);
cudaError_t layout_unpack_cols(cudaStream_t st, const c128 *src, c128 *dst, long rows, int o);
cudaError_t layout_unpack_ring(cudaStream_t st, const c128 *src, c128 *dst, int v, int o);
cudaError_t layout_transpose_pair(cudaStream_t st, const c128 *src, c128 *dst, long ncol, int o);
cudaError_t layout_final_pack(cudaStream_t st, c128 *out2, const c128 *x2, c128 nz, const c128 *Y, const c128 *Q, const c128 *Z,
                              int v, int o);
constexpr size_t LAYOUT_MAX_SMEM = 200 * 1024;   // final_pack stages 3 o^2 complex numbers (o <= 65)

// ---- vecops.cu: bandwidth kernels of the solver / property contraction ------------------------------------------
// out[ia*nb+ib] = sum_i op(A[ia][i]) * B[ib][i]  (op = conj if conjA); diag != 0: out[ia] = sum_i op(A[ia][i]) B[ia][i].
// partial is a device scratch of at least dots_scratch_elems(na*nb) complex numbers; out is a DEVICE array.
size_t dots_scratch_elems(int npairs);
cudaError_t multi_dot(cudaStream_t st, const c128 *A, long lda, int na, const c128 *B, long ldb, int nb, long n,
                      bool conjA, bool diag, c128 *partial, c128 *out);
// y[i] = beta * y[i] + sum_{j<m} coef[j] * V[j*ldv + i]   (coef: DEVICE array of m complex numbers)
cudaError_t lincomb(cudaStream_t st, c128 *y, c128 beta, const c128 *coef, const c128 *V, long ldv, int m, long n);
// Y[r][i] = xs * X[r][i] + sum_j coef[r][j] V0[j][i] + sum_j coef[r][m0+j] V1[j][i] for R <= BLOCK_LINCOMB_MAX rows in one pass
// over the m0 + m1 vectors, with optional fused squared norms (nrm2: device [R]; nrm_scratch: block_lincomb_grid(n) * R doubles)
// and optional preconditioned output P[r][i] = Y[r][i] / (z[r] - D[i]) (z: device [R]); see vecops.cu
constexpr int BLOCK_LINCOMB_MAX = 8;
int block_lincomb_grid(long n);
cudaError_t block_lincomb(cudaStream_t st, int R, c128 *Y, long ldy, const c128 *X, long ldx, c128 xs, const c128 *coef, int ldc,
                          const c128 *V0, long ldv0, int m0, const c128 *V1, long ldv1, int m1, long n, double *nrm2,
                          double *nrm_scratch, const double *D, const c128 *z, c128 *P, long ldp);
// y[i] = alpha * x[i] / (z - D[i])      (orbital-energy preconditioner)
cudaError_t precondition(cudaStream_t st, c128 *y, const c128 *x, const double *D, c128 z, c128 alpha, long n);
cudaError_t scale_vec(cudaStream_t st, c128 *y, c128 alpha, long n);
// out[0] += sum_i |s[i] - D[i] b[i]|^2 (device double, zeroed by the caller)
cudaError_t offdiag_norm2(cudaStream_t st, const c128 *s, const c128 *b, const double *D, long n, double *out);
// out[i] = src[i] + alpha * x[i]
cudaError_t shifted_copy(cudaStream_t st, c128 *out, const c128 *src, c128 alpha, const c128 *x, long n);
// D1[a,i] = eps_a - eps_i, D2[(ab),(ij)] = eps_a + eps_b - eps_i - eps_j from the diagonal of fock ([n][n])
cudaError_t denominators(cudaStream_t st, const c128 *fock, int o, int v, double *D);
