// subspace.cuh — the trial space shared by the response solver (solver.cu) and the EOM-EE eigen-solver (eom.cu): an
// orthonormal block {b_j} in packed unique storage with sigma_j = A b_j and the projected Jacobian G = b^H sigma
// (Eq. 29).  Device work: cclr_sigma_one, tall-skinny dots, linear combinations (vecops.cu).
#pragma once
#include "context.cuh"
#include "small_dense.h"
#include <algorithm>
#include <cmath>

namespace subspace {

typedef small_dense::cplx cplx;

inline void check(cudaError_t e, const char *where) {
  if (e != cudaSuccess)
    throw PlanError(e == cudaErrorMemoryAllocation ? CCLR_ENOMEM : CCLR_ECUDA, std::string(where) + ": " + cudaGetErrorString(e), e);
}

struct DeviceBuf {
  c128 *p = nullptr;
  ~DeviceBuf() { if (p) cudaFree(p); }
  void alloc(size_t elems, const char *what) { check(cudaMalloc(&p, (elems ? elems : 1) * sizeof(c128)), what); }
};

struct Space {
  cclr_ctx *ctx;
  cudaStream_t st;
  long n, n1, n2;
  int maxdim = 0, L = 0;
  DeviceBuf Bm, Sm, coef;
  std::vector<cplx> G;        // maxdim x maxdim, row-major: G[i][j] = b_i^H sigma_j
  int sigma_calls = 0;
  bool left = false;          // sigma_j = A^T b_j (left transform) instead of A b_j
  // Precision on demand (solver.cu; contexts whose ladder / ring run as integer-slice products, zgemm_oz.cu): a trial vector
  // added when the residuals have fallen to relres enters the solutions with coefficients of that size, so its sigma vector may
  // carry a relative error ~ tol / relres without moving the converged residual (inexact-Krylov argument) -- sigma_j is then
  // formed with fewer slices (15, 10, 6 pair products instead of 21).  adapt_tol = 0: always all slices.
  double adapt_tol = 0.0, adapt_relres = 1.0;
  std::vector<double> sig_err;   // per basis vector: estimated 2-norm error of sigma_j from the dropped slices (0 with all slices)
  int reduced_sigma = 0;         // how many sigma vectors were formed with fewer slices

  double offdiag_max = 1.0;      // largest || sigma_j - D b_j || seen so far (unit b_j): the size of the contractions' contribution

  // slices for the next sigma vectors.  The vector enters the solutions with |beta_j| ~ relres ||xi||; its sigma error
  // eps_j ||sigma_j - D b_j|| (only the contractions are inexact, the diagonal part is FP64) is to stay a small part of the budget
  // tol ||xi|| / 2 shared by ~50 such vectors adding in quadrature with a safety factor 3: eps_j <= tol / (50 w relres),
  // w = offdiag_max, eps(s) = 16 * 2^(-7 s) (the measured size of the truncation error of an s-slice product).
  int slices_for_next() const {
    const OzWorkspace *oz = ctx->ws.oz;
    if (!oz || !(adapt_tol > 0.0) || (ctx->graph_enabled && !ctx->graph_failed)) return 0;   // a replayed graph has its slices baked in
    int se = oz->slices;
    while (se > 2 && std::ldexp(16.0, -7 * (se - 1)) * 50.0 * offdiag_max * std::max(adapt_relres, 1e-300) <= adapt_tol) --se;
    return se < oz->slices ? se : 0;
  }

  c128 *b(int j) { return Bm.p + (size_t)j * n; }
  c128 *s(int j) { return Sm.p + (size_t)j * n; }

  // out[ia*nb+ib] = <A_ia | B_ib> (sesquilinear) on the host.  Blocks (na, nb >= 2) run as ONE split-K DMMA GEMM
  // conj(A)[na x n] . B[nb x n]^T, which reads every vector once; single rows / columns and the diagonal use the chunked
  // reduction kernel of vecops.cu.  Both are deterministic (fixed split / chunk order).
  std::vector<cplx> dots(const c128 *A, int na, const c128 *Bp, int nb, bool diag = false) {
    const int np = diag ? na : na * nb;
    std::vector<cplx> out(np);
    if (np == 0) return out;
    cclr_ensure_dot_scratch(ctx, np);
    if (!diag && na >= 2 && nb >= 2 && n >= 4096)
      check(zgemm(st, na, nb, (int)n, make_double2(1.0, 0.0), A, n, true, Bp, n, false, false, make_double2(0.0, 0.0),
                  ctx->dot_out, nb, 1, 0, 0, 0, &ctx->ws), "zgemm(dots)");
    else
      check(multi_dot(st, A, n, na, Bp, n, nb, n, true, diag, ctx->dot_partial, ctx->dot_out), "multi_dot");
    check(cudaMemcpyAsync(out.data(), ctx->dot_out, (size_t)np * sizeof(c128), cudaMemcpyDeviceToHost, st), "D2H dots");
    check(cudaStreamSynchronize(st), "sync dots");
    return out;
  }

  void upload(const std::vector<cplx> &h, c128 *d) {
    check(cudaMemcpyAsync(d, h.data(), h.size() * sizeof(c128), cudaMemcpyHostToDevice, st), "H2D coefficients");
    check(cudaStreamSynchronize(st), "sync H2D");   // h is pageable and may die right after
  }

  // y = beta * y + sum_j coef_j V_j, coefficients given on the host
  void add_combination(c128 *y, c128 beta, const std::vector<cplx> &co, const c128 *V, int m, long len, long ldv) {
    if (m == 0) return;
    upload(co, coef.p);
    check(lincomb(st, y, beta, coef.p, V, ldv, m, len), "lincomb");
  }

  // orthonormalise v against b_from..b_{L-1} (Gram-Schmidt, two passes) and append it; false if (numerically) dependent.
  // n0 = the norm the vector had before any projection (the dependence test is relative to it)
  bool append_range(c128 *v, int from, double n0) {
    if (!(n0 > 0.0) || !std::isfinite(n0)) return false;
    for (int pass = 0; pass < 2 && L > from; ++pass) {
      std::vector<cplx> h = dots(b(from), L - from, v, 1);
      for (auto &x : h) x = -x;
      add_combination(v, make_double2(1.0, 0.0), h, b(from), L - from, n, n);
    }
    const double n1_ = std::sqrt(std::max(0.0, dots(v, 1, v, 1)[0].real()));
    if (!(n1_ > 1e-10 * n0)) return false;
    check(scale_vec(st, v, make_double2(1.0 / n1_, 0.0), n), "scale");
    check(cudaMemcpyAsync(b(L), v, (size_t)n * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy trial vector");
    ++L;
    return true;
  }

  bool append(c128 *v) { return append_range(v, 0, std::sqrt(std::max(0.0, dots(v, 1, v, 1)[0].real()))); }

  // Block version (step 5 of PAPER.md:966 for all new correction vectors of an iteration at once): V holds nv vectors
  // (leading dimension n).  Two passes of block classical Gram-Schmidt against the current basis -- H = b^H V as one GEMM,
  // V -= b H as one multi-row update, each reading the basis once for all nv vectors -- then the vectors are orthonormalised
  // among themselves one by one and appended.  Returns how many were accepted.
  int append_block(c128 *V, int nv) {
    if (nv <= 0) return 0;
    std::vector<cplx> nn0 = dots(V, nv, V, nv, true);
    const int L_old = L;
    for (int pass = 0; pass < 2 && L_old > 0; ++pass) {
      std::vector<cplx> H = dots(Bm.p, L_old, V, nv);                       // [L_old][nv]
      for (int r0 = 0; r0 < nv; r0 += BLOCK_LINCOMB_MAX) {
        const int R = std::min(BLOCK_LINCOMB_MAX, nv - r0);
        std::vector<cplx> co((size_t)R * L_old);
        for (int r = 0; r < R; ++r)
          for (int j = 0; j < L_old; ++j) co[(size_t)r * L_old + j] = -H[(size_t)j * nv + r0 + r];
        upload(co, coef.p);
        check(block_lincomb(st, R, V + (size_t)r0 * n, n, V + (size_t)r0 * n, n, make_double2(1.0, 0.0), coef.p, L_old, Bm.p, n,
                            L_old, nullptr, 0, 0, n, nullptr, nullptr, nullptr, nullptr, nullptr, 0), "block_lincomb(GS)");
      }
    }
    int added = 0;
    for (int k = 0; k < nv && L < maxdim; ++k)
      if (append_range(V + (size_t)k * n, L_old, std::sqrt(std::max(0.0, nn0[k].real())))) ++added;
    return added;
  }

  // sigma_j = A b_j for j in [L0, L) and the new rows / columns of G
  void extend_sigma(int L0) {
    const int se = slices_for_next();
    if (se) ctx->ws.oz->active = se;
    try {
      for (int j = L0; j < L; ++j) {
        cclr_sigma_one(ctx, b(j), b(j) + n1, make_double2(0.0, 0.0), s(j), s(j) + n1, false, left);
        ++sigma_calls;
      }
    } catch (...) {
      if (se) ctx->ws.oz->active = 0;
      throw;
    }
    if (se) ctx->ws.oz->active = 0;
    const int nn = L - L0;
    if (nn == 0) return;
    if ((int)sig_err.size() < maxdim) sig_err.resize(maxdim, 0.0);
    if (ctx->ws.oz && adapt_tol > 0.0 && ctx->D) {
      // || sigma_j - D b_j || of the new vectors (one pass each), through the dot scratch of the context
      cclr_ensure_dot_scratch(ctx, nn);
      double *acc = (double *)ctx->dot_out;
      check(cudaMemsetAsync(acc, 0, (size_t)nn * sizeof(double), st), "memset");
      for (int j = 0; j < nn; ++j) check(offdiag_norm2(st, s(L0 + j), b(L0 + j), ctx->D, n, acc + j), "offdiag_norm2");
      std::vector<double> w(nn);
      check(cudaMemcpyAsync(w.data(), acc, (size_t)nn * sizeof(double), cudaMemcpyDeviceToHost, st), "D2H norms");
      check(cudaStreamSynchronize(st), "sync norms");
      for (int j = 0; j < nn; ++j) {
        const double wj = std::sqrt(std::max(0.0, w[j]));
        offdiag_max = std::max(offdiag_max, wj);
        sig_err[L0 + j] = se ? std::ldexp(16.0, -7 * se) * wj : 0.0;
      }
      if (se) reduced_sigma += nn;
    } else {
      for (int j = 0; j < nn; ++j) sig_err[L0 + j] = 0.0;
    }
    std::vector<cplx> cols = dots(Bm.p, L, s(L0), nn);           // G[0:L, L0:L]
    for (int i = 0; i < L; ++i)
      for (int j = 0; j < nn; ++j) G[(size_t)i * maxdim + L0 + j] = cols[(size_t)i * nn + j];
    if (L0 > 0) {
      std::vector<cplx> rows = dots(b(L0), nn, Sm.p, L0);        // G[L0:L, 0:L0]
      for (int i = 0; i < nn; ++i)
        for (int j = 0; j < L0; ++j) G[(size_t)(L0 + i) * maxdim + j] = rows[(size_t)i * L0 + j];
    }
  }
};

}  // namespace subspace
