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

  c128 *b(int j) { return Bm.p + (size_t)j * n; }
  c128 *s(int j) { return Sm.p + (size_t)j * n; }

  // out[ia*nb+ib] = <A_ia | B_ib> (sesquilinear) on the host
  std::vector<cplx> dots(const c128 *A, int na, const c128 *Bp, int nb, bool diag = false) {
    const int np = diag ? na : na * nb;
    std::vector<cplx> out(np);
    if (np == 0) return out;
    cclr_ensure_dot_scratch(ctx, np);
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

  // orthonormalise v against b_0..b_{L-1} (classical Gram-Schmidt, two passes) and append it; false if dependent
  bool append(c128 *v) {
    const double n0 = std::sqrt(std::max(0.0, dots(v, 1, v, 1)[0].real()));
    if (!(n0 > 0.0) || !std::isfinite(n0)) return false;
    for (int pass = 0; pass < 2 && L > 0; ++pass) {
      std::vector<cplx> h = dots(Bm.p, L, v, 1);
      for (auto &x : h) x = -x;
      add_combination(v, make_double2(1.0, 0.0), h, Bm.p, L, n, n);
    }
    const double n1_ = std::sqrt(std::max(0.0, dots(v, 1, v, 1)[0].real()));
    if (!(n1_ > 1e-10 * n0)) return false;
    check(scale_vec(st, v, make_double2(1.0 / n1_, 0.0), n), "scale");
    check(cudaMemcpyAsync(b(L), v, (size_t)n * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy trial vector");
    ++L;
    return true;
  }

  // sigma_j = A b_j for j in [L0, L) and the new rows / columns of G
  void extend_sigma(int L0) {
    for (int j = L0; j < L; ++j) {
      cclr_sigma_one(ctx, b(j), b(j) + n1, make_double2(0.0, 0.0), s(j), s(j) + n1, false, left);
      ++sigma_calls;
    }
    const int nn = L - L0;
    if (nn == 0) return;
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
