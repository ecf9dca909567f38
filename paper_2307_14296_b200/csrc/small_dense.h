// small_dense.h — the reduced-space algebra of the response solver (step 3 of PAPER.md:955, Eq. 29; Fig. 1
// PAPER.md:971 "reduced system solved on the host"): G' beta = C' with G' = G - z I for MANY shifts z sharing one
// projected Jacobian G = b^H A b.  One Householder reduction to Hessenberg form G = Q H Q^H (O(L^3), once per
// subspace) makes every shifted system an O(L^2) Hessenberg solve:  beta(z) = Q (H - z)^{-1} Q^H c.
// Host-only, plain C++ (no CUDA); L is the subspace dimension (<= a few hundred).
#pragma once
#include <cmath>
#include <complex>
#include <vector>

namespace small_dense {

typedef std::complex<double> cplx;

struct Hessenberg {
  int n = 0;
  std::vector<cplx> H, Q;   // row-major n x n; G = Q H Q^H

  // G: row-major n x n (copied)
  void factor(const cplx *G, int n_) {
    n = n_;
    H.assign(G, G + (size_t)n * n);
    Q.assign((size_t)n * n, cplx(0.0));
    for (int i = 0; i < n; ++i) Q[(size_t)i * n + i] = 1.0;
    std::vector<cplx> v(n), w(n);
    for (int k = 0; k + 2 < n; ++k) {
      double nx = 0.0;
      for (int i = k + 1; i < n; ++i) nx += std::norm(H[(size_t)i * n + k]);
      nx = std::sqrt(nx);
      if (nx == 0.0) continue;
      const cplx x0 = H[(size_t)(k + 1) * n + k];
      const cplx phase = std::abs(x0) > 0.0 ? x0 / std::abs(x0) : cplx(1.0);
      const cplx alpha = -phase * nx;
      double nv = 0.0;
      for (int i = k + 1; i < n; ++i) {
        v[i] = H[(size_t)i * n + k] - (i == k + 1 ? alpha : cplx(0.0));
        nv += std::norm(v[i]);
      }
      nv = std::sqrt(nv);
      if (nv == 0.0) continue;
      for (int i = k + 1; i < n; ++i) v[i] /= nv;
      // H <- P H, P = I - 2 v v^H (rows k+1..)
      for (int j = 0; j < n; ++j) {
        cplx s = 0.0;
        for (int i = k + 1; i < n; ++i) s += std::conj(v[i]) * H[(size_t)i * n + j];
        w[j] = 2.0 * s;
      }
      for (int i = k + 1; i < n; ++i)
        for (int j = 0; j < n; ++j) H[(size_t)i * n + j] -= v[i] * w[j];
      // H <- H P (columns k+1..), Q <- Q P
      for (int i = 0; i < n; ++i) {
        cplx s = 0.0, t = 0.0;
        for (int j = k + 1; j < n; ++j) {
          s += H[(size_t)i * n + j] * v[j];
          t += Q[(size_t)i * n + j] * v[j];
        }
        s *= 2.0;
        t *= 2.0;
        for (int j = k + 1; j < n; ++j) {
          H[(size_t)i * n + j] -= s * std::conj(v[j]);
          Q[(size_t)i * n + j] -= t * std::conj(v[j]);
        }
      }
      for (int i = k + 2; i < n; ++i) H[(size_t)i * n + k] = 0.0;
    }
  }

  // beta = (G - z)^{-1} rhs; returns false if a pivot vanishes (z is numerically an eigenvalue of G)
  bool solve(cplx z, const cplx *rhs, cplx *beta) const {
    std::vector<cplx> M((size_t)n * n), y(n);
    for (int i = 0; i < n; ++i) {
      cplx s = 0.0;
      for (int j = 0; j < n; ++j) s += std::conj(Q[(size_t)j * n + i]) * rhs[j];   // Q^H rhs
      y[i] = s;
    }
    M = H;
    for (int i = 0; i < n; ++i) M[(size_t)i * n + i] -= z;
    // Gaussian elimination of the single subdiagonal with row exchanges
    for (int k = 0; k + 1 < n; ++k) {
      if (std::abs(M[(size_t)(k + 1) * n + k]) > std::abs(M[(size_t)k * n + k])) {
        for (int j = k; j < n; ++j) std::swap(M[(size_t)k * n + j], M[(size_t)(k + 1) * n + j]);
        std::swap(y[k], y[k + 1]);
      }
      const cplx piv = M[(size_t)k * n + k];
      if (std::abs(piv) == 0.0) return false;
      const cplx f = M[(size_t)(k + 1) * n + k] / piv;
      if (f != cplx(0.0)) {
        for (int j = k; j < n; ++j) M[(size_t)(k + 1) * n + j] -= f * M[(size_t)k * n + j];
        y[k + 1] -= f * y[k];
      }
    }
    for (int i = n - 1; i >= 0; --i) {
      cplx s = y[i];
      for (int j = i + 1; j < n; ++j) s -= M[(size_t)i * n + j] * y[j];
      const cplx piv = M[(size_t)i * n + i];
      if (std::abs(piv) == 0.0) return false;
      y[i] = s / piv;
    }
    for (int i = 0; i < n; ++i) {
      cplx s = 0.0;
      for (int j = 0; j < n; ++j) s += Q[(size_t)i * n + j] * y[j];
      beta[i] = s;
    }
    return true;
  }
};

}  // namespace small_dense
