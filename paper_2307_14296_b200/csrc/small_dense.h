// small_dense.h — the reduced-space algebra of the response solver (step 3 of PAPER.md:955, Eq. 29; Fig. 1
// PAPER.md:971 "reduced system solved on the host"): G' beta = C' with G' = G - z I for MANY shifts z sharing one
// projected Jacobian G = b^H A b.  One Householder reduction to Hessenberg form G = Q H Q^H (O(L^3), once per
// subspace) makes every shifted system an O(L^2) Hessenberg solve:  beta(z) = Q (H - z)^{-1} Q^H c.
// Host-only, plain C++ (no CUDA); L is the subspace dimension (<= a few hundred).
#pragma once
#include <algorithm>
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

// Eigenvalues w[k] and right eigenvectors (columns of V, row-major n x n, unit 2-norm) of a general complex matrix G
// (row-major n x n): Householder reduction to Hessenberg form, single-shift complex QR with Givens rotations to the
// Schur form G = U T U^H, back-substitution for the eigenvectors of T.  The reduced eigenproblem of the EOM-EE Davidson
// solver (the sigma routine is shared with the eigen-solver).  Returns false if QR does not converge.
inline bool eigen(const cplx *G, int n, std::vector<cplx> &w, std::vector<cplx> &V) {
  Hessenberg hs;
  hs.factor(G, n);
  std::vector<cplx> &H = hs.H, &U = hs.Q;
  auto h = [&](int i, int j) -> cplx & { return H[(size_t)i * n + j]; };
  const double eps = 2.2e-16;
  int hi = n - 1, iter = 0;
  std::vector<cplx> cs(n), sn(n);
  while (hi > 0) {
    int l = hi;
    for (; l > 0; --l) {
      double sc = std::abs(h(l - 1, l - 1)) + std::abs(h(l, l));
      if (sc == 0.0) sc = 1.0;
      if (std::abs(h(l, l - 1)) <= eps * sc) { h(l, l - 1) = 0.0; break; }
    }
    if (l == hi) { --hi; iter = 0; continue; }
    if (++iter > 300) return false;
    // Wilkinson shift: the eigenvalue of the trailing 2 x 2 block closer to its last diagonal element
    const cplx a = h(hi - 1, hi - 1), b = h(hi - 1, hi), c = h(hi, hi - 1), d = h(hi, hi);
    const cplx tr2 = 0.5 * (a + d), disc = std::sqrt(tr2 * tr2 - (a * d - b * c));
    cplx mu = std::abs(tr2 + disc - d) < std::abs(tr2 - disc - d) ? tr2 + disc : tr2 - disc;
    if (iter % 11 == 10) mu = d + cplx(std::abs(h(hi, hi - 1)), std::abs(h(hi - 1, hi > 1 ? hi - 2 : 0)));   // exceptional
    for (int k = l; k <= hi; ++k) h(k, k) -= mu;
    for (int k = l; k < hi; ++k) {            // R = G_k^H ... G_l^H (H - mu)
      const cplx x = h(k, k), y = h(k + 1, k);
      const double r = std::sqrt(std::norm(x) + std::norm(y));
      cs[k] = r > 0.0 ? x / r : cplx(1.0);
      sn[k] = r > 0.0 ? y / r : cplx(0.0);
      for (int j = k; j < n; ++j) {
        const cplx t1 = h(k, j), t2 = h(k + 1, j);
        h(k, j) = std::conj(cs[k]) * t1 + std::conj(sn[k]) * t2;
        h(k + 1, j) = -sn[k] * t1 + cs[k] * t2;
      }
    }
    for (int k = l; k < hi; ++k) {            // H = R G_l ... G_k + mu, U = U G_l ... G_k
      for (int i = 0; i <= std::min(hi, k + 1); ++i) {
        const cplx t1 = h(i, k), t2 = h(i, k + 1);
        h(i, k) = t1 * cs[k] + t2 * sn[k];
        h(i, k + 1) = -t1 * std::conj(sn[k]) + t2 * std::conj(cs[k]);
      }
      for (int i = 0; i < n; ++i) {
        const cplx t1 = U[(size_t)i * n + k], t2 = U[(size_t)i * n + k + 1];
        U[(size_t)i * n + k] = t1 * cs[k] + t2 * sn[k];
        U[(size_t)i * n + k + 1] = -t1 * std::conj(sn[k]) + t2 * std::conj(cs[k]);
      }
    }
    for (int k = l; k <= hi; ++k) h(k, k) += mu;
  }
  w.resize(n);
  V.assign((size_t)n * n, cplx(0.0));
  double tnorm = 0.0;
  for (int i = 0; i < n; ++i)
    for (int j = i; j < n; ++j) tnorm = std::max(tnorm, std::abs(h(i, j)));
  const double tiny = std::max(tnorm, 1e-300) * eps;
  std::vector<cplx> x(n);
  for (int k = 0; k < n; ++k) {
    w[k] = h(k, k);
    for (int i = 0; i < n; ++i) x[i] = 0.0;
    x[k] = 1.0;
    for (int i = k - 1; i >= 0; --i) {
      cplx sacc = 0.0;
      for (int j = i + 1; j <= k; ++j) sacc += h(i, j) * x[j];
      cplx den = h(i, i) - w[k];
      if (std::abs(den) < tiny) den = tiny;
      x[i] = -sacc / den;
    }
    double nv = 0.0;
    for (int i = 0; i < n; ++i) {
      cplx sacc = 0.0;
      for (int j = 0; j <= k; ++j) sacc += U[(size_t)i * n + j] * x[j];
      V[(size_t)i * n + k] = sacc;
      nv += std::norm(sacc);
    }
    nv = std::sqrt(nv);
    if (nv > 0.0)
      for (int i = 0; i < n; ++i) V[(size_t)i * n + k] /= nv;
  }
  return true;
}

}  // namespace small_dense
