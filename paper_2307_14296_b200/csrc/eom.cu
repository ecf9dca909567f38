// eom.cu — cclr_eom: the lowest EOM-EE excitation energies and right eigenvectors of the CCSD Jacobian A (PAPER.md:131
// Eq. 14), i.e. the poles of the linear response function ("the poles of alpha(omega) coincide with the
// EOM-EE energies" is the paper's own check of its LR solver).  SURVEY.md 8(f) row f4.  The sigma routine, the trial-space
// kernels and the packed storage are those of the response solver (both solvers share the sigma vector).
//
// Block Davidson for a non-Hermitian matrix: orthonormal trial space {b_j}, sigma_j = A b_j, projected matrix G = b^H sigma;
// the reduced eigenproblem G y = theta y is solved on the host (small_dense::eigen: Hessenberg + complex QR); roots are the
// nroots Ritz values of lowest real part; residual r = sigma y - theta b y, correction r / (theta - D) with the orbital-energy
// diagonal, two-pass Gram-Schmidt, collapse onto the current Ritz vectors when the space is full.
// Start vectors: unit vectors on the smallest orbital-energy differences D.
#include "subspace.cuh"
#include <chrono>
#include <numeric>

namespace {

using subspace::check;
using subspace::cplx;
using subspace::DeviceBuf;

__global__ void unit_vector_kernel(c128 *v, long n, long pos) {
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x)
    v[i] = make_double2(i == pos ? 1.0 : 0.0, 0.0);
}

}  // namespace

extern "C" int cclr_eom(cclr_ctx *ctx, int nroots, double tol, int maxiter, cclr_c128 *eig, cclr_c128 *r1_out,
                        cclr_c128 *r2_out, cclr_eom_info *info) {
  if (!ctx || nroots < 1 || !(tol > 0.0) || maxiter < 1 || !eig || !r1_out || !r2_out) {
    cclr_set_error("cclr_eom: null pointer, nroots < 1, tol <= 0 or maxiter < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  const auto wall0 = std::chrono::steady_clock::now();
  cclr_eom_info res{};
  int rc = CCLR_ENOTCONV;
  try {
    const long n1 = ctx->n1, n2 = ctx->n2, n = n1 + n2;
    if (nroots > n) throw PlanError(CCLR_EINVAL, "cclr_eom: more roots than unique excitations");
    cudaStream_t st = ctx->st;
    // ---- trial-space size from the free device memory ----
    size_t free_b = 0, total_b = 0;
    check(cudaMemGetInfo(&free_b, &total_b), "cudaMemGetInfo");
    const double vec_b = (double)n * sizeof(c128);
    int maxdim = (int)std::min<double>(std::min<double>((double)n, std::max(12 * nroots, 48)),
                                       std::floor((0.85 * (double)free_b - (2.0 * nroots + 2.0) * vec_b) / (2.0 * vec_b)));
    if (ctx->max_subspace > 0) maxdim = std::min(maxdim, std::max(ctx->max_subspace, 2 * nroots + 2));
    if (maxdim < std::min<long>(n, 2 * nroots + 2))
      throw PlanError(CCLR_ENOMEM, "cclr_eom: not enough free device memory for the trial space");
    subspace::Space S;
    S.ctx = ctx; S.st = st; S.n = n; S.n1 = n1; S.n2 = n2; S.maxdim = maxdim;
    S.Bm.alloc((size_t)maxdim * n, "cudaMalloc(trial space)");
    S.Sm.alloc((size_t)maxdim * n, "cudaMalloc(sigma space)");
    S.coef.alloc((size_t)2 * maxdim, "cudaMalloc(coefficients)");
    S.G.assign((size_t)maxdim * maxdim, cplx(0.0));
    DeviceBuf R, tmp;
    R.alloc((size_t)nroots * n, "cudaMalloc(residuals / Ritz vectors)");
    tmp.alloc((size_t)nroots * n, "cudaMalloc(collapse scratch)");

    // ---- start vectors: unit vectors on the smallest denominators ----
    std::vector<double> D((size_t)n);
    check(cudaMemcpyAsync(D.data(), ctx->D, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, st), "D2H denominators");
    check(cudaStreamSynchronize(st), "sync");
    const int nguess = (int)std::min<long>(std::min<long>(n, maxdim), std::max(2 * nroots, nroots + 4));
    std::vector<long> order((size_t)n);
    std::iota(order.begin(), order.end(), 0L);
    std::partial_sort(order.begin(), order.begin() + nguess, order.end(), [&](long a, long b) { return D[a] < D[b] || (D[a] == D[b] && a < b); });
    for (int g = 0; g < nguess; ++g) {
      unit_vector_kernel<<<zgemm_num_sms() * 8, 256, 0, st>>>(R.p, n, order[g]);
      cclr_count_launch();
      S.append(R.p);
    }
    std::vector<cplx> theta(nroots), Y;     // Y: L x nroots Ritz coefficient vectors (column k at Y[j*nroots + k])
    std::vector<double> rnorm(nroots, 0.0);
    int L0 = 0;
    for (int iter = 1; iter <= maxiter; ++iter) {
      res.iterations = iter;
      S.extend_sigma(L0);
      L0 = S.L;
      const int L = S.L;
      // ---- reduced eigenproblem ----
      std::vector<cplx> Gc((size_t)L * L), w, V;
      for (int i = 0; i < L; ++i)
        for (int j = 0; j < L; ++j) Gc[(size_t)i * L + j] = S.G[(size_t)i * maxdim + j];
      if (!small_dense::eigen(Gc.data(), L, w, V)) throw PlanError(CCLR_EINVAL, "cclr_eom: reduced eigenproblem did not converge");
      std::vector<int> idx(L);
      std::iota(idx.begin(), idx.end(), 0);
      std::sort(idx.begin(), idx.end(), [&](int a, int b) { return w[a].real() < w[b].real() || (w[a].real() == w[b].real() && w[a].imag() < w[b].imag()); });
      const int nr = std::min(nroots, L);
      Y.assign((size_t)L * nroots, cplx(0.0));
      for (int k = 0; k < nr; ++k) {
        theta[k] = w[idx[k]];
        for (int j = 0; j < L; ++j) Y[(size_t)j * nroots + k] = V[(size_t)j * L + idx[k]];
      }
      // ---- residuals r_k = sum_j y_jk (sigma_j - theta_k b_j) ----
      bool all = nr == nroots;
      std::vector<cplx> co(L);
      for (int k = 0; k < nr; ++k) {
        c128 *r = R.p + (size_t)k * n;
        for (int j = 0; j < L; ++j) co[j] = Y[(size_t)j * nroots + k];
        S.upload(co, S.coef.p);
        check(lincomb(st, r, make_double2(0.0, 0.0), S.coef.p, S.Sm.p, n, L, n), "lincomb(residual sigma)");
        for (int j = 0; j < L; ++j) co[j] = -theta[k] * Y[(size_t)j * nroots + k];
        S.add_combination(r, make_double2(1.0, 0.0), co, S.Bm.p, L, n, n);
      }
      std::vector<cplx> nr2 = S.dots(R.p, nr, R.p, nr, true);
      res.max_residual = 0.0;
      for (int k = 0; k < nr; ++k) {
        rnorm[k] = std::sqrt(std::max(0.0, nr2[k].real()));
        res.max_residual = std::max(res.max_residual, rnorm[k]);
        if (!(rnorm[k] <= tol)) all = false;
      }
      if (all) { res.converged = 1; rc = CCLR_OK; break; }
      if (iter == maxiter) break;
      // ---- collapse onto the Ritz vectors if the corrections do not fit ----
      int nnew = 0;
      bool collapsed = false;
      for (int k = 0; k < nr; ++k) nnew += rnorm[k] > tol;
      if (S.L + nnew > maxdim) {
        collapsed = true;
        // orthonormalise the nr coefficient vectors (b is orthonormal, so B C stays orthonormal)
        std::vector<std::vector<cplx>> C;
        for (int k = 0; k < nr; ++k) {
          std::vector<cplx> vv(L);
          for (int j = 0; j < L; ++j) vv[j] = Y[(size_t)j * nroots + k];
          for (int pass = 0; pass < 2; ++pass)
            for (auto &u : C) {
              cplx d = 0.0;
              for (int j = 0; j < L; ++j) d += std::conj(u[j]) * vv[j];
              for (int j = 0; j < L; ++j) vv[j] -= d * u[j];
            }
          double nv = 0.0;
          for (int j = 0; j < L; ++j) nv += std::norm(vv[j]);
          nv = std::sqrt(nv);
          if (nv < 1e-10) continue;
          for (int j = 0; j < L; ++j) vv[j] /= nv;
          C.push_back(vv);
        }
        const int m = (int)C.size();
        for (int pass = 0; pass < 2; ++pass) {
          c128 *src = pass == 0 ? S.Bm.p : S.Sm.p;
          for (int i = 0; i < m; ++i) {
            S.upload(C[i], S.coef.p);
            check(lincomb(st, tmp.p + (size_t)i * n, make_double2(0.0, 0.0), S.coef.p, src, n, L, n), "lincomb(collapse)");
          }
          check(cudaMemcpyAsync(src, tmp.p, (size_t)m * n * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy collapsed");
        }
        std::vector<cplx> GC((size_t)L * m, cplx(0.0)), Gn((size_t)m * m, cplx(0.0));
        for (int i = 0; i < L; ++i)
          for (int q = 0; q < m; ++q)
            for (int j = 0; j < L; ++j) GC[(size_t)i * m + q] += S.G[(size_t)i * maxdim + j] * C[q][j];
        for (int a = 0; a < m; ++a)
          for (int q = 0; q < m; ++q)
            for (int i = 0; i < L; ++i) Gn[(size_t)a * m + q] += std::conj(C[a][i]) * GC[(size_t)i * m + q];
        std::fill(S.G.begin(), S.G.end(), cplx(0.0));
        for (int a = 0; a < m; ++a)
          for (int q = 0; q < m; ++q) S.G[(size_t)a * maxdim + q] = Gn[(size_t)a * m + q];
        S.L = m;
        L0 = m;
      }
      // ---- corrections r / (theta - D), orthonormalised and appended ----
      int added = 0;
      for (int k = 0; k < nr && S.L < maxdim; ++k) {
        if (rnorm[k] <= tol) continue;
        c128 *r = R.p + (size_t)k * n;
        check(precondition(st, r, r, ctx->D, make_double2(theta[k].real(), theta[k].imag()), make_double2(1.0, 0.0), n), "precondition");
        if (S.append(r)) ++added;
      }
      if (added == 0) {         // no new direction: numerically converged as far as this space allows
        if (collapsed) continue;  // (re-diagonalise in the collapsed basis first so that Y matches the stored vectors)
        break;
      }
    }
    // ---- output: Ritz values and vectors x_k = B y_k (unit 2-norm over unique elements) ----
    const int L = (int)(Y.size() / nroots);
    std::vector<cplx> co(L);
    for (int k = 0; k < nroots; ++k) {
      eig[k].re = theta[k].real();
      eig[k].im = theta[k].imag();
      for (int j = 0; j < L; ++j) co[j] = Y[(size_t)j * nroots + k];
      S.upload(co, S.coef.p);
      check(lincomb(st, (c128 *)r1_out + (size_t)k * n1, make_double2(0.0, 0.0), S.coef.p, S.Bm.p, n, L, n1), "lincomb(r1)");
      check(lincomb(st, (c128 *)r2_out + (size_t)k * n2, make_double2(0.0, 0.0), S.coef.p, S.Bm.p + n1, n, L, n2), "lincomb(r2)");
      check(cudaStreamSynchronize(st), "sync");
    }
    res.sigma_calls = S.sigma_calls;
    res.subspace = S.L;
  } catch (const PlanError &e) {
    return cclr_fail(e);
  } catch (const std::exception &e) {
    cclr_set_error(e.what(), cudaSuccess);
    return CCLR_EINVAL;
  }
  res.seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - wall0).count();
  if (info) *info = res;
  if (rc == CCLR_ENOTCONV) cclr_set_error("cclr_eom: maxiter reached before every root met tol", cudaSuccess);
  return rc;
}

// Host-only: eigenvalues and right eigenvectors of a general complex L x L matrix (tests of the reduced eigenproblem).
extern "C" int cclr_host_eigen(int L, const cclr_c128 *G, cclr_c128 *w, cclr_c128 *V) {
  if (L < 1 || !G || !w || !V) return CCLR_EINVAL;
  std::vector<cplx> ww, VV;
  if (!small_dense::eigen(reinterpret_cast<const cplx *>(G), L, ww, VV)) return CCLR_ENOTCONV;
  for (int k = 0; k < L; ++k) { w[k].re = ww[k].real(); w[k].im = ww[k].imag(); }
  for (size_t k = 0; k < VV.size(); ++k) { V[k].re = VV[k].real(); V[k].im = VV[k].imag(); }
  return CCLR_OK;
}
