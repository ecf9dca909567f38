// response.cu — cclr_response_ci: the CC-CI (EOM-CC) linear response function <<X;Y>>_z of PAPER.md:142 Eq. 16 with the
// symmetriser of Eq. 17 for a complex frequency z = omega + i gamma (Eq. 20-21), assembled
// entirely from this library's device routines (workflow steps 2-4 of PAPER.md:195-203):
//
//     g(w) = EOMeta^X . t^Y(w) - (lambda . t^X(-w)) (lambda . xi^Y) + EOMeta^Y . t^X(-w) - (lambda . t^Y(w)) (lambda . xi^X)
//     <<X;Y>>_z = 1/2 [ g(z) + conj g(-conj z) ]                                   (readings 7, 8)
//
// lambda (cclr_lambda, cached in the context), xi (cclr_xi), EOM-eta (cclr_eta), t (cclr_solve: the two shifts each operator
// needs share one trial space), and bilinear dots over unique elements (cclr_property).
#include "subspace.cuh"

using subspace::check;
using subspace::DeviceBuf;

extern "C" int cclr_response_ci(cclr_ctx *ctx, const cclr_c128 *X, const cclr_c128 *Y, double omega, double gamma, double tol,
                                int maxiter, cclr_c128 *result, cclr_solve_info *info) {
  if (!ctx || !X || !Y || !result || !(tol > 0.0) || maxiter < 1) {
    cclr_set_error("cclr_response_ci: null pointer, tol <= 0 or maxiter < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  typedef std::complex<double> cplx;
  cclr_solve_info total{};
  total.converged = 1;
  try {
    const long n1 = ctx->n1, n2 = ctx->n2, n = n1 + n2;
    auto acc = [&](const cclr_solve_info &i) {
      total.iterations += i.iterations; total.sigma_calls += i.sigma_calls; total.subspace = std::max(total.subspace, i.subspace);
      total.converged = total.converged && i.converged; total.max_residual = std::max(total.max_residual, i.max_residual);
      total.seconds += i.seconds;
    };
    int rc;
    if (!ctx->lambda) {
      check(cudaMalloc(&ctx->lambda, (size_t)n * sizeof(c128)), "cudaMalloc(lambda)");
      ctx->extra_bytes += (size_t)n * sizeof(c128);
      ctx->have_lambda = false;
    }
    cclr_c128 *lam1 = (cclr_c128 *)ctx->lambda, *lam2 = (cclr_c128 *)(ctx->lambda + n1);
    if (!ctx->have_lambda) {
      cclr_solve_info li{};
      rc = cclr_lambda(ctx, tol, maxiter, lam1, lam2, &li);
      acc(li);
      if (rc != CCLR_OK && rc != CCLR_ENOTCONV) return rc;
      ctx->have_lambda = rc == CCLR_OK;
    }
    DeviceBuf xiX, xiY, eX, eY, tX, tY;
    xiX.alloc(n, "cudaMalloc(xi X)"); xiY.alloc(n, "cudaMalloc(xi Y)"); eX.alloc(n, "cudaMalloc(eta X)"); eY.alloc(n, "cudaMalloc(eta Y)");
    tX.alloc(2 * n, "cudaMalloc(t X)"); tY.alloc(2 * n, "cudaMalloc(t Y)");
    auto p1 = [&](DeviceBuf &b) { return (cclr_c128 *)b.p; };
    auto p2 = [&](DeviceBuf &b) { return (cclr_c128 *)(b.p + n1); };
    if ((rc = cclr_xi(ctx, X, p1(xiX), p2(xiX))) != CCLR_OK) return rc;
    if ((rc = cclr_xi(ctx, Y, p1(xiY), p2(xiY))) != CCLR_OK) return rc;
    if ((rc = cclr_eta(ctx, X, lam1, lam2, 1, p1(eX), p2(eX))) != CCLR_OK) return rc;
    if ((rc = cclr_eta(ctx, Y, lam1, lam2, 1, p1(eY), p2(eY))) != CCLR_OK) return rc;
    // response amplitudes: t^Y at {z, -conj z} = ({omega, -omega}, +gamma); t^X at {-z, conj z} = ({-omega, omega}, -gamma);
    // outputs are [shift][n1] and [shift][n2]
    cclr_c128 *tY1 = (cclr_c128 *)tY.p, *tY2 = (cclr_c128 *)(tY.p + 2 * n1);
    cclr_c128 *tX1 = (cclr_c128 *)tX.p, *tX2 = (cclr_c128 *)(tX.p + 2 * n1);
    const double wY[2] = {omega, -omega}, wX[2] = {-omega, omega};
    cclr_solve_info si{};
    rc = cclr_solve(ctx, p1(xiY), p2(xiY), 1, wY, 2, gamma, tol, maxiter, tY1, tY2, &si);
    acc(si);
    if (rc != CCLR_OK && rc != CCLR_ENOTCONV) return rc;
    rc = cclr_solve(ctx, p1(xiX), p2(xiX), 1, wX, 2, -gamma, tol, maxiter, tX1, tX2, &si);
    acc(si);
    if (rc != CCLR_OK && rc != CCLR_ENOTCONV) return rc;
    cclr_c128 a[2], b[2], c[2], d[2], e, f;
    if ((rc = cclr_property(ctx, p1(eX), p2(eX), tY1, tY2, 2, a)) != CCLR_OK) return rc;
    if ((rc = cclr_property(ctx, p1(eY), p2(eY), tX1, tX2, 2, b)) != CCLR_OK) return rc;
    if ((rc = cclr_property(ctx, lam1, lam2, tX1, tX2, 2, c)) != CCLR_OK) return rc;
    if ((rc = cclr_property(ctx, lam1, lam2, tY1, tY2, 2, d)) != CCLR_OK) return rc;
    if ((rc = cclr_property(ctx, lam1, lam2, p1(xiY), p2(xiY), 1, &e)) != CCLR_OK) return rc;
    if ((rc = cclr_property(ctx, lam1, lam2, p1(xiX), p2(xiX), 1, &f)) != CCLR_OK) return rc;
    auto C = [](const cclr_c128 &q) { return cplx(q.re, q.im); };
    const cplx g0 = C(a[0]) - C(c[0]) * C(e) + C(b[0]) - C(d[0]) * C(f);
    const cplx g1 = C(a[1]) - C(c[1]) * C(e) + C(b[1]) - C(d[1]) * C(f);
    const cplx r = 0.5 * (g0 + std::conj(g1));
    result->re = r.real();
    result->im = r.imag();
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  if (info) *info = total;
  return total.converged ? CCLR_OK : CCLR_ENOTCONV;
}
