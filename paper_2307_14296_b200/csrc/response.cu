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

// The stencil route to x . F . y, kept as the independent cross-check of the direct plan (cclr_f_transform, CCLR_PLAN_FY):
// x . F . y = d/da [ (eta0 + lambda A)(t + a x) . y ] at a = 0  (F = CC Hessian of Table 1; S-Eq. 8, PAPER.md:855-857;
// the printed contraction formulas PAPER.md:861-879 are unrecoverable, reading 6).  The bracket is a cubic polynomial
// in a (A is cubic in t, eta0 linear), so the 4-point stencil [w(-2h) - 8 w(-h) + 8 w(h) - w(2h)] / 12h is exact; every w is one
// cclr_create at shifted amplitudes plus one left transform of lambda: "F is never formed, only t.F".
extern "C" int cclr_xfy(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, const cclr_c128 *t1, const cclr_c128 *t2,
                        const cclr_c128 *lam1, const cclr_c128 *lam2, const cclr_c128 *x1, const cclr_c128 *x2,
                        const cclr_c128 *y1, const cclr_c128 *y2, void *cuda_stream, cclr_c128 *result) {
  if (o < 2 || v < 2 || !fock || !eri || !t1 || !t2 || !lam1 || !lam2 || !x1 || !x2 || !y1 || !y2 || !result) {
    cclr_set_error("cclr_xfy: null pointer or o < 2 or v < 2", cudaSuccess);
    return CCLR_EINVAL;
  }
  typedef std::complex<double> cplx;
  try {
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long n1 = (long)o * v, n2 = npair(o) * npair(v), n = n1 + n2;
    DeviceBuf T, Xc, TS, W, coef, dpart, dout;
    T.alloc(n, "cudaMalloc(t)"); Xc.alloc(n, "cudaMalloc(x)"); TS.alloc(n, "cudaMalloc(t + a x)"); W.alloc(n, "cudaMalloc(w)");
    coef.alloc(1, "cudaMalloc(coef)"); dpart.alloc(dots_scratch_elems(2), "cudaMalloc(dot scratch)"); dout.alloc(2, "cudaMalloc(dot out)");
    check(cudaMemcpyAsync(T.p, t1, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t1");
    check(cudaMemcpyAsync(T.p + n1, t2, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t2");
    check(cudaMemcpyAsync(Xc.p, x1, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy x1");
    check(cudaMemcpyAsync(Xc.p + n1, x2, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy x2");
    cplx nrm[2];
    check(multi_dot(st, T.p, n, 1, T.p, n, 1, n, true, false, dpart.p, dout.p), "multi_dot");
    check(multi_dot(st, Xc.p, n, 1, Xc.p, n, 1, n, true, false, dpart.p + dots_scratch_elems(1), dout.p + 1), "multi_dot");
    check(cudaMemcpyAsync(nrm, dout.p, 2 * sizeof(c128), cudaMemcpyDeviceToHost, st), "D2H norms");
    check(cudaStreamSynchronize(st), "sync");
    const double nt = std::sqrt(std::max(0.0, nrm[0].real())), nx = std::sqrt(std::max(0.0, nrm[1].real()));
    if (!(nx > 0.0)) { result->re = result->im = 0.0; return CCLR_OK; }
    const double h = std::max(nt, 0.1) / nx;      // steps of the size of t itself balance round-off
    const double cs[4] = {1.0, -8.0, 8.0, -1.0}, ss[4] = {-2.0, -1.0, 1.0, 2.0};
    cplx acc = 0.0;
    for (int k = 0; k < 4; ++k) {
      const cplx step(ss[k] * h, 0.0);
      check(cudaMemcpyAsync(coef.p, &step, sizeof(c128), cudaMemcpyHostToDevice, st), "H2D step");
      check(cudaMemcpyAsync(TS.p, T.p, (size_t)n * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t");
      check(lincomb(st, TS.p, make_double2(1.0, 0.0), coef.p, Xc.p, n, 1, n), "t + a x");
      check(cudaStreamSynchronize(st), "sync");
      cclr_ctx *ck = nullptr;
      int rc = cclr_create(o, v, fock, eri, (const cclr_c128 *)TS.p, (const cclr_c128 *)(TS.p + n1), 0, cuda_stream, &ck);
      if (rc != CCLR_OK) return rc;
      cclr_c128 a, b;
      rc = cclr_sigma_left(ck, lam1, lam2, 1, 0.0, 0.0, (cclr_c128 *)W.p, (cclr_c128 *)(W.p + n1));
      if (rc == CCLR_OK) rc = cclr_property(ck, (const cclr_c128 *)W.p, (const cclr_c128 *)(W.p + n1), y1, y2, 1, &a);
      if (rc == CCLR_OK)
        rc = cclr_property(ck, (const cclr_c128 *)ck->plan->buf(ck->plan->find("FmeT")).ptr,
                           (const cclr_c128 *)ck->plan->buf(ck->plan->find("eta02")).ptr, y1, y2, 1, &b);
      cclr_destroy(ck);
      if (rc != CCLR_OK) return rc;
      acc += cs[k] * (cplx(a.re, a.im) + cplx(b.re, b.im));
    }
    acc /= 12.0 * h;
    result->re = acc.real();
    result->im = acc.imag();
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}

static int response_impl(cclr_ctx *ctx, const cclr_c128 *X, const cclr_c128 *Y, double omega, double gamma, double tol,
                         int maxiter, cclr_c128 *result, cclr_solve_info *info, const cclr_eri_packed *gs) {
  if (!ctx || !X || !Y || !result || !(tol > 0.0) || maxiter < 1) {
    cclr_set_error("cclr_response: null pointer, tol <= 0 or maxiter < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  const int eom = gs ? 0 : 1;
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
    if (!ctx->have_lambda || tol < ctx->lambda_tol) {
      cclr_solve_info li{};
      rc = cclr_lambda(ctx, tol, maxiter, lam1, lam2, &li);
      acc(li);
      if (rc != CCLR_OK && rc != CCLR_ENOTCONV) return rc;
      ctx->have_lambda = rc == CCLR_OK;
      ctx->lambda_tol = tol;
    }
    DeviceBuf xiX, xiY, eX, eY, tX, tY;
    xiX.alloc(n, "cudaMalloc(xi X)"); xiY.alloc(n, "cudaMalloc(xi Y)"); eX.alloc(n, "cudaMalloc(eta X)"); eY.alloc(n, "cudaMalloc(eta Y)");
    tX.alloc(2 * n, "cudaMalloc(t X)"); tY.alloc(2 * n, "cudaMalloc(t Y)");
    auto p1 = [&](DeviceBuf &b) { return (cclr_c128 *)b.p; };
    auto p2 = [&](DeviceBuf &b) { return (cclr_c128 *)(b.p + n1); };
    if ((rc = cclr_xi(ctx, X, p1(xiX), p2(xiX))) != CCLR_OK) return rc;
    if ((rc = cclr_xi(ctx, Y, p1(xiY), p2(xiY))) != CCLR_OK) return rc;
    if ((rc = cclr_eta(ctx, X, lam1, lam2, eom, p1(eX), p2(eX))) != CCLR_OK) return rc;
    if ((rc = cclr_eta(ctx, Y, lam1, lam2, eom, p1(eY), p2(eY))) != CCLR_OK) return rc;
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
    auto C = [](const cclr_c128 &q) { return cplx(q.re, q.im); };
    cplx g0, g1;
    if (!gs) {   // CC-CI, Eq. 16
      if ((rc = cclr_property(ctx, lam1, lam2, tX1, tX2, 2, c)) != CCLR_OK) return rc;
      if ((rc = cclr_property(ctx, lam1, lam2, tY1, tY2, 2, d)) != CCLR_OK) return rc;
      if ((rc = cclr_property(ctx, lam1, lam2, p1(xiY), p2(xiY), 1, &e)) != CCLR_OK) return rc;
      if ((rc = cclr_property(ctx, lam1, lam2, p1(xiX), p2(xiX), 1, &f)) != CCLR_OK) return rc;
      g0 = C(a[0]) - C(c[0]) * C(e) + C(b[0]) - C(d[0]) * C(f);
      g1 = C(a[1]) - C(c[1]) * C(e) + C(b[1]) - C(d[1]) * C(f);
    } else {     // CC-CC, Eq. 15: g(w) = eta^X . t^Y(w) + eta^Y . t^X(-w) + t^X(-w) . F . t^Y(w)
      // F t^Y for both shifts in one call of the direct plan (one lambda-only ladder, then ~3 sigma-equivalents per vector)
      DeviceBuf FY;
      FY.alloc(2 * n, "cudaMalloc(F t)");
      cclr_c128 *fy1 = (cclr_c128 *)FY.p, *fy2 = (cclr_c128 *)(FY.p + 2 * n1);
      if ((rc = cclr_f_transform(ctx, gs, lam1, lam2, tY1, tY2, 2, fy1, fy2)) != CCLR_OK) return rc;
      for (int k = 0; k < 2; ++k)
        if ((rc = cclr_property(ctx, tX1 + (size_t)k * n1, tX2 + (size_t)k * n2, fy1 + (size_t)k * n1, fy2 + (size_t)k * n2, 1, &c[k])) != CCLR_OK)
          return rc;
      g0 = C(a[0]) + C(b[0]) + C(c[0]);
      g1 = C(a[1]) + C(b[1]) + C(c[1]);
    }
    const cplx r = 0.5 * (g0 + std::conj(g1));
    result->re = r.real();
    result->im = r.imag();
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  if (info) *info = total;
  return total.converged ? CCLR_OK : CCLR_ENOTCONV;
}

extern "C" int cclr_response_ci(cclr_ctx *ctx, const cclr_c128 *X, const cclr_c128 *Y, double omega, double gamma, double tol,
                                int maxiter, cclr_c128 *result, cclr_solve_info *info) {
  return response_impl(ctx, X, Y, omega, gamma, tol, maxiter, result, info, nullptr);
}

extern "C" int cclr_response_cc(cclr_ctx *ctx, const cclr_eri_packed *eri, const cclr_c128 *X, const cclr_c128 *Y, double omega,
                                double gamma, double tol, int maxiter, cclr_c128 *result, cclr_solve_info *info) {
  if (!eri) {
    cclr_set_error("cclr_response_cc: null pointer", cudaSuccess);
    return CCLR_EINVAL;
  }
  return response_impl(ctx, X, Y, omega, gamma, tol, maxiter, result, info, eri);
}


// The whole CC-CI linear response tensor <<X_r; X_s>>_{z_k}, z_k = omegas[k] + i gamma, for nop one-body operators and nomega
// frequencies in one call: steps 3 and 4 of the paper's workflow with ONE shared trial space for all
// operators and frequencies.  Eq. 16 + Eq. 17 (readings 7, 8) need, per operator, t(z_k) and t(-conj z_k) (shifts +-omega_k at
// +gamma) and t(-z_k), t(conj z_k) (shifts -+omega_k at -gamma); for gamma = 0 the two sets coincide and one solve serves both.
//   g_rs(w) = EOMeta_r . t_s(w) - (lambda . t_r(-w)) (lambda . xi_s) + EOMeta_s . t_r(-w) - (lambda . t_s(w)) (lambda . xi_r)
//   <<X_r;X_s>>_z = 1/2 [ g_rs(z) + conj g_rs(-conj z) ]
extern "C" int cclr_response_ci_tensor(cclr_ctx *ctx, const cclr_c128 *X, int nop, const double *omegas, int nomega, double gamma,
                                       double tol, int maxiter, cclr_c128 *result, cclr_solve_info *info) {
  if (!ctx || !X || !omegas || !result || nop < 1 || nomega < 1 || !(tol > 0.0) || maxiter < 1) {
    cclr_set_error("cclr_response_ci_tensor: null pointer, nop < 1, nomega < 1, tol <= 0 or maxiter < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  typedef std::complex<double> cplx;
  cclr_solve_info total{};
  total.converged = 1;
  try {
    const long n1 = ctx->n1, n2 = ctx->n2, n = n1 + n2;
    const size_t nn = (size_t)(ctx->o + ctx->v) * (size_t)(ctx->o + ctx->v);
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
    if (!ctx->have_lambda || tol < ctx->lambda_tol) {
      cclr_solve_info li{};
      rc = cclr_lambda(ctx, tol, maxiter, lam1, lam2, &li);
      acc(li);
      if (rc != CCLR_OK && rc != CCLR_ENOTCONV) return rc;
      ctx->have_lambda = rc == CCLR_OK;
      ctx->lambda_tol = tol;
    }
    // xi and EOM-eta of every operator: [nop][n1] and [nop][n2] blocks
    DeviceBuf XI, ETA;
    XI.alloc((size_t)nop * n, "cudaMalloc(xi)");
    ETA.alloc((size_t)nop * n, "cudaMalloc(eta)");
    cclr_c128 *xi1 = (cclr_c128 *)XI.p, *xi2 = (cclr_c128 *)(XI.p + (size_t)nop * n1);
    cclr_c128 *et1 = (cclr_c128 *)ETA.p, *et2 = (cclr_c128 *)(ETA.p + (size_t)nop * n1);
    for (int r = 0; r < nop; ++r) {
      if ((rc = cclr_xi(ctx, X + (size_t)r * nn, xi1 + (size_t)r * n1, xi2 + (size_t)r * n2)) != CCLR_OK) return rc;
      if ((rc = cclr_eta(ctx, X + (size_t)r * nn, lam1, lam2, 1, et1 + (size_t)r * n1, et2 + (size_t)r * n2)) != CCLR_OK) return rc;
    }
    // shifts needed: +-w_k at +gamma (set P) and at -gamma (set M); equal shifts (w = 0, repeated frequencies) are solved once
    std::vector<double> sh;
    std::vector<int> idx_pos(nomega), idx_neg(nomega);
    auto shift_index = [&](double w) {
      for (size_t q = 0; q < sh.size(); ++q)
        if (sh[q] == w) return (int)q;
      sh.push_back(w);
      return (int)sh.size() - 1;
    };
    for (int k = 0; k < nomega; ++k) idx_pos[k] = shift_index(omegas[k]);
    for (int k = 0; k < nomega; ++k) idx_neg[k] = shift_index(omegas[k] == 0.0 ? 0.0 : -omegas[k]);
    const int ns = (int)sh.size();
    const bool two_sets = gamma != 0.0;
    DeviceBuf TP, TM;
    TP.alloc((size_t)nop * ns * n, "cudaMalloc(t, +gamma)");
    cclr_c128 *tp1 = (cclr_c128 *)TP.p, *tp2 = (cclr_c128 *)(TP.p + (size_t)nop * ns * n1);
    cclr_solve_info si{};
    rc = cclr_solve(ctx, xi1, xi2, nop, sh.data(), ns, gamma, tol, maxiter, tp1, tp2, &si);
    acc(si);
    if (rc != CCLR_OK && rc != CCLR_ENOTCONV) return rc;
    cclr_c128 *tm1 = tp1, *tm2 = tp2;
    if (two_sets) {
      TM.alloc((size_t)nop * ns * n, "cudaMalloc(t, -gamma)");
      tm1 = (cclr_c128 *)TM.p; tm2 = (cclr_c128 *)(TM.p + (size_t)nop * ns * n1);
      rc = cclr_solve(ctx, xi1, xi2, nop, sh.data(), ns, -gamma, tol, maxiter, tm1, tm2, &si);
      acc(si);
      if (rc != CCLR_OK && rc != CCLR_ENOTCONV) return rc;
    }
    // dots: E?[r][s][j] = EOMeta_r . t_s(shift j), L?[s][j] = lambda . t_s(shift j), Lx[s] = lambda . xi_s
    const int nv = nop * ns;
    std::vector<cclr_c128> EP((size_t)nop * nv), EM, LP(nv), LM, Lx(nop);
    for (int r = 0; r < nop; ++r)
      if ((rc = cclr_property(ctx, et1 + (size_t)r * n1, et2 + (size_t)r * n2, tp1, tp2, nv, EP.data() + (size_t)r * nv)) != CCLR_OK) return rc;
    if ((rc = cclr_property(ctx, lam1, lam2, tp1, tp2, nv, LP.data())) != CCLR_OK) return rc;
    if ((rc = cclr_property(ctx, lam1, lam2, xi1, xi2, nop, Lx.data())) != CCLR_OK) return rc;
    if (two_sets) {
      EM.resize((size_t)nop * nv); LM.resize(nv);
      for (int r = 0; r < nop; ++r)
        if ((rc = cclr_property(ctx, et1 + (size_t)r * n1, et2 + (size_t)r * n2, tm1, tm2, nv, EM.data() + (size_t)r * nv)) != CCLR_OK) return rc;
      if ((rc = cclr_property(ctx, lam1, lam2, tm1, tm2, nv, LM.data())) != CCLR_OK) return rc;
    }
    auto C = [](const cclr_c128 &q) { return cplx(q.re, q.im); };
    const std::vector<cclr_c128> &EMr = two_sets ? EM : EP, &LMr = two_sets ? LM : LP;
    for (int k = 0; k < nomega; ++k)
      for (int r = 0; r < nop; ++r)
        for (int s = 0; s < nop; ++s) {
          // shift indices: +gamma set: z_k -> jz, -conj z_k -> jzc;  -gamma set: -z_k -> jzc, conj z_k -> jz
          const int jz = idx_pos[k], jzc = idx_neg[k];
          const cplx g0 = C(EP[((size_t)r * nop + s) * ns + jz]) - C(LMr[(size_t)r * ns + jzc]) * C(Lx[s]) +
                          C(EMr[((size_t)s * nop + r) * ns + jzc]) - C(LP[(size_t)s * ns + jz]) * C(Lx[r]);
          const cplx g1 = C(EP[((size_t)r * nop + s) * ns + jzc]) - C(LMr[(size_t)r * ns + jz]) * C(Lx[s]) +
                          C(EMr[((size_t)s * nop + r) * ns + jz]) - C(LP[(size_t)s * ns + jzc]) * C(Lx[r]);
          const cplx val = 0.5 * (g0 + std::conj(g1));
          result[((size_t)k * nop + r) * nop + s].re = val.real();
          result[((size_t)k * nop + r) * nop + s].im = val.imag();
        }
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  if (info) *info = total;
  return total.converged ? CCLR_OK : CCLR_ENOTCONV;
}
