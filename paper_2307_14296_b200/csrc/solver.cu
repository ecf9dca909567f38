// solver.cu — cclr_solve: the right response equations (A - z_k) t = -xi_r (Eq. 19, 183-187 Eq. 20-21)
// by the Davidson-type subspace method of PAPER.md:944-967 (steps 1-5; Fig. 1) in the readings of
// DESIGN.md (G = A - z, C = -xi, residual r = (A - z) t + xi, correction r / (z - D)).
//
// What differs from the paper's scheme, and why:
//   * ONE orthonormal trial space {b_j} with sigma_j = A b_j serves every right-hand side and every shift of the
//     call: A does not depend on z, so the reduced matrix G = b^H sigma is shift independent and
//     each (r, k) only needs the tiny system (G - z_k) beta = -b^H xi_r.  A 64-frequency damped sweep costs a few
//     tens of sigma products per right-hand side instead of 64 separate solves.
//   * trial vectors live in packed unique storage (a<b, i<j): the explicit antisymmetrisation step of
//     PAPER.md:217-219 does not exist, and every dot / norm is over unique elements.
//   * the reduced systems for all shifts are solved on the host through one Hessenberg reduction (small_dense.h);
//     only O(L^2) numbers cross PCIe per iteration.
// Device work: sigma (cclr_sigma_one), tall-skinny dots, linear combinations, preconditioner (vecops.cu) and, for
// many simultaneous systems, the residual block R = xi + beta^T [sigma; -z b] as two DMMA GEMMs.
#include "subspace.cuh"
#include <chrono>

namespace {

using subspace::check;
using subspace::cplx;
using subspace::DeviceBuf;

struct Solver : subspace::Space {
  int rcap = 0;
  DeviceBuf XI, R, tmp;
  std::vector<cplx> c;        // maxdim x nrhs: c[j][r] = b_j^H xi_r
  int nrhs = 0;

  c128 *xi(int r) { return XI.p + (size_t)r * n; }
  c128 *r(int i) { return R.p + (size_t)i * n; }

  // sigma_j = A b_j for j in [L0, L) and the new rows / columns of G and c
  void extend(int L0) {
    extend_sigma(L0);
    const int nn = L - L0;
    if (nn == 0) return;
    std::vector<cplx> cx = dots(b(L0), nn, XI.p, nrhs);          // c[L0:L, :]
    for (int i = 0; i < nn; ++i)
      for (int rr = 0; rr < nrhs; ++rr) c[(size_t)(L0 + i) * nrhs + rr] = cx[(size_t)i * nrhs + rr];
  }
};

}  // namespace

static int solve_impl(cclr_ctx *ctx, const cclr_c128 *xi1, const cclr_c128 *xi2, int nrhs, const double *omegas,
                      int nomega, double gamma, double tol, int maxiter, cclr_c128 *t1_out, cclr_c128 *t2_out,
                      cclr_solve_info *info, bool left) {
  if (!ctx || !xi1 || !xi2 || !omegas || !t1_out || !t2_out || nrhs < 1 || nomega < 1 || !(tol > 0.0) || maxiter < 1) {
    cclr_set_error("cclr_solve: null pointer, nrhs < 1, nomega < 1, tol <= 0 or maxiter < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  const auto wall0 = std::chrono::steady_clock::now();
  cclr_solve_info res{};
  res.converged = 1;
  int rc = CCLR_OK;
  try {
    const long n1 = ctx->n1, n2 = ctx->n2, n = n1 + n2;
    cudaStream_t st = ctx->st;
    std::vector<cplx> z(nomega);
    for (int k = 0; k < nomega; ++k) z[k] = cplx(omegas[k], gamma);

    // ---- size the subspace from the free device memory; right-hand sides are processed in blocks if needed ----
    size_t free_b = 0, total_b = 0;
    check(cudaMemGetInfo(&free_b, &total_b), "cudaMemGetInfo");
    const double vec_b = (double)n * sizeof(c128);
    const double budget = 0.85 * (double)free_b;
    int rhs_block = nrhs;
    int maxdim = 0, rcap = 0;
    for (;; rhs_block = (rhs_block + 1) / 2) {
      const int nsys_b = rhs_block * nomega;
      rcap = std::min(nsys_b, 256);
      double left = budget - (double)(rhs_block + rcap + 1) * vec_b;
      while (left < 8 * vec_b && rcap > 1) {            // shrink the residual block before the subspace
        left += (rcap - rcap / 2) * vec_b;
        rcap /= 2;
      }
      maxdim = (int)std::min(3000.0, std::floor(left / (2.0 * vec_b)));
      const int want = std::min(3000, 24 * rhs_block + 4 * std::min(nomega, 16) * rhs_block);
      if (maxdim >= want || rhs_block == 1) {
        maxdim = std::min(maxdim, std::max(want, 8));
        break;
      }
    }
    if (ctx->max_subspace > 0) maxdim = std::min(maxdim, std::max(ctx->max_subspace, 8));
    if (maxdim < 8) throw PlanError(CCLR_ENOMEM, "cclr_solve: not enough free device memory for a trial space of 8 vectors");

    for (int r0 = 0; r0 < nrhs; r0 += rhs_block) {
      const int nr = std::min(rhs_block, nrhs - r0);
      const int nsys = nr * nomega;
      Solver S;
      S.ctx = ctx; S.st = st; S.n = n; S.n1 = n1; S.n2 = n2;
      S.maxdim = maxdim; S.rcap = rcap; S.nrhs = nr; S.left = left;
      S.Bm.alloc((size_t)maxdim * n, "cudaMalloc(trial space)");
      S.Sm.alloc((size_t)maxdim * n, "cudaMalloc(sigma space)");
      S.XI.alloc((size_t)nr * n, "cudaMalloc(xi)");
      S.R.alloc((size_t)rcap * n, "cudaMalloc(residual block)");
      S.tmp.alloc((size_t)n, "cudaMalloc(tmp)");
      S.coef.alloc((size_t)std::max(maxdim, 1) * std::max(rcap, 1) * 2, "cudaMalloc(coefficients)");
      S.G.assign((size_t)maxdim * maxdim, cplx(0.0));
      S.c.assign((size_t)maxdim * nr, cplx(0.0));

      for (int r = 0; r < nr; ++r) {
        check(cudaMemcpyAsync(S.xi(r), (const c128 *)xi1 + (size_t)(r0 + r) * n1, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy xi1");
        check(cudaMemcpyAsync(S.xi(r) + n1, (const c128 *)xi2 + (size_t)(r0 + r) * n2, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy xi2");
      }
      std::vector<double> norm_xi(nr);
      {
        std::vector<cplx> d = S.dots(S.XI.p, nr, S.XI.p, nr, true);
        for (int r = 0; r < nr; ++r) norm_xi[r] = std::sqrt(std::max(0.0, d[r].real()));
      }

      // ---- step 1: start vectors = preconditioned right-hand sides at the first and last shift ----
      std::vector<int> done(nsys, 0);
      std::vector<double> relres(nsys, 0.0);
      auto out1 = [&](int r, int k) { return (c128 *)t1_out + ((size_t)(r0 + r) * nomega + k) * n1; };
      auto out2 = [&](int r, int k) { return (c128 *)t2_out + ((size_t)(r0 + r) * nomega + k) * n2; };
      for (int r = 0; r < nr; ++r) {
        if (norm_xi[r] == 0.0) {
          for (int k = 0; k < nomega; ++k) {
            done[r * nomega + k] = 1;
            check(cudaMemsetAsync(out1(r, k), 0, (size_t)n1 * sizeof(c128), st), "memset");
            check(cudaMemsetAsync(out2(r, k), 0, (size_t)n2 * sizeof(c128), st), "memset");
          }
          continue;
        }
        std::vector<int> ks{0};
        if (nomega > 1) ks.push_back(nomega - 1);
        for (int k : ks) {
          check(precondition(st, S.tmp.p, S.xi(r), ctx->D, make_double2(z[k].real(), z[k].imag()), make_double2(-1.0, 0.0), n), "precondition");
          S.append(S.tmp.p);
        }
      }
      int L0 = 0;
      int iter = 0;
      bool all_done = std::all_of(done.begin(), done.end(), [](int d) { return d != 0; });
      small_dense::Hessenberg hess;
      std::vector<cplx> beta((size_t)nsys * maxdim, cplx(0.0));

      while (!all_done) {
        ++iter;
        // ---- step 2: sigma vectors of the new trial vectors, reduced matrix (Eq. 29) ----
        S.extend(L0);
        L0 = S.L;
        const int L = S.L;
        // ---- step 3: reduced systems (G - z_k) beta = -c_r for every unconverged (r, k) ----
        std::vector<cplx> Gc((size_t)L * L);
        for (int i = 0; i < L; ++i)
          for (int j = 0; j < L; ++j) Gc[(size_t)i * L + j] = S.G[(size_t)i * maxdim + j];
        hess.factor(Gc.data(), L);
        std::vector<int> active;
        for (int sidx = 0; sidx < nsys; ++sidx)
          if (!done[sidx]) active.push_back(sidx);
        std::vector<cplx> rhs(L);
        for (int sidx : active) {
          const int r = sidx / nomega, k = sidx % nomega;
          for (int j = 0; j < L; ++j) rhs[j] = -S.c[(size_t)j * nr + r];
          if (!hess.solve(z[k], rhs.data(), &beta[(size_t)sidx * maxdim]))
            for (int j = 0; j < L; ++j) beta[(size_t)sidx * maxdim + j] = 0.0;
        }
        // ---- step 4: residuals r = xi + sum_j beta_j (sigma_j - z b_j), in blocks of rcap systems ----
        const bool single_block = (int)active.size() <= rcap;
        for (size_t a0 = 0; a0 < active.size(); a0 += rcap) {
          const int nb = (int)std::min<size_t>(rcap, active.size() - a0);
          for (int i = 0; i < nb; ++i) {
            const int r = active[a0 + i] / nomega;
            check(cudaMemcpyAsync(S.r(i), S.xi(r), (size_t)n * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy xi");
          }
          if (nb >= 16) {
            std::vector<cplx> co((size_t)2 * nb * L);
            for (int i = 0; i < nb; ++i) {
              const int sidx = active[a0 + i];
              const cplx zz = z[sidx % nomega];
              for (int j = 0; j < L; ++j) {
                co[(size_t)i * L + j] = beta[(size_t)sidx * maxdim + j];
                co[(size_t)(nb + i) * L + j] = -zz * beta[(size_t)sidx * maxdim + j];
              }
            }
            S.upload(co, S.coef.p);
            const c128 one = make_double2(1.0, 0.0);
            check(zgemm(st, nb, (int)n, L, one, S.coef.p, L, false, S.Sm.p, n, true, false, one, S.R.p, n), "zgemm(residual sigma)");
            check(zgemm(st, nb, (int)n, L, one, S.coef.p + (size_t)nb * L, L, false, S.Bm.p, n, true, false, one, S.R.p, n), "zgemm(residual b)");
          } else {
            for (int i = 0; i < nb; ++i) {
              const int sidx = active[a0 + i];
              const cplx zz = z[sidx % nomega];
              std::vector<cplx> co(L);
              for (int j = 0; j < L; ++j) co[j] = beta[(size_t)sidx * maxdim + j];
              S.add_combination(S.r(i), make_double2(1.0, 0.0), co, S.Sm.p, L, n, n);
              for (int j = 0; j < L; ++j) co[j] = -zz * beta[(size_t)sidx * maxdim + j];
              S.add_combination(S.r(i), make_double2(1.0, 0.0), co, S.Bm.p, L, n, n);
            }
          }
          std::vector<cplx> nr2 = S.dots(S.R.p, nb, S.R.p, nb, true);
          for (int i = 0; i < nb; ++i) {
            const int sidx = active[a0 + i];
            relres[sidx] = std::sqrt(std::max(0.0, nr2[i].real())) / norm_xi[sidx / nomega];
          }
        }
        // ---- convergence and step 5: solutions t = sum_j beta_j b_j of the converged systems ----
        const bool last = iter >= maxiter;
        for (int sidx : active) {
          if (relres[sidx] <= tol || last) {
            const int r = sidx / nomega, k = sidx % nomega;
            std::vector<cplx> co(L);
            for (int j = 0; j < L; ++j) co[j] = beta[(size_t)sidx * maxdim + j];
            S.upload(co, S.coef.p);
            check(lincomb(st, out1(r, k), make_double2(0.0, 0.0), S.coef.p, S.Bm.p, n, L, n1), "lincomb(t1)");
            check(lincomb(st, out2(r, k), make_double2(0.0, 0.0), S.coef.p, S.Bm.p + n1, n, L, n2), "lincomb(t2)");
            check(cudaStreamSynchronize(st), "sync");
            if (relres[sidx] <= tol) done[sidx] = 1;
          }
        }
        all_done = std::all_of(done.begin(), done.end(), [](int d) { return d != 0; });
        if (all_done || last) break;

        // ---- new trial vectors: the worst systems of every right-hand side, preconditioned ----
        const int per_rhs = nomega >= 16 ? 4 : std::min(nomega, 2);
        std::vector<int> picks;
        for (int r = 0; r < nr; ++r) {
          std::vector<int> cand;
          for (int k = 0; k < nomega; ++k)
            if (!done[r * nomega + k]) cand.push_back(r * nomega + k);
          std::sort(cand.begin(), cand.end(), [&](int a, int b_) { return relres[a] > relres[b_]; });
          // spread the picks over the frequency range: worst first, then the worst at least nomega/8 away
          std::vector<int> chosen;
          for (int sidx : cand) {
            if ((int)chosen.size() >= per_rhs) break;
            bool far = true;
            for (int c0 : chosen)
              if (std::abs(c0 % nomega - sidx % nomega) < std::max(1, nomega / 8)) far = false;
            if (far) chosen.push_back(sidx);
          }
          picks.insert(picks.end(), chosen.begin(), chosen.end());
        }
        // collapse the trial space if the new vectors do not fit: keep the current solutions of the unconverged systems
        int Lc = L;                       // dimension the betas refer to
        bool have_residuals = single_block;
        if (S.L + (int)picks.size() > maxdim) {
          std::vector<int> keep = picks;
          for (int sidx : active)
            if (!done[sidx] && std::find(keep.begin(), keep.end(), sidx) == keep.end()) keep.push_back(sidx);
          const size_t m_max = (size_t)std::max(1, std::min(rcap, maxdim / 2));
          if (keep.size() > m_max) keep.resize(m_max);
          if (picks.size() > keep.size()) picks.resize(keep.size());
          // orthonormalise the coefficient vectors beta_s in C^L (b is orthonormal, so the vectors B C are orthonormal too)
          std::vector<std::vector<cplx>> Cc;
          for (int sidx : keep) {
            std::vector<cplx> vv(beta.begin() + (size_t)sidx * maxdim, beta.begin() + (size_t)sidx * maxdim + L);
            for (int pass = 0; pass < 2; ++pass)
              for (auto &u : Cc) {
                cplx d = 0.0;
                for (int j = 0; j < L; ++j) d += std::conj(u[j]) * vv[j];
                for (int j = 0; j < L; ++j) vv[j] -= d * u[j];
              }
            double nv = 0.0;
            for (int j = 0; j < L; ++j) nv += std::norm(vv[j]);
            nv = std::sqrt(nv);
            if (nv < 1e-10) continue;
            for (int j = 0; j < L; ++j) vv[j] /= nv;
            Cc.push_back(vv);
          }
          const int m = (int)Cc.size();
          // b' = B C and sigma' = S C, staged in the residual block (m <= rcap), then copied to the front rows
          for (int pass = 0; pass < 2; ++pass) {
            c128 *src = pass == 0 ? S.Bm.p : S.Sm.p;
            for (int i = 0; i < m; ++i) {
              S.upload(Cc[i], S.coef.p);
              check(lincomb(st, S.r(i), make_double2(0.0, 0.0), S.coef.p, src, n, L, n), "lincomb(collapse)");
            }
            check(cudaMemcpyAsync(src, S.R.p, (size_t)m * n * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy collapsed");
          }
          // G' = C^H G C, c' = C^H c, beta' = C^H beta
          std::vector<cplx> GC((size_t)L * m, cplx(0.0));
          for (int i = 0; i < L; ++i)
            for (int bq = 0; bq < m; ++bq) {
              cplx acc = 0.0;
              for (int j = 0; j < L; ++j) acc += S.G[(size_t)i * maxdim + j] * Cc[bq][j];
              GC[(size_t)i * m + bq] = acc;
            }
          std::vector<cplx> Gn((size_t)m * m, cplx(0.0)), cn((size_t)m * nr, cplx(0.0));
          for (int a = 0; a < m; ++a) {
            for (int bq = 0; bq < m; ++bq) {
              cplx acc = 0.0;
              for (int i = 0; i < L; ++i) acc += std::conj(Cc[a][i]) * GC[(size_t)i * m + bq];
              Gn[(size_t)a * m + bq] = acc;
            }
            for (int rr = 0; rr < nr; ++rr) {
              cplx acc = 0.0;
              for (int i = 0; i < L; ++i) acc += std::conj(Cc[a][i]) * S.c[(size_t)i * nr + rr];
              cn[(size_t)a * nr + rr] = acc;
            }
          }
          for (int sidx : active) {
            std::vector<cplx> g(m, cplx(0.0));
            for (int a = 0; a < m; ++a)
              for (int j = 0; j < L; ++j) g[a] += std::conj(Cc[a][j]) * beta[(size_t)sidx * maxdim + j];
            for (int j = 0; j < maxdim; ++j) beta[(size_t)sidx * maxdim + j] = j < m ? g[j] : cplx(0.0);
          }
          std::fill(S.G.begin(), S.G.end(), cplx(0.0));
          std::fill(S.c.begin(), S.c.end(), cplx(0.0));
          for (int a = 0; a < m; ++a) {
            for (int bq = 0; bq < m; ++bq) S.G[(size_t)a * maxdim + bq] = Gn[(size_t)a * m + bq];
            for (int rr = 0; rr < nr; ++rr) S.c[(size_t)a * nr + rr] = cn[(size_t)a * nr + rr];
          }
          S.L = m;
          L0 = m;
          Lc = m;
          have_residuals = false;          // the residual block was used as scratch
        }
        int added = 0;
        for (int sidx : picks) {
          if (S.L >= maxdim) break;
          const int r = sidx / nomega, k = sidx % nomega;
          c128 *rv;
          if (have_residuals) {
            rv = S.r((int)(std::find(active.begin(), active.end(), sidx) - active.begin()));
          } else {
            // r = xi + sum_j beta_j (sigma_j - z b_j) in the current basis
            rv = S.tmp.p;
            check(cudaMemcpyAsync(rv, S.xi(r), (size_t)n * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy xi");
            std::vector<cplx> co(Lc);
            for (int j = 0; j < Lc; ++j) co[j] = beta[(size_t)sidx * maxdim + j];
            S.add_combination(rv, make_double2(1.0, 0.0), co, S.Sm.p, Lc, n, n);
            for (int j = 0; j < Lc; ++j) co[j] = -z[k] * beta[(size_t)sidx * maxdim + j];
            S.add_combination(rv, make_double2(1.0, 0.0), co, S.Bm.p, Lc, n, n);
          }
          check(precondition(st, rv, rv, ctx->D, make_double2(z[k].real(), z[k].imag()), make_double2(1.0, 0.0), n), "precondition");
          if (S.append(rv)) ++added;
        }
        if (added == 0 && S.L == L0) {
          // no new direction could be added (numerically dependent corrections): stop with what we have
          rc = CCLR_ENOTCONV;
          for (int sidx : active)
            if (!done[sidx]) {
              const int r = sidx / nomega, k = sidx % nomega;
              std::vector<cplx> co(Lc);
              for (int j = 0; j < Lc; ++j) co[j] = beta[(size_t)sidx * maxdim + j];
              S.upload(co, S.coef.p);
              check(lincomb(st, out1(r, k), make_double2(0.0, 0.0), S.coef.p, S.Bm.p, n, Lc, n1), "lincomb(t1)");
              check(lincomb(st, out2(r, k), make_double2(0.0, 0.0), S.coef.p, S.Bm.p + n1, n, Lc, n2), "lincomb(t2)");
            }
          break;
        }
      }
      check(cudaStreamSynchronize(st), "cclr_solve sync");
      res.iterations += iter;
      res.sigma_calls += S.sigma_calls;
      res.subspace = std::max(res.subspace, S.L);
      for (int sidx = 0; sidx < nsys; ++sidx) {
        if (!done[sidx]) { res.converged = 0; rc = CCLR_ENOTCONV; }
        res.max_residual = std::max(res.max_residual, relres[sidx]);
      }
    }
  } catch (const PlanError &e) {
    return cclr_fail(e);
  } catch (const std::exception &e) {
    cclr_set_error(e.what(), cudaSuccess);
    return CCLR_EINVAL;
  }
  res.seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - wall0).count();
  if (info) *info = res;
  if (rc == CCLR_ENOTCONV) cclr_set_error("cclr_solve: maxiter reached before every system met tol", cudaSuccess);
  return rc;
}

extern "C" int cclr_solve(cclr_ctx *ctx, const cclr_c128 *xi1, const cclr_c128 *xi2, int nrhs, const double *omegas,
                          int nomega, double gamma, double tol, int maxiter, cclr_c128 *t1_out, cclr_c128 *t2_out,
                          cclr_solve_info *info) {
  return solve_impl(ctx, xi1, xi2, nrhs, omegas, nomega, gamma, tol, maxiter, t1_out, t2_out, info, false);
}

// l (A - z) = -eta: the same subspace method on the left transform (the reduced matrix is b^H A^T b)
extern "C" int cclr_solve_left(cclr_ctx *ctx, const cclr_c128 *eta1, const cclr_c128 *eta2, int nrhs, const double *omegas,
                               int nomega, double gamma, double tol, int maxiter, cclr_c128 *l1_out, cclr_c128 *l2_out,
                               cclr_solve_info *info) {
  return solve_impl(ctx, eta1, eta2, nrhs, omegas, nomega, gamma, tol, maxiter, l1_out, l2_out, info, true);
}

// lambda A = -eta0, eta0 = (F_me[i,a], <ij||ab>)  (Eq. 13)
extern "C" int cclr_lambda(cclr_ctx *ctx, double tol, int maxiter, cclr_c128 *lam1, cclr_c128 *lam2, cclr_solve_info *info) {
  if (!ctx || !lam1 || !lam2) return CCLR_EINVAL;
  const int i1 = ctx->plan->find("FmeT"), i2 = ctx->plan->find("eta02");
  if (i1 < 0 || i2 < 0 || !ctx->plan->buf(i1).ptr || !ctx->plan->buf(i2).ptr) return CCLR_EINVAL;
  const double zero = 0.0;
  const int rc = solve_impl(ctx, (const cclr_c128 *)ctx->plan->buf(i1).ptr, (const cclr_c128 *)ctx->plan->buf(i2).ptr, 1, &zero, 1,
                            0.0, tol, maxiter, lam1, lam2, info, true);
  // keep a copy in the context: cclr_response_ci / _cc reuse multipliers solved to a tolerance at least as tight
  if (rc == CCLR_OK && (c128 *)lam1 != ctx->lambda) {
    const size_t n1 = (size_t)ctx->n1, n2 = (size_t)ctx->n2;
    if (!ctx->lambda) {
      if (cudaMalloc(&ctx->lambda, (n1 + n2) * sizeof(c128)) != cudaSuccess) { cudaGetLastError(); ctx->lambda = nullptr; return rc; }
      ctx->extra_bytes += (n1 + n2) * sizeof(c128);
    }
    cudaMemcpyAsync(ctx->lambda, lam1, n1 * sizeof(c128), cudaMemcpyDeviceToDevice, ctx->st);
    cudaMemcpyAsync(ctx->lambda + n1, lam2, n2 * sizeof(c128), cudaMemcpyDeviceToDevice, ctx->st);
    cudaStreamSynchronize(ctx->st);
    ctx->have_lambda = true;
    ctx->lambda_tol = tol;
  }
  return rc;
}

// Host-only entry point used by the CPU tests of the reduced-space algebra: beta_k = (G - z_k)^{-1} rhs for nz shifts.
extern "C" int cclr_host_shifted_solve(int L, const cclr_c128 *G, const cclr_c128 *rhs, int nz, const cclr_c128 *z,
                                       cclr_c128 *beta) {
  if (L < 1 || !G || !rhs || nz < 1 || !z || !beta) return CCLR_EINVAL;
  small_dense::Hessenberg h;
  h.factor(reinterpret_cast<const cplx *>(G), L);
  for (int k = 0; k < nz; ++k)
    if (!h.solve(cplx(z[k].re, z[k].im), reinterpret_cast<const cplx *>(rhs), reinterpret_cast<cplx *>(beta) + (size_t)k * L))
      return CCLR_EINVAL;
  return CCLR_OK;
}
