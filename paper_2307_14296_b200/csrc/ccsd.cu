// ccsd.cu — cclr_ccsd: the ground-state CCSD amplitudes (paper step 1) on the GPU, built ONLY from the
// response machinery of this library.
//
// The CCSD residual Omega(t) is a polynomial of degree <= 4 in t and the Jacobian of PAPER.md:131 Eq. 14 is its derivative,
// A(t) = dOmega/dt, so along the ray s -> s*t
//
//     Omega(t) = Omega(0) + int_0^1 A(s t) . t ds = Omega(0) + 1/2 [ A(s_1 t) . t + A(s_2 t) . t ],   s_k = 1/2 -+ 1/(2 sqrt 3)
//
// exactly (2-point Gauss-Legendre integrates the cubic s -> A(s t) . t exactly), with Omega(0) = (f[a,i], <ab||ij>).  One residual
// is therefore two cclr_create + cclr_sigma pairs at scaled amplitudes; no separate residual code exists.  The amplitude update is
// the quasi-Newton step t -= Omega / D with DIIS extrapolation (the paper uses CROP; the fixed point is the same).
// The energy uses the same idea: dE/dt . x = eta0(t) . x with eta0 linear in t, so E(t) = eta0(t/2) . t; here it is evaluated
// directly as  sum_ia f[i,a] t1[a,i] + sum_{a<b,i<j} <ij||ab> tau[ab,ij]  (tau of S-Eq. 28).
#include "context.cuh"
#include "small_dense.h"
#include <chrono>
#include <cmath>
#include <complex>

namespace {

typedef small_dense::cplx cplx;

void check(cudaError_t e, const char *where) {
  if (e != cudaSuccess)
    throw PlanError(e == cudaErrorMemoryAllocation ? CCLR_ENOMEM : CCLR_ECUDA, std::string(where) + ": " + cudaGetErrorString(e), e);
}

struct Buf {
  c128 *p = nullptr;
  ~Buf() { if (p) cudaFree(p); }
  void alloc(size_t elems, const char *what) { check(cudaMalloc(&p, (elems ? elems : 1) * sizeof(c128)), what); }
};

const char *const PLAN_OMEGA0 = R"PLAN(
buf W0 (ab)(ij) persist
perm W0[(ab)(ij)] = 1 conj oovv[(ij)(ab)]
buf fovT ai persist
perm fovT[ai] = 1 fov[ia]
)PLAN";

const char *const PLAN_TAU = R"PLAN(
buf tt aibj temp
gemm tt[ai;bj] = 1 t1[ai;1] t1[bj;1] nk
buf tau (ab)(ij) temp
perm tau[(ab)(ij)] = 1 t2[(ab)(ij)] 1 tt[aibj] -1 tt[biaj]
free tt
)PLAN";

}  // namespace

extern "C" int cclr_ccsd(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, cclr_c128 *t1, cclr_c128 *t2,
                         double tol, int maxiter, void *cuda_stream, cclr_ccsd_info *info) {
  if (o < 2 || v < 2 || !fock || !eri || !t1 || !t2 || !(tol > 0.0) || maxiter < 1 || !eri->oooo || !eri->ooov || !eri->oovv ||
      !eri->ovvo || !eri->ovvv || !eri->vvvv) {
    cclr_set_error("cclr_ccsd: null pointer, o < 2, v < 2, tol <= 0 or maxiter < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  const auto wall0 = std::chrono::steady_clock::now();
  cclr_ccsd_info res{};
  int rc = CCLR_ENOTCONV;
  try {
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const long oo = npair(o), vv = npair(v), n1 = (long)o * v, n2 = oo * vv, n = n1 + n2;
    const int ndiis = 8;
    const size_t nf = (size_t)o + v;
    const c128 *F = (const c128 *)fock;
    Buf T, OM, S, TS, HT, HE, fov, om0_1, coef, dpart, dout;
    T.alloc(n, "cudaMalloc(t)"); OM.alloc(n, "cudaMalloc(omega)"); S.alloc(n, "cudaMalloc(sigma)"); TS.alloc(n, "cudaMalloc(scaled t)");
    HT.alloc((size_t)ndiis * n, "cudaMalloc(DIIS t)"); HE.alloc((size_t)ndiis * n, "cudaMalloc(DIIS e)");
    fov.alloc(n1, "cudaMalloc(fov)"); om0_1.alloc(n1, "cudaMalloc(fvo)"); coef.alloc(ndiis + 1, "cudaMalloc(coef)");
    const int npairs_max = ndiis * ndiis;
    dpart.alloc(dots_scratch_elems(npairs_max), "cudaMalloc(dot scratch)"); dout.alloc(npairs_max, "cudaMalloc(dot out)");
    double *D = nullptr;
    check(cudaMalloc(&D, (size_t)n * sizeof(double)), "cudaMalloc(D)");
    struct FreeD { double *p; ~FreeD() { cudaFree(p); } } freeD{D};
    check(denominators(st, F, o, v, D), "denominators");
    // Omega(0): f[a,i] and <ab||ij> = conj <ij||ab>;  f[i,a] transposed for the energy
    check(cudaMemcpy2DAsync(om0_1.p, (size_t)o * sizeof(c128), F + (size_t)o * nf, nf * sizeof(c128), (size_t)o * sizeof(c128), v,
                            cudaMemcpyDeviceToDevice, st), "copy f_vo");
    check(cudaMemcpy2DAsync(fov.p, (size_t)v * sizeof(c128), F + o, nf * sizeof(c128), (size_t)v * sizeof(c128), o,
                            cudaMemcpyDeviceToDevice, st), "copy f_ov");
    Plan P(o, v, st);
    P.bind("oovv", "(ij)(ab)", (c128 *)eri->oovv);
    P.bind("fov", "ia", fov.p);
    P.execute(PLAN_OMEGA0);
    const c128 *W0 = P.buf(P.find("W0")).ptr, *fovT = P.buf(P.find("fovT")).ptr;

    check(cudaMemcpyAsync(T.p, t1, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t1");
    check(cudaMemcpyAsync(T.p + n1, t2, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t2");

    auto host_dots = [&](const c128 *A, long lda, int na, const c128 *B, long ldb, int nb, long len, bool conjA, bool diag) {
      const int np = diag ? na : na * nb;
      std::vector<cplx> out(np);
      check(multi_dot(st, A, lda, na, B, ldb, nb, len, conjA, diag, dpart.p, dout.p), "multi_dot");
      check(cudaMemcpyAsync(out.data(), dout.p, (size_t)np * sizeof(c128), cudaMemcpyDeviceToHost, st), "D2H dots");
      check(cudaStreamSynchronize(st), "sync dots");
      return out;
    };
    auto set_coef = [&](const std::vector<cplx> &h) {
      check(cudaMemcpyAsync(coef.p, h.data(), h.size() * sizeof(c128), cudaMemcpyHostToDevice, st), "H2D coef");
      check(cudaStreamSynchronize(st), "sync coef");
    };
    const double sq[2] = {0.5 - 0.5 / std::sqrt(3.0), 0.5 + 0.5 / std::sqrt(3.0)};
    int nhist = 0;
    for (int it = 0; it < maxiter; ++it) {
      res.iterations = it;
      // ---- Omega(t) = Omega(0) + 1/2 sum_k A(s_k t) . t ----
      check(cudaMemcpyAsync(OM.p, om0_1.p, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy Omega1(0)");
      check(cudaMemcpyAsync(OM.p + n1, W0, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy Omega2(0)");
      for (int k = 0; k < 2; ++k) {
        set_coef({cplx(sq[k], 0.0)});
        check(lincomb(st, TS.p, make_double2(0.0, 0.0), coef.p, T.p, n, 1, n), "scale t");
        cclr_ctx *ctx = nullptr;
        const int e = cclr_create(o, v, fock, eri, (const cclr_c128 *)TS.p, (const cclr_c128 *)(TS.p + n1), 0, cuda_stream, &ctx);
        if (e != CCLR_OK) return e;
        try {
          cclr_sigma_one(ctx, T.p, T.p + n1, make_double2(0.0, 0.0), S.p, S.p + n1, false);
          ++res.sigma_calls;
          set_coef({cplx(0.5, 0.0)});
          check(lincomb(st, OM.p, make_double2(1.0, 0.0), coef.p, S.p, n, 1, n), "accumulate Omega");
          check(cudaStreamSynchronize(st), "sync");
        } catch (...) {
          cclr_destroy(ctx);
          throw;
        }
        cclr_destroy(ctx);
      }
      // ---- convergence on the full-tensor 2-norm: ||Omega1||^2 + 4 ||Omega2 (unique)||^2 ----
      const double d1 = host_dots(OM.p, n, 1, OM.p, n, 1, n1, true, false)[0].real();
      const double d2 = host_dots(OM.p + n1, n, 1, OM.p + n1, n, 1, n2, true, false)[0].real();
      res.residual = std::sqrt(std::max(0.0, d1 + 4.0 * d2));
      if (!std::isfinite(res.residual) || res.residual > 1e6) break;
      if (res.residual <= tol) { res.converged = 1; rc = CCLR_OK; break; }
      if (it == maxiter - 1) { res.iterations = maxiter; break; }
      // ---- quasi-Newton step and DIIS (error vector e = Omega / D) ----
      const int slot = it % ndiis;
      c128 *e_new = HE.p + (size_t)slot * n, *t_new = HT.p + (size_t)slot * n;
      check(precondition(st, e_new, OM.p, D, make_double2(0.0, 0.0), make_double2(1.0, 0.0), n), "Omega / D");   // = -Omega/D
      set_coef({cplx(1.0, 0.0)});
      check(lincomb(st, T.p, make_double2(1.0, 0.0), coef.p, e_new, n, 1, n), "t -= Omega/D");
      check(cudaMemcpyAsync(t_new, T.p, (size_t)n * sizeof(c128), cudaMemcpyDeviceToDevice, st), "store t");
      nhist = std::min(nhist + 1, ndiis);
      if (nhist >= 2) {
        const int m = nhist;
        std::vector<cplx> Bm = host_dots(HE.p, n, m, HE.p, n, m, n, true, false);
        std::vector<cplx> M((size_t)(m + 1) * (m + 1), cplx(0.0)), rhs(m + 1, cplx(0.0)), c(m + 1, cplx(0.0));
        for (int p = 0; p < m; ++p) {
          for (int q = 0; q < m; ++q) M[(size_t)p * (m + 1) + q] = Bm[(size_t)p * m + q];
          M[(size_t)p * (m + 1) + m] = M[(size_t)m * (m + 1) + p] = -1.0;
        }
        rhs[m] = -1.0;
        small_dense::Hessenberg h;
        h.factor(M.data(), m + 1);
        if (h.solve(cplx(0.0), rhs.data(), c.data())) {
          bool finite = true;
          for (int p = 0; p < m; ++p) finite = finite && std::isfinite(c[p].real()) && std::isfinite(c[p].imag());
          if (finite) {
            c.resize(m);
            set_coef(c);
            check(lincomb(st, T.p, make_double2(0.0, 0.0), coef.p, HT.p, n, m, n), "DIIS extrapolation");
          }
        }
      }
    }
    // ---- energy and output ----
    P.bind("t1", "ai", T.p);
    P.bind("t2", "(ab)(ij)", T.p + n1);
    P.execute(PLAN_TAU);
    const c128 *tau = P.buf(P.find("tau")).ptr;
    const cplx e1 = host_dots(fovT, n1, 1, T.p, n1, 1, n1, false, false)[0];
    const cplx e2 = host_dots(W0, n2, 1, tau, n2, 1, n2, true, false)[0];     // conj(W0[(ab)(ij)]) = <ij||ab>
    res.energy_re = (e1 + e2).real();
    res.energy_im = (e1 + e2).imag();
    check(cudaMemcpyAsync(t1, T.p, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t1 out");
    check(cudaMemcpyAsync(t2, T.p + n1, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t2 out");
    check(cudaStreamSynchronize(st), "cclr_ccsd sync");
  } catch (const PlanError &e) {
    return cclr_fail(e);
  } catch (const std::exception &e) {
    cclr_set_error(e.what(), cudaSuccess);
    return CCLR_EINVAL;
  }
  res.seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - wall0).count();
  if (info) *info = res;
  if (rc == CCLR_ENOTCONV) cclr_set_error("cclr_ccsd: maxiter reached (or divergence) before ||Omega|| met tol", cudaSuccess);
  return rc;
}
