// ccsd.cu — cclr_ccsd: the ground-state CCSD amplitudes (paper step 1) on the GPU.
//
// Residual, two independent routes (cclr_ccsd_residual exposes both; cclr_ccsd iterates on the first):
//   mode 0  the direct residual plan CCLR_PLAN_OMEGA (plans.inc): the textbook spin-orbital CCSD equations as ~60 GEMM / layout
//           statements on the library's kernels, <ab||ef> only read (the vvvv term is applied factorised); about 4.3
//           ladder-equivalents per evaluation;
//   mode 1  the quadrature of the Jacobian: Omega is a quartic polynomial in t and A(t) = dOmega/dt, so
//               Omega(t) = Omega(0) + int_0^1 A(s t) . t ds = Omega(0) + 1/2 [ A(s_1 t) . t + A(s_2 t) . t ],  s = 1/2 -+ 1/(2 sqrt 3)
//           exactly (2-point Gauss-Legendre integrates the cubic s -> A(s t) . t), with Omega(0) = (f[a,i], <ab||ij>): two
//           cclr_create + cclr_sigma pairs, no residual code of its own (about 25 ladder-equivalents) -- the cross-check.
// Amplitude update: quasi-Newton step t -= Omega / D with DIIS (the paper uses CROP; the fixed point is the same).
// Energy: sum_ia f[i,a] t1[a,i] + sum_{a<b,i<j} <ij||ab> tau[ab,ij]  (tau of S-Eq. 28).
#include "context.cuh"
#include "small_dense.h"
#include "plans.inc"
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

// Everything a residual evaluation needs: the plan object with the integral classes and Fock blocks bound, Omega(0), scratch.
struct Engine {
  int o, v;
  long n1, n2, n;
  cudaStream_t st;
  void *stream_arg;
  const cclr_c128 *fock;
  const cclr_eri_packed *eri;
  Plan P;
  ZgemmWorkspace ws;
  OzWorkspace oz;      // integer-slice product (zgemm_oz.cu) for the contractions of the residual that dominate an iteration
  Buf fblocks, S, TS, coef;
  const c128 *W0 = nullptr, *fovT = nullptr, *fvo = nullptr;
  int t1_id = -1, t2_id = -1;
  int sigma_calls = 0;

  Engine(int o_, int v_, const cclr_c128 *fock_, const cclr_eri_packed *eri_, void *stream)
      : o(o_), v(v_), n1((long)o_ * v_), n2(npair(o_) * npair(v_)), n(n1 + n2), st((cudaStream_t)stream), stream_arg(stream),
        fock(fock_), eri(eri_), P(o_, v_, (cudaStream_t)stream) {
    const size_t no = (size_t)o, nv = (size_t)v, nf = no + nv;
    const c128 *F = (const c128 *)fock;
    fblocks.alloc(no * no + 2 * no * nv + nv * nv, "cudaMalloc(fock blocks)");
    coef.alloc(1, "cudaMalloc(coef)");
    struct { const char *name, *spec; size_t off, r0, c0, rows, cols; } blocks[4] = {
        {"foo", "mi", 0, 0, 0, no, no}, {"fov", "me", no * no, 0, no, no, nv},
        {"fvo", "ai", no * no + no * nv, no, 0, nv, no}, {"fvv", "ae", no * no + 2 * no * nv, no, no, nv, nv}};
    for (auto &b : blocks) {
      check(cudaMemcpy2DAsync(fblocks.p + b.off, b.cols * sizeof(c128), F + b.r0 * nf + b.c0, nf * sizeof(c128),
                              b.cols * sizeof(c128), b.rows, cudaMemcpyDeviceToDevice, st), "copy fock block");
      P.bind(b.name, b.spec, fblocks.p + b.off);
    }
    fvo = fblocks.p + no * no + no * nv;
    P.bind("oooo", "(mn)(ij)", (c128 *)eri->oooo);
    P.bind("ooov", "(mn)ie", (c128 *)eri->ooov);
    P.bind("oovv", "(mn)(ef)", (c128 *)eri->oovv);
    P.bind("ovvo", "mbej", (c128 *)eri->ovvo);
    P.bind("ovvv", "mb(ef)", (c128 *)eri->ovvv);
    P.bind("vvvv", "(ab)(ef)", (c128 *)eri->vvvv);
    P.bind("t1", "ai", nullptr);
    P.bind("t2", "(ab)(ij)", nullptr);
    t1_id = P.find("t1");
    t2_id = P.find("t2");
    P.execute(PLAN_OMEGA0);
    // split-K workspace of the GEMM engine: the one-index intermediates of the residual are M, N <= v contractions over K = v oo
    // ... o vv (1 - 25 output tiles); without the K split each of them runs on a handful of SMs (130 ms each at config 4)
    ws.elems = (size_t)8 << 20;
    if (cudaMalloc(&ws.buf, ws.elems * sizeof(c128)) != cudaSuccess) { cudaGetLastError(); ws.buf = nullptr; ws.elems = 0; }
    P.set_workspace(&ws);
    W0 = P.buf(P.find("W0")).ptr;
    fovT = P.buf(P.find("fovT")).ptr;
  }

  ~Engine() {
    zgemm_oz_release(&oz);
    if (ws.buf) cudaFree(ws.buf);
  }

  // The iteration of cclr_ccsd evaluates the residual ~100 times on the same integrals: the two contractions with a constant big
  // A operand -- <ab||ef> tau (the pp ladder) and <ma||ef> tau -- get registered integer slices, the three ring-shaped ones slice
  // their operands per call (zgemm.cu dispatch).  7 slices (48 bits below the row maxima, ~1e-13 norm-wise) so that the fixed point
  // of the iteration is the fixed point of the FP64 residual to well below the 1e-10 convergence threshold.  Skipped when the
  // shapes are not eligible or the slices (7/8 of the operands) do not fit comfortably.
  void enable_integer_slices() {
    const long vv = npair(v), oo = npair(o), ov = (long)o * v;
    if (!zgemm_oz_eligible((int)vv, (int)oo, (int)vv)) return;
    const size_t need = (size_t)14 * vv * vv + (size_t)14 * ov * vv;
    size_t free_b = 0, total_b = 0;
    if (cudaMemGetInfo(&free_b, &total_b) != cudaSuccess || free_b < 2 * need) return;
    int s_need = 0;      // one slice more than the range inside the rows asks for (zgemm_oz_suggest_slices: 6 for this task's integrals)
    check(zgemm_oz_suggest_slices(st, (const c128 *)eri->vvvv, vv, vv, vv, &s_need, nullptr), "row statistics of <ab||ef>");
    if (s_need == 0 || s_need + 1 > 8) return;
    oz.slices = s_need + 1;
    check(zgemm_oz_register(st, &oz, (const c128 *)eri->vvvv, vv, vv, vv), "integer slices of <ab||ef>");
    if (zgemm_oz_eligible((int)ov, (int)oo, (int)vv))
      check(zgemm_oz_register(st, &oz, (const c128 *)eri->ovvv, vv, ov, vv), "integer slices of <ma||ef>");
    ws.oz = &oz;
  }

  // mode 0: OM = Omega(T) by the direct residual plan
  void direct(const c128 *T, c128 *OM) {
    P.rebind(t1_id, const_cast<c128 *>(T));
    P.rebind(t2_id, const_cast<c128 *>(T) + n1);
    P.execute(CCLR_PLAN_OMEGA);
    check(cudaMemcpyAsync(OM, P.buf(P.find("om1")).ptr, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy Omega1");
    check(cudaMemcpyAsync(OM + n1, P.buf(P.find("om2")).ptr, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy Omega2");
    check(cudaStreamSynchronize(st), "sync");
    P.free_class(BUF_TEMP);
  }

  // mode 1: OM = Omega(0) + 1/2 sum_k A(s_k T) . T; returns a CCLR_* code
  int quadrature(const c128 *T, c128 *OM) {
    if (!S.p) { S.alloc(n, "cudaMalloc(sigma)"); TS.alloc(n, "cudaMalloc(scaled t)"); }
    const double sq[2] = {0.5 - 0.5 / std::sqrt(3.0), 0.5 + 0.5 / std::sqrt(3.0)};
    check(cudaMemcpyAsync(OM, fvo, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy Omega1(0)");
    check(cudaMemcpyAsync(OM + n1, W0, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy Omega2(0)");
    auto set_coef = [&](cplx c) {
      check(cudaMemcpyAsync(coef.p, &c, sizeof(c128), cudaMemcpyHostToDevice, st), "H2D coef");
      check(cudaStreamSynchronize(st), "sync coef");
    };
    for (int k = 0; k < 2; ++k) {
      set_coef(cplx(sq[k], 0.0));
      check(lincomb(st, TS.p, make_double2(0.0, 0.0), coef.p, T, n, 1, n), "scale t");
      cclr_ctx *ctx = nullptr;
      const int e = cclr_create(o, v, fock, eri, (const cclr_c128 *)TS.p, (const cclr_c128 *)(TS.p + n1), 0, stream_arg, &ctx);
      if (e != CCLR_OK) return e;
      try {
        cclr_sigma_one(ctx, T, T + n1, make_double2(0.0, 0.0), S.p, S.p + n1, false);
        ++sigma_calls;
        set_coef(cplx(0.5, 0.0));
        check(lincomb(st, OM, make_double2(1.0, 0.0), coef.p, S.p, n, 1, n), "accumulate Omega");
        check(cudaStreamSynchronize(st), "sync");
      } catch (...) {
        cclr_destroy(ctx);
        throw;
      }
      cclr_destroy(ctx);
    }
    return CCLR_OK;
  }
};

bool valid_inputs(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, const void *t1, const void *t2) {
  return o >= 2 && v >= 2 && fock && eri && t1 && t2 && eri->oooo && eri->ooov && eri->oovv && eri->ovvo && eri->ovvv && eri->vvvv;
}

}  // namespace

extern "C" int cclr_ccsd_residual(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, const cclr_c128 *t1,
                                  const cclr_c128 *t2, int mode, void *cuda_stream, cclr_c128 *om1, cclr_c128 *om2) {
  if (!valid_inputs(o, v, fock, eri, t1, t2) || !om1 || !om2 || mode < 0 || mode > 1) {
    cclr_set_error("cclr_ccsd_residual: null pointer, o < 2, v < 2 or unknown mode", cudaSuccess);
    return CCLR_EINVAL;
  }
  try {
    Engine E(o, v, fock, eri, cuda_stream);
    Buf T, OM;
    T.alloc(E.n, "cudaMalloc(t)");
    OM.alloc(E.n, "cudaMalloc(omega)");
    check(cudaMemcpyAsync(T.p, t1, (size_t)E.n1 * sizeof(c128), cudaMemcpyDeviceToDevice, E.st), "copy t1");
    check(cudaMemcpyAsync(T.p + E.n1, t2, (size_t)E.n2 * sizeof(c128), cudaMemcpyDeviceToDevice, E.st), "copy t2");
    if (mode == 0) {
      E.direct(T.p, OM.p);
    } else {
      const int rc = E.quadrature(T.p, OM.p);
      if (rc != CCLR_OK) return rc;
    }
    check(cudaMemcpyAsync(om1, OM.p, (size_t)E.n1 * sizeof(c128), cudaMemcpyDeviceToDevice, E.st), "copy Omega1 out");
    check(cudaMemcpyAsync(om2, OM.p + E.n1, (size_t)E.n2 * sizeof(c128), cudaMemcpyDeviceToDevice, E.st), "copy Omega2 out");
    check(cudaStreamSynchronize(E.st), "cclr_ccsd_residual sync");
  } catch (const PlanError &e) {
    return cclr_fail(e);
  } catch (const std::exception &e) {
    cclr_set_error(e.what(), cudaSuccess);
    return CCLR_EINVAL;
  }
  return CCLR_OK;
}

extern "C" int cclr_ccsd(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, cclr_c128 *t1, cclr_c128 *t2,
                         double tol, int maxiter, void *cuda_stream, cclr_ccsd_info *info) {
  if (!valid_inputs(o, v, fock, eri, t1, t2) || !(tol > 0.0) || maxiter < 1) {
    cclr_set_error("cclr_ccsd: null pointer, o < 2, v < 2, tol <= 0 or maxiter < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  const auto wall0 = std::chrono::steady_clock::now();
  cclr_ccsd_info res{};
  int rc = CCLR_ENOTCONV;
  try {
    Engine E(o, v, fock, eri, cuda_stream);
    cudaStream_t st = E.st;
    const long n1 = E.n1, n2 = E.n2, n = E.n;
    const int ndiis = 8;
    Buf T, OM, HT, HE, coef, dpart, dout;
    T.alloc(n, "cudaMalloc(t)"); OM.alloc(n, "cudaMalloc(omega)");
    HT.alloc((size_t)ndiis * n, "cudaMalloc(DIIS t)"); HE.alloc((size_t)ndiis * n, "cudaMalloc(DIIS e)");
    coef.alloc(ndiis + 1, "cudaMalloc(coef)");
    const int npairs_max = ndiis * ndiis;
    dpart.alloc(dots_scratch_elems(npairs_max), "cudaMalloc(dot scratch)"); dout.alloc(npairs_max, "cudaMalloc(dot out)");
    double *D = nullptr;
    check(cudaMalloc(&D, (size_t)n * sizeof(double)), "cudaMalloc(D)");
    struct FreeD { double *p; ~FreeD() { cudaFree(p); } } freeD{D};
    check(denominators(st, (const c128 *)fock, o, v, D), "denominators");
    E.enable_integer_slices();
    check(cudaMemcpyAsync(T.p, t1, (size_t)n1 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t1");
    check(cudaMemcpyAsync(T.p + n1, t2, (size_t)n2 * sizeof(c128), cudaMemcpyDeviceToDevice, st), "copy t2");

    auto host_dots = [&](const c128 *A, long lda, int na, const c128 *B, long ldb, int nb, long len, bool conjA) {
      std::vector<cplx> out((size_t)na * nb);
      check(multi_dot(st, A, lda, na, B, ldb, nb, len, conjA, false, dpart.p, dout.p), "multi_dot");
      check(cudaMemcpyAsync(out.data(), dout.p, out.size() * sizeof(c128), cudaMemcpyDeviceToHost, st), "D2H dots");
      check(cudaStreamSynchronize(st), "sync dots");
      return out;
    };
    auto set_coef = [&](const std::vector<cplx> &h) {
      check(cudaMemcpyAsync(coef.p, h.data(), h.size() * sizeof(c128), cudaMemcpyHostToDevice, st), "H2D coef");
      check(cudaStreamSynchronize(st), "sync coef");
    };
    int nhist = 0;
    // Precision on demand on the integer-slice path: a residual of size r only has to be known to a fraction of r, so the
    // contractions of an evaluation use the fewest slices with 16 * 2^(-7 s) * 10 <= r_prev / 100 (10 = a bound on the size of the
    // contracted terms); 2 slices at the start, all of them near convergence.  A residual that meets tol with fewer than all
    // slices is evaluated again with all of them before it is accepted.
    double prev_res = 1.0;
    auto evaluate = [&](int active) {
      E.oz.active = active;
      try {
        E.direct(T.p, OM.p);
      } catch (...) {
        E.oz.active = 0;
        throw;
      }
      E.oz.active = 0;
      ++res.sigma_calls;     // (residual evaluations)
      // ---- the full-tensor 2-norm: ||Omega1||^2 + 4 ||Omega2 (unique)||^2 ----
      const double d1 = host_dots(OM.p, n, 1, OM.p, n, 1, n1, true)[0].real();
      const double d2 = host_dots(OM.p + n1, n, 1, OM.p + n1, n, 1, n2, true)[0].real();
      res.residual = std::sqrt(std::max(0.0, d1 + 4.0 * d2));
    };
    for (int it = 0; it < maxiter; ++it) {
      res.iterations = it;
      int active = 0;
      if (E.ws.oz && E.oz.slices > 2) {
        int se = 2;
        while (se < E.oz.slices && std::ldexp(160.0, -7 * se) > 0.01 * prev_res) ++se;
        active = se < E.oz.slices ? se : 0;
      }
      evaluate(active);
      if (active && std::isfinite(res.residual) && res.residual <= tol) evaluate(0);
      prev_res = std::isfinite(res.residual) ? std::max(res.residual, 1e-300) : 1.0;
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
        std::vector<cplx> Bm = host_dots(HE.p, n, m, HE.p, n, m, n, true);
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
    E.P.rebind(E.t1_id, T.p);
    E.P.rebind(E.t2_id, T.p + n1);
    E.P.execute(PLAN_TAU);
    const c128 *tau = E.P.buf(E.P.find("tau")).ptr;
    const cplx e1 = host_dots(E.fovT, n1, 1, T.p, n1, 1, n1, false)[0];
    const cplx e2 = host_dots(E.W0, n2, 1, tau, n2, 1, n2, true)[0];     // conj(W0[(ab)(ij)]) = <ij||ab>
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
