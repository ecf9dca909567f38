// context.cu — C ABI of the CC-LR hot path (include/cclr.h): cclr_create / cclr_sigma / cclr_property and the
// kernel-level entry points.  Every arithmetic step is a launch of zgemm.cu (DMMA GEMM), permute.cu (layout) or
// vecops.cu (bandwidth kernels); this file only orchestrates them through the plans of plans.inc.
#include "context.cuh"
#include "plans.inc"
#include <cstring>
#include <new>

extern thread_local int g_last_cuda_error;   // probes.cu
static thread_local std::string g_last_message;

void cclr_set_error(const std::string &msg, cudaError_t e) {
  g_last_message = msg;
  if (e != cudaSuccess) g_last_cuda_error = (int)e;
}

int cclr_fail(const PlanError &e) {
  cclr_set_error(e.what(), e.cuda);
  cudaGetLastError();   // clear the sticky-free error state
  return e.code;
}

extern "C" const char *cclr_last_error_message(void) { return g_last_message.c_str(); }

namespace {

// the ring term alone and the ladder alone, on the buffers of the sigma plan
const char *const PLAN_LADDER = R"PLAN(
@ladder
gemm out2[(ab);(ij)] = 1 Wabef[(ab);(ef)] x2[(ef);(ij)] kn
)PLAN";
const char *const PLAN_RING = R"PLAN(
@layout
perm R[aiem] = 1 x2[(ae)(im)]
@ring
gemm Z[bj;ai] = 1 Wring[bj;em] R[ai;em] nk
@layout
perm out2[(ab)(ij)] = 1 Z[bjai] -1 Z[ajbi] -1 Z[biaj] 1 Z[aibj]
)PLAN";

void check(cudaError_t e, const char *where) {
  if (e != cudaSuccess)
    throw PlanError(e == cudaErrorMemoryAllocation ? CCLR_ENOMEM : CCLR_ECUDA, std::string(where) + ": " + cudaGetErrorString(e), e);
}

void run_ops(cclr_ctx *ctx, const std::vector<ResolvedOp> &ops, bool profile) {
  if (!profile) {
    for (const ResolvedOp &op : ops) ctx->plan->launch(op);
    return;
  }
  while (ctx->events.size() < ops.size() + 1) {
    cudaEvent_t ev;
    check(cudaEventCreate(&ev), "cudaEventCreate");
    ctx->events.push_back(ev);
  }
  check(cudaEventRecord(ctx->events[0], ctx->st), "cudaEventRecord");
  for (size_t k = 0; k < ops.size(); ++k) {
    ctx->plan->launch(ops[k]);
    check(cudaEventRecord(ctx->events[k + 1], ctx->st), "cudaEventRecord");
  }
  check(cudaEventSynchronize(ctx->events[ops.size()]), "cudaEventSynchronize");
  for (size_t k = 0; k < ops.size(); ++k) {
    float ms = 0.f;
    check(cudaEventElapsedTime(&ms, ctx->events[k], ctx->events[k + 1]), "cudaEventElapsedTime");
    ctx->ms[0] += ms;
    if (&ops == &ctx->sigma_ops) {
      if (ctx->op_ms.size() != ops.size()) ctx->op_ms.assign(ops.size(), 0.0);
      ctx->op_ms[k] += ms;
    }
    const int ph = ops[k].phase;
    if (ph >= PHASE_LADDER && ph <= PHASE_LAYOUT) ctx->ms[ph] += ms;
  }
}

void bind_vectors(cclr_ctx *ctx, const c128 *x1, const c128 *x2, c128 *out1, c128 *out2) {
  ctx->plan->rebind(ctx->x1_id, const_cast<c128 *>(x1));
  ctx->plan->rebind(ctx->x2_id, const_cast<c128 *>(x2));
  ctx->plan->rebind(ctx->out1_id, out1);
  ctx->plan->rebind(ctx->out2_id, out2);
}

void destroy(cclr_ctx *ctx) {
  if (!ctx) return;
  if (ctx->st) cudaStreamSynchronize(ctx->st);
  delete ctx->plan;
  if (ctx->ws.buf) cudaFree(ctx->ws.buf);
  if (ctx->ws.plane) cudaFree(ctx->ws.plane);
  if (ctx->wplane) cudaFree(ctx->wplane);
  zgemm_oz_release(&ctx->oz);
  if (ctx->D) cudaFree(ctx->D);
  if (ctx->dot_partial) cudaFree(ctx->dot_partial);
  if (ctx->dot_out) cudaFree(ctx->dot_out);
  if (ctx->host_stage) cudaFree(ctx->host_stage);
  if (ctx->copy_stream) cudaStreamDestroy(ctx->copy_stream);
  if (ctx->copy_done) cudaEventDestroy(ctx->copy_done);
  if (ctx->xblocks) cudaFree(ctx->xblocks);
  if (ctx->lambda) cudaFree(ctx->lambda);
  for (cudaEvent_t ev : ctx->events) cudaEventDestroy(ev);
  if (ctx->sigma_graph) cudaGraphExecDestroy(ctx->sigma_graph);
  if (ctx->graph_stream) cudaStreamDestroy(ctx->graph_stream);
  if (ctx->graph_io) cudaFree(ctx->graph_io);
  delete ctx;
}

}  // namespace

extern unsigned long long cclr_launch_counter();   // probes.cu

// Capture the sigma plan once into a CUDA graph bound to the staging vectors graph_io (shift 0); false if capture is impossible
static bool build_sigma_graph(cclr_ctx *ctx) {
  const size_t n = (size_t)(ctx->n1 + ctx->n2);
  if (cudaMalloc(&ctx->graph_io, 2 * n * sizeof(c128)) != cudaSuccess) { cudaGetLastError(); ctx->graph_io = nullptr; return false; }
  ctx->extra_bytes += 2 * n * sizeof(c128);
  if (cudaStreamCreateWithFlags(&ctx->graph_stream, cudaStreamNonBlocking) != cudaSuccess) { cudaGetLastError(); return false; }
  c128 *g = ctx->graph_io;
  bind_vectors(ctx, g, g + ctx->n1, g + n, g + n + ctx->n1);
  ctx->plan->set_scalar(0, make_double2(0.0, 0.0));
  cudaStreamSynchronize(ctx->st);
  cudaGraph_t graph = nullptr;
  bool ok = cudaStreamBeginCapture(ctx->graph_stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess;
  if (ok) {
    const unsigned long long c0 = cclr_launch_counter();
    ctx->plan->set_stream(ctx->graph_stream);
    try {
      for (const ResolvedOp &op : ctx->sigma_ops) ctx->plan->launch(op);
    } catch (const PlanError &) {
      ok = false;
    }
    ctx->plan->set_stream(ctx->st);
    ctx->graph_kernels = (int)(cclr_launch_counter() - c0);
    if (cudaStreamEndCapture(ctx->graph_stream, &graph) != cudaSuccess || !graph) ok = false;
  }
  if (ok && cudaGraphInstantiate(&ctx->sigma_graph, graph, 0) != cudaSuccess) { ctx->sigma_graph = nullptr; ok = false; }
  if (graph) cudaGraphDestroy(graph);
  if (!ok) cudaGetLastError();
  return ok;
}

void cclr_sigma_one(cclr_ctx *ctx, const c128 *x1, const c128 *x2, c128 z, c128 *out1, c128 *out2, bool profile, bool left) {
  if (ctx->graph_enabled && !ctx->graph_failed && !profile && !left) {
    if (!ctx->sigma_graph && ctx->plain_sigma_calls > 0 && !build_sigma_graph(ctx)) ctx->graph_failed = true;
    if (ctx->sigma_graph) {
      // replay: x -> staging, the captured kernels, out = (A x) - z x
      const size_t n = (size_t)(ctx->n1 + ctx->n2);
      c128 *g = ctx->graph_io;
      check(cudaMemcpyAsync(g, x1, (size_t)ctx->n1 * sizeof(c128), cudaMemcpyDeviceToDevice, ctx->st), "stage x1");
      check(cudaMemcpyAsync(g + ctx->n1, x2, (size_t)ctx->n2 * sizeof(c128), cudaMemcpyDeviceToDevice, ctx->st), "stage x2");
      check(cudaGraphLaunch(ctx->sigma_graph, ctx->st), "cudaGraphLaunch(sigma)");
      cclr_count_launch(ctx->graph_kernels);
      const c128 nz = make_double2(-z.x, -z.y);
      check(shifted_copy(ctx->st, out1, g + n, nz, x1, ctx->n1), "shift sigma1");
      check(shifted_copy(ctx->st, out2, g + n + ctx->n1, nz, x2, ctx->n2), "shift sigma2");
      return;
    }
    ++ctx->plain_sigma_calls;
  }
  bind_vectors(ctx, x1, x2, out1, out2);
  ctx->plan->set_scalar(0, make_double2(-z.x, -z.y));
  run_ops(ctx, left ? ctx->left_ops : ctx->sigma_ops, profile);
}

void cclr_ensure_dot_scratch(cclr_ctx *ctx, int npairs) {
  if (npairs <= ctx->dot_pairs_cap) return;
  check(cudaStreamSynchronize(ctx->st), "sync");
  if (ctx->dot_partial) { cudaFree(ctx->dot_partial); ctx->extra_bytes -= dots_scratch_elems(ctx->dot_pairs_cap) * sizeof(c128); }
  if (ctx->dot_out) { cudaFree(ctx->dot_out); ctx->extra_bytes -= (size_t)ctx->dot_pairs_cap * sizeof(c128); }
  ctx->dot_partial = ctx->dot_out = nullptr;
  ctx->dot_pairs_cap = 0;
  int cap = 256;
  while (cap < npairs) cap *= 2;
  check(cudaMalloc(&ctx->dot_partial, dots_scratch_elems(cap) * sizeof(c128)), "cudaMalloc(dot scratch)");
  check(cudaMalloc(&ctx->dot_out, (size_t)cap * sizeof(c128)), "cudaMalloc(dot out)");
  ctx->dot_pairs_cap = cap;
  ctx->extra_bytes += dots_scratch_elems(cap) * sizeof(c128) + (size_t)cap * sizeof(c128);
}

// ---------------------------------------------------------------------------------------------------------------
extern "C" int cclr_create(int o, int v, const cclr_c128 *fock, const cclr_eri_packed *eri, const cclr_c128 *t1,
                           const cclr_c128 *t2, unsigned flags, void *cuda_stream, cclr_ctx **out) {
  if (!out) return CCLR_EINVAL;
  *out = nullptr;
  if (o < 2 || v < 2 || !fock || !eri || !t1 || !t2 || !eri->oooo || !eri->ooov || !eri->oovv || !eri->ovvo ||
      !eri->ovvv || !eri->vvvv) {
    cclr_set_error("cclr_create: null pointer or o < 2 or v < 2", cudaSuccess);
    return CCLR_EINVAL;
  }
  int dev = 0;
  cudaDeviceProp prop;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&prop, dev) != cudaSuccess || prop.major != 10) {
    cudaGetLastError();
    cclr_set_error("cclr_create: no sm_100 device", cudaSuccess);
    return CCLR_ENODEV;
  }
  cclr_ctx *ctx = new (std::nothrow) cclr_ctx();
  if (!ctx) return CCLR_ENOMEM;
  try {
    ctx->o = o; ctx->v = v;
    ctx->oo = npair(o); ctx->vv = npair(v);
    ctx->n1 = (long)o * v; ctx->n2 = ctx->oo * ctx->vv;
    ctx->st = (cudaStream_t)cuda_stream;
    ctx->plan = new Plan(o, v, ctx->st);
    Plan &P = *ctx->plan;
    if (flags & CCLR_SMALL_CHUNKS) P.set_chunk_override(3);

    // split-K workspace of the GEMM engine
    ctx->ws.elems = (size_t)8 << 20;
    check(cudaMalloc(&ctx->ws.buf, ctx->ws.elems * sizeof(c128)), "cudaMalloc(split-K workspace)");
    ctx->extra_bytes += ctx->ws.elems * sizeof(c128);
    ctx->ws.three_m = (flags & CCLR_GEMM_4M) ? 0 : 1;
    if (ctx->ws.three_m && !(flags & CCLR_NO_SUM_PLANES)) {
      // scratch for the per-call sum planes of the 3M product: both operands of the ring-sized contractions
      const size_t ov = (size_t)o * v;
      ctx->ws.plane_elems = 2 * ov * (ov + 1);
      if (cudaMalloc(&ctx->ws.plane, ctx->ws.plane_elems * sizeof(double)) != cudaSuccess) {
        cudaGetLastError();
        ctx->ws.plane = nullptr;
        ctx->ws.plane_elems = 0;
      } else {
        ctx->extra_bytes += ctx->ws.plane_elems * sizeof(double);
      }
    }
    P.set_workspace(&ctx->ws);

    // borrowed inputs
    P.bind("oooo", "(mn)(ij)", (c128 *)eri->oooo);
    P.bind("ooov", "(mn)ie", (c128 *)eri->ooov);
    P.bind("oovv", "(mn)(ef)", (c128 *)eri->oovv);
    P.bind("ovvo", "mbej", (c128 *)eri->ovvo);
    P.bind("ovvv", "mb(ef)", (c128 *)eri->ovvv);
    P.bind("t1", "ai", (c128 *)t1);
    P.bind("t2", "(ab)(ij)", (c128 *)t2);

    // Fock blocks f_oo, f_ov, f_vv out of the [n][n] matrix
    const size_t nf = (size_t)o + v;
    const c128 *F = (const c128 *)fock;
    struct { const char *name, *spec; size_t r0, c0, rows, cols; } blocks[3] = {
        {"foo", "mi", 0, 0, (size_t)o, (size_t)o}, {"fov", "me", 0, (size_t)o, (size_t)o, (size_t)v},
        {"fvv", "ae", (size_t)o, (size_t)o, (size_t)v, (size_t)v}};
    for (auto &b : blocks) {
      c128 *p = nullptr;
      check(cudaMalloc(&p, b.rows * b.cols * sizeof(c128)), "cudaMalloc(fock block)");
      P.adopt(b.name, b.spec, p, BUF_TEMP, true);
      check(cudaMemcpy2DAsync(p, b.cols * sizeof(c128), F + b.r0 * nf + b.c0, nf * sizeof(c128), b.cols * sizeof(c128),
                              b.rows, cudaMemcpyDeviceToDevice, ctx->st),
            "copy fock block");
    }

    // <ab||ef>: adopted and dressed in place, or copied
    const size_t nvvvv = (size_t)ctx->vv * (size_t)ctx->vv;
    if (flags & CCLR_ERI_INPLACE) {
      P.adopt("Wabef", "(ab)(ef)", (c128 *)eri->vvvv, BUF_PERSIST, false);
    } else {
      c128 *p = nullptr;
      check(cudaMalloc(&p, nvvvv * sizeof(c128)), "cudaMalloc(Wabef)");
      P.adopt("Wabef", "(ab)(ef)", p, BUF_PERSIST, true);
      check(cudaMemcpyAsync(p, eri->vvvv, nvvvv * sizeof(c128), cudaMemcpyDeviceToDevice, ctx->st), "copy vvvv");
    }

    P.execute(CCLR_PLAN_CREATE);
    P.free_class(BUF_TEMP);

    // persistent sum plane of W_vvvv (Re + Im, 8 bytes per element): the ladder's big operand cannot be pre-passed per call
    // (N = oo is small), so the plane is formed once here -- when it fits comfortably (it is 1/2 of W_vvvv)
    if (ctx->ws.plane && ctx->vv >= 512 && ctx->oo >= 24) {
      size_t free_b = 0, total_b = 0;
      const long pld = (ctx->vv + 1) & ~1L;            // TMA needs 16-byte row strides
      const size_t bytes = (size_t)ctx->vv * pld * sizeof(double);
      if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && free_b > 3 * bytes && cudaMalloc(&ctx->wplane, bytes) == cudaSuccess) {
        const c128 *W = P.buf(P.find("Wabef")).ptr;
        check(zgemm_sum_plane(ctx->st, W, ctx->vv, ctx->vv, ctx->vv, false, ctx->wplane, pld), "sum plane of W_vvvv");
        ctx->ws.persist_key[0] = W;
        ctx->ws.persist_plane[0] = ctx->wplane;
        ctx->ws.persist_ld[0] = ctx->vv;
        ctx->ws.persist_pld[0] = pld;
        ctx->extra_bytes += bytes;
      } else {
        cudaGetLastError();
        ctx->wplane = nullptr;
      }
    }

    // integer slices of the two big constant operands of sigma -- the A operands of the ladder and of the ring -- for the INT8
    // tensor path (zgemm_oz.cu), when the shapes are eligible and the slices (3/4 of the operands) fit comfortably
    const bool any_size = (flags & CCLR_GEMM_INT8_ANY_SIZE) != 0;
    if (!(flags & (CCLR_GEMM_DMMA | CCLR_GEMM_4M)) &&
        (any_size ? zgemm_oz_supported((int)ctx->vv, (int)ctx->oo, (int)ctx->vv) : zgemm_oz_eligible((int)ctx->vv, (int)ctx->oo, (int)ctx->vv))) {
      const long ov = (long)o * v;
      const bool ring_too = any_size ? zgemm_oz_supported((int)ov, (int)ov, (int)ov) : zgemm_oz_eligible((int)ov, (int)ov, (int)ov);
      ctx->oz.any_size = any_size;
      const size_t need = (size_t)12 * ctx->vv * ctx->vv + (ring_too ? (size_t)12 * ov * ov : 0);
      size_t free_b = 0, total_b = 0;
      // slice count from the range inside the rows of the two operands (6 for integrals without outliers; more slices are more
      // products: 7 -> 28 pairs instead of 21; beyond 8 the contractions stay on the FP64 tensor cores)
      int s_lad = 0, s_ring = 0;
      check(zgemm_oz_suggest_slices(ctx->st, P.buf(P.find("Wabef")).ptr, ctx->vv, ctx->vv, ctx->vv, &s_lad, nullptr), "row statistics of W_vvvv");
      if (ring_too) check(zgemm_oz_suggest_slices(ctx->st, P.buf(P.find("Wring")).ptr, ov, ov, ov, &s_ring, nullptr), "row statistics of W_ovvo");
      const int s_need = (s_lad == 0 || (ring_too && s_ring == 0)) ? 0 : std::max(s_lad, s_ring);
      if (s_need > 0 && cudaMemGetInfo(&free_b, &total_b) == cudaSuccess && free_b > need * s_need / 6 + need / 2) {
        ctx->oz.slices = s_need;
        check(zgemm_oz_register(ctx->st, &ctx->oz, P.buf(P.find("Wabef")).ptr, ctx->vv, ctx->vv, ctx->vv), "integer slices of W_vvvv");
        if (ring_too) check(zgemm_oz_register(ctx->st, &ctx->oz, P.buf(P.find("Wring")).ptr, ov, ov, ov), "integer slices of W_ovvo");
        // ... and of W_vvvv's transpose for the transposed ladder of the left transform (lambda, left response equations, the F
        // transform), when another 3/4 of W_vvvv still leaves room for the solvers' trial spaces
        const size_t need_t = (size_t)2 * s_need * ctx->vv * ctx->vv;
        if (!(flags & CCLR_NO_LEFT_SLICES) && cudaMemGetInfo(&free_b, &total_b) == cudaSuccess &&
            free_b > need_t + std::max<size_t>((size_t)32 << 30, 64 * (size_t)(ctx->n1 + ctx->n2) * sizeof(c128)))
          check(zgemm_oz_register_t(ctx->st, &ctx->oz, P.buf(P.find("Wabef")).ptr, ctx->vv, ctx->vv, ctx->vv), "integer slices of W_vvvv^T");
        ctx->extra_bytes += ctx->oz.persist_bytes;
        ctx->ws.oz = &ctx->oz;
      }
    }

    check(cudaMalloc(&ctx->D, (size_t)(ctx->n1 + ctx->n2) * sizeof(double)), "cudaMalloc(D)");
    ctx->extra_bytes += (size_t)(ctx->n1 + ctx->n2) * sizeof(double);
    check(denominators(ctx->st, F, o, v, ctx->D), "denominators");

    // the borrowed inputs end here
    check(cudaStreamSynchronize(ctx->st), "cclr_create sync");
    for (const char *name : {"oooo", "ooov", "oovv", "ovvo", "ovvv", "t1", "t2"}) P.rebind(P.find(name), nullptr);

    // resolve the sigma plan once (allocates its workspace)
    P.bind("x1", "ai", nullptr);
    P.bind("x2", "(ab)(ij)", nullptr);
    P.bind("out1", "ai", nullptr);
    P.bind("out2", "(ab)(ij)", nullptr);
    ctx->x1_id = P.find("x1"); ctx->x2_id = P.find("x2");
    ctx->out1_id = P.find("out1"); ctx->out2_id = P.find("out2");
    P.compile(CCLR_PLAN_SIGMA, ctx->sigma_ops);
    ctx->first_x2_op = (int)ctx->sigma_ops.size();
    for (size_t k = 0; k < ctx->sigma_ops.size(); ++k) {
      const ResolvedOp &op = ctx->sigma_ops[k];
      bool reads = false;
      if (op.type == 0) reads = op.a == ctx->x2_id || op.b == ctx->x2_id || (op.acc && op.c == ctx->x2_id);
      else
        for (int q = 0; q < op.args.nsrc; ++q) reads = reads || op.srcbuf[q] == ctx->x2_id;
      if (reads) { ctx->first_x2_op = (int)k; break; }
    }
    P.compile(PLAN_LADDER, ctx->ladder_ops);
    P.compile(PLAN_RING, ctx->ring_ops);
    // the xi plan works on blocks of the operator matrix kept in a small context buffer
    const size_t no = (size_t)o, nv = (size_t)v;
    check(cudaMalloc(&ctx->xblocks, (no * no + 2 * no * nv + nv * nv) * sizeof(c128)), "cudaMalloc(X blocks)");
    ctx->extra_bytes += (no * no + 2 * no * nv + nv * nv) * sizeof(c128);
    P.bind("xoo", "mi", ctx->xblocks);
    P.bind("xov", "me", ctx->xblocks + no * no);
    P.bind("xvo", "ai", ctx->xblocks + no * no + no * nv);
    P.bind("xvv", "ae", ctx->xblocks + no * no + 2 * no * nv);
    P.compile(CCLR_PLAN_XI, ctx->xi_ops);
    P.compile(CCLR_PLAN_SIGMA_LEFT, ctx->left_ops);
    P.compile(CCLR_PLAN_ETA, ctx->eta_ops);
    P.compile(CCLR_PLAN_ETA_EOM, ctx->eta_eom_ops);
    cclr_ensure_dot_scratch(ctx, 256);
    // launch-bound sizes replay the sigma plan as one CUDA graph (configs 1, 2, 5; above ~2M unique elements the ~40 launches
    // of a sigma evaluation are noise)
    ctx->graph_enabled = !(flags & CCLR_NO_GRAPH) && (ctx->n1 + ctx->n2) <= (2L << 20);
  } catch (const PlanError &e) {
    destroy(ctx);
    return cclr_fail(e);
  } catch (const std::exception &e) {
    destroy(ctx);
    cclr_set_error(e.what(), cudaSuccess);
    return CCLR_EINVAL;
  }
  *out = ctx;
  return CCLR_OK;
}

extern "C" void cclr_destroy(cclr_ctx *ctx) { destroy(ctx); }

extern "C" int cclr_gemm_slices(const cclr_ctx *ctx) { return (ctx && ctx->ws.oz) ? ctx->oz.slices : 0; }

extern "C" int cclr_set_gemm_path(cclr_ctx *ctx, int path) {
  if (!ctx) return CCLR_EINVAL;
  if (ctx->st) cudaStreamSynchronize(ctx->st);
  OzWorkspace *want = (path != 0 && ctx->oz.slices > 0 && !ctx->oz.persist.empty()) ? &ctx->oz : nullptr;
  if (want != ctx->ws.oz) {
    ctx->ws.oz = want;
    if (ctx->sigma_graph) { cudaGraphExecDestroy(ctx->sigma_graph); ctx->sigma_graph = nullptr; }   // captured with the other path
    if (ctx->graph_io) { cudaFree(ctx->graph_io); ctx->graph_io = nullptr; ctx->extra_bytes -= 2 * (size_t)(ctx->n1 + ctx->n2) * sizeof(c128); }
    if (ctx->graph_stream) { cudaStreamDestroy(ctx->graph_stream); ctx->graph_stream = nullptr; }
  }
  return ctx->ws.oz ? 1 : 0;
}

extern "C" size_t cclr_ctx_bytes(const cclr_ctx *ctx) {
  return ctx ? ctx->plan->owned_bytes() + ctx->extra_bytes : 0;
}

extern "C" int cclr_sigma(cclr_ctx *ctx, const cclr_c128 *x1, const cclr_c128 *x2, int nvec, double omega,
                          double gamma, cclr_c128 *out1, cclr_c128 *out2) {
  if (!ctx || !x1 || !x2 || !out1 || !out2 || nvec < 1 || x1 == out1 || x2 == out2) {
    cclr_set_error("cclr_sigma: null pointer, nvec < 1 or aliased output", cudaSuccess);
    return CCLR_EINVAL;
  }
  try {
    if (ctx->profiling) {
      for (double &m : ctx->ms) m = 0.0;
      ctx->op_ms.assign(ctx->sigma_ops.size(), 0.0);
    }
    for (int k = 0; k < nvec; ++k)
      cclr_sigma_one(ctx, (const c128 *)x1 + (size_t)k * ctx->n1, (const c128 *)x2 + (size_t)k * ctx->n2,
                     make_double2(omega, gamma), (c128 *)out1 + (size_t)k * ctx->n1, (c128 *)out2 + (size_t)k * ctx->n2,
                     ctx->profiling);
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}

extern "C" int cclr_sigma_left(cclr_ctx *ctx, const cclr_c128 *l1, const cclr_c128 *l2, int nvec, double omega,
                               double gamma, cclr_c128 *out1, cclr_c128 *out2) {
  if (!ctx || !l1 || !l2 || !out1 || !out2 || nvec < 1 || l1 == out1 || l2 == out2) {
    cclr_set_error("cclr_sigma_left: null pointer, nvec < 1 or aliased output", cudaSuccess);
    return CCLR_EINVAL;
  }
  try {
    for (int k = 0; k < nvec; ++k)
      cclr_sigma_one(ctx, (const c128 *)l1 + (size_t)k * ctx->n1, (const c128 *)l2 + (size_t)k * ctx->n2,
                     make_double2(omega, gamma), (c128 *)out1 + (size_t)k * ctx->n1, (c128 *)out2 + (size_t)k * ctx->n2,
                     false, true);
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}

extern "C" int cclr_sigma_host(cclr_ctx *ctx, const cclr_c128 *x1, const cclr_c128 *x2, int nvec, double omega,
                               double gamma, cclr_c128 *out1, cclr_c128 *out2) {
  if (!ctx || !x1 || !x2 || !out1 || !out2 || nvec < 1) {
    cclr_set_error("cclr_sigma_host: null pointer or nvec < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  try {
    const size_t n = (size_t)(ctx->n1 + ctx->n2), need = 2 * n * (size_t)nvec;
    if (ctx->host_stage_elems < need) {
      check(cudaStreamSynchronize(ctx->st), "sync");
      if (ctx->host_stage) { cudaFree(ctx->host_stage); ctx->extra_bytes -= ctx->host_stage_elems * sizeof(c128); }
      ctx->host_stage = nullptr;
      ctx->host_stage_elems = 0;
      check(cudaMalloc(&ctx->host_stage, need * sizeof(c128)), "cudaMalloc(host staging)");
      ctx->host_stage_elems = need;
      ctx->extra_bytes += need * sizeof(c128);
    }
    c128 *dx1 = ctx->host_stage, *dx2 = dx1 + (size_t)nvec * ctx->n1;
    c128 *do1 = dx2 + (size_t)nvec * ctx->n2, *do2 = do1 + (size_t)nvec * ctx->n1;
    check(cudaMemcpyAsync(dx1, x1, (size_t)nvec * ctx->n1 * sizeof(c128), cudaMemcpyHostToDevice, ctx->st), "H2D x1");
    const bool overlap = !ctx->graph_enabled && !ctx->profiling && ctx->first_x2_op > 0 && ctx->first_x2_op < (int)ctx->sigma_ops.size();
    if (!overlap) {
      check(cudaMemcpyAsync(dx2, x2, (size_t)nvec * ctx->n2 * sizeof(c128), cudaMemcpyHostToDevice, ctx->st), "H2D x2");
      const int rc = cclr_sigma(ctx, (cclr_c128 *)dx1, (cclr_c128 *)dx2, nvec, omega, gamma, (cclr_c128 *)do1, (cclr_c128 *)do2);
      if (rc != CCLR_OK) return rc;
    } else {
      // the doubles part of the trial block (99.9 % of the bytes) travels on a second stream while the statements of the plan that
      // read x1 only run (the plan lists them first); the first statement that reads x2 waits for the copy
      if (!ctx->copy_stream) check(cudaStreamCreateWithFlags(&ctx->copy_stream, cudaStreamNonBlocking), "cudaStreamCreate(copy)");
      if (!ctx->copy_done) check(cudaEventCreateWithFlags(&ctx->copy_done, cudaEventDisableTiming), "cudaEventCreate(copy)");
      check(cudaStreamSynchronize(ctx->st), "sync before the overlapped copy");      // earlier work on st may still read the staging block
      check(cudaMemcpyAsync(dx2, x2, (size_t)nvec * ctx->n2 * sizeof(c128), cudaMemcpyHostToDevice, ctx->copy_stream), "H2D x2");
      check(cudaEventRecord(ctx->copy_done, ctx->copy_stream), "cudaEventRecord(copy)");
      for (int k = 0; k < nvec; ++k) {
        bind_vectors(ctx, dx1 + (size_t)k * ctx->n1, dx2 + (size_t)k * ctx->n2, do1 + (size_t)k * ctx->n1, do2 + (size_t)k * ctx->n2);
        ctx->plan->set_scalar(0, make_double2(-omega, -gamma));
        for (int i = 0; i < (int)ctx->sigma_ops.size(); ++i) {
          if (i == ctx->first_x2_op && k == 0) check(cudaStreamWaitEvent(ctx->st, ctx->copy_done, 0), "cudaStreamWaitEvent(copy)");
          ctx->plan->launch(ctx->sigma_ops[i]);
        }
      }
    }
    check(cudaMemcpyAsync(out1, do1, (size_t)nvec * ctx->n1 * sizeof(c128), cudaMemcpyDeviceToHost, ctx->st), "D2H out1");
    check(cudaMemcpyAsync(out2, do2, (size_t)nvec * ctx->n2 * sizeof(c128), cudaMemcpyDeviceToHost, ctx->st), "D2H out2");
    check(cudaStreamSynchronize(ctx->st), "cclr_sigma_host sync");
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}

extern "C" int cclr_ladder(cclr_ctx *ctx, const cclr_c128 *x2, int nvec, cclr_c128 *out2) {
  if (!ctx || !x2 || !out2 || nvec < 1 || x2 == out2) return CCLR_EINVAL;
  try {
    for (int k = 0; k < nvec; ++k) {
      bind_vectors(ctx, nullptr, (const c128 *)x2 + (size_t)k * ctx->n2, nullptr, (c128 *)out2 + (size_t)k * ctx->n2);
      run_ops(ctx, ctx->ladder_ops, false);
    }
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}

extern "C" int cclr_ring(cclr_ctx *ctx, const cclr_c128 *x2, cclr_c128 *out2) {
  if (!ctx || !x2 || !out2 || x2 == out2) return CCLR_EINVAL;
  try {
    bind_vectors(ctx, nullptr, (const c128 *)x2, nullptr, (c128 *)out2);
    run_ops(ctx, ctx->ring_ops, false);
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}

static void load_x_blocks(cclr_ctx *ctx, const cclr_c128 *X);

extern "C" int cclr_xi(cclr_ctx *ctx, const cclr_c128 *X, cclr_c128 *xi1, cclr_c128 *xi2) {
  if (!ctx || !X || !xi1 || !xi2) {
    cclr_set_error("cclr_xi: null pointer", cudaSuccess);
    return CCLR_EINVAL;
  }
  try {
    load_x_blocks(ctx, X);
    bind_vectors(ctx, nullptr, nullptr, (c128 *)xi1, (c128 *)xi2);
    run_ops(ctx, ctx->xi_ops, false);
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}

static void load_x_blocks(cclr_ctx *ctx, const cclr_c128 *X) {
  const size_t o = (size_t)ctx->o, v = (size_t)ctx->v, nf = o + v;
  const c128 *F = (const c128 *)X;
  struct { size_t off, r0, c0, rows, cols; } blocks[4] = {
      {0, 0, 0, o, o}, {o * o, 0, o, o, v}, {o * o + o * v, o, 0, v, o}, {o * o + 2 * o * v, o, o, v, v}};
  for (auto &b : blocks)
    check(cudaMemcpy2DAsync(ctx->xblocks + b.off, b.cols * sizeof(c128), F + b.r0 * nf + b.c0, nf * sizeof(c128),
                            b.cols * sizeof(c128), b.rows, cudaMemcpyDeviceToDevice, ctx->st),
          "copy X block");
}

extern "C" int cclr_eta(cclr_ctx *ctx, const cclr_c128 *X, const cclr_c128 *lam1, const cclr_c128 *lam2, int eom,
                        cclr_c128 *eta1, cclr_c128 *eta2) {
  if (!ctx || !X || !lam1 || !lam2 || !eta1 || !eta2 || lam1 == eta1 || lam2 == eta2) {
    cclr_set_error("cclr_eta: null pointer or aliased output", cudaSuccess);
    return CCLR_EINVAL;
  }
  try {
    load_x_blocks(ctx, X);
    if (eom) {   // xi^X into the work buffers xiw1 / xiw2 first (the EOM term contracts lambda2 with xi1)
      c128 *w1 = ctx->plan->buf(ctx->plan->find("xiw1")).ptr, *w2 = ctx->plan->buf(ctx->plan->find("xiw2")).ptr;
      bind_vectors(ctx, nullptr, nullptr, w1, w2);
      run_ops(ctx, ctx->xi_ops, false);
    }
    bind_vectors(ctx, (const c128 *)lam1, (const c128 *)lam2, (c128 *)eta1, (c128 *)eta2);
    run_ops(ctx, ctx->eta_ops, false);
    if (eom) run_ops(ctx, ctx->eta_eom_ops, false);
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}

// out = F y (CCLR_PLAN_FY, csrc/plans.inc) for nvec vectors y and one set of multipliers; the lambda-only left ladder M
// (CCLR_PLAN_FY_M) is evaluated once per call.  The plan holds chunk loops and frees its temporaries as it goes, so it is
// executed statement by statement on the context's plan (like cclr_create), not compiled.
extern "C" int cclr_f_transform(cclr_ctx *ctx, const cclr_eri_packed *eri, const cclr_c128 *lam1, const cclr_c128 *lam2,
                                const cclr_c128 *y1, const cclr_c128 *y2, int nvec, cclr_c128 *out1, cclr_c128 *out2) {
  if (!ctx || !eri || !eri->ooov || !eri->oovv || !eri->ovvo || !eri->ovvv || !lam1 || !lam2 || !y1 || !y2 || !out1 || !out2 ||
      nvec < 1 || y1 == out1 || y2 == out2) {
    cclr_set_error("cclr_f_transform: null pointer, nvec < 1 or aliased output", cudaSuccess);
    return CCLR_EINVAL;
  }
  Plan &P = *ctx->plan;
  auto unbind = [&]() {
    for (const char *name : {"ooov", "oovv", "ovvo", "ovvv", "y1", "y2"}) {
      const int id = P.find(name);
      if (id >= 0) P.rebind(id, nullptr);
    }
  };
  try {
    P.bind("ooov", "(mn)ie", (c128 *)eri->ooov);
    P.bind("oovv", "(mn)(ef)", (c128 *)eri->oovv);
    P.bind("ovvo", "mbej", (c128 *)eri->ovvo);
    P.bind("ovvv", "mb(ef)", (c128 *)eri->ovvv);
    bind_vectors(ctx, (const c128 *)lam1, (const c128 *)lam2, nullptr, nullptr);
    P.execute(CCLR_PLAN_FY_M);
    for (int k = 0; k < nvec; ++k) {
      P.bind("y1", "ai", (c128 *)y1 + (size_t)k * ctx->n1);
      P.bind("y2", "(ab)(ij)", (c128 *)y2 + (size_t)k * ctx->n2);
      bind_vectors(ctx, (const c128 *)lam1, (const c128 *)lam2, (c128 *)out1 + (size_t)k * ctx->n1, (c128 *)out2 + (size_t)k * ctx->n2);
      P.execute(CCLR_PLAN_FY);
      P.free_class(BUF_TEMP);
    }
    check(cudaStreamSynchronize(ctx->st), "cclr_f_transform sync");   // the borrowed integrals end here
    unbind();
  } catch (const PlanError &e) {
    try { P.free_class(BUF_TEMP); } catch (...) {}
    unbind();
    return cclr_fail(e);
  }
  return CCLR_OK;
}

extern "C" long cclr_get_intermediate(cclr_ctx *ctx, const char *name, cclr_c128 *out, long capacity) {
  if (!ctx || !name) return CCLR_EINVAL;
  long n = 0;
  const void *src = nullptr;
  const int id = ctx->plan->find(name);
  if (id >= 0 && ctx->plan->buf(id).ptr && ctx->plan->buf(id).cls != BUF_EXTERNAL) {
    n = (long)ctx->plan->buf_elems(id);
    src = ctx->plan->buf(id).ptr;
  } else if (id >= 0 && std::strcmp(name, "Wabef") == 0 && ctx->plan->buf(id).ptr) {
    n = (long)ctx->plan->buf_elems(id);
    src = ctx->plan->buf(id).ptr;
  }
  if (!src) {
    cclr_set_error(std::string("cclr_get_intermediate: unknown intermediate ") + name, cudaSuccess);
    return CCLR_EINVAL;
  }
  if (!out) return n;
  if (capacity < n) return CCLR_EINVAL;
  cudaError_t e = cudaMemcpyAsync(out, src, (size_t)n * sizeof(c128), cudaMemcpyDeviceToDevice, ctx->st);
  if (e != cudaSuccess) { cclr_set_error("cclr_get_intermediate copy", e); return CCLR_ECUDA; }
  return n;
}

extern "C" long cclr_get_intermediate_slice(cclr_ctx *ctx, const char *name, long offset, long count, cclr_c128 *out) {
  if (!ctx || !name || !out || offset < 0 || count < 0) return CCLR_EINVAL;
  const long n = cclr_get_intermediate(ctx, name, nullptr, 0);
  if (n < 0) return n;
  if (offset + count > n) {
    cclr_set_error(std::string("cclr_get_intermediate_slice: range outside ") + name, cudaSuccess);
    return CCLR_EINVAL;
  }
  const c128 *src = ctx->plan->buf(ctx->plan->find(name)).ptr + offset;
  cudaError_t e = cudaMemcpyAsync(out, src, (size_t)count * sizeof(c128), cudaMemcpyDeviceToDevice, ctx->st);
  if (e != cudaSuccess) { cclr_set_error("cclr_get_intermediate_slice copy", e); return CCLR_ECUDA; }
  return count;
}

extern "C" int cclr_set_max_subspace(cclr_ctx *ctx, int dim) {
  if (!ctx || dim < 0) return CCLR_EINVAL;
  ctx->max_subspace = dim;
  return CCLR_OK;
}

extern "C" int cclr_set_profiling(cclr_ctx *ctx, int on) {
  if (!ctx) return CCLR_EINVAL;
  ctx->profiling = on != 0;
  return CCLR_OK;
}

extern "C" int cclr_last_sigma_ms(const cclr_ctx *ctx, double ms[5]) {
  if (!ctx || !ms) return CCLR_EINVAL;
  for (int k = 0; k < 5; ++k) ms[k] = ctx->ms[k];
  return CCLR_OK;
}

extern "C" int cclr_sigma_op_count(const cclr_ctx *ctx) { return ctx ? (int)ctx->sigma_ops.size() : CCLR_EINVAL; }

extern "C" const char *cclr_sigma_op_text(const cclr_ctx *ctx, int k) {
  if (!ctx || k < 0 || k >= (int)ctx->sigma_ops.size()) return "";
  return ctx->sigma_ops[k].text.c_str();
}

extern "C" int cclr_last_sigma_op_ms(const cclr_ctx *ctx, double *ms, int capacity) {
  if (!ctx || !ms || capacity < (int)ctx->sigma_ops.size()) return CCLR_EINVAL;
  for (size_t k = 0; k < ctx->sigma_ops.size(); ++k) ms[k] = k < ctx->op_ms.size() ? ctx->op_ms[k] : 0.0;
  return (int)ctx->sigma_ops.size();
}

extern "C" int cclr_property(cclr_ctx *ctx, const cclr_c128 *eta1, const cclr_c128 *eta2, const cclr_c128 *x1,
                             const cclr_c128 *x2, int nvec, cclr_c128 *result) {
  if (!ctx || !eta1 || !eta2 || !x1 || !x2 || !result || nvec < 1 || nvec > 16384) return CCLR_EINVAL;
  try {
    cclr_ensure_dot_scratch(ctx, 2 * nvec);
    // bilinear dots over unique elements: singles then packed doubles (Eq. 15)
    check(multi_dot(ctx->st, (const c128 *)eta1, ctx->n1, 1, (const c128 *)x1, ctx->n1, nvec, ctx->n1, false, false,
                    ctx->dot_partial, ctx->dot_out),
          "multi_dot(singles)");
    check(multi_dot(ctx->st, (const c128 *)eta2, ctx->n2, 1, (const c128 *)x2, ctx->n2, nvec, ctx->n2, false, false,
                    ctx->dot_partial + dots_scratch_elems(nvec), ctx->dot_out + nvec),
          "multi_dot(doubles)");
    std::vector<c128> host(2 * (size_t)nvec);
    check(cudaMemcpyAsync(host.data(), ctx->dot_out, host.size() * sizeof(c128), cudaMemcpyDeviceToHost, ctx->st), "D2H dots");
    check(cudaStreamSynchronize(ctx->st), "cclr_property sync");
    for (int k = 0; k < nvec; ++k) {
      result[k].re = host[k].x + host[nvec + k].x;
      result[k].im = host[k].y + host[nvec + k].y;
    }
  } catch (const PlanError &e) {
    return cclr_fail(e);
  }
  return CCLR_OK;
}
