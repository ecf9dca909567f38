// context.cuh — the opaque cclr_ctx of include/cclr.h (shared by context.cu and solver.cu).
#pragma once
#include "plan.cuh"
#include "../../include/cclr.h"
#include <string>
#include <vector>

struct cclr_ctx {
  int o = 0, v = 0;
  long oo = 0, vv = 0, n1 = 0, n2 = 0;
  cudaStream_t st = nullptr;
  Plan *plan = nullptr;
  ZgemmWorkspace ws;
  OzWorkspace oz;                 // integer-slice product of ladder / ring (CCLR_GEMM_OZAKI): slices of W_vvvv, W_ovvo + scratch
  double *wplane = nullptr;       // persistent sum plane Re + Im of W_vvvv for the 3M ladder (ws.persist_*), or null
  std::vector<ResolvedOp> sigma_ops, ladder_ops, ring_ops, xi_ops, left_ops, eta_ops, eta_eom_ops;
  c128 *xblocks = nullptr;        // X_oo, X_ov, X_vo, X_vv of cclr_xi, contiguous
  int x1_id = -1, x2_id = -1, out1_id = -1, out2_id = -1;
  double *D = nullptr;            // orbital-energy denominators over unique elements, [n1 + n2]
  // small device scratch for dot products (vecops.cu)
  c128 *dot_partial = nullptr, *dot_out = nullptr;
  int dot_pairs_cap = 0;
  // profiling of the last cclr_sigma call
  bool profiling = false;
  double ms[5] = {0, 0, 0, 0, 0};
  std::vector<double> op_ms;      // per operation of the sigma plan, summed over the vectors of the last call
  std::vector<cudaEvent_t> events;
  // staging buffers of cclr_sigma_host
  cudaStream_t copy_stream = nullptr;   // cclr_sigma_host: x2 goes to the device here while the x1-only statements of the plan run
  cudaEvent_t copy_done = nullptr;
  int first_x2_op = 0;                  // index of the first statement of the sigma plan that reads x2
  c128 *host_stage = nullptr;
  size_t host_stage_elems = 0;
  c128 *lambda = nullptr;         // ground-state multipliers [n1 + n2], solved on first use by cclr_response_ci
  bool have_lambda = false;
  double lambda_tol = 0.0;        // tolerance the cached multipliers were solved to (a tighter request re-solves)
  // CUDA graph of the sigma plan (small problems are launch bound: ~35 kernels + 2 tensor-map encodes per GEMM per vector)
  bool graph_enabled = false, graph_failed = false;
  int plain_sigma_calls = 0;      // the first call runs plainly (it also configures the kernels' shared-memory attributes)
  cudaStream_t graph_stream = nullptr;
  cudaGraphExec_t sigma_graph = nullptr;
  c128 *graph_io = nullptr;       // staging [x1 | x2 | out1 | out2] the captured kernels are bound to
  int graph_kernels = 0;          // kernels per replay (added to the launch counter)
  int max_subspace = 0;           // cclr_set_max_subspace (0 = automatic)
  size_t extra_bytes = 0;         // device bytes owned outside the plan
};

// thread-local error reporting (context.cu)
void cclr_set_error(const std::string &msg, cudaError_t e);
int cclr_fail(const PlanError &e);

// out = A x for one vector on the context's stream (no shift when z == 0); throws PlanError
// left = true: out = l (A - z), the left transform (CCLR_PLAN_SIGMA_LEFT)
void cclr_sigma_one(cclr_ctx *ctx, const c128 *x1, const c128 *x2, c128 z, c128 *out1, c128 *out2, bool profile,
                    bool left = false);
void cclr_ensure_dot_scratch(cclr_ctx *ctx, int npairs);
