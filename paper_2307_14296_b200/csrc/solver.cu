// solver.cu — placeholder until the response solver lands
#include "context.cuh"
extern "C" int cclr_solve(cclr_ctx *ctx, const cclr_c128 *xi1, const cclr_c128 *xi2, int nrhs, const double *omegas,
                          int nomega, double gamma, double tol, int maxiter, cclr_c128 *t1_out, cclr_c128 *t2_out,
                          cclr_solve_info *info) {
  cclr_set_error("cclr_solve: not implemented yet", cudaSuccess);
  return CCLR_EINVAL;
}
