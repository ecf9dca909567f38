// probes.cu — roofline denominators measured by the library itself (include/cclr.h: cclr_fp64_tensor_peak,
// cclr_hbm_copy_peak) and the C-ABI wrapper of the GEMM engine (cclr_zgemm).
#include "common.cuh"
#include "../../include/cclr.h"

thread_local int g_last_cuda_error = 0;

#include <atomic>
static std::atomic<unsigned long long> g_kernel_launches{0};
void cclr_count_launch(int n) { g_kernel_launches.fetch_add((unsigned long long)n, std::memory_order_relaxed); }
unsigned long long cclr_launch_counter() { return g_kernel_launches.load(std::memory_order_relaxed); }
extern "C" unsigned long long cclr_kernel_launches(void) { return g_kernel_launches.load(std::memory_order_relaxed); }

namespace {

// 8 independent accumulator pairs per warp, no memory traffic: the DMMA issue-rate ceiling.
__global__ void __launch_bounds__(256) dmma_peak_kernel(double *out, int iters, double seed) {
  double c[16][2];
  double a = seed * (threadIdx.x + 1), b = seed * 3.0;
#pragma unroll
  for (int j = 0; j < 16; ++j) c[j][0] = c[j][1] = 0.0;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int j = 0; j < 16; ++j)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                   : "+d"(c[j][0]), "+d"(c[j][1])
                   : "d"(a), "d"(b));
  }
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < 16; ++j) s += c[j][0] + c[j][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

// mode 1: vector DFMA only; mode 2: even warps DMMA, odd warps DFMA (do the two FP64 paths overlap? on B200 they do not)
template <int MODE>
__global__ void __launch_bounds__(256) fp64_mix_kernel(double *out, int iters, double seed) {
  double c[8][2], d[16];
  const double a = seed * (threadIdx.x + 1), b = seed * 3.0;
#pragma unroll
  for (int j = 0; j < 8; ++j) c[j][0] = c[j][1] = 0.0;
#pragma unroll
  for (int j = 0; j < 16; ++j) d[j] = seed * j;
  const bool odd = (threadIdx.x >> 5) & 1;
  for (int it = 0; it < iters; ++it) {
    if (MODE == 2 && !odd) {
#pragma unroll
      for (int j = 0; j < 8; ++j)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                     : "+d"(c[j][0]), "+d"(c[j][1]) : "d"(a), "d"(b));
    }
    if (MODE == 1 || (MODE == 2 && odd)) {
#pragma unroll
      for (int r = 0; r < 4; ++r)
#pragma unroll
        for (int j = 0; j < 16; ++j) asm volatile("fma.rn.f64 %0, %1, %2, %0;" : "+d"(d[j]) : "d"(a), "d"(b));
    }
  }
  double s = 0.0;
#pragma unroll
  for (int j = 0; j < 8; ++j) s += c[j][0] + c[j][1];
#pragma unroll
  for (int j = 0; j < 16; ++j) s += d[j];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__global__ void copy_kernel(const double2 *__restrict__ src, double2 *__restrict__ dst, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x)
    dst[i] = src[i];
}

}  // namespace

extern "C" int cclr_last_cuda_error(void) { return g_last_cuda_error; }

extern "C" const char *cclr_strerror(int code) {
  switch (code) {
    case CCLR_OK: return "ok";
    case CCLR_EINVAL: return "invalid argument";
    case CCLR_ENOMEM: return "device allocation failed";
    case CCLR_ECUDA: return "CUDA error (see cclr_last_cuda_error)";
    case CCLR_ENOTCONV: return "solver did not converge within maxiter";
    case CCLR_ENODEV: return "no sm_100 CUDA device";
    default: return "unknown error";
  }
}

extern "C" int cclr_fp64_tensor_peak(void *cuda_stream, int iters, double *tflops) {
  if (!tflops || iters < 1) return CCLR_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int sms = zgemm_num_sms();
  const int grid = sms * 2, threads = 256;
  double *out = nullptr;
  cudaError_t e = cudaMalloc(&out, sizeof(double) * grid * threads);
  if (e != cudaSuccess) { g_last_cuda_error = e; return CCLR_ENOMEM; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  dmma_peak_kernel<<<grid, threads, 0, st>>>(out, iters / 4 + 1, 1e-9);  // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, st);
    dmma_peak_kernel<<<grid, threads, 0, st>>>(out, iters, 1e-9);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (e != cudaSuccess) { g_last_cuda_error = e; return CCLR_ECUDA; }
  const double flops = (double)grid * (threads / 32) * (double)iters * 16.0 * (8.0 * 8.0 * 4.0 * 2.0);
  *tflops = flops / (best * 1e-3) / 1e12;
  return CCLR_OK;
}

extern "C" int cclr_fp64_pipe_probe(void *cuda_stream, int mode, int iters, double *tflops) {
  if (!tflops || iters < 1 || mode < 0 || mode > 2) return CCLR_EINVAL;
  if (mode == 0) return cclr_fp64_tensor_peak(cuda_stream, iters, tflops);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int grid = zgemm_num_sms() * 2, threads = 256;
  double *out = nullptr;
  cudaError_t e = cudaMalloc(&out, sizeof(double) * grid * threads);
  if (e != cudaSuccess) { g_last_cuda_error = e; return CCLR_ENOMEM; }
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {   // first repetition is the warm-up
    cudaEventRecord(e0, st);
    if (mode == 1) fp64_mix_kernel<1><<<grid, threads, 0, st>>>(out, iters, 1e-9);
    else fp64_mix_kernel<2><<<grid, threads, 0, st>>>(out, iters, 1e-9);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(out);
  if (e != cudaSuccess) { g_last_cuda_error = e; return CCLR_ECUDA; }
  const double warps = (double)grid * (threads / 32);
  // per warp and iteration: DMMA warps 8 x 512 flop, DFMA warps 64 fma x 32 lanes x 2 flop (both 4096)
  *tflops = warps * (double)iters * 4096.0 / (best * 1e-3) / 1e12;
  return CCLR_OK;
}

extern "C" int cclr_hbm_copy_peak(void *cuda_stream, size_t bytes, double *gbs) {
  if (!gbs || bytes < (1u << 20)) return CCLR_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const size_t n = bytes / 32;  // n double2 read + n double2 written = bytes
  double2 *src = nullptr, *dst = nullptr;
  cudaError_t e = cudaMalloc(&src, n * 16);
  if (e == cudaSuccess) e = cudaMalloc(&dst, n * 16);
  if (e != cudaSuccess) { cudaFree(src); g_last_cuda_error = e; return CCLR_ENOMEM; }
  cudaMemsetAsync(src, 0, n * 16, st);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int grid = zgemm_num_sms() * 16;
  copy_kernel<<<grid, 512, 0, st>>>(src, dst, n);
  float best = 1e30f;
  for (int rep = 0; rep < 5; ++rep) {
    cudaEventRecord(e0, st);
    copy_kernel<<<grid, 512, 0, st>>>(src, dst, n);
    cudaEventRecord(e1, st);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(src);
  cudaFree(dst);
  if (e != cudaSuccess) { g_last_cuda_error = e; return CCLR_ECUDA; }
  *gbs = (double)(2 * n * 16) / (best * 1e-3) / 1e9;
  return CCLR_OK;
}

extern "C" int cclr_zgemm(void *cuda_stream, int M, int N, int K, const cclr_c128 *alpha, const cclr_c128 *A,
                          long lda, int conj_a, const cclr_c128 *B, long ldb, int b_is_kn, int conj_b,
                          const cclr_c128 *beta, cclr_c128 *C, long ldc, int batch, long sa, long sb, long sc, int three_m) {
  if (!alpha || !beta || !C || M < 0 || N < 0 || K < 0 || batch < 1) return CCLR_EINVAL;
  if (K > 0 && (!A || !B)) return CCLR_EINVAL;
  if (lda < K || ldc < N || (b_is_kn ? ldb < N : ldb < K)) return CCLR_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  // K-split workspace for this stand-alone entry point (the context keeps its own): room for 3 partial tiles per SM
  ZgemmWorkspace ws;
  ws.elems = (size_t)3 * zgemm_num_sms() * 128 * 64;
  ws.three_m = three_m != 0;
  if (ws.three_m && batch == 1 && M >= 512 && N >= 24 && K >= 64) {   // room for the sum planes of both operands (3M product)
    ws.plane_elems = ((size_t)M + (size_t)N + 16) * ((size_t)K + 2) + ((size_t)K + 16) * ((size_t)N + 2);
    if (cudaMalloc(&ws.plane, ws.plane_elems * sizeof(double)) != cudaSuccess) { ws.plane = nullptr; ws.plane_elems = 0; cudaGetLastError(); }
  }
  if (cudaMalloc(&ws.buf, ws.elems * sizeof(c128)) != cudaSuccess) { ws.buf = nullptr; ws.elems = 0; cudaGetLastError(); }
  cudaError_t e = zgemm(st, M, N, K, make_double2(alpha->re, alpha->im), (const c128 *)A, lda, conj_a != 0,
                        (const c128 *)B, ldb, b_is_kn != 0, conj_b != 0, make_double2(beta->re, beta->im), (c128 *)C,
                        ldc, batch, sa, sb, sc, &ws);
  if (ws.buf || ws.plane) {
    cudaStreamSynchronize(st);
    if (ws.buf) cudaFree(ws.buf);
    if (ws.plane) cudaFree(ws.plane);
  }
  if (e != cudaSuccess) { g_last_cuda_error = e; return CCLR_ECUDA; }
  return CCLR_OK;
}

extern "C" int cclr_zgemm_oz(void *cuda_stream, int M, int N, int K, const cclr_c128 *alpha, const cclr_c128 *A, long lda, int conj_a,
                             const cclr_c128 *B, long ldb, int b_is_kn, int conj_b, const cclr_c128 *beta, cclr_c128 *C, long ldc,
                             int slices, int bn, int reps, double *ms) {
  const bool b_side = slices >= 100;      // slices + 100: B ([K][N]) is the constant operand, C^T = B^T A^T route (zgemm_oz_bt)
  if (b_side) slices -= 100;
  if (!alpha || !beta || !A || !B || !C || reps < 1 || slices < 2 || slices > 8 || !zgemm_oz_supported(M, N, K)) return CCLR_EINVAL;
  if (b_side && !b_is_kn) return CCLR_EINVAL;
  if (lda < K || ldc < N || (b_is_kn ? ldb < N : ldb < K)) return CCLR_EINVAL;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  OzWorkspace ow;
  ow.slices = slices;
  ow.force_bn = bn % 1000;                  // bn + 1000 * c_n + 10000 * c_m forces the cluster shape as well (tuning runs)
  ow.force_cn = (bn / 1000) % 10;
  ow.force_cm = bn >= 1000 ? (bn / 10000 > 0 ? bn / 10000 : 1) : 0;
  cudaEvent_t ev[6];
  for (auto &e : ev) cudaEventCreate(&e);
  ow.ev_b[0] = ev[4]; ow.ev_b[1] = ev[5];
  cudaEventRecord(ev[0], st);
  cudaError_t e = b_side ? zgemm_oz_register_t(st, &ow, (const c128 *)B, ldb, K, N) : zgemm_oz_register(st, &ow, (const c128 *)A, lda, M, K);
  cudaEventRecord(ev[1], st);
  // reps > 1: the first product is an untimed warm-up (it allocates the B scratch); reps == 1 runs exactly one product
  const int first = reps > 1 ? 1 : 0;
  for (int r = 0; r < reps + first && e == cudaSuccess; ++r) {
    if (r == first) cudaEventRecord(ev[2], st);
    e = b_side ? zgemm_oz_bt(st, M, N, K, make_double2(alpha->re, alpha->im), (const c128 *)A, lda, conj_a != 0, (const c128 *)B, ldb,
                             conj_b != 0, make_double2(beta->re, beta->im), (c128 *)C, ldc, &ow)
               : zgemm_oz(st, M, N, K, make_double2(alpha->re, alpha->im), (const c128 *)A, lda, conj_a != 0, (const c128 *)B, ldb,
                          b_is_kn != 0, conj_b != 0, make_double2(beta->re, beta->im), (c128 *)C, ldc, &ow);
  }
  cudaEventRecord(ev[3], st);
  const cudaError_t e2 = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = e2;
  if (e == cudaSuccess && ms) {
    float t = 0.f;
    cudaEventElapsedTime(&t, ev[0], ev[1]); ms[0] = t;
    cudaEventElapsedTime(&t, ev[2], ev[3]); ms[1] = t / reps;
    cudaEventElapsedTime(&t, ev[4], ev[5]); ms[2] = t;
  }
  for (auto &x : ev) cudaEventDestroy(x);
  zgemm_oz_release(&ow);
  if (e != cudaSuccess) { g_last_cuda_error = e; return CCLR_ECUDA; }
  return CCLR_OK;
}
