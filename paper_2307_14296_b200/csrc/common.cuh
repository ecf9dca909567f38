// common.cuh — shared declarations of the CC-LR library (sm_100a only).
#pragma once
#include <cuda_runtime.h>
#include <cuda.h>
#include <stdint.h>
#include <stddef.h>

typedef double2 c128;  // complex128, interleaved (re, im)

#define CCLR_HOST_DEVICE __host__ __device__ __forceinline__

CCLR_HOST_DEVICE c128 cmul(c128 a, c128 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
CCLR_HOST_DEVICE c128 cadd(c128 a, c128 b) { return make_double2(a.x + b.x, a.y + b.y); }
CCLR_HOST_DEVICE c128 csub(c128 a, c128 b) { return make_double2(a.x - b.x, a.y - b.y); }
CCLR_HOST_DEVICE c128 cneg(c128 a) { return make_double2(-a.x, -a.y); }
CCLR_HOST_DEVICE c128 cconj(c128 a) { return make_double2(a.x, -a.y); }
CCLR_HOST_DEVICE c128 cscale(double s, c128 a) { return make_double2(s * a.x, s * a.y); }
CCLR_HOST_DEVICE c128 czero() { return make_double2(0.0, 0.0); }
// a += b * c
CCLR_HOST_DEVICE void cfma(c128 &a, c128 b, c128 c) {
  a.x = fma(b.x, c.x, a.x); a.x = fma(-b.y, c.y, a.x);
  a.y = fma(b.x, c.y, a.y); a.y = fma(b.y, c.x, a.y);
}

// pair index P(p<q) = q(q-1)/2 + p   (include/cclr.h)
CCLR_HOST_DEVICE long pair_index(long p, long q) { return q * (q - 1) / 2 + p; }
CCLR_HOST_DEVICE long npair(long n) { return n * (n - 1) / 2; }

// ---- zgemm.cu -------------------------------------------------------------------------------------------------
struct ZgemmWorkspace {
  c128 *buf = nullptr;   // split-K partial sums
  size_t elems = 0;      // capacity in complex elements
};
// C = alpha * opA(A) * opB(B) + beta * C; see include/cclr.h (cclr_zgemm).  ws may be null (no split-K then).
cudaError_t zgemm(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA,
                  const c128 *B, long ldb, bool b_is_kn, bool conjB, c128 beta, c128 *C, long ldc, int batch = 1,
                  long sa = 0, long sb = 0, long sc = 0, const ZgemmWorkspace *ws = nullptr);
int zgemm_num_sms();
