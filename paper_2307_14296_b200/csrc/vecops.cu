// vecops.cu — bandwidth kernels of the response solver (steps 2-5 of PAPER.md:952-967) and of the property
// contraction eta . t (PAPER.md:137 Eq. 15, :203): tall-skinny dot products with warp-shuffle + block reductions,
// linear combinations of subspace vectors, the orbital-energy preconditioner r / (z - D) and the
// denominators D1, D2.  All are pure streaming kernels over packed unique elements, 16-byte vectorised accesses.
#include "common.cuh"

namespace {

constexpr int DOT_THREADS = 256;
constexpr int DOT_MAX_CHUNKS = 296;   // 2 x 148 SMs

__device__ __forceinline__ c128 warp_sum(c128 v) {
#pragma unroll
  for (int s = 16; s > 0; s >>= 1) {
    v.x += __shfl_xor_sync(0xffffffffu, v.x, s);
    v.y += __shfl_xor_sync(0xffffffffu, v.y, s);
  }
  return v;
}

// partial[pair][chunk]: each block reduces one chunk of one (ia, ib) pair; fixed chunking -> deterministic result
__global__ void __launch_bounds__(DOT_THREADS) dot_partial_kernel(const c128 *__restrict__ A, long lda,
                                                                  const c128 *__restrict__ B, long ldb, int nb, long n,
                                                                  int conjA, int diag, long chunk_len,
                                                                  c128 *__restrict__ partial) {
  const int pair = blockIdx.y;
  const int ia = diag ? pair : pair / nb, ib = diag ? pair : pair % nb;
  const c128 *a = A + (size_t)ia * lda, *b = B + (size_t)ib * ldb;
  const long i0 = (long)blockIdx.x * chunk_len;
  long i1 = i0 + chunk_len;
  if (i1 > n) i1 = n;
  double sx = 0.0, sy = 0.0;
  const double sgn = conjA ? -1.0 : 1.0;
  // four independent 16-byte loads per operand in flight per thread (memory-level parallelism), fixed summation order
  double tx[4] = {0.0, 0.0, 0.0, 0.0}, ty[4] = {0.0, 0.0, 0.0, 0.0};
  long i = i0 + threadIdx.x;
  for (; i + 3 * DOT_THREADS < i1; i += 4 * DOT_THREADS) {
    c128 x[4], y[4];
#pragma unroll
    for (int u = 0; u < 4; ++u) { x[u] = a[i + u * DOT_THREADS]; y[u] = b[i + u * DOT_THREADS]; }
#pragma unroll
    for (int u = 0; u < 4; ++u) {
      x[u].y *= sgn;
      tx[u] = fma(x[u].x, y[u].x, tx[u]); tx[u] = fma(-x[u].y, y[u].y, tx[u]);
      ty[u] = fma(x[u].x, y[u].y, ty[u]); ty[u] = fma(x[u].y, y[u].x, ty[u]);
    }
  }
  for (; i < i1; i += DOT_THREADS) {
    c128 x = a[i];
    const c128 y = b[i];
    x.y *= sgn;
    tx[0] = fma(x.x, y.x, tx[0]); tx[0] = fma(-x.y, y.y, tx[0]);
    ty[0] = fma(x.x, y.y, ty[0]); ty[0] = fma(x.y, y.x, ty[0]);
  }
  sx = (tx[0] + tx[1]) + (tx[2] + tx[3]);
  sy = (ty[0] + ty[1]) + (ty[2] + ty[3]);
  __shared__ c128 red[DOT_THREADS / 32];
  c128 w = warp_sum(make_double2(sx, sy));
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = w;
  __syncthreads();
  if (threadIdx.x < 32) {
    c128 t = threadIdx.x < DOT_THREADS / 32 ? red[threadIdx.x] : czero();
    t = warp_sum(t);
    if (threadIdx.x == 0) partial[(size_t)pair * gridDim.x + blockIdx.x] = t;
  }
}

__global__ void dot_final_kernel(const c128 *__restrict__ partial, int nchunks, int npairs, c128 *__restrict__ out) {
  const int pair = blockIdx.x * blockDim.x + threadIdx.x;
  if (pair >= npairs) return;
  c128 s = czero();
  for (int c = 0; c < nchunks; ++c) s = cadd(s, partial[(size_t)pair * nchunks + c]);
  out[pair] = s;
}

__global__ void __launch_bounds__(256) lincomb_kernel(c128 *__restrict__ y, c128 beta, const c128 *__restrict__ coef,
                                                      const c128 *__restrict__ V, long ldv, int m, long n) {
  extern __shared__ c128 cs[];
  for (int j = threadIdx.x; j < m; j += blockDim.x) cs[j] = coef[j];
  __syncthreads();
  const bool has_beta = beta.x != 0.0 || beta.y != 0.0;
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
    c128 acc = has_beta ? cmul(beta, y[i]) : czero();
    for (int j = 0; j < m; ++j) cfma(acc, cs[j], V[(size_t)j * ldv + i]);
    y[i] = acc;
  }
}

__global__ void __launch_bounds__(256) precondition_kernel(c128 *__restrict__ y, const c128 *__restrict__ x,
                                                           const double *__restrict__ D, c128 z, c128 alpha, long n) {
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
    const double dr = z.x - D[i], di = z.y;          // 1 / (dr + i di) = (dr - i di) / (dr^2 + di^2)
    const double inv = 1.0 / (dr * dr + di * di);
    const c128 q = cmul(alpha, x[i]);
    y[i] = make_double2((q.x * dr + q.y * di) * inv, (q.y * dr - q.x * di) * inv);
  }
}

__global__ void __launch_bounds__(256) scale_kernel(c128 *__restrict__ y, c128 alpha, long n) {
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x)
    y[i] = cmul(alpha, y[i]);
}

__global__ void __launch_bounds__(256) denominators_kernel(const c128 *__restrict__ fock, int o, int v,
                                                           double *__restrict__ D) {
  const long nf = o + v, n1 = (long)o * v, oo = npair(o), n2 = npair(v) * oo;
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n1 + n2; i += (long)gridDim.x * blockDim.x) {
    double d;
    if (i < n1) {
      const long a = i / o, ii = i % o;
      d = fock[(o + a) * nf + (o + a)].x - fock[ii * nf + ii].x;
    } else {
      const long r = i - n1, ab = r / oo, ij = r % oo;
      long b = (long)((1.0 + sqrt(1.0 + 8.0 * (double)ab)) * 0.5);
      while (b * (b - 1) / 2 > ab) --b;
      while ((b + 1) * b / 2 <= ab) ++b;
      const long a = ab - b * (b - 1) / 2;
      long j = (long)((1.0 + sqrt(1.0 + 8.0 * (double)ij)) * 0.5);
      while (j * (j - 1) / 2 > ij) --j;
      while ((j + 1) * j / 2 <= ij) ++j;
      const long ii = ij - j * (j - 1) / 2;
      d = fock[(o + a) * nf + (o + a)].x + fock[(o + b) * nf + (o + b)].x - fock[ii * nf + ii].x - fock[j * nf + j].x;
    }
    D[i] = d;
  }
}

int stream_grid(long n) {
  long blocks = (n + 255) / 256;
  const long cap = (long)zgemm_num_sms() * 16;
  if (blocks > cap) blocks = cap;
  if (blocks < 1) blocks = 1;
  return (int)blocks;
}

int dot_chunks(long n) {
  long c = (n + 4095) / 4096;   // at least 4096 elements per chunk
  if (c > DOT_MAX_CHUNKS) c = DOT_MAX_CHUNKS;
  if (c < 1) c = 1;
  return (int)c;
}

}  // namespace

size_t dots_scratch_elems(int npairs) { return (size_t)npairs * DOT_MAX_CHUNKS; }

cudaError_t multi_dot(cudaStream_t st, const c128 *A, long lda, int na, const c128 *B, long ldb, int nb, long n,
                      bool conjA, bool diag, c128 *partial, c128 *out) {
  const int npairs = diag ? na : na * nb;
  if (npairs <= 0) return cudaSuccess;
  const int chunks = dot_chunks(n);
  const long chunk_len = (n + chunks - 1) / chunks;
  // blockIdx.y is limited to 65535 pairs per launch
  for (int p0 = 0; p0 < npairs; p0 += 32768) {
    const int np = npairs - p0 < 32768 ? npairs - p0 : 32768;
    if (!diag && p0 != 0) return cudaErrorInvalidValue;   // callers keep na*nb below the limit
    dim3 grid(chunks, np);
    const c128 *Ap = diag ? A + (size_t)p0 * lda : A, *Bp = diag ? B + (size_t)p0 * ldb : B;
    dot_partial_kernel<<<grid, DOT_THREADS, 0, st>>>(Ap, lda, Bp, ldb, nb, n, conjA ? 1 : 0, diag ? 1 : 0, chunk_len,
                                                     partial + (size_t)p0 * chunks);
    cclr_count_launch();
  }
  dot_final_kernel<<<(npairs + 127) / 128, 128, 0, st>>>(partial, chunks, npairs, out);
  cclr_count_launch();
  return cudaGetLastError();
}

cudaError_t lincomb(cudaStream_t st, c128 *y, c128 beta, const c128 *coef, const c128 *V, long ldv, int m, long n) {
  if (n <= 0) return cudaSuccess;
  if ((size_t)m * sizeof(c128) > 48 * 1024) return cudaErrorInvalidValue;
  lincomb_kernel<<<stream_grid(n), 256, (size_t)m * sizeof(c128), st>>>(y, beta, coef, V, ldv, m, n);
  cclr_count_launch();
  return cudaGetLastError();
}

cudaError_t precondition(cudaStream_t st, c128 *y, const c128 *x, const double *D, c128 z, c128 alpha, long n) {
  if (n <= 0) return cudaSuccess;
  precondition_kernel<<<stream_grid(n), 256, 0, st>>>(y, x, D, z, alpha, n);
  cclr_count_launch();
  return cudaGetLastError();
}

cudaError_t scale_vec(cudaStream_t st, c128 *y, c128 alpha, long n) {
  if (n <= 0) return cudaSuccess;
  scale_kernel<<<stream_grid(n), 256, 0, st>>>(y, alpha, n);
  cclr_count_launch();
  return cudaGetLastError();
}

cudaError_t denominators(cudaStream_t st, const c128 *fock, int o, int v, double *D) {
  const long n = (long)o * v + npair(o) * npair(v);
  denominators_kernel<<<stream_grid(n), 256, 0, st>>>(fock, o, v, D);
  cclr_count_launch();
  return cudaGetLastError();
}
