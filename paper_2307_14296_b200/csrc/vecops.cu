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

__global__ void __launch_bounds__(256) shifted_copy_kernel(c128 *__restrict__ out, const c128 *__restrict__ src, c128 alpha,
                                                           const c128 *__restrict__ x, long n) {
  for (long i = (long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long)gridDim.x * blockDim.x) {
    c128 acc = src[i];
    cfma(acc, alpha, x[i]);
    out[i] = acc;
  }
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

// Y[r][i] = xs * X[r][i] + sum_{j<m0} coef[r][j] V0[j][i] + sum_{j<m1} coef[r][m0+j] V1[j][i]   for r < R rows at once:
// every element of the m0 + m1 subspace vectors is read ONCE for all R outputs (the per-row kernel above reads them R times).
// This is the residual block r_k = xi + sum_j beta_kj (sigma_j - z_k b_j) (step 4), the solutions t_k = sum_j
// beta_kj b_j (step 5), the subspace collapse and the block Gram-Schmidt update of PAPER.md:966.  Fused outputs
// (each optional): nrm2[r] = sum_i |Y[r][i]|^2 (deterministic two-level reduction: per-CTA partials in fixed order), and the
// preconditioned vector P[r][i] = Y[r][i] / (z[r] - D[i]) -- residual, norm and correction in one pass.
constexpr int BL_JT = 32;   // coefficient tile (columns j) staged in shared memory
struct BlockLincombArgs {
  c128 *Y; long ldy;
  const c128 *X; long ldx; c128 xs;
  const c128 *coef; int ldc;               // device [R][ldc]
  const c128 *V0; long ldv0; int m0;
  const c128 *V1; long ldv1; int m1;
  long n;
  double *nrm_partial;                      // [gridDim.x][R] or null
  const double *D; const c128 *z;           // preconditioner (z: device [R]) or null
  c128 *P; long ldp;
};

template <int R, int BL_E>
__global__ void __launch_bounds__(256) block_lincomb_kernel(const BlockLincombArgs a) {
  __shared__ c128 cs[R][BL_JT];
  const int m = a.m0 + a.m1;
  double nr[R];
#pragma unroll
  for (int r = 0; r < R; ++r) nr[r] = 0.0;
  const long tile = 256L * BL_E;
  for (long t0 = (long)blockIdx.x * tile; t0 < a.n; t0 += (long)gridDim.x * tile) {
    c128 acc[R][BL_E];
    long idx[BL_E];
#pragma unroll
    for (int e = 0; e < BL_E; ++e) {
      idx[e] = t0 + e * 256 + threadIdx.x;
#pragma unroll
      for (int r = 0; r < R; ++r)
        acc[r][e] = (a.X && idx[e] < a.n) ? cmul(a.xs, a.X[(size_t)r * a.ldx + idx[e]]) : czero();
    }
    for (int j0 = 0; j0 < m; j0 += BL_JT) {
      __syncthreads();
      for (int q = threadIdx.x; q < R * BL_JT; q += 256) {
        const int r = q / BL_JT, j = j0 + q % BL_JT;
        cs[r][q % BL_JT] = j < m ? a.coef[(size_t)r * a.ldc + j] : czero();
      }
      __syncthreads();
      const int jn = m - j0 < BL_JT ? m - j0 : BL_JT;
#pragma unroll 4
      for (int jj = 0; jj < jn; ++jj) {
        const int j = j0 + jj;
        const c128 *vrow = j < a.m0 ? a.V0 + (size_t)j * a.ldv0 : a.V1 + (size_t)(j - a.m0) * a.ldv1;
        c128 v[BL_E];
#pragma unroll
        for (int e = 0; e < BL_E; ++e) v[e] = idx[e] < a.n ? vrow[idx[e]] : czero();
#pragma unroll
        for (int r = 0; r < R; ++r) {
          const c128 c = cs[r][jj];
#pragma unroll
          for (int e = 0; e < BL_E; ++e) cfma(acc[r][e], c, v[e]);
        }
      }
    }
#pragma unroll
    for (int e = 0; e < BL_E; ++e) {
      if (idx[e] >= a.n) continue;
      const double d = a.P ? a.D[idx[e]] : 0.0;
#pragma unroll
      for (int r = 0; r < R; ++r) {
        const c128 y = acc[r][e];
        a.Y[(size_t)r * a.ldy + idx[e]] = y;
        nr[r] += y.x * y.x + y.y * y.y;
        if (a.P) {
          const c128 z = a.z[r];
          const double dr = z.x - d, di = z.y, inv = 1.0 / (dr * dr + di * di);
          a.P[(size_t)r * a.ldp + idx[e]] = make_double2((y.x * dr + y.y * di) * inv, (y.y * dr - y.x * di) * inv);
        }
      }
    }
  }
  if (a.nrm_partial) {
    __shared__ double red[R][8];
#pragma unroll
    for (int r = 0; r < R; ++r) {
      double w = nr[r];
#pragma unroll
      for (int s = 16; s > 0; s >>= 1) w += __shfl_xor_sync(0xffffffffu, w, s);
      if ((threadIdx.x & 31) == 0) red[r][threadIdx.x >> 5] = w;
    }
    __syncthreads();
    if (threadIdx.x < R) {
      double w = 0.0;
      for (int k = 0; k < 8; ++k) w += red[threadIdx.x][k];
      a.nrm_partial[(size_t)blockIdx.x * R + threadIdx.x] = w;
    }
  }
}

__global__ void block_norm_final_kernel(const double *__restrict__ partial, int nblocks, int R, double *__restrict__ out) {
  const int r = threadIdx.x;
  if (r >= R) return;
  double s = 0.0;
  for (int b = 0; b < nblocks; ++b) s += partial[(size_t)b * R + r];
  out[r] = s;
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
  // blockIdx.y is limited to 65535: launch in slabs of at most 32768 (ia, ib) pairs -- whole rows ia of the pair matrix in the
  // general case, consecutive pairs in the diagonal case; every slab writes its partial sums at its own offset
  if (!diag && nb > 32768) return cudaErrorInvalidValue;
  const int rows_per = diag ? 32768 : (32768 / nb > 0 ? 32768 / nb : 1);
  for (int r0 = 0; r0 < na; r0 += rows_per) {
    const int nr = na - r0 < rows_per ? na - r0 : rows_per;
    const int np = diag ? nr : nr * nb;
    const size_t p0 = diag ? (size_t)r0 : (size_t)r0 * nb;
    dim3 grid(chunks, np);
    dot_partial_kernel<<<grid, DOT_THREADS, 0, st>>>(A + (size_t)r0 * lda, lda, diag ? B + (size_t)r0 * ldb : B, ldb, nb, n,
                                                     conjA ? 1 : 0, diag ? 1 : 0, chunk_len, partial + p0 * chunks);
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

// out[0] += sum_i |s_i - D_i b_i|^2 : the part of a sigma vector that does not come from the orbital-energy diagonal (what the
// contractions contribute; the solver scales its error estimate of reduced-precision sigma vectors with it).  out zeroed by the caller.
__global__ void __launch_bounds__(256) offdiag_norm2_kernel(const c128 *__restrict__ s, const c128 *__restrict__ b,
                                                            const double *__restrict__ D, long n, double *out) {
  double acc = 0.0;
  for (long i = (long)blockIdx.x * 256 + threadIdx.x; i < n; i += (long)gridDim.x * 256) {
    const c128 sv = s[i], bv = b[i];
    const double d = D[i], re = sv.x - d * bv.x, im = sv.y - d * bv.y;
    acc += re * re + im * im;
  }
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  __shared__ double red[8];
  if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    for (int w = 1; w < 8; ++w) acc += red[w];
    atomicAdd(out, acc);
  }
}
cudaError_t offdiag_norm2(cudaStream_t st, const c128 *s, const c128 *b, const double *D, long n, double *out) {
  if (n <= 0) return cudaSuccess;
  offdiag_norm2_kernel<<<stream_grid(n), 256, 0, st>>>(s, b, D, n, out);
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

static int block_lincomb_e(int R) { return R <= 4 ? 4 : 2; }   // elements per thread: more loads in flight when few accumulators

int block_lincomb_grid(long n) {
  long tiles = (n + 511) / 512;
  const long cap = (long)zgemm_num_sms() * 8;
  if (tiles > cap) tiles = cap;
  if (tiles < 1) tiles = 1;
  return (int)tiles;
}

// see block_lincomb_kernel; R <= BLOCK_LINCOMB_MAX rows per call; nrm2 (device [R]) / nrm_scratch (device, block_lincomb_grid(n) * R
// doubles) and D / z / P are optional (null)
cudaError_t block_lincomb(cudaStream_t st, int R, c128 *Y, long ldy, const c128 *X, long ldx, c128 xs, const c128 *coef, int ldc,
                          const c128 *V0, long ldv0, int m0, const c128 *V1, long ldv1, int m1, long n, double *nrm2,
                          double *nrm_scratch, const double *D, const c128 *z, c128 *P, long ldp) {
  if (n <= 0 || R <= 0) return cudaSuccess;
  if (R > BLOCK_LINCOMB_MAX) return cudaErrorInvalidValue;
  BlockLincombArgs a{Y, ldy, X, ldx, xs, coef, ldc, V0, ldv0, m0, V1, ldv1, m1, n, nrm2 ? nrm_scratch : nullptr, D, z, P, ldp};
  int grid = block_lincomb_grid(n);
  const long tiles = (n + 256L * block_lincomb_e(R) - 1) / (256L * block_lincomb_e(R));
  if (grid > tiles) grid = (int)tiles;
  switch (R) {
    case 1: block_lincomb_kernel<1, 4><<<grid, 256, 0, st>>>(a); break;
    case 2: block_lincomb_kernel<2, 4><<<grid, 256, 0, st>>>(a); break;
    case 3: block_lincomb_kernel<3, 4><<<grid, 256, 0, st>>>(a); break;
    case 4: block_lincomb_kernel<4, 4><<<grid, 256, 0, st>>>(a); break;
    case 5: block_lincomb_kernel<5, 2><<<grid, 256, 0, st>>>(a); break;
    case 6: block_lincomb_kernel<6, 2><<<grid, 256, 0, st>>>(a); break;
    case 7: block_lincomb_kernel<7, 2><<<grid, 256, 0, st>>>(a); break;
    default: block_lincomb_kernel<8, 2><<<grid, 256, 0, st>>>(a); break;
  }
  cclr_count_launch();
  if (nrm2) {
    block_norm_final_kernel<<<1, 32, 0, st>>>(nrm_scratch, grid, R, nrm2);
    cclr_count_launch();
  }
  return cudaGetLastError();
}

cudaError_t shifted_copy(cudaStream_t st, c128 *out, const c128 *src, c128 alpha, const c128 *x, long n) {
  if (n <= 0) return cudaSuccess;
  shifted_copy_kernel<<<stream_grid(n), 256, 0, st>>>(out, src, alpha, x, n);
  cclr_count_launch();
  return cudaGetLastError();
}

// ---- cclr_property_noalloc: the property contraction without a context and without any allocation (include/cclr.h) ----------
// Callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid it) get the
// partial-sum scratch of the two-pass dot from this file-scope device array instead of a context's heap buffer: 2 (singles,
// doubles) x CCLR_NOALLOC_MAX_VECS pairs x DOT_MAX_CHUNKS partial sums = 151,552 bytes, held by every GPU that loads the
// library until the process exits.  Every call shares it: calls that overlap on the GPU (two streams, two threads) race.
// Nothing in it has to start at zero -- dot_partial_kernel writes every slot dot_final reads -- so stale contents are harmless.
#include "../../include/cclr.h"
#include <mutex>
#include <string>

void cclr_set_error(const std::string &msg, cudaError_t e);   // context.cu

static __device__ __align__(256) c128 g_noalloc_scratch[2 * CCLR_NOALLOC_MAX_VECS * DOT_MAX_CHUNKS];

namespace {

// out[k] = (sum_c p1[k][c]) + (sum_c p2[k][c]): the same two fixed-order sums cclr_property forms, added in the same order
__global__ void noalloc_final_kernel(const c128 *__restrict__ p1, int c1, const c128 *__restrict__ p2, int c2, int nvec,
                                     c128 *__restrict__ out) {
  const int k = blockIdx.x * blockDim.x + threadIdx.x;
  if (k >= nvec) return;
  c128 s1 = czero(), s2 = czero();
  for (int c = 0; c < c1; ++c) s1 = cadd(s1, p1[(size_t)k * c1 + c]);
  for (int c = 0; c < c2; ++c) s2 = cadd(s2, p2[(size_t)k * c2 + c]);
  out[k] = cadd(s1, s2);
}

// device address of g_noalloc_scratch, looked up once per device with that device current (in host code the array's name is a
// host-side stand-in, not a device address)
cudaError_t noalloc_scratch_address(c128 **ptr) {
  static std::mutex mu;
  static c128 *addr[64] = {};
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  std::lock_guard<std::mutex> lock(mu);
  if (dev >= 0 && dev < 64 && addr[dev]) { *ptr = addr[dev]; return cudaSuccess; }
  void *p = nullptr;
  e = cudaGetSymbolAddress(&p, g_noalloc_scratch);
  if (e != cudaSuccess) return e;
  if (dev >= 0 && dev < 64) addr[dev] = (c128 *)p;
  *ptr = (c128 *)p;
  return cudaSuccess;
}

}  // namespace

extern "C" int cclr_property_noalloc(void *cuda_stream, const cclr_c128 *eta1, const cclr_c128 *eta2, const cclr_c128 *x1,
                                     const cclr_c128 *x2, long n1, long n2, int nvec, cclr_c128 *result) {
  if (!eta1 || !eta2 || !x1 || !x2 || !result || n1 < 1 || n2 < 1 || nvec < 1) {
    cclr_set_error("cclr_property_noalloc: null pointer, n1 < 1, n2 < 1 or nvec < 1", cudaSuccess);
    return CCLR_EINVAL;
  }
  if (nvec > CCLR_NOALLOC_MAX_VECS) {
    cclr_set_error("cclr_property_noalloc: nvec exceeds CCLR_NOALLOC_MAX_VECS (" + std::to_string(CCLR_NOALLOC_MAX_VECS) +
                       "), the size of the static scratch; split the call or use cclr_property",
                   cudaSuccess);
    return CCLR_EINVAL;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  c128 *scratch = nullptr;
  cudaError_t e = noalloc_scratch_address(&scratch);
  if (e != cudaSuccess) {
    cclr_set_error(std::string("cclr_property_noalloc: cudaGetSymbolAddress: ") + cudaGetErrorString(e), e);
    return CCLR_ECUDA;
  }
  c128 *p1 = scratch, *p2 = scratch + (size_t)CCLR_NOALLOC_MAX_VECS * DOT_MAX_CHUNKS;
  const int c1 = dot_chunks(n1), c2 = dot_chunks(n2);
  dot_partial_kernel<<<dim3(c1, nvec), DOT_THREADS, 0, st>>>((const c128 *)eta1, n1, (const c128 *)x1, n1, nvec, n1, 0, 0,
                                                             (n1 + c1 - 1) / c1, p1);
  dot_partial_kernel<<<dim3(c2, nvec), DOT_THREADS, 0, st>>>((const c128 *)eta2, n2, (const c128 *)x2, n2, nvec, n2, 0, 0,
                                                             (n2 + c2 - 1) / c2, p2);
  noalloc_final_kernel<<<1, 32, 0, st>>>(p1, c1, p2, c2, nvec, (c128 *)result);
  cclr_count_launch(3);
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    cclr_set_error(std::string("cclr_property_noalloc: ") + cudaGetErrorString(e), e);
    return CCLR_ECUDA;
  }
  return CCLR_OK;
}
