// layout.cu — the five hot layout kernels of one sigma evaluation (SURVEY 8(a)B "layout", "shift"), specialised.
//
// The generic gather kernel of permute.cu decodes every element's indices (divisions, a sqrt per packed pair) and is
// instruction bound at ~0.3 of the HBM copy rate.  The five statements below run once per trial vector and move 90 % of
// sigma's layout bytes, so each gets a kernel whose index work is done once per ROW of the packed pair axis:
//   unpack_rows     Ur[e][a][(ij)]   =  x2[(ea)][(ij)]                     sign / pair index per row, then a row copy
//   unpack_cols     Xo[(ab)][i][n]   =  x2[(ab)][(in)]                     row staged in shared memory, o x o signed gather
//   unpack_ring     R[a][i][e][m]    =  x2[(ae)][(im)]                     same, written as runs of o elements to (a,e) and (e,a)
//   transpose_pair  Xt[i][m][(ef)]   =  x2[(ef)][(im)]                     32 x 32 shared-memory tile transpose
//   final_pack      out2[(ab)][(ij)] += -z x2 + P(ab) Y + P(ij) Q + P(ab)P(ij) Z     (the antisymmetrised packing and the shift)
// plan.cu recognises the statements by their index specs and routes them here; everything else stays with permute.cu.
#include "common.cuh"
#include <atomic>

namespace {

__device__ __forceinline__ c128 csign(c128 x, int s) { return s > 0 ? x : make_double2(-x.x, -x.y); }

// dst[p][q][0:len] = sign(p,q) * src[P(min,max)][0:len], zero rows for p = q.  One warp per destination row.
__global__ void __launch_bounds__(256) unpack_rows_kernel(const c128 *__restrict__ src, c128 *__restrict__ dst, int n, long len) {
  const int lane = threadIdx.x & 31;
  const long row = (long)blockIdx.x * 8 + (threadIdx.x >> 5);
  if (row >= (long)n * n) return;
  const int p = (int)(row / n), q = (int)(row % n);
  c128 *d = dst + row * len;
  if (p == q) {
    for (long k = lane; k < len; k += 32) d[k] = czero();
    return;
  }
  const long lo = p < q ? p : q, hi = p < q ? q : p;
  const c128 *s = src + (hi * (hi - 1) / 2 + lo) * len;
  const int sg = p < q ? 1 : -1;
  for (long k = lane; k < len; k += 32) d[k] = csign(s[k], sg);
}

// dst[r][i][n] = sign(i,n) * src[r][P(i,n)] for every packed row r (o x o block per row).  One warp per row.
__global__ void __launch_bounds__(256) unpack_cols_kernel(const c128 *__restrict__ src, c128 *__restrict__ dst, long rows, int o) {
  // (8 warps per block when 8 rows fit the default 48 KB of shared memory, fewer otherwise)
  extern __shared__ c128 sm[];                       // (warps per block) x oo
  const int oo = o * (o - 1) / 2, lane = threadIdx.x & 31, w = threadIdx.x >> 5;
  const long row = (long)blockIdx.x * (blockDim.x >> 5) + w;
  if (row >= rows) return;
  c128 *buf = sm + (size_t)w * oo;
  const c128 *s = src + row * oo;
  for (int k = lane; k < oo; k += 32) buf[k] = s[k];
  __syncwarp();
  c128 *d = dst + row * (long)o * o;
  for (int t = lane; t < o * o; t += 32) {
    const int i = t / o, m = t - i * o;
    c128 x = czero();
    if (i != m) {
      const int lo = i < m ? i : m, hi = i < m ? m : i;
      x = csign(buf[hi * (hi - 1) / 2 + lo], i < m ? 1 : -1);
    }
    d[t] = x;
  }
}

// R[a][i][e][m] = x2[(ae)][(im)]: one block per ordered pair (a, e): the row of (a<e or e<a) is staged once, then written as o runs
// of o elements (i fixed, m contiguous); a = e gives zero runs.
__global__ void __launch_bounds__(128) unpack_ring_kernel(const c128 *__restrict__ src, c128 *__restrict__ dst, int v, int o) {
  extern __shared__ c128 sm[];                       // oo
  const int oo = o * (o - 1) / 2;
  const int a = blockIdx.x / v, e = blockIdx.x % v;
  const int sab = a < e ? 1 : -1;
  if (a != e) {
    const long lo = a < e ? a : e, hi = a < e ? e : a;
    const c128 *s = src + (hi * (hi - 1) / 2 + lo) * oo;
    for (int k = threadIdx.x; k < oo; k += blockDim.x) sm[k] = s[k];
  }
  __syncthreads();
  for (int t = threadIdx.x; t < o * o; t += blockDim.x) {
    const int i = t / o, m = t - i * o;
    c128 x = czero();
    if (a != e && i != m) {
      const int lo = i < m ? i : m, hi = i < m ? m : i;
      x = csign(sm[hi * (hi - 1) / 2 + lo], (i < m ? 1 : -1) * sab);
    }
    dst[(((long)a * o + i) * v + e) * o + m] = x;
  }
}

// dst[i][m][c] = sign(i,m) * src[c][P(i,m)] (c < ncol): 32 x 32 tile transpose through shared memory; the tiles of the first
// column block also clear the rows (i,i).
__global__ void __launch_bounds__(256) transpose_pair_kernel(const c128 *__restrict__ src, c128 *__restrict__ dst, long ncol, int o) {
  __shared__ c128 tile[32][33];
  __shared__ int pi[32], pm[32];
  const int oo = o * (o - 1) / 2;
  const long c0 = (long)blockIdx.x * 32;
  const int p0 = blockIdx.y * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;          // 32 x 8
  if (threadIdx.x < 32) {
    const int p = p0 + threadIdx.x;
    int q = (int)((1.0 + sqrt(1.0 + 8.0 * (double)p)) * 0.5);
    while (q * (q - 1) / 2 > p) --q;
    while ((q + 1) * q / 2 <= p) ++q;
    pi[threadIdx.x] = p - q * (q - 1) / 2;
    pm[threadIdx.x] = q;
  }
  for (int r = ty; r < 32; r += 8) {
    const long c = c0 + r;
    const int p = p0 + tx;
    tile[r][tx] = (c < ncol && p < oo) ? src[c * oo + p] : czero();
  }
  __syncthreads();
  for (int r = ty; r < 32; r += 8) {                                 // r indexes the pair inside the tile, tx the column c
    const int p = p0 + r;
    const long c = c0 + tx;
    if (p < oo && c < ncol) {
      const c128 x = tile[tx][r];
      const int i = pi[r], m = pm[r];
      dst[((long)i * o + m) * ncol + c] = x;
      dst[((long)m * o + i) * ncol + c] = make_double2(-x.x, -x.y);
    }
  }
  if (blockIdx.y == 0)
    for (int i = ty; i < o; i += 8) {
      const long c = c0 + tx;
      if (c < ncol) dst[((long)i * o + i) * ncol + c] = czero();
    }
}

// out2[(ab)][(ij)] += nz * x2[(ab)][(ij)] + Y[a][b][(ij)] - Y[b][a][(ij)] + Q[(ab)][i][j] - Q[(ab)][j][i]
//                     + Z[b][j][a][i] - Z[a][j][b][i] - Z[b][i][a][j] + Z[a][i][b][j]
// One block per packed row (ab): the Q row and the two o x o slabs of Z it needs are staged in shared memory (runs of o
// contiguous elements), then the oo outputs are formed with the pair (i<j) decoded incrementally.
__global__ void __launch_bounds__(128) final_pack_kernel(c128 *__restrict__ out2, const c128 *__restrict__ x2, c128 nz,
                                                         const c128 *__restrict__ Y, const c128 *__restrict__ Q,
                                                         const c128 *__restrict__ Z, int v, int o) {
  extern __shared__ c128 sm[];                       // Q row [o*o], Zba [o*o], Zab [o*o]
  const int oo = o * (o - 1) / 2, o2 = o * o;
  c128 *q = sm, *zba = sm + o2, *zab = sm + 2 * o2;
  const long ab = blockIdx.x;
  int b = (int)((1.0 + sqrt(1.0 + 8.0 * (double)ab)) * 0.5);
  while ((long)b * (b - 1) / 2 > ab) --b;
  while ((long)(b + 1) * b / 2 <= ab) ++b;
  const int a = (int)(ab - (long)b * (b - 1) / 2);
  const c128 *qs = Q + ab * o2;
  for (int t = threadIdx.x; t < o2; t += blockDim.x) {
    const int j = t / o, i = t - j * o;
    q[t] = qs[t];
    zba[t] = Z[(((long)b * o + j) * v + a) * o + i];               // [j][i]
    zab[t] = Z[(((long)a * o + j) * v + b) * o + i];
  }
  __syncthreads();
  const c128 *yab = Y + ((long)a * v + b) * oo, *yba = Y + ((long)b * v + a) * oo;
  const c128 *xr = x2 + ab * oo;
  c128 *dr = out2 + ab * oo;
  for (int p = threadIdx.x; p < oo; p += blockDim.x) {
    int j = (int)((1.0f + sqrtf(1.0f + 8.0f * (float)p)) * 0.5f);
    while (j * (j - 1) / 2 > p) --j;
    while ((j + 1) * j / 2 <= p) ++j;
    const int i = p - j * (j - 1) / 2;
    const c128 x = xr[p], y1 = yab[p], y2 = yba[p], old = dr[p];
    const int ij = i * o + j, ji = j * o + i;
    double re = old.x + nz.x * x.x - nz.y * x.y + y1.x - y2.x + q[ij].x - q[ji].x + zba[ji].x - zab[ji].x - zba[ij].x + zab[ij].x;
    double im = old.y + nz.x * x.y + nz.y * x.x + y1.y - y2.y + q[ij].y - q[ji].y + zba[ji].y - zab[ji].y - zba[ij].y + zab[ij].y;
    dr[p] = make_double2(re, im);
  }
}

}  // namespace

cudaError_t layout_unpack_rows(cudaStream_t st, const c128 *src, c128 *dst, int n, long len) {
  const long rows = (long)n * n;
  unpack_rows_kernel<<<(unsigned)((rows + 7) / 8), 256, 0, st>>>(src, dst, n, len);
  cclr_count_launch();
  return cudaGetLastError();
}

cudaError_t layout_unpack_cols(cudaStream_t st, const c128 *src, c128 *dst, long rows, int o) {
  const size_t row_bytes = (size_t)(o * (o - 1) / 2) * sizeof(c128);
  int wpb = (int)((48 * 1024) / (row_bytes ? row_bytes : 1));
  if (wpb > 8) wpb = 8;
  if (wpb < 1) return cudaErrorInvalidValue;
  unpack_cols_kernel<<<(unsigned)((rows + wpb - 1) / wpb), 32 * wpb, wpb * row_bytes, st>>>(src, dst, rows, o);
  cclr_count_launch();
  return cudaGetLastError();
}

cudaError_t layout_unpack_ring(cudaStream_t st, const c128 *src, c128 *dst, int v, int o) {
  const size_t smem = (size_t)(o * (o - 1) / 2) * sizeof(c128);
  if (smem > 48 * 1024) return cudaErrorInvalidValue;
  unpack_ring_kernel<<<(unsigned)(v * v), 128, smem, st>>>(src, dst, v, o);
  cclr_count_launch();
  return cudaGetLastError();
}

cudaError_t layout_transpose_pair(cudaStream_t st, const c128 *src, c128 *dst, long ncol, int o) {
  const int oo = o * (o - 1) / 2;
  dim3 grid((unsigned)((ncol + 31) / 32), (unsigned)((oo + 31) / 32));
  transpose_pair_kernel<<<grid, 256, 0, st>>>(src, dst, ncol, o);
  cclr_count_launch();
  return cudaGetLastError();
}

cudaError_t layout_final_pack(cudaStream_t st, c128 *out2, const c128 *x2, c128 nz, const c128 *Y, const c128 *Q, const c128 *Z,
                              int v, int o) {
  const size_t smem = (size_t)3 * o * o * sizeof(c128);
  const long vv = (long)v * (v - 1) / 2;
  static std::atomic<unsigned long long> configured{0};
  if (smem > 48 * 1024) {
    int dev = 0;
    cudaGetDevice(&dev);
    if (dev >= 64 || !((configured.load() >> dev) & 1ull)) {
      cudaError_t e = cudaFuncSetAttribute(final_pack_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
      if (e != cudaSuccess) return e;
      if (dev < 64) configured.fetch_or(1ull << dev);
    }
  }
  final_pack_kernel<<<(unsigned)vv, 128, smem, st>>>(out2, x2, nz, Y, Q, Z, v, o);
  cclr_count_launch();
  return cudaGetLastError();
}
