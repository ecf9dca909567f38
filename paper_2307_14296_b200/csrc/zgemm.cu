// zgemm.cu — complex128 GEMM on the FP64 tensor cores of sm_100a.
//
//   C[M][N] = alpha * opA(A)[M][K] * opB(B)[K][N] + beta * C
//
// This is the contraction engine behind every dense term of the CC-LR sigma vector (S-Eq. 11-12)
// and of the intermediates (S-Eq. 15-25): pp ladder, ring, hole ladder, W/F builds.
//
// Design (B200):
//   * sm_100a has no FP64 kind in tcgen05; the FP64 tensor path is warp-level DMMA (mma.sync m8n8k4 f64).  Measured
//     issue-rate peak on B200: 36.9 TFLOP/s (profiles/r01_fp64_peak.md).
//   * 4M complex product without expanding any operand in memory: per complex k, a lane holds a = A[m][k] and
//     b = B[k][n]; the 8 real columns of one DMMA are 4 complex columns x {re, im}, so
//         acc += a.re * (parity ? b.im :  b.re)      acc += a.im * (parity ? b.re : -b.im)
//     where parity = "this lane feeds an imaginary output column".  conj(A)/conj(B) only flip sign bits.
//     The C fragment of m8n8k4 (row g, real columns 2t, 2t+1) is then exactly one complex number per lane.
//   * operands are staged by TMA (cp.async.bulk.tensor, FLOAT64 tensor maps over the interleaved data, boxes of
//     128 B x rows, SWIZZLE_128B) into a STAGES-deep ring guarded by full/empty mbarriers; one producer warp,
//     (BM/WM)*(BN/WN) consumer warps.  Fragment loads are single conflict-free LDS.128 per complex element:
//       - K-contiguous operand rows: the 8 rows a quarter-warp touches are permuted (rmap) so the two rows of a
//         quarter-warp differ in address bit 9 and the swizzle separates them;
//       - N-contiguous B ([K][N]): the four k rows of a quarter-warp are separated by the swizzle directly.
//   * ragged M, N, K: TMA zero-fills out-of-bounds loads; stores are guarded.
//   * optional split-K (partials in a workspace + a deterministic reduce kernel) for tall-K / tiny-MN contractions.
#include "common.cuh"
#include <mutex>

namespace {

// ---------------------------------------------------------------------------------------------------------------
// PTX wrappers
// ---------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done;
  do {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  } while (!done);
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
      ::"r"(dst), "l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
      : "memory");
}
__device__ __forceinline__ void dmma884(double &c0, double &c1, double a, double b) {
  asm("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
               : "+d"(c0), "+d"(c1)
               : "d"(a), "d"(b));
}
__device__ __forceinline__ double2 lds128(uint32_t addr) {
  double2 v;
  asm volatile("ld.shared.v2.f64 {%0,%1}, [%2];" : "=d"(v.x), "=d"(v.y) : "r"(addr));
  return v;
}
__device__ __forceinline__ double flip_sign(double x, uint32_t mask) {
  return __hiloint2double(__double2hiint(x) ^ (int)mask, __double2loint(x));
}

struct ZgemmArgs {
  int M, N, K;
  c128 *C;
  long ldc, sc;
  c128 alpha, beta;
  int conjA, conjB;
  int splits;          // >= 1
  int chunks_per_split;
  c128 *partial;       // [batch*splits][M][N] when splits > 1
};

// ---------------------------------------------------------------------------------------------------------------
// kernel
// ---------------------------------------------------------------------------------------------------------------
template <int BM, int BN, int BK, int WM, int WN, int STAGES, bool BKN>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32 + 128, 1)
zgemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const ZgemmArgs p) {
  constexpr int WARPS_M = BM / WM, WARPS_N = BN / WN, NCW = WARPS_M * WARPS_N;
  constexpr int MI = WM / 8, NG = WN / 4;          // DMMA tiles per warp: MI row groups x NG column groups
  constexpr int A_BYTES = BM * BK * 16, B_BYTES = BN * BK * 16, STAGE_BYTES = A_BYTES + B_BYTES;
  static_assert(BK % 8 == 0 && BM % 8 == 0 && BN % 8 == 0 && WM % 8 == 0 && WN % 8 == 0, "tile shape");
  static_assert(NCW % 4 == 0, "consumer warps must form whole warpgroups (setmaxnreg)");
  constexpr int CONSUMER_REGS = (NCW == 8) ? 232 : 200;

  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte alignment is required by SWIZZLE_128B; dynamic smem base is only guaranteed 16 B, so align by hand.
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;   // full[STAGES], empty[STAGES], 8 B each

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tile_n = blockIdx.x, tile_m = blockIdx.y;
  const int batch = blockIdx.z / p.splits, split = blockIdx.z % p.splits;
  const int nchunks_total = (p.K + BK - 1) / BK;
  const int chunk0 = split * p.chunks_per_split;
  int nchunks = nchunks_total - chunk0;
  if (nchunks > p.chunks_per_split) nchunks = p.chunks_per_split;
  if (nchunks < 0) nchunks = 0;

  if (threadIdx.x == 0) {
    for (int s = 0; s < STAGES; ++s) {
      mbar_init(bar_base + 8 * s, 1);                 // full: one arrive (the producer's expect_tx) + tx bytes
      mbar_init(bar_base + 8 * (STAGES + s), NCW);    // empty: one arrive per consumer warp
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();

  if (warp >= NCW) {
    // ===== producer warpgroup: gives its registers to the consumers; one elected lane drives TMA =====
    asm volatile("setmaxnreg.dec.sync.aligned.u32 40;");
    if (warp == NCW && lane == 0) {
      for (int c = 0; c < nchunks; ++c) {
        const int s = c % STAGES;
        const uint32_t ph = (c / STAGES) & 1;
        mbar_wait(bar_base + 8 * (STAGES + s), ph ^ 1);
        const uint32_t full = bar_base + 8 * s;
        mbar_expect_tx(full, STAGE_BYTES);
        const uint32_t sA = smem_base + s * STAGE_BYTES, sB = sA + A_BYTES;
        const int k0 = (chunk0 + c) * BK;
#pragma unroll
        for (int kb = 0; kb < BK / 8; ++kb)   // A boxes: [BM rows][8 complex]
          tma_load_3d(sA + kb * (BM * 128), &tmA, 2 * (k0 + kb * 8), tile_m * BM, batch, full);
        if (!BKN) {
#pragma unroll
          for (int kb = 0; kb < BK / 8; ++kb) // B boxes: [BN rows][8 complex]
            tma_load_3d(sB + kb * (BN * 128), &tmB, 2 * (k0 + kb * 8), tile_n * BN, batch, full);
        } else {
#pragma unroll
          for (int nb = 0; nb < BN / 8; ++nb) // B boxes: [BK rows][8 complex]
            tma_load_3d(sB + nb * (BK * 128), &tmB, 2 * (tile_n * BN + nb * 8), k0, batch, full);
        }
      }
    }
    return;
  }

  // ===== consumers =====
  asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(CONSUMER_REGS));
  const int gid = lane >> 2, tig = lane & 3;
  const int rmap = ((gid & 1) << 2) | (gid >> 1);   // row permutation inside an 8-row group (bank-conflict free)
  const int par = gid & 1, nb4 = gid >> 1;
  const int wm = warp / WARPS_N, wn = warp % WARPS_N;
  // sign masks (see header comment): f1 = m1 ^ (par ? b.im : b.re), f2 = m2 ^ (par ? b.re : b.im)
  const uint32_t sa = p.conjA ? 0x80000000u : 0u, sb = p.conjB ? 0x80000000u : 0u;
  const uint32_t m1 = par ? sb : 0u;
  const uint32_t m2 = par ? sa : (0x80000000u ^ sa ^ sb);

  // per-lane byte offsets inside one 8-complex box, for the two k4 steps (k = 4*s4 + tig)
  uint32_t a_off[2], b_off[2];
#pragma unroll
  for (int s4 = 0; s4 < 2; ++s4) {
    const int k = 4 * s4 + tig;
    a_off[s4] = (uint32_t)((wm * WM + rmap) * 128 + ((k ^ rmap) << 4));
    if (!BKN) {
      // row n = wn*WN + 4g + nb4 ; (n & 7) = ((g & 1) << 2) | nb4 -> handled per g below
      b_off[s4] = (uint32_t)((wn * WN + nb4) * 128 + (k << 4));
    } else {
      // row k (inside a box of BK rows: + kb*8*128 per 8-k block), col n = wn*WN + 4g + nb4
      b_off[s4] = (uint32_t)(k * 128);
    }
  }

  double acc[MI][NG][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int g = 0; g < NG; ++g) acc[i][g][0] = acc[i][g][1] = 0.0;

  for (int c = 0; c < nchunks; ++c) {
    const int s = c % STAGES;
    const uint32_t ph = (c / STAGES) & 1;
    mbar_wait(bar_base + 8 * s, ph);
    const uint32_t sA = smem_base + s * STAGE_BYTES, sB = sA + A_BYTES;
#pragma unroll
    for (int kb = 0; kb < BK / 8; ++kb) {
#pragma unroll
      for (int s4 = 0; s4 < 2; ++s4) {
        double2 a[MI];
#pragma unroll
        for (int i = 0; i < MI; ++i) a[i] = lds128(sA + kb * (BM * 128) + a_off[s4] + i * 1024);
#pragma unroll
        for (int g = 0; g < NG; ++g) {
          uint32_t addr;
          if (!BKN) {
            const int n7 = ((g & 1) << 2) | nb4;
            addr = sB + kb * (BN * 128) + g * 512 + (b_off[s4] ^ (uint32_t)(n7 << 4));
          } else {
            const int n = wn * WN + 4 * g + nb4;
            const int k7 = 4 * s4 + tig;
            addr = sB + (n >> 3) * (BK * 128) + kb * 1024 + b_off[s4] + (uint32_t)((((n & 7) ^ k7)) << 4);
          }
          const double2 b = lds128(addr);
          const double f1 = flip_sign(par ? b.y : b.x, m1);
          const double f2 = flip_sign(par ? b.x : b.y, m2);
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][g][0], acc[i][g][1], a[i].x, f1);
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][g][0], acc[i][g][1], a[i].y, f2);
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + s));
  }

  // ===== epilogue =====
  const bool partial = p.splits > 1;
  c128 *Cb = partial ? p.partial + (size_t)blockIdx.z * (size_t)p.M * (size_t)p.N : p.C + (size_t)batch * p.sc;
  const long ldc = partial ? (long)p.N : p.ldc;
  const c128 alpha = partial ? make_double2(1.0, 0.0) : p.alpha;
  const c128 beta = partial ? make_double2(0.0, 0.0) : p.beta;
  const bool has_beta = (beta.x != 0.0) || (beta.y != 0.0);
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    const int row = tile_m * BM + wm * WM + i * 8 + rmap;
    if (row >= p.M) continue;
#pragma unroll
    for (int g = 0; g < NG; ++g) {
      const int col = tile_n * BN + wn * WN + g * 4 + tig;
      if (col >= p.N) continue;
      c128 *dst = Cb + (size_t)row * ldc + col;
      c128 r = cmul(alpha, make_double2(acc[i][g][0], acc[i][g][1]));
      if (has_beta) {
        const c128 old = *dst;
        r = cadd(r, cmul(beta, old));
      }
      *dst = r;
    }
  }
}

// C = alpha * sum_s partial[s] + beta * C
__global__ void zgemm_reduce_kernel(const c128 *__restrict__ partial, int splits, int M, int N, c128 alpha, c128 beta,
                                    c128 *C, long ldc, long sc, int batch) {
  const size_t mn = (size_t)M * N;
  const size_t total = mn * batch;
  for (size_t idx = blockIdx.x * (size_t)blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
    const size_t b = idx / mn, r = idx % mn;
    const size_t row = r / N, col = r % N;
    c128 s = czero();
    for (int k = 0; k < splits; ++k) s = cadd(s, partial[(b * splits + k) * mn + r]);
    c128 *dst = C + b * sc + row * ldc + col;
    c128 out = cmul(alpha, s);
    if (beta.x != 0.0 || beta.y != 0.0) out = cadd(out, cmul(beta, *dst));
    *dst = out;
  }
}

// ---------------------------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------------------------
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn get_encode() {
  static EncodeTiledFn fn = nullptr;
  static std::once_flag once;
  std::call_once(once, [] {
    void *ptr = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)ptr;
  });
  return fn;
}

// tensor map over a [rows][inner complex] (x batch) operand viewed as FLOAT64, box = [box_rows][8 complex = 128 B]
bool make_map(CUtensorMap *tm, const c128 *base, long inner_complex, long rows, long ld, int batch, long stride,
              int box_rows) {
  EncodeTiledFn enc = get_encode();
  if (!enc) return false;
  cuuint64_t dims[3] = {(cuuint64_t)(2 * inner_complex), (cuuint64_t)rows, (cuuint64_t)batch};
  cuuint64_t strides[2] = {(cuuint64_t)ld * 16ull, (cuuint64_t)(batch > 1 ? stride : ld * rows) * 16ull};
  if (strides[1] == 0) strides[1] = 16;
  cuuint32_t box[3] = {16u, (cuuint32_t)box_rows, 1u};
  cuuint32_t es[3] = {1u, 1u, 1u};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void *)base, dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
}

template <int BM, int BN, int BK, int WM, int WN, int STAGES, bool BKN>
cudaError_t launch(cudaStream_t st, const CUtensorMap &tmA, const CUtensorMap &tmB, const ZgemmArgs &args, int batch) {
  constexpr int threads = (BM / WM) * (BN / WN) * 32 + 128;
  constexpr int smem = STAGES * (BM + BN) * BK * 16 + 2 * STAGES * 8 + 1024;
  auto kern = zgemm_kernel<BM, BN, BK, WM, WN, STAGES, BKN>;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((args.N + BN - 1) / BN, (args.M + BM - 1) / BM, batch * args.splits);
  kern<<<grid, threads, smem, st>>>(tmA, tmB, args);
  cclr_count_launch();
  return cudaGetLastError();
}

}  // namespace

int zgemm_num_sms() {
  static int n = 0;
  if (!n) {
    int dev = 0;
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
    if (n <= 0) n = 148;
  }
  return n;
}

cudaError_t zgemm(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA,
                  const c128 *B, long ldb, bool b_is_kn, bool conjB, c128 beta, c128 *C, long ldc, int batch, long sa,
                  long sb, long sc, const ZgemmWorkspace *ws) {
  if (M <= 0 || N <= 0 || batch <= 0) return cudaSuccess;
  constexpr int BM = 128, BN = 64, BK = 16, WM = 32, WN = 32, STAGES = 4;
  if (K <= 0) {  // C = beta * C
    zgemm_reduce_kernel<<<256, 256, 0, st>>>(nullptr, 0, M, N, alpha, beta, C, ldc, sc, batch);
    cclr_count_launch();
    return cudaGetLastError();
  }
  ZgemmArgs args{};
  args.M = M; args.N = N; args.K = K;
  args.C = C; args.ldc = ldc; args.sc = sc;
  args.alpha = alpha; args.beta = beta;
  args.conjA = conjA; args.conjB = conjB;
  const int nchunks = (K + BK - 1) / BK;
  // split-K when the MN tile grid cannot fill the chip and K is long
  int splits = 1;
  const long tiles = (long)((M + BM - 1) / BM) * ((N + BN - 1) / BN) * batch;
  const int sms = zgemm_num_sms();
  if (ws && ws->buf && tiles < sms && nchunks >= 16) {
    splits = (int)((2L * sms + tiles - 1) / tiles);
    if (splits > nchunks / 4) splits = nchunks / 4;
    const size_t per = (size_t)M * N * batch;
    if ((size_t)splits * per > ws->elems) splits = (int)(ws->elems / per);
    if (splits < 1) splits = 1;
  }
  args.splits = splits;
  args.chunks_per_split = (nchunks + splits - 1) / splits;
  args.partial = splits > 1 ? ws->buf : nullptr;

  CUtensorMap tmA, tmB;
  if (!make_map(&tmA, A, K, M, lda, batch, sa, BM)) return cudaErrorInvalidValue;
  if (!b_is_kn) {
    if (!make_map(&tmB, B, K, N, ldb, batch, sb, BN)) return cudaErrorInvalidValue;
  } else {
    if (!make_map(&tmB, B, N, K, ldb, batch, sb, BK)) return cudaErrorInvalidValue;
  }
  cudaError_t e = b_is_kn ? launch<BM, BN, BK, WM, WN, STAGES, true>(st, tmA, tmB, args, batch)
                          : launch<BM, BN, BK, WM, WN, STAGES, false>(st, tmA, tmB, args, batch);
  if (e != cudaSuccess) return e;
  if (splits > 1) {
    const size_t total = (size_t)M * N * batch;
    int blocks = (int)((total + 255) / 256);
    if (blocks > 4 * sms) blocks = 4 * sms;
    zgemm_reduce_kernel<<<blocks, 256, 0, st>>>(ws->buf, splits, M, N, alpha, beta, C, ldc, sc, batch);
    cclr_count_launch();
    e = cudaGetLastError();
  }
  return e;
}
