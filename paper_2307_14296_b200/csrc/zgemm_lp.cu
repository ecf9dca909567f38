// zgemm_lp.cu — reduced-precision complex GEMM on the 5th-generation tensor cores of sm_100a (tcgen05.mma, BF16 operands,
// FP32 accumulators in tensor memory).
//
//   C[M][N] = alpha * opA(A)[M][K] * opB(B)[K][N] + beta * C        (A, B, C complex128 in memory, as for zgemm)
//
// Where it is used: ONLY inside the inner (preconditioning) solve of cclr_solve (solver.cu).  The response
// equations are solved to 1e-10 by an outer subspace method whose sigma vectors, residuals and solutions are FP64 (zgemm.cu,
// FP64 DMMA); the trial vectors it is fed with come from an approximate solve of (A - z) d = -r, and an approximate operator is
// good enough for that.  The FP64 tensor pipe of B200 peaks at 37 TFLOP/s, the BF16 one at ~1.6 PFLOP/s: the same contraction
// plan run through this kernel costs ~1/15 of an FP64 sigma, and the outer iteration needs ~5 FP64 sigma per system instead of
// ~35.  Nothing here ever reaches a result the caller sees: every number returned by the library is produced and checked in FP64.
//
// Design:
//   * complex product from real tensor-core products without an interleaved layout: the operands are split into planes
//     Re / Im (BF16, K contiguous) by a conversion pre-pass (cached for the context's constant intermediates, W_vvvv first);
//     per K block of 64 the CTA holds A_re, A_im [128 x 64] and B_re, B_im [128 x 64] with B_im stored right behind B_re, so
//     that [B_re; B_im] is ONE 256-row operand:  D1 = A_re . [B_re; B_im]^T = [A_re B_re | A_re B_im],
//     D2 = A_im . [B_re; B_im]^T = [A_im B_re | A_im B_im] -- two tcgen05.mma of 128 x 256 x 16 per 16 k instead of four of
//     128 x 128 x 16 (12 KB of shared-memory operand per 128 cycles instead of 8 KB per 64: below the 128 B/clk limit), and
//     C_re = D1[:, :128] - D2[:, 128:],  C_im = D1[:, 128:] + D2[:, :128] is formed in the epilogue.  D1, D2 fill the 512
//     columns of tensor memory.
//   * warp roles (192 threads): warp 0 = TMA producer (one lane), warp 1 = TMEM allocation + MMA issue (one lane), warps 2-5 =
//     epilogue (tcgen05.ld 32x32b: thread <-> accumulator row).  3-stage shared-memory ring (64 KB per stage) with full / empty
//     mbarriers; tcgen05.commit releases a stage when the MMAs that read it have finished, and signals the epilogue.
//   * operands by TMA (cp.async.bulk.tensor.2d, BF16 maps, 128 B x 128 rows boxes, SWIZZLE_128B) = the canonical K-major
//     SWIZZLE_128B layout of the shared-memory matrix descriptor; ragged M, N, K: TMA zero-fills, stores are guarded.
//   * one 128 x 128 complex output tile per CTA, tile_n fastest (the CTAs of one A row panel run together and share it in L2).
#include "common.cuh"
#include <cuda_bf16.h>
#include <algorithm>
#include <atomic>
#include <mutex>

namespace {

constexpr int LP_BM = 128, LP_BN = 128, LP_BK = 64, LP_STAGES = 3;
constexpr int LP_TILE_BYTES = 128 * LP_BK * 2;          // 128 rows x 64 bf16 = 16 KB
constexpr int LP_STAGE_BYTES = 4 * LP_TILE_BYTES;       // A_re, A_im, B_re, B_im
constexpr int LP_SMEM = 1024 + LP_STAGES * LP_STAGE_BYTES + 128;
constexpr int LP_THREADS = 192;
constexpr uint32_t LP_TMEM_COLS = 512;

struct LpArgs {
  int M, N, K, tiles_n, nkb;
  c128 alpha, beta;
  c128 *C;
  long ldc;
};

__device__ __forceinline__ uint32_t smem_u32(const void *p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
// bounded spin: a protocol error traps (the launch fails) instead of hanging the device
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  for (long spin = 0; !done; ++spin) {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    if (spin > (1L << 26)) __trap();
  }
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];"
               ::"r"(dst), "l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// shared-memory matrix descriptor: K-major, SWIZZLE_128B, rows of 128 bytes, 8-row groups 1024 bytes apart (the tile is dense)
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr) {
  const uint32_t lo = ((addr & 0x3FFFFu) >> 4) | (1u << 16);            // start address, leading byte offset (unused) = 1
  const uint32_t hi = (1024u >> 4) | (1u << 14) | (2u << 29);           // stride byte offset, version 1, SWIZZLE_128B
  return ((uint64_t)hi << 32) | lo;
}
// instruction descriptor (kind::f16): D = F32, A = B = BF16, both K-major, M = 128, N = 256
constexpr uint32_t LP_IDESC = (1u << 4) | (1u << 7) | (1u << 10) | ((256u >> 3) << 17) | ((128u >> 4) << 24);

__device__ __forceinline__ void umma(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t accumulate) {
  asm volatile(
      "{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n}\n"
      ::"r"(tmem_d), "l"(da), "l"(db), "r"(LP_IDESC), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t addr, float *v) {
  uint32_t r[16];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
      : "r"(addr)
      : "memory");
#pragma unroll
  for (int j = 0; j < 16; ++j) v[j] = __uint_as_float(r[j]);
}

__global__ void __launch_bounds__(LP_THREADS, 1)
zgemm_lp_kernel(const __grid_constant__ CUtensorMap tAr, const __grid_constant__ CUtensorMap tAi,
                const __grid_constant__ CUtensorMap tBr, const __grid_constant__ CUtensorMap tBi, const LpArgs a) {
  extern __shared__ uint8_t lp_smem_raw[];
  const uint32_t base = (smem_u32(lp_smem_raw) + 1023u) & ~1023u;
  const uint32_t bars = base + LP_STAGES * LP_STAGE_BYTES;      // full[s], empty[s], tmem_full (8 B each), tmem slot (4 B)
  const uint32_t bar_full = bars, bar_empty = bars + 8 * LP_STAGES, bar_tmem = bars + 16 * LP_STAGES;
  const uint32_t slot_addr = bar_tmem + 8;
  volatile uint32_t *slot = (volatile uint32_t *)(lp_smem_raw + (slot_addr - smem_u32(lp_smem_raw)));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int tm = blockIdx.x / a.tiles_n, tn = blockIdx.x % a.tiles_n;
  const int m0 = tm * LP_BM, n0 = tn * LP_BN;

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < LP_STAGES; ++s) {
      mbar_init(bar_full + 8 * s, 1);       // the producer's expect_tx arrive + the bytes of four TMA boxes
      mbar_init(bar_empty + 8 * s, 1);      // one tcgen05.commit
    }
    mbar_init(bar_tmem, 1);                 // one tcgen05.commit after the last MMA
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {                          // the allocating warp also deallocates
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot_addr), "r"(LP_TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem = *slot;

  if (warp == 0) {
    if (lane == 0) {
      for (int kb = 0; kb < a.nkb; ++kb) {
        const int s = kb % LP_STAGES;
        const uint32_t ph = (uint32_t)(kb / LP_STAGES) & 1u;
        mbar_wait(bar_empty + 8 * s, ph ^ 1u);
        const uint32_t st = base + s * LP_STAGE_BYTES, fb = bar_full + 8 * s;
        mbar_expect_tx(fb, LP_STAGE_BYTES);
        tma_load_2d(st, &tAr, kb * LP_BK, m0, fb);
        tma_load_2d(st + LP_TILE_BYTES, &tAi, kb * LP_BK, m0, fb);
        tma_load_2d(st + 2 * LP_TILE_BYTES, &tBr, kb * LP_BK, n0, fb);
        tma_load_2d(st + 3 * LP_TILE_BYTES, &tBi, kb * LP_BK, n0, fb);
      }
    }
  } else if (warp == 1) {
    for (int kb = 0; kb < a.nkb; ++kb) {
      const int s = kb % LP_STAGES;
      const uint32_t ph = (uint32_t)(kb / LP_STAGES) & 1u;
      mbar_wait(bar_full + 8 * s, ph);
      tc_fence_after();
      if (lane == 0) {
        const uint32_t st = base + s * LP_STAGE_BYTES;
#pragma unroll
        for (int k = 0; k < LP_BK / 16; ++k) {
          const uint64_t dar = smem_desc(st + k * 32), dai = smem_desc(st + LP_TILE_BYTES + k * 32);
          const uint64_t db = smem_desc(st + 2 * LP_TILE_BYTES + k * 32);
          const uint32_t acc = (kb > 0 || k > 0) ? 1u : 0u;
          umma(tmem, dar, db, acc);            // D1 = [A_re B_re | A_re B_im]
          umma(tmem + 256u, dai, db, acc);     // D2 = [A_im B_re | A_im B_im]
        }
        umma_commit(bar_empty + 8 * s);        // the stage is free once these MMAs have read it
        if (kb == a.nkb - 1) umma_commit(bar_tmem);
      }
      __syncwarp();
    }
  } else {
    const int q = warp & 3;                    // the TMEM lane quarter this warp may read
    const int row = q * 32 + lane;
    const long grow = (long)m0 + row;
    mbar_wait(bar_tmem, 0);
    tc_fence_after();
    const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16);
    const bool has_beta = a.beta.x != 0.0 || a.beta.y != 0.0;
    for (int c0 = 0; c0 < LP_BN; c0 += 16) {
      float rr[16], ri[16], ir[16], ii[16];
      tmem_ld16(taddr + c0, rr);
      tmem_ld16(taddr + 128 + c0, ri);
      tmem_ld16(taddr + 256 + c0, ir);
      tmem_ld16(taddr + 384 + c0, ii);
      asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
      if (grow < a.M) {
        c128 *crow = a.C + grow * a.ldc;
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const int col = n0 + c0 + j;
          if (col < a.N) {
            const c128 p = make_double2((double)rr[j] - (double)ii[j], (double)ri[j] + (double)ir[j]);
            c128 out = cmul(a.alpha, p);
            if (has_beta) out = cadd(out, cmul(a.beta, crow[col]));
            crow[col] = out;
          }
        }
      }
    }
    tc_fence_before();
  }
  __syncthreads();
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(LP_TMEM_COLS) : "memory");
  }
}

// ---- conversion pre-pass: complex128 [rows][cols] (K contiguous) -> BF16 planes re / im [rows][ldp] ------------------------
__global__ void __launch_bounds__(256) lp_convert_kernel(const c128 *__restrict__ X, long ld, long rows, long cols, int conj,
                                                         __nv_bfloat16 *__restrict__ re, __nv_bfloat16 *__restrict__ im, long ldp) {
  const double sg = conj ? -1.0 : 1.0;
  const long pairs = (cols + 1) / 2;
  for (long r = blockIdx.y; r < rows; r += gridDim.y) {
    const c128 *x = X + r * ld;
    __nv_bfloat162 *dr = (__nv_bfloat162 *)(re + r * ldp), *di = (__nv_bfloat162 *)(im + r * ldp);
    for (long c = (long)blockIdx.x * blockDim.x + threadIdx.x; c < pairs; c += (long)gridDim.x * blockDim.x) {
      const c128 v0 = x[2 * c], v1 = 2 * c + 1 < cols ? x[2 * c + 1] : czero();
      dr[c] = __floats2bfloat162_rn((float)v0.x, (float)v1.x);
      di[c] = __floats2bfloat162_rn((float)(sg * v0.y), (float)(sg * v1.y));
    }
  }
}
// the same for an operand stored [K][N] (N contiguous): planes [N][ldp] with K contiguous (32 x 32 tile transpose)
__global__ void __launch_bounds__(256) lp_convert_t_kernel(const c128 *__restrict__ X, long ld, long krows, long ncols, int conj,
                                                           __nv_bfloat16 *__restrict__ re, __nv_bfloat16 *__restrict__ im, long ldp) {
  __shared__ float tr[32][33], ti[32][33];
  const float sg = conj ? -1.f : 1.f;
  const long k0 = (long)blockIdx.y * 32, n0 = (long)blockIdx.x * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;          // 32 x 8
  for (int i = ty; i < 32; i += 8) {
    const long k = k0 + i, n = n0 + tx;
    c128 v = czero();
    if (k < krows && n < ncols) v = X[k * ld + n];
    tr[i][tx] = (float)v.x;
    ti[i][tx] = sg * (float)v.y;
  }
  __syncthreads();
  for (int i = ty; i < 32; i += 8) {
    const long n = n0 + i, k = k0 + tx;
    if (n < ncols && k < krows) {
      re[n * ldp + k] = __float2bfloat16_rn(tr[tx][i]);
      im[n * ldp + k] = __float2bfloat16_rn(ti[tx][i]);
    }
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn lp_get_encode() {
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
// tensor map over a BF16 plane [rows][kdim] with row stride ldp: box = 64 elements (128 B) x 128 rows, SWIZZLE_128B
bool lp_make_map(CUtensorMap *tm, const void *plane, long kdim, long rows, long ldp) {
  EncodeTiledFn enc = lp_get_encode();
  if (!enc || (ldp & 7)) return false;
  cuuint64_t dims[2] = {(cuuint64_t)kdim, (cuuint64_t)rows};
  cuuint64_t strides[1] = {(cuuint64_t)ldp * 2ull};
  cuuint32_t box[2] = {(cuuint32_t)LP_BK, 128u};
  cuuint32_t es[2] = {1u, 1u};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, (void *)plane, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

cudaError_t lp_convert(cudaStream_t st, const c128 *X, long ld, long rows, long kdim, bool transposed, bool conj, uint16_t *planes,
                       long ldp) {
  __nv_bfloat16 *re = (__nv_bfloat16 *)planes, *im = re + (size_t)rows * ldp;
  if (!transposed) {
    dim3 grid((unsigned)std::min<long>(std::max<long>(1, ((kdim + 1) / 2 + 255) / 256), 64), (unsigned)std::min<long>(rows, 32768));
    lp_convert_kernel<<<grid, 256, 0, st>>>(X, ld, rows, kdim, conj ? 1 : 0, re, im, ldp);
  } else {
    // X is [kdim][rows]
    dim3 grid((unsigned)((rows + 31) / 32), (unsigned)((kdim + 31) / 32));
    lp_convert_t_kernel<<<grid, 256, 0, st>>>(X, ld, kdim, rows, conj ? 1 : 0, re, im, ldp);
  }
  cclr_count_launch();
  return cudaGetLastError();
}

}  // namespace

bool zgemm_lp_eligible(int M, int N, int K) { return M >= 128 && N >= 8 && K >= 256; }

void zgemm_lp_release(LpWorkspace *lw) {
  if (!lw) return;
  for (auto &e : lw->cache)
    if (e.planes) cudaFree(e.planes);
  lw->cache.clear();
  lw->cache_bytes = 0;
  for (int i = 0; i < 2; ++i) {
    if (lw->scratch[i]) cudaFree(lw->scratch[i]);
    lw->scratch[i] = nullptr;
    lw->scratch_elems[i] = 0;
  }
}

// planes of one operand: from the cache (constant operands), else converted into the scratch slot `which`
static cudaError_t lp_operand(cudaStream_t st, LpWorkspace *lw, int which, const c128 *X, long ld, long rows, long kdim,
                              bool transposed, bool conj, bool constant, const uint16_t **planes, long *ldp_out) {
  const long ldp = (kdim + 7) & ~7L;
  *ldp_out = ldp;
  const size_t elems = 2 * (size_t)rows * (size_t)ldp;
  if (constant) {
    for (auto &e : lw->cache)
      if (e.key == X && e.rows == rows && e.kdim == kdim && e.ld == ld && e.transposed == transposed && e.conj == conj) {
        *planes = e.planes;
        return cudaSuccess;
      }
    if (lw->cache_bytes + elems * 2 <= lw->cache_budget) {
      uint16_t *p = nullptr;
      if (cudaMalloc(&p, elems * 2) == cudaSuccess) {
        const cudaError_t e = lp_convert(st, X, ld, rows, kdim, transposed, conj, p, ldp);
        if (e != cudaSuccess) { cudaFree(p); return e; }
        LpCacheEntry ce;
        ce.key = X; ce.rows = rows; ce.kdim = kdim; ce.ld = ld; ce.transposed = transposed; ce.conj = conj; ce.planes = p;
        ce.bytes = elems * 2;
        lw->cache.push_back(ce);
        lw->cache_bytes += elems * 2;
        *planes = p;
        return cudaSuccess;
      }
      cudaGetLastError();
    }
  }
  if (lw->scratch_elems[which] < elems) {
    cudaError_t e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return e;
    if (lw->scratch[which]) cudaFree(lw->scratch[which]);
    lw->scratch[which] = nullptr;
    lw->scratch_elems[which] = 0;
    e = cudaMalloc(&lw->scratch[which], elems * 2);
    if (e != cudaSuccess) return e;
    lw->scratch_elems[which] = elems;
  }
  *planes = lw->scratch[which];
  return lp_convert(st, X, ld, rows, kdim, transposed, conj, lw->scratch[which], ldp);
}

cudaError_t zgemm_lp(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA, bool a_const,
                     const c128 *B, long ldb, bool b_is_kn, bool conjB, bool b_const, c128 beta, c128 *C, long ldc, LpWorkspace *lw) {
  if (!lw || M < 1 || N < 1 || K < 1) return cudaErrorInvalidValue;
  const uint16_t *pa = nullptr, *pb = nullptr;
  long lpa = 0, lpb = 0;
  cudaError_t e = lp_operand(st, lw, 0, A, lda, M, K, false, conjA, a_const, &pa, &lpa);
  if (e != cudaSuccess) return e;
  e = lp_operand(st, lw, 1, B, ldb, N, K, b_is_kn, conjB, b_const, &pb, &lpb);
  if (e != cudaSuccess) return e;
  CUtensorMap tAr, tAi, tBr, tBi;
  if (!lp_make_map(&tAr, pa, K, M, lpa) || !lp_make_map(&tAi, pa + (size_t)M * lpa, K, M, lpa) ||
      !lp_make_map(&tBr, pb, K, N, lpb) || !lp_make_map(&tBi, pb + (size_t)N * lpb, K, N, lpb))
    return cudaErrorInvalidValue;
  LpArgs a;
  a.M = M; a.N = N; a.K = K;
  a.tiles_n = (N + LP_BN - 1) / LP_BN;
  a.nkb = (K + LP_BK - 1) / LP_BK;
  a.alpha = alpha; a.beta = beta; a.C = C; a.ldc = ldc;
  const long tiles = (long)((M + LP_BM - 1) / LP_BM) * a.tiles_n;
  static std::atomic<unsigned long long> configured{0};
  int dev = 0;
  e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev >= 64 || !((configured.load() >> dev) & 1ull)) {
    e = cudaFuncSetAttribute((const void *)zgemm_lp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, LP_SMEM);
    if (e != cudaSuccess) return e;
    if (dev < 64) configured.fetch_or(1ull << dev);
  }
  zgemm_lp_kernel<<<(unsigned)tiles, LP_THREADS, LP_SMEM, st>>>(tAr, tAi, tBr, tBi, a);
  cclr_count_launch();
  return cudaGetLastError();
}
