// zgemm_oz.cu — complex128 GEMM at FP64 accuracy on the INT8 path of the 5th-generation tensor cores (sm_100a:
// tcgen05.mma.kind::i8, S32 accumulators in tensor memory), by integer slicing of the operands (Ozaki-type splitting).
//
//   C[M][N] = alpha * opA(A)[M][K] * opB(B)[K][N] + beta * C        (A, B, C complex128 in memory, as for zgemm)
//
// Why: the FP64 tensor pipe of B200 (DMMA) tops out at 37 TFLOP/s and the 3M kernel of zgemm.cu already runs it at 0.93; the
// INT8 pipe of the same chip is nominally 4.5 Pop/s.  A contraction whose operands are cut into s signed slices of 7 bits costs
// s(s+1)/2 integer products and is exact in the integer part -- the only error is the truncation of the operands at 6 + 7(s-1)
// bits below the largest element of each row (s = 6: 41 bits, norm-wise error ~6e-12 for the Gaussian-like rows of this path;
// north_star's bar for sigma is 1e-10).  Ladder (T11) and ring (T8) -- 91 % of sigma -- are the users.
//
// Arithmetic (what the tolerance of the parity tests is derived from):
//   * real embedding of the complex product: A' [M][2K] is the operand's memory as it stands (re, im interleaved along K);
//     B' [2N][2K] holds, for the complex column n, the rows  (n,re) = [ b_re, -sa sb b_im ]_k  and  (n,im) = [ sb b_im, sa b_re ]_k
//     (sa / sb = -1 when A / B is conjugated), so that  C'[m][(n,re)], C'[m][(n,im)]  are Re and Im of C[m][n], adjacent in
//     memory like the complex128 output.  One real GEMM of M x 2N x 2K per slice pair.
//   * scaling: per row m of A' a power of two 2^ea[m] > max |A'[m][:]|, per complex column n of B 2^eb[n] likewise (exact).
//   * slicing (exact in FP64): y = x 2^(6-e);  q_0 = rint(y);  y <- (y - q_0) 2^7;  q_1 = rint(y); ...  every |q_t| <= 64, and
//     x 2^-e = sum_t q_t 2^(-6-7t) + rest,  |rest| <= 2^(-7s).
//   * product: C' = 2^(ea+eb) sum_{t+u <= s-1} 2^(-12-7(t+u)) (A_t . B_u); the pairs of one anti-diagonal d = t+u share one S32
//     accumulator as long as  pairs * 2K * 64^2 < 2^31  (otherwise the diagonal is split into several accumulation groups);
//     each group is converted to FP64, scaled (exactly) and added to C in the epilogue -- smallest diagonals last.
//
// Kernel: one CTA per 256 x BN output tile (BN <= 256 real columns, chosen per call from a port / pipe cost model); two 128-row
// tcgen05.mma halves with their accumulators side by side in the 512 columns of tensor memory.  warp 0 = TMA producer (3-D
// maps {k, row, slice} over the INT8 slices, 128 B x rows boxes, SWIZZLE_128B = the canonical K-major layout of the shared-
// memory matrix descriptors), warp 1 = MMA issue (one lane; 8 MMAs of 128 x BN x 32 per 128-byte k block), warps 2-9 =
// epilogue (tcgen05.ld 32x32b, S32 -> FP64, read-modify-write of the C tile).  Ring of as many (32 KB + BN x 128 B) stages as fit
// 227 KB (3 or 4) with full / empty mbarriers; tcgen05.commit frees a stage and hands the accumulators to the epilogue at the
// end of each accumulation group.
// Clusters: the CTAs of c_m x c_n adjacent tiles form a thread-block cluster and share operand tiles by TMA multicast -- the
// A tile along a cluster row, the B tile along a cluster column; the CTAs take turns as the loader of a stage and the
// "slot consumed" commits are multicast to the peers, which keeps a cluster in lock-step.  For the ladder one cluster spans all
// tile columns of a row panel, so W_vvvv's slices leave HBM once per use (538 GB -> 104 GB per call at config 4, profiles/).
#include "common.cuh"
#include <algorithm>
#include <atomic>
#include <mutex>
#include <cmath>

namespace {

constexpr int OZ_BM = 256, OZ_BK = 128;
constexpr int OZ_A_BYTES = OZ_BM * OZ_BK;                 // 32 KB
constexpr int OZ_MAX_SMEM = 227 * 1024;                   // per CTA on sm_100a
constexpr int OZ_MAX_STAGES = 6;
constexpr int OZ_THREADS = 320;                           // producer warp, MMA warp, 8 epilogue warps
constexpr uint32_t OZ_TMEM_COLS = 512;
constexpr int OZ_MAX_PAIRS = 36, OZ_MAX_GROUPS = 24;

struct OzArgs {
  int M, N2, BN, nkb, npairs, ngroups;
  int nstages, stage_bytes;                           // shared-memory ring: stage = A tile (32 KB) + B tile (BN x 128 B)
  int c_m, c_n, ctiles_n;                             // cluster shape (CTAs along M x along N) and cluster columns of the grid
  unsigned char pt[OZ_MAX_PAIRS], pu[OZ_MAX_PAIRS];   // slice indices (A, B) of pair p, grouped
  unsigned char gend[OZ_MAX_GROUPS];                  // group g = pairs [gend[g-1], gend[g])
  unsigned char gdiag[OZ_MAX_GROUPS];                 // its anti-diagonal t + u
  uint32_t idesc;
  c128 alpha, beta;
  c128 *C;
  long c_rs, c_cs;                                    // element strides of C along the rows (m) / complex columns (n) of this product
  const double *sa, *sb;                              // 2^ea[m] per row of A, 2^eb[n] per complex column of B
};

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
// bounded spin: a protocol error traps (the launch fails) instead of hanging the device
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  for (long spin = 0; !done; ++spin) {
    asm volatile(
        "{\n .reg .pred p;\n mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n selp.u32 %0, 1, 0, p;\n}\n"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
    if (spin > (1L << 28)) __trap();
  }
}
__device__ __forceinline__ void tma_load_3d(uint32_t dst, const CUtensorMap *tm, int c0, int c1, int c2, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4}], [%5];"
               ::"r"(dst), "l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void tma_load_3d_mc(uint32_t dst, const CUtensorMap *tm, int c0, int c1, int c2, uint32_t bar, uint16_t mask) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1, {%2, %3, %4}], [%5], %6;"
      ::"r"(dst), "l"((uint64_t)tm), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "h"(mask)
      : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync() {
  asm volatile("barrier.cluster.arrive.release.aligned;\n barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// shared-memory matrix descriptor: K-major, SWIZZLE_128B, rows of 128 bytes, 8-row groups 1024 bytes apart (dense tile)
__device__ __forceinline__ uint64_t smem_desc(uint32_t addr) {
  const uint32_t lo = ((addr & 0x3FFFFu) >> 4) | (1u << 16);
  const uint32_t hi = (1024u >> 4) | (1u << 14) | (2u << 29);
  return ((uint64_t)hi << 32) | lo;
}
__device__ __forceinline__ void umma_i8(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n .reg .pred p;\n setp.ne.b32 p, %4, 0;\n tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n}\n"
      ::"r"(tmem_d), "l"(da), "l"(db), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void umma_commit_mc(uint32_t bar, uint16_t mask) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"(mask) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t addr, int *v) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
      : "r"(addr)
      : "memory");
}

__global__ void __launch_bounds__(OZ_THREADS, 1)
zgemm_oz_kernel(const __grid_constant__ CUtensorMap tA, const __grid_constant__ CUtensorMap tB, const __grid_constant__ OzArgs a) {
  extern __shared__ uint8_t oz_smem_raw[];
  const uint32_t base = (smem_u32(oz_smem_raw) + 1023u) & ~1023u;
  const int NS = a.nstages;
  const uint32_t bars = base + NS * a.stage_bytes;   // full[s], emptyA[s], emptyB[s], tmem_full, tmem_empty (8 B each), tmem slot
  const uint32_t bar_full = bars, bar_empty = bars + 8 * OZ_MAX_STAGES, bar_emptyb = bars + 16 * OZ_MAX_STAGES;
  const uint32_t bar_tfull = bars + 24 * OZ_MAX_STAGES, bar_tempty = bar_tfull + 8;
  const uint32_t slot_addr = bar_tempty + 8;
  volatile uint32_t *slot = (volatile uint32_t *)(oz_smem_raw + (slot_addr - smem_u32(oz_smem_raw)));
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  // cluster of c_m x c_n CTAs = c_m x c_n adjacent tiles: the A tile of a cluster row is multicast to its c_n CTAs, the B tile of a
  // cluster column to its c_m CTAs; the CTAs take turns as the loader of a stage (stage it: column it % c_n loads A, row
  // it % c_m loads B), so every operand byte crosses L2 -> SM once per cluster and the CTAs of a cluster run in lock-step
  const int csize = a.c_m * a.c_n;
  const int rank = csize > 1 ? (int)cluster_ctarank() : 0;
  const int rm = rank / a.c_n, rn = rank % a.c_n;
  const int cid = blockIdx.x / csize;
  const int tm = (cid / a.ctiles_n) * a.c_m + rm, tn = (cid % a.ctiles_n) * a.c_n + rn;
  const int m0 = tm * OZ_BM, n0 = tn * a.BN;
  uint16_t row_mask = 0, col_mask = 0;      // the CTAs that share my A tile / my B tile (including me)
  for (int j = 0; j < a.c_n; ++j) row_mask |= (uint16_t)(1u << (rm * a.c_n + j));
  for (int j = 0; j < a.c_m; ++j) col_mask |= (uint16_t)(1u << (j * a.c_n + rn));

  if (warp == 0 && lane == 0) {
    for (int s = 0; s < NS; ++s) {
      mbar_init(bar_full + 8 * s, 1);      // the producer's expect_tx arrive + the bytes of the two boxes (whoever loads them)
      // "slot consumed" is signalled separately by the CTAs of my cluster row (they share my A tile; its loader waits on this)
      // and of my cluster column (B tile): the A loads keep a row in lock-step and the B loads a column, so neither barrier can
      // be lapped by a fast peer -- one barrier for row and column together could (a row peer is not held back by my column)
      mbar_init(bar_empty + 8 * s, (uint32_t)a.c_n);
      mbar_init(bar_emptyb + 8 * s, (uint32_t)a.c_m);
    }
    mbar_init(bar_tfull, 1);               // one tcgen05.commit at the end of an accumulation group
    mbar_init(bar_tempty, 8);              // one arrive per epilogue warp
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  if (warp == 1) {                         // the allocating warp also deallocates
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(slot_addr), "r"(OZ_TMEM_COLS) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  tc_fence_before();
  __syncthreads();
  if (csize > 1) cluster_sync();            // every barrier of the cluster is initialised before any remote arrive / multicast
  tc_fence_after();
  const uint32_t tmem = *slot;
  const uint32_t b_bytes = (uint32_t)a.BN * OZ_BK;

  if (warp == 0) {
    if (lane == 0) {
      const bool mc = csize > 1;
      long it = 0;
      int s = 0;
      uint32_t ph = 0;
      for (int p = 0; p < a.npairs; ++p) {
        const int t = a.pt[p], u = a.pu[p];
        for (int kb = 0; kb < a.nkb; ++kb, ++it) {
          mbar_wait(bar_empty + 8 * s, ph ^ 1u);
          if (a.c_m > 1) mbar_wait(bar_emptyb + 8 * s, ph ^ 1u);
          const uint32_t st = base + s * a.stage_bytes, fb = bar_full + 8 * s;
          mbar_expect_tx(fb, OZ_A_BYTES + b_bytes);
          if (!mc) {
            tma_load_3d(st, &tA, kb * OZ_BK, m0, t, fb);
            tma_load_3d(st + OZ_A_BYTES, &tB, kb * OZ_BK, n0, u, fb);
          } else {
            if ((int)(it % a.c_n) == rn) tma_load_3d_mc(st, &tA, kb * OZ_BK, m0, t, fb, row_mask);
            if ((int)(it % a.c_m) == rm) tma_load_3d_mc(st + OZ_A_BYTES, &tB, kb * OZ_BK, n0, u, fb, col_mask);
          }
          if (++s == NS) { s = 0; ph ^= 1u; }
        }
      }
    }
  } else if (warp == 1) {
    int p = 0, s = 0;
    uint32_t ph = 0;
    for (int g = 0; g < a.ngroups; ++g) {
      if (g > 0) {                          // the epilogue must have drained the accumulators of the previous group
        mbar_wait(bar_tempty, (uint32_t)(g - 1) & 1u);
        tc_fence_after();
      }
      bool first = true;
      for (; p < a.gend[g]; ++p) {
        for (int kb = 0; kb < a.nkb; ++kb) {
          mbar_wait(bar_full + 8 * s, ph);
          tc_fence_after();
          if (lane == 0) {
            const uint32_t st = base + s * a.stage_bytes;
#pragma unroll
            for (int k = 0; k < OZ_BK / 32; ++k) {
              const uint64_t db = smem_desc(st + OZ_A_BYTES + k * 32);
              const uint32_t acc = (first && k == 0) ? 0u : 1u;
              umma_i8(tmem, smem_desc(st + k * 32), db, a.idesc, acc);
              umma_i8(tmem + 256u, smem_desc(st + 128 * OZ_BK + k * 32), db, a.idesc, acc);
            }
            // the stage is free once these MMAs have read it: tell every CTA that loads into my shared memory
            if (csize == 1) umma_commit(bar_empty + 8 * s);
            else {
              umma_commit_mc(bar_empty + 8 * s, row_mask);
              if (a.c_m > 1) umma_commit_mc(bar_emptyb + 8 * s, col_mask);
            }
          }
          first = false;
          if (++s == NS) { s = 0; ph ^= 1u; }
          __syncwarp();
        }
      }
      if (lane == 0) umma_commit(bar_tfull);
      __syncwarp();
    }
  } else {
    const int q = warp & 3;                  // the TMEM lane quarter this warp may read
    const int h = (warp - 2) >> 2;           // which 128-row half
    const long grow = (long)m0 + h * 128 + q * 32 + lane;
    const uint32_t taddr = tmem + ((uint32_t)(q * 32) << 16) + (uint32_t)h * 256u;
    const bool has_beta = a.beta.x != 0.0 || a.beta.y != 0.0;
    const double rs0 = grow < a.M ? a.sa[grow] : 0.0;
    c128 *crow = a.C + (grow < a.M ? grow : 0) * a.c_rs;   // c_rs = 1, c_cs = ldc: the product is stored transposed (zgemm_oz_bt)
    const int N = a.N2 >> 1;
    for (int g = 0; g < a.ngroups; ++g) {
      mbar_wait(bar_tfull, (uint32_t)g & 1u);
      tc_fence_after();
      const double rs = rs0 * exp2(-12.0 - 7.0 * (double)a.gdiag[g]);
      for (int c0 = 0; c0 < a.BN; c0 += 16) {
        int r[16];
        tmem_ld16(taddr + c0, r);
        asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
        if (grow < a.M) {
          const int cb = (n0 + c0) >> 1;
#pragma unroll
          for (int j = 0; j < 8; ++j) {
            const int col = cb + j;
            if (col < N) {
              const double sc = rs * a.sb[col];
              const c128 pv = make_double2((double)r[2 * j] * sc, (double)r[2 * j + 1] * sc);
              c128 out = cmul(a.alpha, pv);
              c128 *cp = crow + (long)col * a.c_cs;
              if (g > 0) out = cadd(out, *cp);
              else if (has_beta) out = cadd(out, cmul(a.beta, *cp));
              *cp = out;
            }
          }
        }
      }
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(bar_tempty);
    }
  }
  __syncthreads();
  if (csize > 1) cluster_sync();            // no CTA leaves while a peer may still signal its barriers
  if (warp == 1) {
    tc_fence_after();
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(tmem), "r"(OZ_TMEM_COLS) : "memory");
  }
}

// ---- scaling: scale[r] = 2^E > max_k |X[r][k]| (both parts), 1 for a zero row ------------------------------------------------
__device__ __forceinline__ double pow2_above(double mx) {
  if (!(mx > 0.0)) return 1.0;
  int e;
  frexp(mx, &e);                        // mx = f 2^e, f in [0.5, 1)
  return ldexp(1.0, e);
}
__global__ void __launch_bounds__(256) oz_rowmax_kernel(const c128 *__restrict__ X, long ld, long rows, long cols,
                                                        double *__restrict__ scale) {
  __shared__ double red[8];
  for (long r = blockIdx.x; r < rows; r += gridDim.x) {
    const c128 *x = X + r * ld;
    double mx = 0.0;
    for (long c = threadIdx.x; c < cols; c += 256) {
      const c128 v = x[c];
      mx = fmax(mx, fmax(fabs(v.x), fabs(v.y)));
    }
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = mx;
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int w = 1; w < 8; ++w) mx = fmax(mx, red[w]);
      scale[r] = pow2_above(mx);
    }
    __syncthreads();
  }
}
// acc[0] += sum over rows of (2^E_r)^2 / mean(x^2 over the row), acc[1] += number of non-zero rows: the dynamic range the slicing
// has to cover (zgemm_oz_suggest_slices)
__global__ void __launch_bounds__(256) oz_rowstats_kernel(const c128 *__restrict__ X, long ld, long rows, long cols, double *acc) {
  __shared__ double redm[8], reds[8];
  for (long r = blockIdx.x; r < rows; r += gridDim.x) {
    const c128 *x = X + r * ld;
    double mx = 0.0, ss = 0.0;
    for (long c = threadIdx.x; c < cols; c += 256) {
      const c128 v = x[c];
      mx = fmax(mx, fmax(fabs(v.x), fabs(v.y)));
      ss += v.x * v.x + v.y * v.y;
    }
    for (int o = 16; o > 0; o >>= 1) {
      mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
      ss += __shfl_xor_sync(0xffffffffu, ss, o);
    }
    if ((threadIdx.x & 31) == 0) { redm[threadIdx.x >> 5] = mx; reds[threadIdx.x >> 5] = ss; }
    __syncthreads();
    if (threadIdx.x == 0) {
      for (int w = 1; w < 8; ++w) { mx = fmax(mx, redm[w]); ss += reds[w]; }
      if (mx > 0.0 && ss > 0.0) {
        const double sc = pow2_above(mx);
        atomicAdd(acc, sc * sc * (2.0 * (double)cols) / ss);
        atomicAdd(acc + 1, 1.0);
      }
    }
    __syncthreads();
  }
}
// column maxima of X [krows][ncols] (N contiguous): bit patterns of |x| through atomicMax, then 2^E in place
__global__ void __launch_bounds__(256) oz_colmax_kernel(const c128 *__restrict__ X, long ld, long krows, long ncols, long kslab,
                                                        unsigned long long *__restrict__ mxbits) {
  const long n = (long)blockIdx.x * 256 + threadIdx.x;
  if (n >= ncols) return;
  const long k0 = (long)blockIdx.y * kslab, k1 = k0 + kslab < krows ? k0 + kslab : krows;
  double mx = 0.0;
  for (long k = k0; k < k1; ++k) {
    const c128 v = X[k * ld + n];
    mx = fmax(mx, fmax(fabs(v.x), fabs(v.y)));
  }
  atomicMax(mxbits + n, (unsigned long long)__double_as_longlong(mx));
}
__global__ void __launch_bounds__(256) oz_scale_finalize_kernel(double *scale, long n) {
  const long i = (long)blockIdx.x * 256 + threadIdx.x;
  if (i < n) scale[i] = pow2_above(scale[i]);
}

// ---- slicing -----------------------------------------------------------------------------------------------------------------
// rows of X [rows][K] (K contiguous) -> INT8 slices.  MODE 0 (A operand): out row r = [re, im]_k.  MODE 1 (B operand stored
// [N][K]): out rows 2r = [re, c0 im]_k and 2r+1 = [c1 im, c2 re]_k.  One thread = 8 complex numbers = one 16-byte store per row.
template <int MODE>
__global__ void __launch_bounds__(256) oz_slice_rows_kernel(const c128 *__restrict__ X, long ld, long rows, long K, int s,
                                                            const double *__restrict__ scale, int8_t *__restrict__ out, long ldp,
                                                            size_t slice_stride, int c0, int c1, int c2) {
  const long chunks = (K + 7) / 8;
  for (long r = blockIdx.y; r < rows; r += gridDim.y) {
    const double inv = 64.0 / scale[r];
    const c128 *x = X + r * ld;
    for (long ch = (long)blockIdx.x * 256 + threadIdx.x; ch < chunks; ch += (long)gridDim.x * 256) {
      double y[16];
#pragma unroll
      for (int j = 0; j < 8; ++j) {
        const long k = ch * 8 + j;
        const c128 v = k < K ? x[k] : czero();
        y[2 * j] = v.x * inv;
        y[2 * j + 1] = v.y * inv;
      }
      for (int t = 0; t < s; ++t) {
        int q[16];
#pragma unroll
        for (int j = 0; j < 16; ++j) {
          const double qq = rint(y[j]);
          y[j] = (y[j] - qq) * 128.0;
          q[j] = (int)qq;
        }
        uint32_t w0[4], w1[4];
#pragma unroll
        for (int j = 0; j < 4; ++j) {
          // complex numbers 2j, 2j+1 -> four bytes per 32-bit word
          const int ar = q[4 * j], ai = q[4 * j + 1], br = q[4 * j + 2], bi = q[4 * j + 3];
          if (MODE == 0) {
            w0[j] = (uint32_t)(ar & 0xff) | ((uint32_t)(ai & 0xff) << 8) | ((uint32_t)(br & 0xff) << 16) | ((uint32_t)(bi & 0xff) << 24);
          } else {
            w0[j] = (uint32_t)(ar & 0xff) | ((uint32_t)((c0 * ai) & 0xff) << 8) | ((uint32_t)(br & 0xff) << 16) |
                    ((uint32_t)((c0 * bi) & 0xff) << 24);
            w1[j] = (uint32_t)((c1 * ai) & 0xff) | ((uint32_t)((c2 * ar) & 0xff) << 8) | ((uint32_t)((c1 * bi) & 0xff) << 16) |
                    ((uint32_t)((c2 * br) & 0xff) << 24);
          }
        }
        if (MODE == 0) {
          *(uint4 *)(out + (size_t)t * slice_stride + (size_t)r * ldp + ch * 16) = make_uint4(w0[0], w0[1], w0[2], w0[3]);
        } else {
          *(uint4 *)(out + (size_t)t * slice_stride + (size_t)(2 * r) * ldp + ch * 16) = make_uint4(w0[0], w0[1], w0[2], w0[3]);
          *(uint4 *)(out + (size_t)t * slice_stride + (size_t)(2 * r + 1) * ldp + ch * 16) = make_uint4(w1[0], w1[1], w1[2], w1[3]);
        }
      }
    }
  }
}
// B operand stored [K][N] (N contiguous): 64 k x 32 n tiles transposed through shared memory into the same two-rows-per-column
// K-major layout.  256 threads: tx = column in the tile, ty = 0..7 -> k = ty, ty + 8, ...
// AFMT: the A-operand format instead (ONE row [re, im]_k per column n: the slices of the operand's transpose, zgemm_oz_register_t).
template <bool AFMT>
__global__ void __launch_bounds__(256) oz_slice_kn_kernel(const c128 *__restrict__ X, long ld, long krows, long ncols, int s,
                                                          const double *__restrict__ scale, int8_t *__restrict__ out, long ldp,
                                                          size_t slice_stride, int c0, int c1, int c2) {
  __shared__ __align__(16) int8_t tile[64][132];
  const long k0 = (long)blockIdx.y * 64, n0 = (long)blockIdx.x * 32;
  const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;
  const long n = n0 + tx;
  const double inv = n < ncols ? 64.0 / scale[n] : 0.0;
  double yr[8], yi[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    const long k = k0 + ty + 8 * i;
    c128 v = czero();
    if (k < krows && n < ncols) v = X[k * ld + n];
    yr[i] = v.x * inv;
    yi[i] = v.y * inv;
  }
  for (int t = 0; t < s; ++t) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      const double qr = rint(yr[i]), qi = rint(yi[i]);
      yr[i] = (yr[i] - qr) * 128.0;
      yi[i] = (yi[i] - qi) * 128.0;
      const int ir = (int)qr, ii = (int)qi, kk = 2 * (ty + 8 * i);
      if (AFMT) {
        tile[tx][kk] = (int8_t)ir;
        tile[tx][kk + 1] = (int8_t)ii;
      } else {
        tile[2 * tx][kk] = (int8_t)ir;
        tile[2 * tx][kk + 1] = (int8_t)(c0 * ii);
        tile[2 * tx + 1][kk] = (int8_t)(c1 * ii);
        tile[2 * tx + 1][kk + 1] = (int8_t)(c2 * ir);
      }
    }
    __syncthreads();
    // 64 (32) rows x 128 bytes: warp w writes rows w, w + 8, ...; lane = 4 bytes
    const int nrows = AFMT ? 32 : 64;
    for (int row = ty; row < nrows; row += 8) {
      const long nn = (AFMT ? n0 : 2 * n0) + row;
      const long kb = 2 * k0 + 4 * tx;
      if (nn < (AFMT ? ncols : 2 * ncols) && kb < ldp)
        *(uint32_t *)(out + (size_t)t * slice_stride + (size_t)nn * ldp + kb) = *(const uint32_t *)&tile[row][4 * tx];
    }
    __syncthreads();
  }
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
EncodeTiledFn oz_get_encode() {
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
// 3-D map {k (bytes), row, slice} over INT8 slices [s][rows][ldp]: box = 128 bytes x box_rows rows x 1 slice, SWIZZLE_128B;
// out-of-range rows / k read as zero
bool oz_make_map(CUtensorMap *tm, const int8_t *slices, long k2, long rows, long ldp, int s, int box_rows) {
  EncodeTiledFn enc = oz_get_encode();
  if (!enc || (ldp & 15)) return false;
  cuuint64_t dims[3] = {(cuuint64_t)k2, (cuuint64_t)rows, (cuuint64_t)s};
  cuuint64_t strides[2] = {(cuuint64_t)ldp, (cuuint64_t)rows * (cuuint64_t)ldp};
  cuuint32_t box[3] = {(cuuint32_t)OZ_BK, (cuuint32_t)box_rows, 1u};
  cuuint32_t es[3] = {1u, 1u, 1u};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, (void *)slices, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// row stride of the slices: 2K bytes rounded up to 128, so that every 128-byte box row is four whole 32-byte sectors
long oz_ldp(long K) { return (2 * K + 127) & ~127L; }

// slices + scales of the A operand ([rows][K], K contiguous) into caller-provided storage
cudaError_t oz_slice_a(cudaStream_t st, const c128 *A, long lda, long rows, long K, int s, int8_t *slices, double *scale) {
  const long ldp = oz_ldp(K);
  oz_rowmax_kernel<<<(unsigned)std::min<long>(rows, 148 * 16), 256, 0, st>>>(A, lda, rows, K, scale);
  dim3 grid((unsigned)std::min<long>(((K + 7) / 8 + 255) / 256, 64), (unsigned)std::min<long>(rows, 32768));
  oz_slice_rows_kernel<0><<<grid, 256, 0, st>>>(A, lda, rows, K, s, scale, slices, ldp, (size_t)rows * ldp, 1, 1, 1);
  cclr_count_launch(2);
  return cudaGetLastError();
}
// slices + scales of the B operand (N complex columns -> 2N rows of 2K bytes) with the sign pattern of the real embedding
cudaError_t oz_slice_b(cudaStream_t st, const c128 *B, long ldb, bool b_is_kn, long N, long K, int s, bool conjA, bool conjB,
                       int8_t *slices, double *scale) {
  const long ldp = oz_ldp(K);
  const int sa = conjA ? -1 : 1, sb = conjB ? -1 : 1;
  const int c0 = -sa * sb, c1 = sb, c2 = sa;
  if (!b_is_kn) {
    oz_rowmax_kernel<<<(unsigned)std::min<long>(N, 148 * 16), 256, 0, st>>>(B, ldb, N, K, scale);
    dim3 grid((unsigned)std::min<long>(((K + 7) / 8 + 255) / 256, 64), (unsigned)std::min<long>(N, 32768));
    oz_slice_rows_kernel<1><<<grid, 256, 0, st>>>(B, ldb, N, K, s, scale, slices, ldp, (size_t)(2 * N) * ldp, c0, c1, c2);
    cclr_count_launch(2);
  } else {
    cudaError_t e = cudaMemsetAsync(scale, 0, (size_t)N * sizeof(double), st);
    if (e != cudaSuccess) return e;
    const long kslab = 256;
    dim3 g1((unsigned)((N + 255) / 256), (unsigned)((K + kslab - 1) / kslab));
    oz_colmax_kernel<<<g1, 256, 0, st>>>(B, ldb, K, N, kslab, (unsigned long long *)scale);
    oz_scale_finalize_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(scale, N);
    dim3 g2((unsigned)((N + 31) / 32), (unsigned)((K + 63) / 64));
    oz_slice_kn_kernel<false><<<g2, 256, 0, st>>>(B, ldb, K, N, s, scale, slices, ldp, (size_t)(2 * N) * ldp, c0, c1, c2);
    cclr_count_launch(3);
  }
  return cudaGetLastError();
}

cudaError_t oz_ensure(cudaStream_t st, void **ptr, size_t *have, size_t need) {
  if (*have >= need) return cudaSuccess;
  cudaError_t e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return e;
  if (*ptr) cudaFree(*ptr);
  *ptr = nullptr;
  *have = 0;
  e = cudaMalloc(ptr, need);
  if (e != cudaSuccess) return e;
  *have = need;
  return cudaSuccess;
}

}  // namespace

bool zgemm_oz_supported(int M, int N, int K) {
  // what the kernel can do: 2K * 64^2 must leave room for one slice pair in an S32 accumulator
  return M >= 1 && N >= 1 && K >= 1 && (long)K < (1L << 17);
}

bool zgemm_oz_eligible(int M, int N, int K) {
  // large contractions only: at least 64 output tiles of 256 x 256 reals (below that the 148 SMs are not filled and the DMMA kernels
  // with their smaller tiles win: config 2's ladder is 13 tiles), and 2K * 64^2 must leave room for one pair in an S32 accumulator
  if (M < 512 || N < 32 || K < 512 || (long)K >= (1L << 17)) return false;
  return (long)((M + 255) / 256) * ((2L * N + 255) / 256) >= 64;
}

// How many slices a constant operand needs.  The error of the product is ~ 2^(-7s) rho_A rho_B with rho = (power-of-two row scale) /
// (row rms), taken as the rms over the rows (rows without outliers: rho = 4.5 ... 9 for Gaussian entries; measured 1e-11 at s = 6).
// Assuming the other operand is no worse, s is the smallest count with 2^(-7s) rho^2 <= 3e-11 -- 6 for the integrals of this task, 7
// or 8 for operands with a wider range inside their rows, 0 (do not use the integer path) beyond that.
cudaError_t zgemm_oz_suggest_slices(cudaStream_t st, const c128 *A, long lda, long rows, long K, int *slices, double *rho_out) {
  *slices = 0;
  double *acc = nullptr, h[2] = {0.0, 0.0};
  cudaError_t err = cudaMalloc((void **)&acc, 2 * sizeof(double));
  if (err != cudaSuccess) return err;
  err = cudaMemsetAsync(acc, 0, 2 * sizeof(double), st);
  if (err == cudaSuccess) {
    oz_rowstats_kernel<<<(unsigned)std::min<long>(rows, 148 * 16), 256, 0, st>>>(A, lda, rows, K, acc);
    cclr_count_launch();
    err = cudaMemcpyAsync(h, acc, 2 * sizeof(double), cudaMemcpyDeviceToHost, st);
  }
  if (err == cudaSuccess) err = cudaStreamSynchronize(st);
  cudaFree(acc);
  if (err != cudaSuccess) return err;
  const double rho2 = h[1] > 0.0 ? h[0] / h[1] : 1.0;
  if (rho_out) *rho_out = std::sqrt(rho2);
  for (int s = 6; s <= 8; ++s)
    if (std::ldexp(rho2, -7 * s) <= 3e-11) { *slices = s; break; }
  return cudaSuccess;
}

void zgemm_oz_release(OzWorkspace *ow) {
  if (!ow) return;
  for (auto &e : ow->persist) {
    if (e.slices) cudaFree(e.slices);
    if (e.scale) cudaFree(e.scale);
  }
  ow->persist.clear();
  ow->persist_bytes = 0;
  for (int i = 0; i < 2; ++i) {
    if (ow->scratch[i]) cudaFree(ow->scratch[i]);
    if (ow->scale[i]) cudaFree(ow->scale[i]);
    ow->scratch[i] = nullptr; ow->scale[i] = nullptr;
    ow->scratch_bytes[i] = ow->scale_bytes[i] = 0;
  }
}

cudaError_t zgemm_oz_register(cudaStream_t st, OzWorkspace *ow, const c128 *A, long lda, long rows, long K) {
  if (!ow || ow->slices < 2 || ow->slices > 8) return cudaErrorInvalidValue;
  OzEntry e;
  e.key = A; e.ld = lda; e.rows = rows; e.K = K; e.s = ow->slices;
  const long ldp = oz_ldp(K);
  const size_t bytes = (size_t)e.s * (size_t)rows * (size_t)ldp;
  cudaError_t err = cudaMalloc((void **)&e.slices, bytes);
  if (err != cudaSuccess) return err;
  err = cudaMalloc((void **)&e.scale, (size_t)rows * sizeof(double));
  if (err != cudaSuccess) { cudaFree(e.slices); return err; }
  err = oz_slice_a(st, A, lda, rows, K, e.s, e.slices, e.scale);
  if (err != cudaSuccess) { cudaFree(e.slices); cudaFree(e.scale); return err; }
  e.bytes = bytes + (size_t)rows * sizeof(double);
  ow->persist.push_back(e);
  ow->persist_bytes += e.bytes;
  return cudaSuccess;
}

// The product proper: C'[M][N] = alpha * A'[M][K] * opB(B)[K][N] + beta * C' with A' given as slices + scales (the conjugation of A'
// is folded into the sign pattern of the B slices), C' addressed as C[m * c_rs + n * c_cs].
static cudaError_t oz_run(cudaStream_t st, int M, int N, int K, c128 alpha, const int8_t *sa_sl, const double *sa_sc, bool conjA,
                          const c128 *B, long ldb, bool b_is_kn, bool conjB, c128 beta, c128 *C, long c_rs, long c_cs, OzWorkspace *ow) {
  const int s_all = ow->slices;
  // the leading slices of a decomposition are the decomposition with fewer slices (the slicing is sequential), so a product at
  // reduced precision reads the first `active` slices of the registered operands and slices the per-call side that far only
  const int s = (ow->active >= 2 && ow->active < s_all) ? ow->active : s_all;
  const long ldp = oz_ldp(K);
  // ---- B: always sliced per call (the trial vector side) ----
  cudaError_t err = oz_ensure(st, (void **)&ow->scratch[1], &ow->scratch_bytes[1], (size_t)s_all * 2 * N * ldp);
  if (err != cudaSuccess) return err;
  err = oz_ensure(st, (void **)&ow->scale[1], &ow->scale_bytes[1], (size_t)N * sizeof(double));
  if (err != cudaSuccess) return err;
  if (ow->ev_b[0]) cudaEventRecord(ow->ev_b[0], st);
  err = oz_slice_b(st, B, ldb, b_is_kn, N, K, s, conjA, conjB, ow->scratch[1], ow->scale[1]);
  if (err != cudaSuccess) return err;
  if (ow->ev_b[1]) cudaEventRecord(ow->ev_b[1], st);

  OzArgs a{};
  a.M = M; a.N2 = 2 * N;
  // tile width: each CTA receives (256 + BN) x 128 bytes per k block through its ~64 B/clk L2 port and spends 4 BN cycles of the
  // INT8 pipe on them, so the cost of a width is  tile columns x max(4 BN, 2 (256 + BN))  -- wide tiles unless they pad 2N badly
  int BN = ow->force_bn;
  if (BN < 16 || BN > 256 || (BN & 15)) {
    long best = -1;
    for (int bn = 256; bn >= 64; bn -= 16) {
      const long cost = (long)((a.N2 + bn - 1) / bn) * std::max(4 * bn, 2 * (256 + bn));
      if (best < 0 || cost < best) { best = cost; BN = bn; }
    }
  }
  a.BN = BN;
  a.stage_bytes = OZ_A_BYTES + BN * OZ_BK;
  a.nstages = std::min(OZ_MAX_STAGES, (OZ_MAX_SMEM - 1024 - 256) / a.stage_bytes);

  const int smem_bytes = 1024 + a.nstages * a.stage_bytes + 256;
  const int tiles_n = (a.N2 + BN - 1) / BN, tiles_m = (M + OZ_BM - 1) / OZ_BM;
  a.nkb = (int)((2L * K + OZ_BK - 1) / OZ_BK);
  // accumulation groups: anti-diagonals d = t + u <= s - 1, split so that pairs * 2K * 64^2 < 2^31
  const long cap = ((1L << 31) - 1) / (2L * K * 4096L);
  if (cap < 1) return cudaErrorInvalidValue;
  int np = 0, ng = 0;
  for (int d = 0; d < s; ++d) {
    int in_group = 0;
    for (int t = 0; t <= d; ++t) {
      if (in_group == cap) { a.gend[ng] = (unsigned char)np; a.gdiag[ng] = (unsigned char)d; ++ng; in_group = 0; }
      a.pt[np] = (unsigned char)t; a.pu[np] = (unsigned char)(d - t); ++np; ++in_group;
    }
    a.gend[ng] = (unsigned char)np; a.gdiag[ng] = (unsigned char)d; ++ng;
    if (ng >= OZ_MAX_GROUPS - 8) return cudaErrorInvalidValue;
  }
  a.npairs = np; a.ngroups = ng;
  // instruction descriptor (kind::i8): D = S32, A = B = signed 8 bit, both K-major, M = 128, N = BN
  a.idesc = (2u << 4) | (1u << 7) | (1u << 10) | (((uint32_t)BN >> 3) << 17) | ((128u >> 4) << 24);
  a.alpha = alpha; a.beta = beta; a.C = C; a.c_rs = c_rs; a.c_cs = c_cs;
  a.sa = sa_sc; a.sb = ow->scale[1];
  CUtensorMap tA, tB;
  if (!oz_make_map(&tA, sa_sl, 2L * K, M, ldp, s, OZ_BM) || !oz_make_map(&tB, ow->scratch[1], 2L * K, 2L * N, ldp, s, BN))
    return cudaErrorInvalidValue;
  static std::atomic<unsigned long long> configured{0};
  int dev = 0;
  err = cudaGetDevice(&dev);
  if (err != cudaSuccess) return err;
  if (dev >= 64 || !((configured.load() >> dev) & 1ull)) {
    err = cudaFuncSetAttribute((const void *)zgemm_oz_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, OZ_MAX_SMEM);
    if (err != cudaSuccess) return err;
    if (dev < 64) configured.fetch_or(1ull << dev);
  }
  // cluster shape c_m x c_n (tiles along M x along N that share their operand tiles by multicast): up to 8 tile columns can form
  // ONE cluster row (the A panel then leaves HBM exactly once -- without it the tile columns of a panel drift apart in time and
  // re-read it: 538 GB instead of 104 GB at config 4, profiles/r02_oz_*); more tile columns are covered by c_m x 1 or 4 x 2
  // clusters.  Clusters must fit the GPCs (8-, 6-, 5-CTA clusters keep 120, 132, 130 of the 148 SMs busy), and every cluster takes
  // the same time, so at the mid-size configs the shape is picked by the number of WAVES ceil(clusters / resident clusters) -- the
  // last partial wave is what differs (ring of config 5: 3 waves of 4 x 2 clusters, 2 waves of 6 x 1: 2.7 -> 1.9 ms) -- and at
  // large sizes by the operand traffic (below)
  struct Shape { int cm, cn; };
  Shape cand[12];
  int ncand = 0;
  if (ow->force_cm >= 1 && ow->force_cn >= 1 && ow->force_cm * ow->force_cn <= 8) cand[ncand++] = {ow->force_cm, ow->force_cn};
  else if (tiles_n <= 8) {
    for (int d = tiles_n; d >= 1; --d)
      if (tiles_n % d == 0) cand[ncand++] = {1, d};
  } else {
    const Shape all[10] = {{5, 1}, {4, 2}, {6, 1}, {4, 1}, {8, 1}, {3, 1}, {2, 2}, {2, 1}, {1, 2}, {1, 1}};
    for (const Shape &c : all)
      if (c.cm <= tiles_m || c.cm == 1) cand[ncand++] = c;
  }
  auto make_cfg = [&](const Shape &c, cudaLaunchConfig_t &cfg, cudaLaunchAttribute *attr) {
    const int ct_m = (tiles_m + c.cm - 1) / c.cm, ct_n = (tiles_n + c.cn - 1) / c.cn;
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3((unsigned)((long)ct_m * ct_n * c.cm * c.cn), 1, 1);
    cfg.blockDim = dim3(OZ_THREADS, 1, 1);
    cfg.dynamicSmemBytes = (size_t)smem_bytes;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)(c.cm * c.cn);
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = c.cm * c.cn > 1 ? 1 : 0;
    return ct_n;
  };
  int resident[12];
  double waves[12], traffic[12];
  const int sms = zgemm_num_sms();
  for (int i = 0; i < ncand; ++i) {
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[1];
    make_cfg(cand[i], cfg, attr);
    int active = 0;
    if (cand[i].cm * cand[i].cn == 1) active = sms;
    else if (cudaOccupancyMaxActiveClusters(&active, (const void *)zgemm_oz_kernel, &cfg) != cudaSuccess) { cudaGetLastError(); active = 0; }
    resident[i] = std::min(active * cand[i].cm * cand[i].cn, sms);
    const long ncl = (long)((tiles_m + cand[i].cm - 1) / cand[i].cm) * ((tiles_n + cand[i].cn - 1) / cand[i].cn);
    const long res_cl = std::max(1, resident[i] / (cand[i].cm * cand[i].cn));
    waves[i] = resident[i] >= 1 ? (double)((ncl + res_cl - 1) / res_cl) : 1e30;
    // operand bytes a tile pulls through L2 / HBM per k block ~ 1 / c_n (its A tile is shared by c_n CTAs) + 1 / c_m (B tile)
    traffic[i] = 1.0 / cand[i].cn + 1.0 / cand[i].cm;
    // unclustered CTAs re-read their operands from HBM (see above): only when nothing else can be scheduled
    if (cand[i].cm * cand[i].cn == 1 && ncand > 1 && tiles_n > 1) waves[i] = 1e29;
  }
  // Few waves (mid-size products): the last partial wave decides -- fewest waves wins, ties to the shape that shares more.
  // Many waves (>= 16 for every shape: config 4): the chip runs at its power cap and the total rate is the same for every shape
  // that fills 3/4 of the SMs (ring of config 4: 78-80 ms for 4 x 2, 5 x 1, 6 x 1, 8 x 1), falling with the operand traffic
  // (2 x 2: 84 ms, 1 x 2: 92 ms) -- and a shape that reads twice the bytes (5 x 1: 233 GB per call against 124 GB for 4 x 2)
  // takes power from the kernels around it (the ladder after it: 78 -> 86 ms) -- so the shape that shares most wins.
  double minw = 1e30;
  for (int i = 0; i < ncand; ++i) minw = std::min(minw, waves[i]);
  if (minw >= 16.0 && ncand > 1 && !(ow->force_cm >= 1 && ow->force_cn >= 1)) {
    for (int i = 0; i < ncand; ++i)
      waves[i] = (waves[i] < 1e29 && resident[i] * 4 >= sms * 3) ? traffic[i] + 1e-3 * waves[i] : 1e28 + waves[i];
  } else {
    for (int i = 0; i < ncand; ++i)
      if (waves[i] < 1e29) waves[i] += 1e-3 * traffic[i];
  }
  int order[12];
  for (int i = 0; i < ncand; ++i) order[i] = i;
  std::stable_sort(order, order + ncand, [&](int x, int y) { return waves[x] < waves[y]; });
  err = cudaErrorLaunchFailure;
  bool launched = false;
  for (int q = 0; q < ncand && !launched; ++q) {
    {
      const int i = order[q];
      if (resident[i] < 1) continue;
      cudaLaunchConfig_t cfg;
      cudaLaunchAttribute attr[1];
      a.c_m = cand[i].cm; a.c_n = cand[i].cn;
      a.ctiles_n = make_cfg(cand[i], cfg, attr);
      err = cudaLaunchKernelEx(&cfg, zgemm_oz_kernel, tA, tB, a);
      if (err == cudaSuccess) launched = true; else cudaGetLastError();
    }
  }
  if (!launched) return err;
  cclr_count_launch();
  return cudaSuccess;
}

cudaError_t zgemm_oz(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA, const c128 *B, long ldb,
                     bool b_is_kn, bool conjB, c128 beta, c128 *C, long ldc, OzWorkspace *ow) {
  if (!ow || ow->slices < 2 || ow->slices > 8 || !zgemm_oz_supported(M, N, K)) return cudaErrorInvalidValue;
  const int s = ow->slices;
  const long ldp = oz_ldp(K);
  // ---- A: registered slices, else sliced into scratch 0 ----
  const int8_t *sa_sl = nullptr;
  const double *sa_sc = nullptr;
  for (const auto &e : ow->persist)
    if (!e.transposed && e.key == A && e.ld == lda && e.rows == M && e.K == K && e.s == s) { sa_sl = e.slices; sa_sc = e.scale; }
  if (!sa_sl) {
    cudaError_t err = oz_ensure(st, (void **)&ow->scratch[0], &ow->scratch_bytes[0], (size_t)s * M * ldp);
    if (err != cudaSuccess) return err;
    err = oz_ensure(st, (void **)&ow->scale[0], &ow->scale_bytes[0], (size_t)M * sizeof(double));
    if (err != cudaSuccess) return err;
    err = oz_slice_a(st, A, lda, M, K, s, ow->scratch[0], ow->scale[0]);
    if (err != cudaSuccess) return err;
    sa_sl = ow->scratch[0]; sa_sc = ow->scale[0];
  }
  return oz_run(st, M, N, K, alpha, sa_sl, sa_sc, conjA, B, ldb, b_is_kn, conjB, beta, C, ldc, 1, ow);
}

// Slices of the TRANSPOSE of a constant operand stored [K][N] (N contiguous, leading dimension ldb): rows n = [re, im]_k, scaled
// by the column maxima.  For products in which the big constant matrix is the B operand (the transposed ladder of the left
// transform, O2T[(ij);(ef)] = l2T[(ij);(ab)] . W[(ab);(ef)]): zgemm_oz_bt then runs C^T = B^T . A^T with these slices on the A side.
cudaError_t zgemm_oz_register_t(cudaStream_t st, OzWorkspace *ow, const c128 *B, long ldb, long K, long N) {
  if (!ow || ow->slices < 2 || ow->slices > 8) return cudaErrorInvalidValue;
  OzEntry e;
  e.key = B; e.ld = ldb; e.rows = N; e.K = K; e.s = ow->slices; e.transposed = true;
  const long ldp = oz_ldp(K);
  const size_t bytes = (size_t)e.s * (size_t)N * (size_t)ldp;
  cudaError_t err = cudaMalloc((void **)&e.slices, bytes);
  if (err != cudaSuccess) return err;
  err = cudaMalloc((void **)&e.scale, (size_t)N * sizeof(double));
  if (err != cudaSuccess) { cudaFree(e.slices); return err; }
  err = cudaMemsetAsync(e.scale, 0, (size_t)N * sizeof(double), st);
  if (err == cudaSuccess) {
    const long kslab = 256;
    dim3 g1((unsigned)((N + 255) / 256), (unsigned)((K + kslab - 1) / kslab));
    oz_colmax_kernel<<<g1, 256, 0, st>>>(B, ldb, K, N, kslab, (unsigned long long *)e.scale);
    oz_scale_finalize_kernel<<<(unsigned)((N + 255) / 256), 256, 0, st>>>(e.scale, N);
    dim3 g2((unsigned)((N + 31) / 32), (unsigned)((K + 63) / 64));
    oz_slice_kn_kernel<true><<<g2, 256, 0, st>>>(B, ldb, K, N, e.s, e.scale, e.slices, ldp, (size_t)N * ldp, 1, 1, 1);
    cclr_count_launch(3);
    err = cudaGetLastError();
  }
  if (err != cudaSuccess) { cudaFree(e.slices); cudaFree(e.scale); return err; }
  e.bytes = bytes + (size_t)N * sizeof(double);
  ow->persist.push_back(e);
  ow->persist_bytes += e.bytes;
  return cudaSuccess;
}

bool zgemm_oz_has_bt(const OzWorkspace *ow, const c128 *B, long ldb, int N, int K) {
  if (!ow) return false;
  for (const auto &e : ow->persist)
    if (e.transposed && e.key == B && e.ld == ldb && e.rows == N && e.K == K && e.s == ow->slices) return true;
  return false;
}

// C[M][N] = alpha opA(A)[M][K] opB(B)[K][N] + beta C with B stored [K][N] and registered by zgemm_oz_register_t: computed as
// C^T = opB(B)^T . opA(A)^T -- B's transposed slices are the A side, A ([M][K], K contiguous) is the per-call side, and the
// epilogue stores transposed (consecutive lanes = consecutive n: coalesced).
cudaError_t zgemm_oz_bt(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA, const c128 *B, long ldb,
                        bool conjB, c128 beta, c128 *C, long ldc, OzWorkspace *ow) {
  if (!ow || ow->slices < 2 || ow->slices > 8 || !zgemm_oz_supported(N, M, K)) return cudaErrorInvalidValue;
  for (const auto &e : ow->persist)
    if (e.transposed && e.key == B && e.ld == ldb && e.rows == N && e.K == K && e.s == ow->slices)
      return oz_run(st, N, M, K, alpha, e.slices, e.scale, conjB, A, lda, false, conjA, beta, C, 1, ldc, ow);
  return cudaErrorInvalidValue;
}
