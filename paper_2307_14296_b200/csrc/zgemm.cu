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
//   * 3M kernel (zgemm3m_kernel) for the large contractions: T1 = Ar Br, T2 = Ai Bi, T3 = (Ar + Ai)(Br + Bi) on 8 x 8-complex
//     DMMA tiles with three real accumulator tiles per complex tile -- 3 DMMA per 8 x 8 x 4 complex block instead of 4.
//   * operands are staged by TMA (cp.async.bulk.tensor, FLOAT64 tensor maps over the interleaved data, boxes of
//     128 B x rows, SWIZZLE_128B) into a STAGES-deep ring guarded by full/empty mbarriers; one producer warp,
//     (BM/WM)*(BN/WN) consumer warps.  Fragment loads are single conflict-free LDS.128 per complex element:
//       - K-contiguous operand rows: the 8 rows a quarter-warp touches are permuted (rmap) so the two rows of a
//         quarter-warp differ in address bit 9 and the swizzle separates them;
//       - N-contiguous B ([K][N]): the four k rows of a quarter-warp are separated by the swizzle directly.
//   * ragged M, N, K: TMA zero-fills out-of-bounds loads; stores are guarded.
//   * tile shape per call (BM 128 | 64, BN 32..64), a 1-D tile grid whose last partial wave is split along K (partials in a
//     workspace + a deterministic reduce kernel; the same mechanism serves tall-K / tiny-MN contractions), and
//     matrix-vector kernels for N = 1 / M = 1.
#include "common.cuh"
#include <algorithm>
#include <atomic>
#include <cmath>
#include <mutex>

namespace {

constexpr int ZG_BK = 16, ZG_STAGES = 4;   // K chunk, TMA ring depth; CTA tile BM x BN with BM = 128 | 64, BN = 8*NG, NG = 4..8

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
  // launch geometry: a 1-D grid of CTAs over the (batch, tile_m, tile_n) tiles, tile_n fastest.  The first `main_tiles`
  // tiles are computed whole by one CTA each; every remaining ("tail") tile is split along K over `tail_splits` CTAs
  // which write partial tiles to `partial` ([tail tile][split][BM*BN]) for zgemm_tail_reduce_kernel.  This removes the
  // wave-quantisation loss of the last partial wave (and is the split-K path of tall-K / tiny-MN contractions when
  // main_tiles == 0).
  int tiles_m, tiles_n;
  int group_m;         // raster: tiles are walked in groups of group_m tile rows, tile_m fastest inside a group, then tile_n
                       // (1 = tile_n fastest over a whole tile row, tiles_m = tile_m fastest over a whole column): the CTAs
                       // running together cover a group_m x (SMs / group_m) block of tiles and share its panels through L2
  int main_tiles, tail_splits, chunks_per_split;
  c128 *partial;
};

// tile id -> (batch, tile_m, tile_n) in the raster order of ZgemmArgs::group_m
__host__ __device__ __forceinline__ void tile_coords(const ZgemmArgs &p, int tile, int &batch, int &tile_m, int &tile_n) {
  const int tiles_mn = p.tiles_m * p.tiles_n;
  batch = tile / tiles_mn;
  const int t = tile - batch * tiles_mn;
  const int per_group = p.group_m * p.tiles_n;
  const int grp = t / per_group, r = t - grp * per_group;
  const int m0 = grp * p.group_m;
  const int gsz = p.tiles_m - m0 < p.group_m ? p.tiles_m - m0 : p.group_m;
  tile_m = m0 + r % gsz;
  tile_n = r / gsz;
}

// ---------------------------------------------------------------------------------------------------------------
// kernel
// ---------------------------------------------------------------------------------------------------------------
template <int BM, int BN, int BK, int WM, int WN, int STAGES, bool BKN>
__global__ void __launch_bounds__((BM / WM) * (BN / WN) * 32 + 128, 1)
zgemm_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB, const ZgemmArgs p) {
  constexpr int WARPS_M = BM / WM, WARPS_N = BN / WN, NCW = WARPS_M * WARPS_N;
  constexpr int MI = WM / 8, NG = WN / 4;          // DMMA tiles per warp: MI row groups x NG column groups
  constexpr int A_BYTES = BM * BK * 16, B_BYTES = BN * BK * 16, STAGE_BYTES = A_BYTES + B_BYTES;
  static_assert(BK % 8 == 0 && BM % 8 == 0 && BN % 8 == 0 && WM % 8 == 0 && WN % 4 == 0, "tile shape");
  static_assert(NCW % 4 == 0, "consumer warps must form whole warpgroups (setmaxnreg)");
  constexpr int CONSUMER_REGS = (NCW == 8) ? 232 : 200;

  extern __shared__ __align__(1024) uint8_t smem_raw[];
  // 1024-byte alignment is required by SWIZZLE_128B; dynamic smem base is only guaranteed 16 B, so align by hand.
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;   // full[STAGES], empty[STAGES], 8 B each

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int tile = (int)blockIdx.x, split = 0;
  const bool is_tail = tile >= p.main_tiles;
  if (is_tail) {
    const int r = tile - p.main_tiles;
    tile = p.main_tiles + r / p.tail_splits;
    split = r % p.tail_splits;
  }
  int batch, tile_m, tile_n;
  tile_coords(p, tile, batch, tile_m, tile_n);
  const int nchunks_total = (p.K + BK - 1) / BK;
  int chunk0 = 0, nchunks = nchunks_total;
  if (is_tail) {
    chunk0 = split * p.chunks_per_split;
    nchunks = nchunks_total - chunk0;
    if (nchunks > p.chunks_per_split) nchunks = p.chunks_per_split;
    if (nchunks < 0) nchunks = 0;
  }

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
  const int wm = warp / WARPS_N, wn = warp % WARPS_N;
  const int par = gid & 1, nb4 = gid >> 1;
  const int wpar = ((wn * WN) >> 2) & 1;            // WN may be an odd multiple of 4: parity of the warp's first 4-row group
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
      // row k (inside a box of BK rows: + kb*8*128 per 8-k block), col n = wn*WN + 4g + nb4.  For WN a multiple of 8 the box
      // of the warp's first column and the lane part (nb4 ^ k) of the swizzled chunk are folded in here; the loop then only
      // adds compile-time terms and flips bit 6 for odd g
      b_off[s4] = (WN % 8 == 0) ? (uint32_t)(((wn * WN) >> 3) * (BK * 128) + k * 128 + ((nb4 ^ k) << 4)) : (uint32_t)(k * 128);
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
            const int n7 = (((g & 1) ^ wpar) << 2) | nb4;   // (row & 7) of row = wn*WN + 4g + nb4
            addr = sB + kb * (BN * 128) + g * 512 + (b_off[s4] ^ (uint32_t)(n7 << 4));
          } else if constexpr (WN % 8 == 0) {
            // n = wn*WN + 4g + nb4 with wn*WN a multiple of 8: box (n >> 3) = wn*WN/8 + g/2, (n & 7) = 4 (g & 1) + nb4
            addr = sB + (uint32_t)(g >> 1) * (BK * 128) + kb * 1024 + (b_off[s4] ^ (uint32_t)((g & 1) << 6));
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
  // tail tiles: raw partial sums into the workspace tile [BM][BN] of (tail tile, split); main tiles: C directly
  const bool partial = is_tail;
  c128 *Cb = partial ? p.partial + ((size_t)(blockIdx.x - p.main_tiles)) * (size_t)(BM * BN) -
                           ((size_t)tile_m * BM * BN + (size_t)tile_n * BN)
                     : p.C + (size_t)batch * p.sc;
  const long ldc = partial ? (long)BN : p.ldc;
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


// ---------------------------------------------------------------------------------------------------------------
// 3M kernel: T1 = Ar Br, T2 = Ai Bi, T3 = (Ar + Ai)(Br + Bi); C = (T1 - T2) + i (T3 - T1 - T2).
//
// One DMMA tile is 8 rows x 8 COMPLEX columns (no re/im doubling of the columns), three real accumulator tiles per complex
// tile: 3 DMMA per 8 x 8 x 4 complex block instead of 4.  CTA tile 128 x BN (BN = 32 | 48), 8 consumer warps (4 x 2, warp tile
// 32 x BN/2), same TMA ring as the 4M kernel.  The sums Ar + Ai, Br + Bi are formed in registers from the LDS.128 fragments
// (7 DADD per 36 DMMA and k-step).  Physical column of DMMA column g is 8*g3 + rmap(g) (the row permutation) so that the B
// fragment loads stay bank-conflict free under the 128-byte swizzle.
// What the DADDs cost, measured on B200 at config 4 (profiles/r02_3m_sum_experiments.md): ladder 206.4 ms as is, 195.2 ms with
// the sums deleted (wrong results; the bound), 205.5 ms with the sums formed once per CTA one stage ahead through shared-memory
// planes (11 DADD per 144 DMMA and warp, nothing in the DMMAs' dependency chain; ring 195 vs 190 ms), 359 ms with the sums
// formed by the idle producer warps (their DADDs starve behind the consumers' DMMAs).  I.e. the cost is the DADDs' presence on
// the FP64 datapath shared with DMMA, not their latency; only sum planes that arrive from global memory would remove it.
// ---------------------------------------------------------------------------------------------------------------
// PL = true: the sums arrive from GLOBAL memory as "sum planes" (one double Re + Im per complex element, conjugation applied;
// a persistent plane registered for the operand, or a pre-pass of zgemm() over an operand that is small next to the product):
// TMA stages them beside the tiles ([rows][8 doubles] boxes, SWIZZLE_64B, conflict-free LDS.64), the main loop has no DADD at
// all, and 3 stages of [A | B | SA | SB] replace the 4 stages of [A | B] (two stages already hide the TMA latency).
constexpr int Z3_BM = 128, Z3_BK = 16, Z3_WM = 32, Z3_NCW = 8;
__device__ __forceinline__ double lds64(uint32_t addr) {
  double v;
  asm volatile("ld.shared.f64 %0, [%1];" : "=d"(v) : "r"(addr));
  return v;
}

template <int BN, bool BKN, bool PL>
__global__ void __launch_bounds__(Z3_NCW * 32 + 128, 1)
zgemm3m_kernel(const __grid_constant__ CUtensorMap tmA, const __grid_constant__ CUtensorMap tmB,
               const __grid_constant__ CUtensorMap tmSA, const __grid_constant__ CUtensorMap tmSB, const ZgemmArgs p) {
  constexpr int BM = Z3_BM, BK = Z3_BK, STAGES = PL ? 3 : 4, WM = Z3_WM, NCW = Z3_NCW;
  constexpr int WN = BN / 2, WARPS_N = 2, MI = WM / 8, NG3 = WN / 8;
  constexpr int A_BYTES = BM * BK * 16, B_BYTES = BN * BK * 16, SA_BYTES = PL ? BM * BK * 8 : 0, SB_BYTES = PL ? BN * BK * 8 : 0;
  constexpr int STAGE_BYTES = A_BYTES + B_BYTES + SA_BYTES + SB_BYTES;
  static_assert(BN % 16 == 0 && STAGE_BYTES % 1024 == 0, "3M tile shape");

  extern __shared__ __align__(1024) uint8_t smem_raw[];
  const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t bar_base = smem_base + STAGES * STAGE_BYTES;   // full[STAGES], empty[STAGES], 8 B each

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  int tile = (int)blockIdx.x, split = 0;
  const bool is_tail = tile >= p.main_tiles;
  if (is_tail) {
    const int r = tile - p.main_tiles;
    tile = p.main_tiles + r / p.tail_splits;
    split = r % p.tail_splits;
  }
  int batch, tile_m, tile_n;
  tile_coords(p, tile, batch, tile_m, tile_n);
  const int nchunks_total = (p.K + BK - 1) / BK;
  int chunk0 = 0, nchunks = nchunks_total;
  if (is_tail) {
    chunk0 = split * p.chunks_per_split;
    nchunks = nchunks_total - chunk0;
    if (nchunks > p.chunks_per_split) nchunks = p.chunks_per_split;
    if (nchunks < 0) nchunks = 0;
  }

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
        if (PL) {   // sum planes: [rows][8 doubles] boxes
          const uint32_t sSA = sB + B_BYTES, sSB = sSA + SA_BYTES;
#pragma unroll
          for (int kb = 0; kb < BK / 8; ++kb) tma_load_3d(sSA + kb * (BM * 64), &tmSA, k0 + kb * 8, tile_m * BM, 0, full);
          if (!BKN) {
#pragma unroll
            for (int kb = 0; kb < BK / 8; ++kb) tma_load_3d(sSB + kb * (BN * 64), &tmSB, k0 + kb * 8, tile_n * BN, 0, full);
          } else {
#pragma unroll
            for (int nb = 0; nb < BN / 8; ++nb) tma_load_3d(sSB + nb * (BK * 64), &tmSB, tile_n * BN + nb * 8, k0, 0, full);
          }
        }
      }
    }
    return;
  }

  // ===== consumers =====
  asm volatile("setmaxnreg.inc.sync.aligned.u32 232;");
  const int gid = lane >> 2, tig = lane & 3;
  const int rmap = ((gid & 1) << 2) | (gid >> 1);   // row / column permutation inside an 8-group (bank-conflict free)
  const int wm = warp / WARPS_N, wn = warp % WARPS_N;
  const uint32_t sa3 = p.conjA ? 0x80000000u : 0u, sb3 = p.conjB ? 0x80000000u : 0u;
  uint32_t a_off[2], b_off[2], sa_off[2], sb_off[2];
#pragma unroll
  for (int s4 = 0; s4 < 2; ++s4) {
    const int k = 4 * s4 + tig;
    a_off[s4] = (uint32_t)((wm * WM + rmap) * 128 + ((k ^ rmap) << 4));
    b_off[s4] = !BKN ? (uint32_t)((wn * WN + rmap) * 128 + ((k ^ rmap) << 4))
                     : (uint32_t)(((wn * WN) >> 3) * (BK * 128) + k * 128 + ((rmap ^ k) << 4));
    // sum planes under SWIZZLE_64B: 16-byte chunk index ^= bits 7-8 of the address = (row >> 1) & 3 for 64-byte rows
    sa_off[s4] = (uint32_t)((wm * WM + rmap) * 64 + (((k >> 1) ^ ((rmap >> 1) & 3)) << 4) + (k & 1) * 8);
    sb_off[s4] = !BKN ? (uint32_t)((wn * WN + rmap) * 64 + (((k >> 1) ^ ((rmap >> 1) & 3)) << 4) + (k & 1) * 8)
                      : (uint32_t)(((wn * WN) >> 3) * (BK * 64) + k * 64 + (((rmap >> 1) ^ ((k >> 1) & 3)) << 4) + (rmap & 1) * 8);
  }
  double acc[MI][NG3][3][2];
#pragma unroll
  for (int i = 0; i < MI; ++i)
#pragma unroll
    for (int g = 0; g < NG3; ++g)
#pragma unroll
      for (int t = 0; t < 3; ++t) acc[i][g][t][0] = acc[i][g][t][1] = 0.0;
  for (int c = 0; c < nchunks; ++c) {
    const int s = c % STAGES;
    const uint32_t ph = (c / STAGES) & 1;
    mbar_wait(bar_base + 8 * s, ph);
    const uint32_t sA = smem_base + s * STAGE_BYTES, sB = sA + A_BYTES, sSA = sB + B_BYTES, sSB = sSA + SA_BYTES;
#pragma unroll
    for (int kb = 0; kb < BK / 8; ++kb) {
#pragma unroll
      for (int s4 = 0; s4 < 2; ++s4) {
        double ar[MI], ai[MI], as[MI];
#pragma unroll
        for (int i = 0; i < MI; ++i) {
          const double2 a = lds128(sA + kb * (BM * 128) + a_off[s4] + i * 1024);
          ar[i] = a.x;
          ai[i] = flip_sign(a.y, sa3);
          as[i] = PL ? lds64(sSA + kb * (BM * 64) + sa_off[s4] + i * 512) : ar[i] + ai[i];
        }
#pragma unroll
        for (int g = 0; g < NG3; ++g) {
          const uint32_t addr = !BKN ? sB + kb * (BN * 128) + g * 1024 + b_off[s4]
                                     : sB + g * (BK * 128) + kb * 1024 + b_off[s4];
          const double2 b = lds128(addr);
          const double br = b.x, bi = flip_sign(b.y, sb3);
          const double bs = PL ? lds64(!BKN ? sSB + kb * (BN * 64) + g * 512 + sb_off[s4] : sSB + g * (BK * 64) + kb * 512 + sb_off[s4])
                               : br + bi;
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][g][0][0], acc[i][g][0][1], ar[i], br);
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][g][1][0], acc[i][g][1][1], ai[i], bi);
#pragma unroll
          for (int i = 0; i < MI; ++i) dmma884(acc[i][g][2][0], acc[i][g][2][1], as[i], bs);
        }
      }
    }
    __syncwarp();
    if (lane == 0) mbar_arrive(bar_base + 8 * (STAGES + s));
  }
  // ===== epilogue: tail tiles write raw partial sums to the workspace, main tiles write C =====
  c128 *Cb = is_tail ? p.partial + ((size_t)(blockIdx.x - p.main_tiles)) * (size_t)(BM * BN) -
                           ((size_t)tile_m * BM * BN + (size_t)tile_n * BN)
                     : p.C + (size_t)batch * p.sc;
  const long ldc = is_tail ? (long)BN : p.ldc;
  const c128 alpha = is_tail ? make_double2(1.0, 0.0) : p.alpha;
  const c128 beta = is_tail ? make_double2(0.0, 0.0) : p.beta;
  const bool has_beta = (beta.x != 0.0) || (beta.y != 0.0);
#pragma unroll
  for (int i = 0; i < MI; ++i) {
    const int row = tile_m * BM + wm * WM + i * 8 + rmap;
    if (row >= p.M) continue;
#pragma unroll
    for (int g = 0; g < NG3; ++g) {
#pragma unroll
      for (int cc = 0; cc < 2; ++cc) {
        const int col = tile_n * BN + wn * WN + g * 8 + (cc ? 4 + tig : tig);
        if (col >= p.N) continue;
        const double t1 = acc[i][g][0][cc], t2 = acc[i][g][1][cc], t3 = acc[i][g][2][cc];
        c128 *dst = Cb + (size_t)row * ldc + col;
        c128 r = cmul(alpha, make_double2(t1 - t2, t3 - t1 - t2));
        if (has_beta) r = cadd(r, cmul(beta, *dst));
        *dst = r;
      }
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

// plane[r][c] = Re X[r][c] + (conj ? -1 : +1) Im X[r][c]  (the A_r + A_i / B_r + B_i operand of the 3M product)
__global__ void __launch_bounds__(256) sum_plane_kernel(const c128 *__restrict__ X, long ld, long rows, long cols, int conj,
                                                        double *__restrict__ plane, long ldp) {
  const double sg = conj ? -1.0 : 1.0;
  for (long r = blockIdx.y; r < rows; r += gridDim.y) {
    const c128 *x = X + r * ld;
    double *d = plane + r * ldp;
    for (long c = (long)blockIdx.x * blockDim.x + threadIdx.x; c < cols; c += (long)gridDim.x * blockDim.x) {
      const c128 v = x[c];
      d[c] = v.x + sg * v.y;
    }
  }
}

// tensor map over a [rows][cols doubles] sum plane, box = [box_rows][8 doubles = 64 B], SWIZZLE_64B
bool make_plane_map(CUtensorMap *tm, const double *base, long cols, long rows, long ldp, int box_rows) {
  EncodeTiledFn enc = get_encode();
  if (!enc || (ldp & 1)) return false;
  cuuint64_t dims[3] = {(cuuint64_t)cols, (cuuint64_t)rows, 1};
  cuuint64_t strides[2] = {(cuuint64_t)ldp * 8ull, (cuuint64_t)ldp * (cuuint64_t)rows * 8ull};
  cuuint32_t box[3] = {8u, (cuuint32_t)box_rows, 1u};
  cuuint32_t es[3] = {1u, 1u, 1u};
  CUresult r = enc(tm, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, (void *)base, dims, strides, box, es,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_64B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                   CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  return r == CUDA_SUCCESS;
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

// cudaFuncSetAttribute is per device: remember which devices a kernel instantiation has been configured on
inline cudaError_t configure_smem(const void *kern, int smem, unsigned long long &done_mask) {
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 64 && (done_mask >> dev) & 1ull) return cudaSuccess;
  e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, smem);
  if (e == cudaSuccess && dev < 64) done_mask |= 1ull << dev;
  return e;
}

template <int BM, int BN, int BK, int WM, int WN, int STAGES, bool BKN>
cudaError_t launch(cudaStream_t st, const CUtensorMap &tmA, const CUtensorMap &tmB, const ZgemmArgs &args, int ctas) {
  constexpr int threads = (BM / WM) * (BN / WN) * 32 + 128;
  constexpr int smem = STAGES * (BM + BN) * BK * 16 + 2 * STAGES * 8 + 1024;
  auto kern = zgemm_kernel<BM, BN, BK, WM, WN, STAGES, BKN>;
  static std::atomic<unsigned long long> configured{0};
  unsigned long long mask = configured.load();
  const cudaError_t e = configure_smem((const void *)kern, smem, mask);
  if (e != cudaSuccess) return e;
  configured.fetch_or(mask);
  kern<<<ctas, threads, smem, st>>>(tmA, tmB, args);
  cclr_count_launch();
  return cudaGetLastError();
}

// one instantiation per N-tile width BN = 8*NG (NG DMMA column groups per warp), for both B layouts
template <int NG>
cudaError_t launch_ng(cudaStream_t st, const CUtensorMap &tmA, const CUtensorMap &tmB, const ZgemmArgs &args, int ctas,
                      bool kn, int BM) {
  if (BM == 128)
    return kn ? launch<128, 8 * NG, ZG_BK, 32, 4 * NG, ZG_STAGES, true>(st, tmA, tmB, args, ctas)
              : launch<128, 8 * NG, ZG_BK, 32, 4 * NG, ZG_STAGES, false>(st, tmA, tmB, args, ctas);
  return kn ? launch<64, 8 * NG, ZG_BK, 16, 4 * NG, ZG_STAGES, true>(st, tmA, tmB, args, ctas)
            : launch<64, 8 * NG, ZG_BK, 16, 4 * NG, ZG_STAGES, false>(st, tmA, tmB, args, ctas);
}

// 3M kernel: 128 x BN tiles, BN = 32 | 48; PL: with sum planes from global memory
template <int BN, bool BKN, bool PL>
cudaError_t launch_3m(cudaStream_t st, const CUtensorMap &tmA, const CUtensorMap &tmB, const CUtensorMap &tmSA,
                      const CUtensorMap &tmSB, const ZgemmArgs &args, int ctas) {
  constexpr int threads = Z3_NCW * 32 + 128;
  constexpr int stages = PL ? 3 : 4;
  constexpr int smem = stages * (Z3_BM + BN) * Z3_BK * (PL ? 24 : 16) + 2 * stages * 8 + 1024;
  auto kern = zgemm3m_kernel<BN, BKN, PL>;
  static std::atomic<unsigned long long> configured{0};
  unsigned long long mask = configured.load();
  const cudaError_t e = configure_smem((const void *)kern, smem, mask);
  if (e != cudaSuccess) return e;
  configured.fetch_or(mask);
  kern<<<ctas, threads, smem, st>>>(tmA, tmB, tmSA, tmSB, args);
  cclr_count_launch();
  return cudaGetLastError();
}

// C tile = alpha * sum_splits partial + beta * C for the K-split tail tiles
__global__ void __launch_bounds__(256) zgemm_tail_reduce_kernel(const ZgemmArgs p, int BM, int BN) {
  int batch, tile_m, tile_n;
  tile_coords(p, p.main_tiles + (int)blockIdx.x, batch, tile_m, tile_n);
  const c128 *part = p.partial + (size_t)blockIdx.x * p.tail_splits * (size_t)(BM * BN);
  const bool has_beta = p.beta.x != 0.0 || p.beta.y != 0.0;
  for (int e = threadIdx.x; e < BM * BN; e += blockDim.x) {
    const int r = e / BN, c = e % BN;
    const int row = tile_m * BM + r, col = tile_n * BN + c;
    if (row >= p.M || col >= p.N) continue;
    c128 s = czero();
    for (int k = 0; k < p.tail_splits; ++k) s = cadd(s, part[(size_t)k * (BM * BN) + e]);
    c128 *dst = p.C + (size_t)batch * p.sc + (size_t)row * p.ldc + col;
    c128 out = cmul(p.alpha, s);
    if (has_beta) out = cadd(out, cmul(p.beta, *dst));
    *dst = out;
  }
}

// y[n] = sum_{k in slab} opA(a[k]) * opB(B[k][n])  (row vector times a [K][N] matrix: the M = 1 adjoint contractions of the left
// transform): one thread per column, coalesced 16-byte loads along n, K split over gridDim.y slabs whose partial rows go to
// part[slab][N] (fixed order -> deterministic) and are combined by zgemv_t_reduce_kernel.
__global__ void __launch_bounds__(128) zgemv_t_kernel(int N, int K, const c128 *__restrict__ a, int conjA,
                                                      const c128 *__restrict__ B, long ldb, int conjB, int kslab,
                                                      c128 *__restrict__ part) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  const int k0 = blockIdx.y * kslab;
  int k1 = k0 + kslab;
  if (k1 > K) k1 = K;
  const double sa = conjA ? -1.0 : 1.0, sb = conjB ? -1.0 : 1.0;
  double x0 = 0.0, y0 = 0.0, x1 = 0.0, y1 = 0.0;
  int k = k0;
  for (; k + 1 < k1; k += 2) {
    c128 u = a[k], w = B[(size_t)k * ldb + n], u2 = a[k + 1], w2 = B[(size_t)(k + 1) * ldb + n];
    u.y *= sa; w.y *= sb; u2.y *= sa; w2.y *= sb;
    x0 = fma(u.x, w.x, x0); x0 = fma(-u.y, w.y, x0); y0 = fma(u.x, w.y, y0); y0 = fma(u.y, w.x, y0);
    x1 = fma(u2.x, w2.x, x1); x1 = fma(-u2.y, w2.y, x1); y1 = fma(u2.x, w2.y, y1); y1 = fma(u2.y, w2.x, y1);
  }
  if (k < k1) {
    c128 u = a[k], w = B[(size_t)k * ldb + n];
    u.y *= sa; w.y *= sb;
    x0 = fma(u.x, w.x, x0); x0 = fma(-u.y, w.y, x0); y0 = fma(u.x, w.y, y0); y0 = fma(u.y, w.x, y0);
  }
  part[(size_t)blockIdx.y * N + n] = make_double2(x0 + x1, y0 + y1);
}

__global__ void __launch_bounds__(256) zgemv_t_reduce_kernel(int N, int slabs, const c128 *__restrict__ part, c128 alpha,
                                                             c128 beta, c128 *y) {
  const int n = blockIdx.x * blockDim.x + threadIdx.x;
  if (n >= N) return;
  c128 s = czero();
  for (int k = 0; k < slabs; ++k) s = cadd(s, part[(size_t)k * N + n]);
  c128 out = cmul(alpha, s);
  if (beta.x != 0.0 || beta.y != 0.0) out = cadd(out, cmul(beta, y[n]));
  y[n] = out;
}

// y[m] = alpha * sum_k opA(A[m][k]) * opB(b[k]) + beta * y[m]: the N = 1 contractions (S3, S4, G3, G4, F_me) are
// bandwidth-bound GEMVs; one warp per row, 16-byte loads, shuffle reduction (HBM roofline, not the tensor pipe).
__global__ void __launch_bounds__(256) zgemv_kernel(int M, int K, c128 alpha, const c128 *__restrict__ A, long lda,
                                                    int conjA, const c128 *__restrict__ b, long incb, int conjB,
                                                    c128 beta, c128 *C, long ldc) {
  const int lane = threadIdx.x & 31;
  const int warps = (gridDim.x * blockDim.x) >> 5;
  const double sa = conjA ? -1.0 : 1.0, sb = conjB ? -1.0 : 1.0;
  for (int m = (blockIdx.x * blockDim.x + threadIdx.x) >> 5; m < M; m += warps) {
    const c128 *a = A + (size_t)m * lda;
    double x0 = 0.0, y0 = 0.0, x1 = 0.0, y1 = 0.0;
    int k = lane;
    for (; k + 32 < K; k += 64) {
      c128 u = a[k], w = b[(size_t)k * incb], u2 = a[k + 32], w2 = b[(size_t)(k + 32) * incb];
      u.y *= sa; w.y *= sb; u2.y *= sa; w2.y *= sb;
      x0 = fma(u.x, w.x, x0); x0 = fma(-u.y, w.y, x0); y0 = fma(u.x, w.y, y0); y0 = fma(u.y, w.x, y0);
      x1 = fma(u2.x, w2.x, x1); x1 = fma(-u2.y, w2.y, x1); y1 = fma(u2.x, w2.y, y1); y1 = fma(u2.y, w2.x, y1);
    }
    if (k < K) {
      c128 u = a[k], w = b[(size_t)k * incb];
      u.y *= sa; w.y *= sb;
      x0 = fma(u.x, w.x, x0); x0 = fma(-u.y, w.y, x0); y0 = fma(u.x, w.y, y0); y0 = fma(u.y, w.x, y0);
    }
    x0 += x1; y0 += y1;
#pragma unroll
    for (int s = 16; s > 0; s >>= 1) {
      x0 += __shfl_xor_sync(0xffffffffu, x0, s);
      y0 += __shfl_xor_sync(0xffffffffu, y0, s);
    }
    if (lane == 0) {
      c128 out = cmul(alpha, make_double2(x0, y0));
      c128 *dst = C + (size_t)m * ldc;
      if (beta.x != 0.0 || beta.y != 0.0) out = cadd(out, cmul(beta, *dst));
      *dst = out;
    }
  }
}

}  // namespace

cudaError_t zgemm_sum_plane(cudaStream_t st, const c128 *X, long ld, long rows, long cols, bool conj, double *plane, long ldp) {
  if (rows <= 0 || cols <= 0) return cudaSuccess;
  dim3 grid((unsigned)std::min<long>((cols + 255) / 256, 64), (unsigned)std::min<long>(rows, 32768));
  sum_plane_kernel<<<grid, 256, 0, st>>>(X, ld, rows, cols, conj ? 1 : 0, plane, ldp);
  cclr_count_launch();
  return cudaGetLastError();
}

int zgemm_num_sms() {
  static std::atomic<int> cache[64];   // per device ordinal (zero-initialised)
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return 148;
  if (dev >= 0 && dev < 64 && cache[dev].load() > 0) return cache[dev].load();
  int n = 0;
  cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev);
  if (n <= 0) n = 148;
  if (dev >= 0 && dev < 64) cache[dev].store(n);
  return n;
}

// Raster (ZgemmArgs::group_m): the CTAs of one wave cover a block of rows x cols tiles and stream rows A panels and cols B
// panels in k-lockstep; pick the group height that minimises the panel bytes per wave (BM rows + BN cols, per unit of K).
static int pick_group_m(int tiles_m, int tiles_n, int BM, int BN, int sms) {
  int best_g = 1;
  double best = -1.0;
  for (int g = 1; g <= tiles_m; ++g) {
    int cols = (sms + g - 1) / g;
    if (cols > tiles_n) cols = tiles_n;
    double rows = (double)sms / cols;
    if (rows < g) rows = g;
    if (rows > tiles_m) rows = tiles_m;
    const double bytes = rows * BM + (double)cols * BN;
    if (best < 0.0 || bytes < best * 0.999) { best = bytes; best_g = g; }
    if (g >= sms) break;
  }
  return best_g;
}

cudaError_t zgemm(cudaStream_t st, int M, int N, int K, c128 alpha, const c128 *A, long lda, bool conjA,
                  const c128 *B, long ldb, bool b_is_kn, bool conjB, c128 beta, c128 *C, long ldc, int batch, long sa,
                  long sb, long sc, const ZgemmWorkspace *ws) {
  if (M <= 0 || N <= 0 || batch <= 0) return cudaSuccess;
  // integer-slice product on the INT8 tensor path (zgemm_oz.cu): contractions whose A operand has registered slices (the context's
  // W_vvvv and W_ovvo: ladder and ring of sigma), and ring-shaped ones (N >= 1024: slicing A per call costs < 10 % of the product)
  // as long as the per-call slices stay small (the transposed ladder of the left transform, 48 GB of them, stays on DMMA)
  if (ws && ws->oz && ws->oz->slices > 0 && batch == 1 && zgemm_oz_supported(M, N, K)) {
    // the big constant operand on the B side (transposed ladder of the left transform): C^T = B^T A^T on the slices of B^T
    if (b_is_kn && zgemm_oz_has_bt(ws->oz, B, ldb, N, K) && (zgemm_oz_eligible(N, M, K) || ws->oz->any_size) &&
        (size_t)ws->oz->slices * 4 * (size_t)K * (size_t)M <= ((size_t)6 << 30))
      return zgemm_oz_bt(st, M, N, K, alpha, A, lda, conjA, B, ldb, conjB, beta, C, ldc, ws->oz);
    bool registered = false;
    for (const OzEntry &e : ws->oz->persist)
      if (!e.transposed && e.key == A && e.ld == lda && e.rows == M && e.K == K) registered = true;
    const bool pays = zgemm_oz_eligible(M, N, K);
    const size_t per_call = (size_t)ws->oz->slices * 2 * (size_t)K * ((registered ? 0 : (size_t)M) + 2 * (size_t)N);
    if (((registered && (pays || ws->oz->any_size)) || (pays && N >= 1024)) && per_call <= ((size_t)6 << 30))
      return zgemm_oz(st, M, N, K, alpha, A, lda, conjA, B, ldb, b_is_kn, conjB, beta, C, ldc, ws->oz);
  }
  constexpr int BK = ZG_BK;
  const int sms = zgemm_num_sms();
  // 64-row tiles when they cut the padding of M by more than 10 % (M of a few hundred: 300 -> 320 instead of 384)
  const long pad128 = (M + 127L) / 128 * 128, pad64 = (M + 63L) / 64 * 64;
  // 3M complex product (3 real DMMA products per complex one instead of 4) for the large contractions; the 4M kernel keeps
  // the small and skinny ones, where tile padding, not the DMMA count, is the cost
  const bool use3m = (!ws || ws->three_m) && M >= 512 && N >= 24 && K >= 64;
  // "skinny" reductions of the solver (Gram blocks b^H sigma, Gram-Schmidt projections: a few rows and columns, K = the whole
  // amplitude vector): 32 x 8 tiles and an 8-deep ring keep the padding waste and the bytes in flight where HBM, not the
  // tensor pipe, is the limit
  const bool skinny = !use3m && !b_is_kn && batch == 1 && N <= 16 && M <= 256 && K >= 65536;
  const int BM = use3m ? 128 : skinny ? 32 : ((pad64 * 10 <= pad128 * 9) ? 64 : 128);
  if (batch > 1 && (sa == 0 || sb == 0)) {   // a shared operand has no batch stride a tensor map could carry: one launch per batch
    for (int b = 0; b < batch; ++b) {
      const cudaError_t e = zgemm(st, M, N, K, alpha, A + (size_t)b * sa, lda, conjA, B + (size_t)b * sb, ldb, b_is_kn, conjB, beta,
                                  C + (size_t)b * sc, ldc, 1, 0, 0, 0, ws);
      if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
  }
  if (K <= 0) {  // C = beta * C
    zgemm_reduce_kernel<<<256, 256, 0, st>>>(nullptr, 0, M, N, alpha, beta, C, ldc, sc, batch);
    cclr_count_launch();
    return cudaGetLastError();
  }
  // ---- N = 1 or M = 1: bandwidth-bound matrix-vector products ----
  if (batch == 1 && (N == 1 || (M == 1 && !b_is_kn)) && K >= 32) {
    const int rows = N == 1 ? M : N;
    int blocks = (rows + 7) / 8;
    if (blocks > sms * 8) blocks = sms * 8;
    if (N == 1)
      zgemv_kernel<<<blocks, 256, 0, st>>>(M, K, alpha, A, lda, conjA, B, b_is_kn ? ldb : 1, conjB, beta, C, ldc);
    else
      zgemv_kernel<<<blocks, 256, 0, st>>>(N, K, alpha, B, ldb, conjB, A, 1, conjA, beta, C, 1);
    cclr_count_launch();
    return cudaGetLastError();
  }
  if (batch == 1 && M == 1 && b_is_kn && K >= 32 && ws && ws->buf && (size_t)N <= ws->elems) {
    const int nblk = (N + 127) / 128;
    int slabs = (4 * sms + nblk - 1) / nblk;
    if (slabs > K / 16) slabs = K / 16;
    if ((size_t)slabs * N > ws->elems) slabs = (int)(ws->elems / N);
    if (slabs < 1) slabs = 1;
    const int kslab = (K + slabs - 1) / slabs;
    slabs = (K + kslab - 1) / kslab;
    zgemv_t_kernel<<<dim3(nblk, slabs), 128, 0, st>>>(N, K, A, conjA, B, ldb, conjB, kslab, ws->buf);
    zgemv_t_reduce_kernel<<<(N + 255) / 256, 256, 0, st>>>(N, slabs, ws->buf, alpha, beta, C);
    cclr_count_launch(2);
    return cudaGetLastError();
  }
  // ---- N-tile width: the least padded N, widest tile on ties ----
  // (the widest tile within 1 % of the least padding: narrower tiles re-read the A panels more often)
  int NG = 8;
  long best = -1;
  for (int ng = 8; ng >= 4; --ng) {
    const long bn = 8 * ng, padded = (N + bn - 1) / bn * bn;
    if (best < 0 || padded < best) best = padded;
  }
  for (int ng = 8; ng >= 4; --ng) {
    const long bn = 8 * ng, padded = (N + bn - 1) / bn * bn;
    if (padded * 100 <= best * 101) { NG = ng; break; }
  }
  int NG3 = 3;
  if (use3m) {
    const long p48 = (N + 47L) / 48 * 48, p32 = (N + 31L) / 32 * 32;
    NG3 = (p32 * 100 < p48 * 99) ? 2 : 3;
  }
  const int BN = use3m ? 16 * NG3 : skinny ? 8 : 8 * NG;
  ZgemmArgs args{};
  args.M = M; args.N = N; args.K = K;
  args.C = C; args.ldc = ldc; args.sc = sc;
  args.alpha = alpha; args.beta = beta;
  args.conjA = conjA; args.conjB = conjB;
  args.tiles_m = (M + BM - 1) / BM;
  args.tiles_n = (N + BN - 1) / BN;
  args.group_m = pick_group_m(args.tiles_m, args.tiles_n, BM, BN, sms);
  const long tiles = (long)args.tiles_m * args.tiles_n * batch;
  if (tiles > 0x7fffffffL / 2) return cudaErrorInvalidValue;
  const int nchunks = (K + BK - 1) / BK;
  // ---- launch geometry (see ZgemmArgs): whole tiles, then the K-split tail ----
  int main_tiles = (int)tiles, splits = 1;
  const size_t tile_elems = (size_t)BM * BN;
  if (ws && ws->buf) {
    if (tiles < sms && nchunks >= 16) {
      // the MN grid cannot fill the chip: split every tile along K
      splits = (int)(2L * sms / tiles);                 // at most two full waves of CTAs
      if (splits > nchunks / 4) splits = nchunks / 4;
      if ((size_t)splits * tiles * tile_elems > ws->elems) splits = (int)(ws->elems / (tiles * tile_elems));
      if (splits > 1) main_tiles = 0; else splits = 1;
    } else if (tiles > sms) {
      // last partial wave: split its tiles so that it lasts 1/splits of a wave instead of a whole one
      const int rem = (int)(tiles % sms);
      if (rem > 0 && 2 * rem <= sms) {
        splits = sms / rem;
        if (splits > nchunks / 4) splits = nchunks / 4;
        if ((size_t)splits * rem * tile_elems > ws->elems) splits = (int)(ws->elems / (rem * tile_elems));
        if (splits > 1) main_tiles = (int)tiles - rem; else splits = 1;
      }
    }
  }
  args.main_tiles = main_tiles;
  args.tail_splits = splits;
  args.chunks_per_split = (nchunks + splits - 1) / splits;
  args.partial = splits > 1 ? ws->buf : nullptr;
  const int tail_tiles = (int)tiles - main_tiles;
  const int ctas = main_tiles + tail_tiles * splits;

  // ---- 3M: sum planes Re + Im of both operands from global memory, when they can be had cheaply ----
  // an operand's plane is either registered (persistent, unconjugated use) or formed here by a streaming pre-pass, which pays
  // when the operand is small next to the product (the other output dimension >= 2048: < 1.2 % of the GEMM's time)
  CUtensorMap tmSA, tmSB;
  bool planes = false;
  if (use3m && batch == 1 && ws) {
    const double *pa = nullptr, *pb = nullptr;
    long ldpa = 0, ldpb = 0;
    for (int q = 0; q < 2; ++q) {
      if (ws->persist_key[q] == A && !conjA && ws->persist_ld[q] == lda) { pa = ws->persist_plane[q]; ldpa = ws->persist_pld[q]; }
      if (ws->persist_key[q] == B && !conjB && ws->persist_ld[q] == ldb) { pb = ws->persist_plane[q]; ldpb = ws->persist_pld[q]; }
    }
    const long rowsB = b_is_kn ? K : N, colsB = b_is_kn ? N : K;
    const long ldsa = (K + 1) & ~1L, ldsb = (colsB + 1) & ~1L;
    size_t need = 0;
    const bool preA = !pa && N >= 2048, preB = !pb && M >= 2048;
    if (preA) need += (size_t)M * ldsa;
    if (preB) need += (size_t)rowsB * ldsb;
    if ((pa || preA) && (pb || preB) && need <= ws->plane_elems) {
      double *scratch = ws->plane;
      if (preA) {
        dim3 grid((unsigned)std::min<long>((K + 255) / 256, 64), (unsigned)std::min<long>(M, 32768));
        sum_plane_kernel<<<grid, 256, 0, st>>>(A, lda, M, K, conjA ? 1 : 0, scratch, ldsa);
        cclr_count_launch();
        pa = scratch; ldpa = ldsa;
        scratch += (size_t)M * ldsa;
      }
      if (preB) {
        dim3 grid((unsigned)std::min<long>((colsB + 255) / 256, 64), (unsigned)std::min<long>(rowsB, 32768));
        sum_plane_kernel<<<grid, 256, 0, st>>>(B, ldb, rowsB, colsB, conjB ? 1 : 0, scratch, ldsb);
        cclr_count_launch();
        pb = scratch; ldpb = ldsb;
      }
      planes = make_plane_map(&tmSA, pa, K, M, ldpa, BM) &&
               (b_is_kn ? make_plane_map(&tmSB, pb, N, K, ldpb, BK) : make_plane_map(&tmSB, pb, K, N, ldpb, BN));
    }
  }
  CUtensorMap tmA, tmB;
  if (!planes) { tmSA = CUtensorMap{}; tmSB = CUtensorMap{}; }
  if (!make_map(&tmA, A, K, M, lda, batch, sa, BM)) return cudaErrorInvalidValue;
  if (!b_is_kn) {
    if (!make_map(&tmB, B, K, N, ldb, batch, sb, BN)) return cudaErrorInvalidValue;
  } else {
    if (!make_map(&tmB, B, N, K, ldb, batch, sb, BK)) return cudaErrorInvalidValue;
  }
  cudaError_t e;
  if (use3m) {
#define CCLR_L3M(BN_, KN_) (planes ? launch_3m<BN_, KN_, true>(st, tmA, tmB, tmSA, tmSB, args, ctas) \
                                   : launch_3m<BN_, KN_, false>(st, tmA, tmB, tmSA, tmSB, args, ctas))
    if (NG3 == 2) e = b_is_kn ? CCLR_L3M(32, true) : CCLR_L3M(32, false);
    else e = b_is_kn ? CCLR_L3M(48, true) : CCLR_L3M(48, false);
#undef CCLR_L3M
  } else if (skinny) {
    e = launch<32, 8, ZG_BK, 8, 8, 8, false>(st, tmA, tmB, args, ctas);
  } else
  switch (NG) {
    case 4: e = launch_ng<4>(st, tmA, tmB, args, ctas, b_is_kn, BM); break;
    case 5: e = launch_ng<5>(st, tmA, tmB, args, ctas, b_is_kn, BM); break;
    case 6: e = launch_ng<6>(st, tmA, tmB, args, ctas, b_is_kn, BM); break;
    case 7: e = launch_ng<7>(st, tmA, tmB, args, ctas, b_is_kn, BM); break;
    default: e = launch_ng<8>(st, tmA, tmB, args, ctas, b_is_kn, BM); break;
  }
  if (e != cudaSuccess) return e;
  if (tail_tiles > 0 && splits > 1) {
    zgemm_tail_reduce_kernel<<<tail_tiles, 256, 0, st>>>(args, BM, BN);
    cclr_count_launch();
    e = cudaGetLastError();
  }
  return e;
}
