// permute.cu — the layout engine of the CC-LR library: one bandwidth kernel that performs every index permutation,
// unpacking of antisymmetric pairs (a<b -> a,b with sign), antisymmetrised packing P(ab), P(ij) (PAPER.md:217-219,
// 817) and the final sum of the Y / Q / ring pieces of sigma2 with the -(omega + i gamma) x shift.
//
//   gather mode : the iteration space IS the destination (dst_linear): coalesced 16-byte stores, gathered loads
//                 (served by L1/L2: consecutive threads read consecutive or strided elements of the same rows).
//   scatter mode: the iteration space is the source chunk; the destination offset is computed from its slots and an
//                 optional condition p<q / p>q on a destination pair makes the targets unique (no atomics).
//
// The descriptor (PermArgs, common.cuh) is built by plan.cu from the plan text; it is passed by value in the
// kernel parameter space.  Index arithmetic is 32-bit whenever the iteration space allows it.
#include "common.cuh"

namespace {

__device__ __forceinline__ void decode_pair(unsigned P, int &p, int &q) {
  int qq = (int)((1.0 + sqrt(1.0 + 8.0 * (double)P)) * 0.5);
  while ((unsigned)qq * (unsigned)(qq - 1) / 2u > P) --qq;
  while ((unsigned)(qq + 1) * (unsigned)qq / 2u <= P) ++qq;
  q = qq;
  p = (int)(P - (unsigned)qq * (unsigned)(qq - 1) / 2u);
}

// offset and sign (+1, -1, 0) of an operand for the current letter values
__device__ __forceinline__ int slots_offset(const PermSlot *slot, int nslot, const int *val, long &off) {
  int sign = 1;
  off = 0;
  for (int s = 0; s < nslot; ++s) {
    const PermSlot sl = slot[s];
    if (sl.kind == 0) {
      off += (long)(val[sl.l0] - sl.sub) * sl.stride;
    } else if (sl.kind == 1) {
      const int p = val[sl.l0], q = val[sl.l1];
      if (p == q) return 0;
      const long lo = p < q ? p : q, hi = p < q ? q : p;
      if (p > q) sign = -sign;
      off += (hi * (hi - 1) / 2 + lo) * sl.stride;
    }
  }
  return sign;
}

template <typename IndexT>
__global__ void __launch_bounds__(256) permute_kernel(const __grid_constant__ PermArgs p) {
  const IndexT total = (IndexT)p.total;
  const IndexT step = (IndexT)gridDim.x * (IndexT)blockDim.x;
  for (IndexT idx = (IndexT)blockIdx.x * (IndexT)blockDim.x + threadIdx.x; idx < total; idx += step) {
    int val[PERM_MAX_LETTERS];
    IndexT r = idx;
    for (int k = p.naxis - 1; k >= 0; --k) {
      const PermAxis ax = p.axis[k];
      const IndexT e = (IndexT)ax.ext;
      const IndexT q = r / e;
      const unsigned i = (unsigned)(r - q * e);
      r = q;
      if (ax.kind == 0) {
        val[ax.l0] = (int)i + ax.off;
      } else if (ax.kind == 1) {
        int a, b;
        decode_pair(i, a, b);
        val[ax.l0] = a;
        val[ax.l1] = b;
      }
    }
    long doff = (long)idx;
    int dsign = 1;
    if (!p.dst_linear) {
      dsign = slots_offset(p.dslot, p.ndslot, val, doff);
      if (dsign == 0) continue;
      if (p.cond) {
        const bool lt = val[p.cond_l0] < val[p.cond_l1];
        if ((p.cond == 1) != lt) continue;
      }
    }
    double sx = 0.0, sy = 0.0;
    for (int s = 0; s < p.nsrc; ++s) {
      long off;
      const int sg = slots_offset(p.src[s].slot, p.src[s].nslot, val, off);
      if (sg == 0) continue;
      c128 x = p.src[s].ptr[off];
      if (p.src[s].conj) x.y = -x.y;
      if (sg < 0) { x.x = -x.x; x.y = -x.y; }
      const c128 c = p.src[s].coef;
      sx = fma(c.x, x.x, sx); sx = fma(-c.y, x.y, sx);
      sy = fma(c.x, x.y, sy); sy = fma(c.y, x.x, sy);
    }
    if (dsign < 0) { sx = -sx; sy = -sy; }
    c128 *d = p.dst + doff;
    if (p.accumulate) {
      const c128 old = *d;
      sx += old.x; sy += old.y;
    }
    *d = make_double2(sx, sy);
  }
}

}  // namespace

cudaError_t permute(cudaStream_t st, const PermArgs &args) {
  if (args.total <= 0) return cudaSuccess;
  const int threads = 256;
  long blocks = (args.total + threads - 1) / threads;
  const long cap = (long)zgemm_num_sms() * 32;
  if (blocks > cap) blocks = cap;
  if (args.total < (1L << 31))
    permute_kernel<unsigned><<<(unsigned)blocks, threads, 0, st>>>(args);
  else
    permute_kernel<unsigned long long><<<(unsigned)blocks, threads, 0, st>>>(args);
  cclr_count_launch();
  return cudaGetLastError();
}
