"""Time the integer-slice GEMM (cclr_zgemm_oz; csrc/zgemm_oz.cu) alone at a given shape on cuda:0.

    python -m paper_2307_14296_b200.oz_bench M N K [--kn] [--slices 6] [--bn 0] [--reps 3] [--check]

A [M][K], B [N][K] (or [K][N] with --kn), complex128, standard normal entries from a seeded generator.  Prints the time of the
slicing of A (done once for a constant operand), of one product (including the slicing of B) and of the slicing of B, the INT8
op rate of the tensor pipe (slices (slices + 1) / 2 pairs x 8 M N K ops) and the FP64-equivalent rate (8 M N K flop per product).
--bn: tile width / cluster shape override as in include/cclr.h.  --check compares 64 sampled rows with a float64 product of the
same rows formed by torch (a check, not part of the product path).
"""
import argparse

import torch

from . import cclr_zgemm_oz


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("M", type=int)
    ap.add_argument("N", type=int)
    ap.add_argument("K", type=int)
    ap.add_argument("--kn", action="store_true")
    ap.add_argument("--slices", type=int, default=6)
    ap.add_argument("--bn", type=int, default=0)
    ap.add_argument("--reps", type=int, default=3)
    ap.add_argument("--check", action="store_true")
    a = ap.parse_args()
    torch.cuda.set_device(0)
    g = torch.Generator(device="cuda")
    g.manual_seed(5)
    rnd = lambda *s: torch.view_as_complex(torch.randn(*s, 2, dtype=torch.float64, device="cuda", generator=g))
    A = rnd(a.M, a.K)
    B = rnd(a.K, a.N) if a.kn else rnd(a.N, a.K)
    C = torch.empty(a.M, a.N, dtype=torch.complex128, device="cuda")
    _, ms = cclr_zgemm_oz(A, B, C, b_is_kn=a.kn, slices=a.slices, bn=a.bn, reps=a.reps)
    pairs = a.slices * (a.slices + 1) // 2
    mnk = float(a.M) * a.N * a.K
    kern = ms[1] - ms[2]
    print("M=%d N=%d K=%d slices=%d bn=%d: slicing A %.2f ms (once), product %.2f ms (slicing B %.2f ms, kernel %.2f ms) = %.0f Top/s INT8, "
          "%.1f TFLOP/s FP64-equivalent (8 M N K)" % (a.M, a.N, a.K, a.slices, a.bn, ms[0], ms[1], ms[2], kern,
                                                    8.0 * mnk * pairs / kern / 1e9, 8.0 * mnk / ms[1] / 1e9))
    if a.check:
        rows = torch.randint(0, a.M, (64,), device="cuda")
        ref = A[rows] @ (B if a.kn else B.T)
        print("sampled rows: ||C - A B|| / ||A B|| = %.3e" % ((C[rows] - ref).norm() / ref.norm()).item())


if __name__ == "__main__":
    main()
