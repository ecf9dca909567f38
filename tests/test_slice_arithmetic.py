"""The arithmetic of the integer-slice product (csrc/zgemm_oz.cu) restated in numpy and checked against what the
mathematics fixes -- CPU only, no library call: the slicing is an exact decomposition with |q_t| <= 64 and a rest below
2^(-7 s), the leading slices of a decomposition are the decomposition with fewer slices (what precision on demand relies on),
the S32 accumulators cannot overflow under the grouping rule, and the truncated product has the error the tolerances of the GPU
tests are derived from (2^(-7 s + 6) norm-wise for Gaussian operands)."""
import numpy as np
import pytest


def slices_of(x, s):
    """Rows of x scaled by the power of two above the row maximum, cut into s signed 7-bit slices."""
    mx = np.abs(x).max(axis=1, keepdims=True)
    e = np.where(mx > 0, np.frexp(mx)[1], 0)                   # 2^e > max |x| (frexp: mx = f 2^e, f in [0.5, 1))
    y = np.ldexp(x, 6 - e)
    q = []
    for _ in range(s):
        qt = np.rint(y)
        q.append(qt)
        y = (y - qt) * 128.0
    return np.array(q), e, y                                   # y = rest * 2^(7 s), |y| <= 64


@pytest.mark.parametrize("s", [2, 4, 6, 8])
def test_slicing_is_an_exact_decomposition_with_small_digits(s):
    rng = np.random.default_rng(s)
    x = rng.normal(size=(7, 300)) * np.exp(rng.normal(size=(7, 1)) * 5)
    x[3] = 0.0                                                  # a zero row keeps scale 1 and zero digits
    q, e, rest = slices_of(x, s)
    assert np.abs(q).max() <= 64 and np.all(q == np.rint(q))
    recon = sum(np.ldexp(q[t], e - 6 - 7 * t) for t in range(s))          # every term and every partial sum is exact in fp64
    assert np.abs(x - recon).max() <= np.ldexp(np.abs(x).max(axis=1, keepdims=True), -7 * s + 1).max()
    assert np.all(np.abs(x - recon) <= np.ldexp(1.0, e - 7 * s))          # |rest| <= 2^(-7 s) of the row scale, row by row
    assert np.abs(rest).max() <= 64.0


def test_leading_slices_are_the_decomposition_with_fewer_slices():
    rng = np.random.default_rng(1)
    x = rng.normal(size=(5, 200))
    q6, e6, _ = slices_of(x, 6)
    for s in (2, 3, 4, 5):
        qs, es, _ = slices_of(x, s)
        assert np.array_equal(es, e6) and np.array_equal(qs, q6[:s])


@pytest.mark.parametrize("K", [600, 4800, 44850, 131071])
def test_accumulation_groups_cannot_overflow_int32(K):
    """Pairs of one anti-diagonal share an S32 accumulator while pairs * 2K * 64^2 < 2^31 (the real embedding doubles K)."""
    cap = (2 ** 31 - 1) // (2 * K * 4096)
    assert cap >= 1
    assert cap * 2 * K * 64 * 64 < 2 ** 31 <= (cap + 1) * 2 * K * 64 * 64 + 2 * K * 4096
    if K == 44850:
        assert cap == 5                                         # the 6 pairs of the last anti-diagonal of 6 slices run as 5 + 1


@pytest.mark.parametrize("s", [3, 4, 5, 6])
def test_truncated_product_error_matches_the_model(s):
    """C = sum_{t+u<=s-1} A_t B_u 2^(...) against the exact product: norm-wise error below 2^(-7 s + 6) for Gaussian operands (the
    bound the GPU tests assert) and of the order 30 * 2^(-7 s) the design states (between 1/20 and 1 of the bound)."""
    rng = np.random.default_rng(10 + s)
    M, N, K = 48, 40, 2000
    A, B = rng.normal(size=(M, K)), rng.normal(size=(N, K))
    qa, ea, _ = slices_of(A, s)
    qb, eb, _ = slices_of(B, s)
    C = np.zeros((M, N))
    for d in range(s - 1, -1, -1):                              # smallest anti-diagonals first; the integer products are exact
        acc = np.zeros((M, N))
        for t in range(d + 1):
            acc += qa[t] @ qb[d - t].T
        assert np.abs(acc).max() < 2 ** 31
        C += np.ldexp(acc, -12 - 7 * d)
    C = np.ldexp(C, ea + eb.T)
    ref = (A.astype(np.longdouble) @ B.T.astype(np.longdouble)).astype(np.float64)
    err = np.linalg.norm(C - ref) / np.linalg.norm(ref)
    bound = 2.0 ** (-7 * s + 6)
    assert bound / 20 < err < bound, (s, err, bound)
