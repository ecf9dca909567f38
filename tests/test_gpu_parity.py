"""GPU parity tests: the CUDA path (through the C ABI of include/cclr.h and its ctypes binding) against the CPU
oracle on the same seeded synthetic inputs, element by element.

Tolerances (BASELINE.json north_star): sigma vectors ||gpu - oracle||_2 / ||oracle||_2 <= 1e-10
per vector, singles and doubles separately; intermediates max-norm 1e-11 relative; response functions 1e-8.
"""
import numpy as np
import pytest
import torch

import synth
from oracle import ccsd, cclr, packing

pytestmark = pytest.mark.gpu


def _lib():
    import paper_2307_14296_b200 as cc
    return cc


def make_system(o, v, seed=0, t_scale=None, diag_fock=False, eri_scale=None):
    """Synthetic packed inputs (host torch tensors) + the oracle objects built from the same numbers."""
    eri = synth.eri_packed(o, v, seed=seed, scale=eri_scale)
    f = synth.fock(o, v, seed=seed)
    if not diag_fock:
        f = f + 0.05 * torch.from_numpy(synth.hermitian_operator(o + v, seed, 7))
    ts = synth.sigma_v(v) * 2 if t_scale is None else t_scale
    t1, t2 = synth.amplitudes(o, v, seed=seed, scale=ts)
    full = packing.unpack_eri(o, v, {k: x.numpy() for k, x in eri.items()})
    ints = ccsd.Integrals(o, v, f.numpy(), **full)
    t1f, t2f = packing.unpack_amplitudes(t1[0].numpy(), t2[0].numpy(), o, v)
    return dict(o=o, v=v, eri=eri, fock=f, t1=t1[0], t2=t2[0], ints=ints, t1f=t1f, t2f=t2f)


def gpu_context(s, flags=0):
    cc = _lib()
    dev = {k: x.cuda() for k, x in s["eri"].items()}
    ctx = cc.cclr_create(s["o"], s["v"], s["fock"].contiguous().cuda(), dev, s["t1"].cuda(), s["t2"].cuda(), flags)
    return ctx


def rel(a, b):
    return np.linalg.norm(a - b) / max(np.linalg.norm(b), 1e-300)


# ---------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("M,N,K,kn,ca,cb,beta", [
    (1, 1, 1, False, False, False, 0.0), (5, 3, 2, True, True, False, 0.5), (128, 64, 16, False, False, False, 0.0),
    (129, 65, 17, False, False, True, 1.0), (200, 150, 333, True, False, False, 0.0), (37, 190, 190, True, True, True, -1.0),
    (300, 34, 5000, False, False, False, 1.0),     # tall K -> split-K path
    (20, 1, 80, False, False, False, 1.0),         # GEMV shapes of the singles terms
    (1000, 9, 34, True, False, False, 0.0),
    # every N-tile width (BN = 32, 40, 48, 56, 64) in both B layouts, ragged edges
    (300, 34, 70, True, False, False, 1.0), (300, 34, 70, False, True, False, 0.0),
    (257, 45, 100, True, False, True, 0.5), (257, 45, 100, False, False, False, 0.0),
    (130, 153, 64, True, False, False, 0.0), (130, 153, 64, False, False, True, 1.0),
    (260, 276, 48, True, True, False, 0.0), (260, 276, 48, False, False, False, -1.0),
    # more tiles than SMs with a short last wave -> K-split tail tiles (40 x 5 = 200 tiles on 148 SMs)
    (5120, 276, 200, True, False, False, 1.0), (5120, 276, 200, False, True, True, 0.0),
    (19000, 30, 130, True, False, False, 0.5),
    # matrix-vector products (N = 1 in both layouts, M = 1)
    (4000, 1, 481, False, True, False, 1.0), (4000, 1, 481, True, False, True, 0.0), (1, 700, 333, False, False, True, 0.5),
])
def test_zgemm_matches_numpy(M, N, K, kn, ca, cb, beta):
    cc = _lib()
    rng = np.random.default_rng(M * 1000 + N * 10 + K)
    A = rng.normal(size=(M, K)) + 1j * rng.normal(size=(M, K))
    B = rng.normal(size=(K, N) if kn else (N, K)) + 1j * rng.normal(size=(K, N) if kn else (N, K))
    C0 = rng.normal(size=(M, N)) + 1j * rng.normal(size=(M, N))
    alpha = 0.7 - 0.3j
    opA = A.conj() if ca else A
    opB = B.conj() if cb else B
    ref = alpha * (opA @ (opB if kn else opB.T)) + beta * C0
    Cd = torch.from_numpy(C0.copy()).cuda()
    cc.cclr_zgemm(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), Cd, alpha=alpha, beta=beta, conj_a=ca,
                  conj_b=cb, b_is_kn=kn)
    torch.cuda.synchronize()
    assert rel(Cd.cpu().numpy(), ref) < 1e-13


@pytest.mark.parametrize("M,N,K,kn,ca,cb,beta", [
    (640, 100, 300, True, False, False, 0.0), (640, 100, 300, False, True, True, 1.0),
    (513, 24, 64, True, True, False, 0.5), (1300, 561, 96, True, False, False, 0.0),
    (1300, 153, 200, False, False, True, -1.0), (5120, 276, 200, True, False, False, 1.0),
    (700, 10200 // 8, 130, False, False, False, 0.0),
    # both output dimensions >= 2048: the 3M kernel is fed with sum planes Re + Im formed by a pre-pass (even / odd K, conj)
    (2100, 2060, 130, False, False, False, 0.0), (2100, 2060, 131, True, True, False, 1.0),
    (2304, 2100, 96, True, False, True, 0.5), (2050, 2049, 77, False, True, True, 0.0),
])
def test_zgemm_3m_and_4m_modes_match_numpy(M, N, K, kn, ca, cb, beta):
    """The large-contraction path in both complex-product modes (3M: three real DMMA products per complex one; 4M: four),
    both tile widths of the 3M kernel (32, 48), both B layouts, conjugations, K-split tail tiles."""
    cc = _lib()
    rng = np.random.default_rng(M + N + K)
    A = rng.normal(size=(M, K)) + 1j * rng.normal(size=(M, K))
    B = rng.normal(size=(K, N) if kn else (N, K)) + 1j * rng.normal(size=(K, N) if kn else (N, K))
    C0 = rng.normal(size=(M, N)) + 1j * rng.normal(size=(M, N))
    alpha = -0.4 + 0.9j
    opA = A.conj() if ca else A
    opB = B.conj() if cb else B
    ref = alpha * (opA @ (opB if kn else opB.T)) + beta * C0
    for mode in (True, False):
        Cd = torch.from_numpy(C0.copy()).cuda()
        cc.cclr_zgemm(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), Cd, alpha=alpha, beta=beta, conj_a=ca,
                      conj_b=cb, b_is_kn=kn, three_m=mode)
        torch.cuda.synchronize()
        assert rel(Cd.cpu().numpy(), ref) < 1e-13, mode


def test_zgemm_3m_component_accuracy_when_one_part_is_tiny():
    """What the 3M product does to a component that is much smaller than its partner: the imaginary
    part is T3 - T1 - T2, a difference of O(|Re|) numbers, so with |Im| = 1e-8 |Re| operands it carries an ABSOLUTE error of
    a few ulp of |Re C| -- norm-wise 1e-15 like 4M, but only ~7 digits relative to Im C itself; 4M keeps Im C to ~1e-15 of
    its own size.  A purely real B with a complex A: the same statement for the cross terms."""
    cc = _lib()
    rng = np.random.default_rng(77)
    M, N, K = 640, 96, 512
    A = rng.normal(size=(M, K)) + 1e-8j * rng.normal(size=(M, K))
    B = rng.normal(size=(K, N)) + 1e-8j * rng.normal(size=(K, N))
    ref = A @ B
    out = {}
    for mode in (True, False):
        Cd = torch.zeros((M, N), dtype=torch.complex128, device="cuda")
        cc.cclr_zgemm(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), Cd, b_is_kn=True, three_m=mode)
        torch.cuda.synchronize()
        out[mode] = Cd.cpu().numpy()
        assert rel(out[mode], ref) < 1e-14, mode                                    # norm-wise: both at rounding level
    im_err = {m: np.abs(out[m].imag - ref.imag).max() / np.abs(ref.imag).max() for m in out}
    assert im_err[False] < 1e-12                                                     # 4M: Im C relative to itself
    assert im_err[True] < 1e-5                                                       # 3M: absolute error ~ ulp(|Re C|) ...
    assert np.abs(out[True].imag - ref.imag).max() < 1e-13 * np.abs(ref.real).max()   # ... i.e. tiny relative to |C|
    Br = rng.normal(size=(K, N)) + 0j                                                # purely real operand
    Ac = rng.normal(size=(M, K)) + 1j * rng.normal(size=(M, K))
    for mode in (True, False):
        Cd = torch.zeros((M, N), dtype=torch.complex128, device="cuda")
        cc.cclr_zgemm(torch.from_numpy(Ac).cuda(), torch.from_numpy(Br).cuda(), Cd, b_is_kn=True, three_m=mode)
        torch.cuda.synchronize()
        assert rel(Cd.cpu().numpy(), Ac @ Br) < 1e-14, mode


@pytest.mark.parametrize("M,N,K,kn,ca,cb,beta,slices", [
    (66, 6, 66, True, False, False, 0.0, 6), (3, 5, 7, False, True, False, 1.0, 6),      # far below one tile
    (512, 32, 512, False, False, False, 0.0, 6), (700, 77, 1000, True, False, False, 0.0, 6),
    (515, 130, 777, False, True, False, 1.0, 6), (515, 130, 777, True, False, True, -0.5, 6),
    (1300, 561, 1000, True, True, True, 0.0, 6), (1024, 300, 2048, False, False, False, 1.0, 7),
    (2100, 520, 4099, False, False, True, 0.0, 6), (600, 1030, 515, True, False, False, 0.0, 8),
    (1024, 300, 2048, True, False, False, 0.0, 3), (1024, 300, 2048, True, False, False, 0.0, 4),
])
def test_zgemm_integer_slice_product_matches_numpy(M, N, K, kn, ca, cb, beta, slices):
    """zgemm_oz (csrc/zgemm_oz.cu): the complex128 product from INT8 slices on tcgen05.mma.kind::i8 with S32 accumulators in tensor
    memory.  The integer products are exact, so the error is the truncation of the operands 6 + 7 (s - 1) bits below their row /
    column maxima: for Gaussian operands norm-wise ~30 * 2^(-7 s).  Asserted: 2^(-7 s + 6) (s = 6: 1.5e-11, an order
    below north_star's 1e-10 for sigma), ragged M / N / K, both B layouts, conjugations, complex alpha, beta, several tile widths
    and (K = 4099) a split anti-diagonal.  Per 128 x 64 block as well, so that a wrong tile or scale cannot hide in the norm."""
    cc = _lib()
    rng = np.random.default_rng(M + N + K + slices)
    A = rng.normal(size=(M, K)) + 1j * rng.normal(size=(M, K))
    B = rng.normal(size=(K, N) if kn else (N, K)) + 1j * rng.normal(size=(K, N) if kn else (N, K))
    C0 = rng.normal(size=(M, N)) + 1j * rng.normal(size=(M, N))
    alpha = -0.4 + 0.9j
    opA = A.conj() if ca else A
    opB = B.conj() if cb else B
    prod = alpha * (opA @ (opB if kn else opB.T))
    ref = prod + beta * C0
    Cd = torch.from_numpy(C0.copy()).cuda()
    cc.cclr_zgemm_oz(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), Cd, alpha=alpha, beta=beta, conj_a=ca, conj_b=cb,
                     b_is_kn=kn, slices=slices)
    torch.cuda.synchronize()
    got = Cd.cpu().numpy()
    tol = max(2.0 ** (-7 * slices + 6), 2e-14)
    assert np.linalg.norm(got - ref) < tol * np.linalg.norm(prod)
    for i0 in range(0, M, 128):
        for j0 in range(0, N, 64):
            blk = (slice(i0, i0 + 128), slice(j0, j0 + 64))
            assert np.linalg.norm(got[blk] - ref[blk]) < 4 * tol * np.linalg.norm(prod[blk]), (i0, j0)


@pytest.mark.parametrize("M,N,K,ca,cb,beta", [(36, 561, 561, False, False, 0.0), (153, 1400, 1100, True, False, 1.0),
                                              (561, 2100, 777, False, True, -0.5), (40, 300, 4099, True, True, 0.0)])
def test_zgemm_integer_slice_product_with_the_constant_operand_on_the_b_side(M, N, K, ca, cb, beta):
    """zgemm_oz_bt: B stored [K][N] is the big constant operand (the transposed ladder of the left transform); its TRANSPOSE is
    sliced once and the product runs as C^T = B^T A^T with a transposed store.  Same tolerance as the direct route."""
    cc = _lib()
    rng = np.random.default_rng(M + N + K)
    A = rng.normal(size=(M, K)) + 1j * rng.normal(size=(M, K))
    B = rng.normal(size=(K, N)) + 1j * rng.normal(size=(K, N))
    C0 = rng.normal(size=(M, N)) + 1j * rng.normal(size=(M, N))
    alpha = 0.6 + 0.2j
    prod = alpha * ((A.conj() if ca else A) @ (B.conj() if cb else B))
    ref = prod + beta * C0
    Cd = torch.from_numpy(C0.copy()).cuda()
    cc.cclr_zgemm_oz(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), Cd, alpha=alpha, beta=beta, conj_a=ca, conj_b=cb,
                     b_is_kn=True, slices=6, b_side=True)
    torch.cuda.synchronize()
    got = Cd.cpu().numpy()
    assert np.linalg.norm(got - ref) < 2.0 ** -36 * np.linalg.norm(prod)
    for j0 in range(0, N, 256):
        blk = (slice(None), slice(j0, j0 + 256))
        assert np.linalg.norm(got[blk] - ref[blk]) < 4 * 2.0 ** -36 * np.linalg.norm(prod[blk]), j0


def test_zgemm_integer_slice_product_is_limited_by_the_row_maximum():
    """What the slicing does NOT keep: elements far below the largest element of their row (of A) or column (of B)
    are truncated 41 bits below that maximum, not below themselves.  One outlier of 1e6 in every row of A costs six digits --
    stated here so that the limit is documented by a test, like the 3M component test above."""
    cc = _lib()
    rng = np.random.default_rng(9)
    M, N, K = 640, 96, 700
    A = rng.normal(size=(M, K)) + 1j * rng.normal(size=(M, K))
    B = rng.normal(size=(K, N)) + 1j * rng.normal(size=(K, N))
    A[:, 5] *= 1e6
    B[5, :] = 0.0                      # the outlier column meets a zero row: it sets the scale and contributes nothing
    ref = A @ B
    Cd = torch.zeros((M, N), dtype=torch.complex128, device="cuda")
    cc.cclr_zgemm_oz(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), Cd, b_is_kn=True, slices=6)
    torch.cuda.synchronize()
    err = rel(Cd.cpu().numpy(), ref)
    assert 1e-9 < err < 1e-4
    Cd.zero_()
    cc.cclr_zgemm_oz(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), Cd, b_is_kn=True, slices=8)
    torch.cuda.synchronize()
    assert rel(Cd.cpu().numpy(), ref) < 1e-8


def test_zgemm_batched_and_strided():
    cc = _lib()
    rng = np.random.default_rng(5)
    A = rng.normal(size=(3, 70, 40)) + 1j * rng.normal(size=(3, 70, 40))
    B = rng.normal(size=(3, 40, 50)) + 1j * rng.normal(size=(3, 40, 50))
    C = torch.zeros((3, 70, 50), dtype=torch.complex128, device="cuda")
    cc.cclr_zgemm(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, b_is_kn=True)
    torch.cuda.synchronize()
    assert rel(C.cpu().numpy(), A @ B) < 1e-13


def test_zgemm_batched_with_a_shared_operand():
    """batch > 1 with stride 0 on A (one matrix applied to a block of right-hand sides)."""
    cc = _lib()
    rng = np.random.default_rng(6)
    A = rng.normal(size=(70, 40)) + 1j * rng.normal(size=(70, 40))
    B = rng.normal(size=(3, 40, 50)) + 1j * rng.normal(size=(3, 40, 50))
    C = torch.zeros((3, 70, 50), dtype=torch.complex128, device="cuda")
    cc.cclr_zgemm(torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda(), C, b_is_kn=True, M=70, N=50, K=40, lda=40, ldb=50,
                  ldc=50, batch=3, sa=0, sb=40 * 50, sc=70 * 50)
    torch.cuda.synchronize()
    assert rel(C.cpu().numpy(), np.einsum("mk,bkn->bmn", A, B)) < 1e-13


# ---------------------------------------------------------------------------------------------------------------
INTERMEDIATES = {
    # name -> oracle array in the library's layout
    "Fme": lambda c: c.Fme, "Fmi": lambda c: c.Fmi, "Fae": lambda c: c.Fae,
    "Wmnij": lambda c: packing.pack_pair_axes(packing.pack_pair_axes(c.Wmnij, 2), 0),
    "Wabef": lambda c: packing.pack_pair_axes(packing.pack_pair_axes(c.Wabef, 2), 0),
    "Wring": lambda c: c.Wmbej.transpose(1, 3, 2, 0),
    "Wie": lambda c: packing.pack_pair_axes(c.Wmnie, 0).transpose(1, 2, 0),
    "Wnjem": lambda c: c.Wmnie.transpose(0, 2, 3, 1),
    "Wamef": lambda c: packing.pack_pair_axes(c.Wamef, 2),
    "Wx": lambda c: c.Wamef.transpose(0, 2, 3, 1),
    "Wmbij": lambda c: packing.pack_pair_axes(c.Wmbij, 2),
    "Wabej": lambda c: packing.pack_pair_axes(c.Wabej, 0).transpose(0, 2, 1),
}


@pytest.mark.parametrize("o,v,flags", [(3, 5, 0), (4, 7, 2), (4, 20, 0), (5, 33, 2), (5, 33, 4)])
def test_create_intermediates_match_oracle(o, v, flags):
    s = make_system(o, v, seed=o * 100 + v)
    ctx = gpu_context(s, flags)
    c = cclr.CCLR(s["ints"], s["t1f"], s["t2f"])
    bad = []
    for name, fn in INTERMEDIATES.items():
        got = ctx.get_intermediate(name).cpu().numpy()
        want = np.ascontiguousarray(fn(c)).reshape(-1)
        err = np.abs(got - want).max() / max(1.0, np.abs(want).max())
        if not err < 1e-11:
            bad.append((name, err))
    ctx.close()
    assert not bad, bad


@pytest.mark.parametrize("o,v,flags,nvec", [(3, 5, 0, 1), (4, 7, 2, 2), (4, 20, 0, 3), (6, 40, 0, 1), (6, 40, 4, 1),
                                            # CCLR_GEMM_INT8_ANY_SIZE: ladder and ring on the INT8 tensor path at sizes the
                                            # full oracle can do (several tile rows, ragged: vv = 561 / 1326, ov = 306 / 520)
                                            (9, 34, 64, 2), (10, 52, 64, 1), (10, 52, 64 | 2, 1),
                                            (10, 52, 32, 1)])   # CCLR_GEMM_DMMA: the same on the FP64 tensor cores
def test_sigma_matches_oracle(o, v, flags, nvec):
    cc = _lib()
    s = make_system(o, v, seed=o * 100 + v + 1)
    ctx = gpu_context(s, flags)
    c = cclr.CCLR(s["ints"], s["t1f"], s["t2f"])
    x1, x2 = synth.amplitudes(o, v, seed=3, cls1="x1", cls2="x2", nvec=nvec)
    for (w, g) in [(0.0, 0.0), (0.0773, 0.0045)]:
        o1, o2 = cc.cclr_sigma(ctx, x1.cuda(), x2.cuda(), w, g)
        torch.cuda.synchronize()
        for k in range(nvec):
            r1, r2 = c.sigma(*packing.unpack_amplitudes(x1[k].numpy(), x2[k].numpy(), o, v), z=w + 1j * g)
            r1p, r2p = packing.pack_amplitudes(r1, r2)
            assert rel(o1[k].cpu().numpy(), r1p.reshape(-1)) < 1e-10, ("sigma1", k, w, g)
            assert rel(o2[k].cpu().numpy(), r2p.reshape(-1)) < 1e-10, ("sigma2", k, w, g)
    ctx.close()


def test_slice_count_follows_the_range_inside_the_rows():
    """cclr_create picks the slice count of the INT8 tensor path from the data (include/cclr.h: cclr_gemm_slices): 6 for the synthetic
    integrals; with the diagonal of <ab||ef> scaled by 1000 (still Hermitian) every row has one element far above the rest, six slices
    would lose ~3 digits, and the context takes 8 -- sigma keeps north_star's 1e-10 against the oracle on the same integrals."""
    cc = _lib()
    o, v = 9, 34
    s = make_system(o, v, seed=77)
    ctx = gpu_context(s, cc.GEMM_INT8_ANY_SIZE)
    assert ctx.gemm_slices() == 6
    ctx.close()
    vv = v * (v - 1) // 2
    idx = torch.arange(vv)
    s["eri"]["vvvv"] = s["eri"]["vvvv"].clone()
    s["eri"]["vvvv"].view(vv, vv)[idx, idx] *= 1000.0
    full = packing.unpack_eri(o, v, {k: x.numpy() for k, x in s["eri"].items()})
    ints = ccsd.Integrals(o, v, s["fock"].numpy(), **full)
    ctx = gpu_context(s, cc.GEMM_INT8_ANY_SIZE)
    assert ctx.gemm_slices() in (7, 8)
    c = cclr.CCLR(ints, s["t1f"], s["t2f"])
    x1, x2 = synth.amplitudes(o, v, seed=3, cls1="x1", cls2="x2")
    o1, o2 = cc.cclr_sigma(ctx, x1.cuda(), x2.cuda(), 0.0773, 0.0045)
    torch.cuda.synchronize()
    r1, r2 = c.sigma(*packing.unpack_amplitudes(x1[0].numpy(), x2[0].numpy(), o, v), z=0.0773 + 0.0045j)
    r1p, r2p = packing.pack_amplitudes(r1, r2)
    assert rel(o1[0].cpu().numpy(), r1p.reshape(-1)) < 1e-10 and rel(o2[0].cpu().numpy(), r2p.reshape(-1)) < 1e-10
    ctx.close()


def test_solver_with_precision_on_demand_is_certified_by_the_oracle_residual():
    """cclr_solve on the integer-slice path (forced at a size the full oracle can do; CCLR_NO_GRAPH so that the slice count can
    follow the residual, subspace.cuh) -- the solutions are certified by the ORACLE's sigma: ||(A - z) t + xi|| <= 2 tol ||xi||."""
    cc = _lib()
    o, v = 9, 34
    s = make_system(o, v, seed=91, t_scale=0.01, diag_fock=True, eri_scale=0.01)     # weakly coupled: a well-conditioned Jacobian
    ctx = gpu_context(s, cc.GEMM_INT8_ANY_SIZE | cc.NO_GRAPH)
    assert ctx.gemm_slices() == 6
    c = cclr.CCLR(s["ints"], s["t1f"], s["t2f"])
    xi1, xi2 = synth.amplitudes(o, v, seed=92, cls1="x1", cls2="x2")
    gamma, omegas, tol = 0.0045, [0.0773, -0.0773], 1e-10
    t1s, t2s, info = cc.cclr_solve(ctx, xi1.cuda(), xi2.cuda(), omegas, gamma, tol=tol, maxiter=300)
    assert info.converged == 1
    xi = np.concatenate([xi1[0].numpy(), xi2[0].numpy()])
    for k, w in enumerate(omegas):
        g1, g2 = packing.unpack_amplitudes(t1s[0, k].cpu().numpy(), t2s[0, k].cpu().numpy(), o, v)
        q1, q2 = c.sigma(g1, g2, z=w + 1j * gamma)
        res = packing.flat(q1, q2) + xi
        assert np.linalg.norm(res) <= 2 * tol * np.linalg.norm(xi), (w, np.linalg.norm(res) / np.linalg.norm(xi))
    ctx.close()


def test_ladder_and_ring_terms_match_oracle():
    cc = _lib()
    o, v = 4, 20
    s = make_system(o, v, seed=11)
    ctx = gpu_context(s)
    c = cclr.CCLR(s["ints"], s["t1f"], s["t2f"])
    x1, x2 = synth.amplitudes(o, v, seed=4, cls1="x1", cls2="x2", nvec=2)
    lad = cc.cclr_ladder(ctx, x2.cuda()).cpu().numpy()
    ring = cc.cclr_ring(ctx, x2[0].contiguous().cuda()).cpu().numpy()
    for k in range(2):
        _, r2 = packing.unpack_amplitudes(x1[k].numpy(), x2[k].numpy(), o, v)
        want = 0.5 * np.einsum("abef,efij->abij", c.Wabef, r2)                       # T11
        assert rel(lad[k], packing.pack_amplitudes(x1[k].numpy(), want)[1].reshape(-1)) < 1e-12
    _, r2 = packing.unpack_amplitudes(x1[0].numpy(), x2[0].numpy(), o, v)
    t8 = np.einsum("mbej,aeim->abij", c.Wmbej, r2)                                   # T8
    t8 = t8 - t8.transpose(1, 0, 2, 3)
    t8 = t8 - t8.transpose(0, 1, 3, 2)
    assert rel(ring, packing.pack_amplitudes(x1[0].numpy(), t8)[1].reshape(-1)) < 1e-12
    ctx.close()


@pytest.mark.parametrize("flags", [0, 8])     # 8 = CCLR_NO_GRAPH: the host entry copies x2 on a second stream while the x1-only
def test_sigma_host_entry_point_and_inplace_vvvv(flags):     # statements of the plan run
    cc = _lib()
    o, v = 4, 20
    s = make_system(o, v, seed=12)
    dev = {k: x.cuda() for k, x in s["eri"].items()}
    ctx = cc.cclr_create(o, v, s["fock"].contiguous().cuda(), dev, s["t1"].cuda(), s["t2"].cuda(), cc.ERI_INPLACE | flags)
    c = cclr.CCLR(s["ints"], s["t1f"], s["t2f"])
    x1, x2 = synth.amplitudes(o, v, seed=5, cls1="x1", cls2="x2", nvec=2)
    o1, o2 = torch.empty_like(x1), torch.empty_like(x2)
    cc.cclr_sigma_host(ctx, x1, x2, 0.1, -0.02, o1, o2)
    for k in range(2):
        r1, r2 = packing.pack_amplitudes(*c.sigma(*packing.unpack_amplitudes(x1[k].numpy(), x2[k].numpy(), o, v), z=0.1 - 0.02j))
        assert rel(o1[k].numpy(), r1.reshape(-1)) < 1e-10 and rel(o2[k].numpy(), r2.reshape(-1)) < 1e-10
    ctx.close()


def test_property_is_bilinear_dot_over_unique_elements():
    cc = _lib()
    o, v = 4, 20
    s = make_system(o, v, seed=13)
    ctx = gpu_context(s)
    e1, e2 = synth.amplitudes(o, v, seed=6, cls1="x1", cls2="x2")
    x1, x2 = synth.amplitudes(o, v, seed=7, cls1="x1", cls2="x2", nvec=3)
    got = cc.cclr_property(ctx, e1[0].cuda(), e2[0].cuda(), x1.cuda(), x2.cuda())
    for k in range(3):
        want = (e1[0].numpy() * x1[k].numpy()).sum() + (e2[0].numpy() * x2[k].numpy()).sum()
        assert abs(got[k] - want) < 1e-12 * abs(want)
    ctx.close()


# ---------------------------------------------------------------------------------------------------------------
# invariants of the GPU path alone (no oracle): special cases with closed forms
def test_gpu_V_zero_gives_orbital_energy_diagonal():
    cc = _lib()
    o, v = 5, 24
    s = make_system(o, v, seed=14, diag_fock=True, eri_scale=0.0)
    ctx = gpu_context(s)
    x1, x2 = synth.amplitudes(o, v, seed=8, cls1="x1", cls2="x2")
    o1, o2 = cc.cclr_sigma(ctx, x1.cuda(), x2.cuda())
    eps = s["fock"].numpy().diagonal().real
    eo, ev = eps[:o], eps[o:]
    D1 = (ev[:, None] - eo[None, :]).reshape(-1)
    pa, pb = packing.pairs(v)
    pi, pj = packing.pairs(o)
    D2 = ((ev[pa] + ev[pb])[:, None] - (eo[pi] + eo[pj])[None, :]).reshape(-1)
    assert rel(o1[0].cpu().numpy(), D1 * x1[0].numpy()) < 1e-13
    assert rel(o2[0].cpu().numpy(), D2 * x2[0].numpy()) < 1e-13
    ctx.close()


def test_gpu_T_zero_jacobian_is_hermitian():
    cc = _lib()
    o, v = 4, 12
    s = make_system(o, v, seed=15, diag_fock=True, t_scale=0.0)
    ctx = gpu_context(s)
    x1, x2 = synth.amplitudes(o, v, seed=9, cls1="x1", cls2="x2", nvec=2)
    o1, o2 = cc.cclr_sigma(ctx, x1.cuda(), x2.cuda())
    X = torch.cat([x1, x2], dim=1).numpy()
    S = torch.cat([o1.cpu(), o2.cpu()], dim=1).numpy()
    lhs, rhs = np.vdot(X[0], S[1]), np.conj(np.vdot(X[1], S[0]))      # x^H A y = conj(y^H A x)
    assert abs(lhs - rhs) < 1e-12 * abs(lhs)
    ctx.close()


def test_gpu_linearity_and_shift_identity():
    cc = _lib()
    o, v = 4, 20
    s = make_system(o, v, seed=16)
    ctx = gpu_context(s)
    x1, x2 = synth.amplitudes(o, v, seed=10, cls1="x1", cls2="x2", nvec=2)
    a, b = 0.3 - 1.1j, -0.7 + 0.2j
    y1 = (a * x1[0] + b * x1[1])[None].contiguous()
    y2 = (a * x2[0] + b * x2[1])[None].contiguous()
    o1, o2 = cc.cclr_sigma(ctx, x1.cuda(), x2.cuda())
    p1, p2 = cc.cclr_sigma(ctx, y1.cuda(), y2.cuda())
    assert rel(p2[0].cpu().numpy(), (a * o2[0] + b * o2[1]).cpu().numpy()) < 1e-13
    assert rel(p1[0].cpu().numpy(), (a * o1[0] + b * o1[1]).cpu().numpy()) < 1e-13
    z1, z2 = cc.cclr_sigma(ctx, x1.cuda(), x2.cuda(), 0.0773, 0.0045)
    zz = 0.0773 + 0.0045j
    assert rel(z2.cpu().numpy(), (o2.cpu() - zz * x2).numpy()) < 1e-14
    assert rel(z1.cpu().numpy(), (o1.cpu() - zz * x1).numpy()) < 1e-14
    ctx.close()


def test_config2_ground_state_sigma_solve_and_response_function_against_full_oracle():
    """BASELINE.json configs[1] (o=10, v=80, damped gamma=0.0045) at full size, everything against the full-tensor oracle:
    the GPU ground state (cclr_ccsd, 1e-10) is certified by ONE oracle residual evaluation, sigma matches norm-wise to 1e-10,
    the damped response amplitudes of a dipole perturbation satisfy the oracle's (A - z) t + xi = 0 to 2e-10, and the damped
    CC-CI response function <<X;X>>_z (Eq. 16-17) equals the oracle's assembly from certified vectors to 1e-8."""
    cc = _lib()
    o, v = 10, 80
    eri = synth.eri_packed(o, v, seed=0)
    f = synth.fock(o, v, seed=0)
    dev = {k: x.cuda() for k, x in eri.items()}
    t1, t2, info = cc.cclr_ccsd(o, v, f.cuda(), dev, tol=1e-10, maxiter=80)
    assert info.converged == 1
    full = packing.unpack_eri(o, v, {k: x.numpy() for k, x in eri.items()})
    ints = ccsd.Integrals(o, v, f.numpy(), **full)
    t1f, t2f = packing.unpack_amplitudes(t1.cpu().numpy(), t2.cpu().numpy(), o, v)
    w1, w2 = ccsd.residual(ints, t1f, t2f)
    assert np.sqrt(np.linalg.norm(w1) ** 2 + np.linalg.norm(w2) ** 2) <= 2e-10
    assert abs(complex(info.energy_re, info.energy_im) - ccsd.energy(ints, t1f, t2f)) < 1e-11
    c = cclr.CCLR(ints, t1f, t2f)
    ctx = cc.cclr_create(o, v, f.cuda(), dev, t1, t2)
    x1, x2 = synth.amplitudes(o, v, seed=3, cls1="x1", cls2="x2")
    z = 0.0773 + 0.0045j
    o1, o2 = cc.cclr_sigma(ctx, x1.cuda(), x2.cuda(), z.real, z.imag)
    torch.cuda.synchronize()
    r1, r2 = c.sigma(*packing.unpack_amplitudes(x1[0].numpy(), x2[0].numpy(), o, v), z=z)
    r1p, r2p = packing.pack_amplitudes(r1, r2)
    assert rel(o1[0].cpu().numpy(), r1p.reshape(-1)) < 1e-10
    assert rel(o2[0].cpu().numpy(), r2p.reshape(-1)) < 1e-10
    # damped response to a dipole component: xi from the oracle, solve on the GPU, residual by the oracle's sigma
    xi = c.xi(synth.hermitian_operator(o + v, 0, 0))
    a, b = packing.pack_amplitudes(*xi)
    s1, s2, sinfo = cc.cclr_solve(ctx, torch.from_numpy(a.reshape(1, -1)).cuda(), torch.from_numpy(b.reshape(1, -1)).cuda(),
                                  [z.real], z.imag, tol=1e-10, maxiter=100)
    assert sinfo.converged == 1
    g1, g2 = packing.unpack_amplitudes(s1[0, 0].cpu().numpy(), s2[0, 0].cpu().numpy(), o, v)
    q1, q2 = c.sigma(g1, g2, z=z)
    res = packing.flat(q1, q2) + packing.flat(*xi)
    assert np.linalg.norm(res) <= 2e-10 * np.linalg.norm(packing.flat(*xi))
    # the complete CC-CI response function <<X;X>>_z at this size: the device value (cclr_response_ci: lambda, xi, EOM-eta,
    # four response solves, dots) against the oracle's own assembly of Eq. 16-17 from amplitudes it has CERTIFIED -- lambda and
    # every t(z) come from the GPU, and the oracle checks each against its own residual before using it.
    X = synth.hermitian_operator(o + v, 0, 0)
    # (damped, gamma = 0.0045 as BASELINE.json configs[1] asks: four distinct response solves t(z), t(-z), t(-z*), t(z*), each
    # certified by one oracle sigma and cached)
    got, rinfo = cc.cclr_response_ci(ctx, torch.from_numpy(X).cuda(), torch.from_numpy(X).cuda(), z.real, z.imag, tol=1e-10)
    assert rinfo.converged == 1
    lg1, lg2, linfo = cc.cclr_lambda(ctx, tol=1e-10)
    assert linfo.converged == 1
    lam = packing.unpack_amplitudes(lg1.cpu().numpy(), lg2.cpu().numpy(), o, v)
    e0 = packing.flat(*c.eta0())
    assert np.linalg.norm(packing.flat(*c.sigma_left(*lam)) + e0) <= 2e-10 * np.linalg.norm(e0)      # lambda A + eta0 = 0

    cache = {}

    def certified_gpu_solve(x1f, x2f, zz):
        if complex(zz) in cache:
            return cache[complex(zz)]
        pa, pb = packing.pack_amplitudes(x1f, x2f)
        u1, u2, uinfo = cc.cclr_solve(ctx, torch.from_numpy(pa.reshape(1, -1)).cuda(), torch.from_numpy(pb.reshape(1, -1)).cuda(),
                                      [complex(zz).real], complex(zz).imag, tol=1e-10, maxiter=100)
        assert uinfo.converged == 1
        h1, h2 = packing.unpack_amplitudes(u1[0, 0].cpu().numpy(), u2[0, 0].cpu().numpy(), o, v)
        rr = packing.flat(*c.sigma(h1, h2, z=zz)) + packing.flat(x1f, x2f)
        assert np.linalg.norm(rr) <= 2e-10 * np.linalg.norm(packing.flat(x1f, x2f))
        cache[complex(zz)] = (h1, h2)
        return h1, h2

    want = c.response_cc_ci(certified_gpu_solve, X, X, z, *lam)
    assert abs(got - want) <= 1e-8 * abs(want), (got, want)
    ctx.close()


@pytest.mark.parametrize("o,v,flags,nvec", [(3, 5, 0, 1), (4, 7, 2, 2), (4, 20, 0, 2), (6, 40, 0, 1), (6, 40, 4, 1),
                                            # CCLR_GEMM_INT8_ANY_SIZE: the transposed ladder (slices of W_vvvv^T, transposed store)
                                            # and the ring adjoint on the INT8 tensor path; | 128: the ladder back on DMMA
                                            (9, 34, 64, 2), (10, 52, 64, 1), (10, 52, 64 | 128, 1)])
def test_sigma_left_matches_oracle(o, v, flags, nvec):
    """The left transform l (A - z) (cclr_sigma_left) against the oracle's adjoint of S-Eq. 11-12 (pinned by A^T of the dense
    Jacobian), norm-wise 1e-10; and the duality <l, A x> = <l A, x> between the two GPU transforms."""
    cc = _lib()
    s = make_system(o, v, seed=o * 100 + v + 2)
    ctx = gpu_context(s, flags)
    c = cclr.CCLR(s["ints"], s["t1f"], s["t2f"])
    l1, l2 = synth.amplitudes(o, v, seed=13, cls1="x1", cls2="x2", nvec=nvec)
    for (w, g) in [(0.0, 0.0), (0.0773, 0.0045)]:
        o1, o2 = cc.cclr_sigma_left(ctx, l1.cuda(), l2.cuda(), w, g)
        torch.cuda.synchronize()
        for k in range(nvec):
            r1, r2 = c.sigma_left(*packing.unpack_amplitudes(l1[k].numpy(), l2[k].numpy(), o, v), z=w + 1j * g)
            r1p, r2p = packing.pack_amplitudes(r1, r2)
            assert rel(o1[k].cpu().numpy(), r1p.reshape(-1)) < 1e-10, ("left sigma1", k, w, g)
            assert rel(o2[k].cpu().numpy(), r2p.reshape(-1)) < 1e-10, ("left sigma2", k, w, g)
    x1, x2 = synth.amplitudes(o, v, seed=14, cls1="x1", cls2="x2")
    s1, s2 = cc.cclr_sigma(ctx, x1.cuda(), x2.cuda())
    q1, q2 = cc.cclr_sigma_left(ctx, l1[:1].contiguous().cuda(), l2[:1].contiguous().cuda())
    lhs = (l1[0].cuda() * s1[0]).sum() + (l2[0].cuda() * s2[0]).sum()           # bilinear, unique elements
    rhs = (q1[0] * x1[0].cuda()).sum() + (q2[0] * x2[0].cuda()).sum()
    assert abs(complex(lhs - rhs)) <= (1e-10 if flags & 64 else 1e-11) * abs(complex(lhs))
    ctx.close()
