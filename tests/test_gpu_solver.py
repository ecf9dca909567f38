"""GPU parity of cclr_solve / cclr_property against the oracle at config 1 (o=4, v=20, sigma_V = 0.05, diagonal Fock,
ground-state CCSD converged to 1e-10 by the oracle): response amplitudes against the oracle's dense LU solution, the
true residual re-evaluated by the oracle's sigma, and response functions <<X;Y>>_z (CC-CI form Eq. 16 and CC-CC form
Eq. 15) to relative 1e-8."""
import numpy as np
import pytest
import torch

import synth
from oracle import ccsd, cclr, packing
from oracle.packing import flat

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cfg1():
    import paper_2307_14296_b200 as cc
    o, v = 4, 20
    eri = synth.eri_packed(o, v, seed=0, scale=0.05)
    f = synth.fock(o, v, seed=0)
    full = packing.unpack_eri(o, v, {k: x.numpy() for k, x in eri.items()})
    ints = ccsd.Integrals(o, v, f.numpy(), **full)
    t1, t2, info = ccsd.solve_ground_state(ints, tol=1e-10)
    assert info["converged"], info
    c = cclr.CCLR(ints, t1, t2)
    A = c.dense_jacobian()
    lam1, lam2 = c.solve_lambda_dense(A)
    t1p, t2p = packing.pack_amplitudes(t1, t2)
    ctx = cc.cclr_create(o, v, f.cuda(), {k: x.cuda() for k, x in eri.items()}, torch.from_numpy(t1p).cuda(),
                         torch.from_numpy(t2p).cuda())
    ops = [synth.hermitian_operator(o + v, 0, comp) for comp in range(3)]
    ops.append(synth.hermitian_operator(o + v, 0, 3, imaginary_antisymmetric=True))
    xis = [c.xi(X) for X in ops]
    xi1 = torch.from_numpy(np.stack([packing.pack_amplitudes(*x)[0].reshape(-1) for x in xis])).cuda()
    xi2 = torch.from_numpy(np.stack([packing.pack_amplitudes(*x)[1].reshape(-1) for x in xis])).cuda()
    yield dict(cc=cc, o=o, v=v, c=c, A=A, lam=(lam1, lam2), ctx=ctx, ops=ops, xis=xis, xi1=xi1, xi2=xi2)
    ctx.close()


def _unpack(s, t1, t2):
    return packing.unpack_amplitudes(t1.cpu().numpy(), t2.cpu().numpy(), s["o"], s["v"])


@pytest.mark.parametrize("gamma", [0.0, 0.0045, -0.0045])
def test_solutions_match_dense_oracle_and_true_residual(cfg1, gamma):
    s = cfg1
    omegas = [0.0, 0.0773, -0.0773]
    t1, t2, info = s["cc"].cclr_solve(s["ctx"], s["xi1"], s["xi2"], omegas, gamma, tol=1e-10, maxiter=100)
    assert info.converged == 1 and info.max_residual <= 1e-10
    for r in range(4):
        for k, w in enumerate(omegas):
            z = w + 1j * gamma
            want = flat(*s["c"].solve_dense(s["A"], *s["xis"][r], z))
            got1, got2 = _unpack(s, t1[r, k], t2[r, k])
            got = flat(got1, got2)
            assert np.linalg.norm(got - want) <= 1e-8 * np.linalg.norm(want), (r, k)
            res = flat(*s["c"].sigma(got1, got2, z=z)) + flat(*s["xis"][r])       # (A - z) t + xi by the oracle
            assert np.linalg.norm(res) <= 2e-10 * np.linalg.norm(flat(*s["xis"][r])), (r, k)


@pytest.mark.parametrize("z", [0.0, 0.0773, 0.0773 + 0.0045j])
def test_response_functions_match_oracle(cfg1, z):
    """<<X;Y>>_z from GPU response amplitudes vs the all-oracle value; pairs: dipole-dipole (diagonal, off-diagonal)
    and dipole x imaginary-antisymmetric operator (optical-rotation type, Eq. 36)."""
    s = cfg1
    c, A, (l1, l2), ops = s["c"], s["A"], s["lam"], s["ops"]
    cache = {}

    def gpu_solve(x1, x2, zz):
        key = (id(x1), complex(zz))
        a, b = packing.pack_amplitudes(x1, x2)
        t1, t2, info = s["cc"].cclr_solve(s["ctx"], torch.from_numpy(a.reshape(1, -1)).cuda(),
                                          torch.from_numpy(b.reshape(1, -1)).cuda(), [complex(zz).real],
                                          complex(zz).imag, tol=1e-11, maxiter=100)
        assert info.converged == 1
        cache[key] = (t1, t2)
        return _unpack(s, t1[0, 0], t2[0, 0])

    dense = lambda a, b, zz: c.solve_dense(A, a, b, zz)
    for (P, Q) in [(ops[0], ops[0]), (ops[0], ops[1]), (ops[2], ops[3])]:
        want = c.response_cc_ci(dense, P, Q, z, l1, l2)
        got = c.response_cc_ci(gpu_solve, P, Q, z, l1, l2)
        assert abs(got - want) <= 1e-8 * abs(want), ("CC-CI", z)
    want = c.response_cc_cc(dense, ops[0], ops[1], z, l1, l2)
    got = c.response_cc_cc(gpu_solve, ops[0], ops[1], z, l1, l2)
    assert abs(got - want) <= 1e-8 * abs(want), ("CC-CC", z)


def test_property_contraction_of_gpu_amplitudes(cfg1):
    """cclr_property(eta^X, t^Y(z_k)) for all shifts at once vs the oracle's bilinear dot of its own amplitudes."""
    s = cfg1
    c, A, (l1, l2), ops = s["c"], s["A"], s["lam"], s["ops"]
    omegas = [0.0, 0.0773]
    t1, t2, info = s["cc"].cclr_solve(s["ctx"], s["xi1"][1:2].contiguous(), s["xi2"][1:2].contiguous(), omegas, 0.0045,
                                      tol=1e-11)
    assert info.converged == 1
    e1, e2 = c.eta(ops[0], l1, l2)
    e1p, e2p = packing.pack_amplitudes(e1, e2)
    got = s["cc"].cclr_property(s["ctx"], torch.from_numpy(e1p.reshape(-1)).cuda(), torch.from_numpy(e2p.reshape(-1)).cuda(),
                                t1[0].contiguous(), t2[0].contiguous())
    for k, w in enumerate(omegas):
        want = cclr.dot(e1, e2, *c.solve_dense(A, *s["xis"][1], w + 0.0045j))
        assert abs(got[k] - want) <= 1e-8 * abs(want)


def test_frequency_sweep_shares_one_subspace(cfg1):
    """16 damped frequencies x 3 right-hand sides in one call (config-5 pattern) equal the one-by-one dense solutions,
    with far fewer sigma products than 48 separate solves."""
    s = cfg1
    omegas = list(np.linspace(0.05, 0.4, 16))
    t1, t2, info = s["cc"].cclr_solve(s["ctx"], s["xi1"][:3].contiguous(), s["xi2"][:3].contiguous(), omegas, 0.0045,
                                      tol=1e-10, maxiter=100)
    assert info.converged == 1
    assert info.sigma_calls < 48 * 6
    for r in (0, 2):
        for k in (0, 7, 15):
            want = flat(*s["c"].solve_dense(s["A"], *s["xis"][r], omegas[k] + 0.0045j))
            got = flat(*_unpack(s, t1[r, k], t2[r, k]))
            assert np.linalg.norm(got - want) <= 1e-8 * np.linalg.norm(want)


def test_collapse_of_a_full_trial_space_still_converges(cfg1):
    s = cfg1
    s["ctx"].set_max_subspace(8)
    try:
        t1, t2, info = s["cc"].cclr_solve(s["ctx"], s["xi1"][:1].contiguous(), s["xi2"][:1].contiguous(), [0.0, 0.0773],
                                          0.0, tol=1e-10, maxiter=200)
    finally:
        s["ctx"].set_max_subspace(0)
    assert info.converged == 1 and info.subspace <= 8
    for k, w in enumerate([0.0, 0.0773]):
        want = flat(*s["c"].solve_dense(s["A"], *s["xis"][0], w))
        got = flat(*_unpack(s, t1[0, k], t2[0, k]))
        assert np.linalg.norm(got - want) <= 1e-8 * np.linalg.norm(want)


def test_maxiter_reports_not_converged(cfg1):
    s = cfg1
    t1, t2, info = s["cc"].cclr_solve(s["ctx"], s["xi1"][:1].contiguous(), s["xi2"][:1].contiguous(), [0.0], 0.0,
                                      tol=1e-12, maxiter=2)
    assert info.converged == 0 and info.iterations == 2 and info.max_residual > 1e-12
    assert torch.isfinite(t2.abs().sum()).item()


def test_zero_right_hand_side_gives_zero(cfg1):
    s = cfg1
    z1, z2 = torch.zeros_like(s["xi1"][:1]), torch.zeros_like(s["xi2"][:1])
    t1, t2, info = s["cc"].cclr_solve(s["ctx"], z1, z2, [0.0773], 0.0045)
    assert info.converged == 1 and t1.abs().max().item() == 0.0 and t2.abs().max().item() == 0.0


def test_xi_built_on_the_device_matches_oracle(cfg1):
    """cclr_xi (S-Eq. 2-3) for the dipole-type and the imaginary-antisymmetric operators."""
    s = cfg1
    for k, X in enumerate(s["ops"]):
        g1, g2 = s["cc"].cclr_xi(s["ctx"], torch.from_numpy(np.ascontiguousarray(X)).cuda())
        torch.cuda.synchronize()
        w1, w2 = packing.pack_amplitudes(*s["xis"][k])
        assert np.linalg.norm(g1.cpu().numpy() - w1.reshape(-1)) <= 1e-12 * np.linalg.norm(w1)
        assert np.linalg.norm(g2.cpu().numpy() - w2.reshape(-1)) <= 1e-12 * np.linalg.norm(w2)


def test_solver_bandwidth_kernels_match_numpy(cfg1):
    """The multi-row update (residual / solution / Gram-Schmidt block, with the fused norm and preconditioned output) and the
    dot block (split-K DMMA GEMM path and single-row path) against numpy, ragged sizes."""
    s = cfg1
    cc, ctx = s["cc"], s["ctx"]
    n = ctx.n1 + ctx.n2
    rng = np.random.default_rng(5)
    cplx = lambda *shape: rng.normal(size=shape) + 1j * rng.normal(size=shape)
    D = flat(s["c"].D1 + 0j, s["c"].D2 + 0j).real                 # orbital-energy differences over unique elements
    for (R, m, shared_x) in [(1, 3, False), (3, 37, True), (8, 70, False), (5, 1, True)]:
        V, X, coef = cplx(m, n), cplx(n) if shared_x else cplx(R, n), cplx(R, m)
        z = cplx(R) * 0.1 + 0.05
        Y = torch.zeros((R, n), dtype=torch.complex128, device="cuda")
        P = torch.zeros((R, n), dtype=torch.complex128, device="cuda")
        nrm = torch.zeros(R, dtype=torch.float64, device="cuda")
        cc.cclr_vec_block_lincomb(ctx, Y, torch.from_numpy(X).cuda(), torch.from_numpy(coef).cuda().contiguous(),
                                  torch.from_numpy(V).cuda(), nrm2=nrm, z=torch.from_numpy(z).cuda(), P=P)
        torch.cuda.synchronize()
        want = (X[None, :] if shared_x else X) + coef @ V
        assert np.abs(Y.cpu().numpy() - want).max() <= 1e-13 * np.abs(want).max()
        assert np.abs(nrm.cpu().numpy() - (np.abs(want) ** 2).sum(1)).max() <= 1e-13 * (np.abs(want) ** 2).sum(1).max()
        wp = want / (z[:, None] - D[None, :])
        assert np.abs(P.cpu().numpy() - wp).max() <= 1e-13 * np.abs(wp).max()
    for big, na, nb in [(6000, 5, 3), (70001, 37, 6), (66000, 3, 2)]:   # GEMM dot path; long vectors: the 32 x 8 "skinny" tiles, ragged
        A, B = cplx(na, big), cplx(nb, big)
        got = np.array(cc.cclr_vec_dots(ctx, torch.from_numpy(A).cuda(), torch.from_numpy(B).cuda()))
        want = A.conj() @ B.T
        assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max(), (big, na, nb)
    big = 6000
    A, B = cplx(5, big), cplx(3, big)
    for (a, b) in [(A, B[:1]), (A[:1], B)]:
        got = np.array(cc.cclr_vec_dots(ctx, torch.from_numpy(np.ascontiguousarray(a)).cuda(), torch.from_numpy(np.ascontiguousarray(b)).cuda()))
        want = a.conj() @ b.T
        assert np.abs(got - want).max() <= 1e-13 * np.abs(want).max()
