"""SURVEY 8(f) f2 on the device: ground-state multipliers (cclr_lambda: lambda A = -eta0, Eq. 13), eta / EOM-eta
(cclr_eta, S-Eq. 5-7), left response equations (cclr_solve_left) and the complete CC-CI response function of Eq. 16-17
(cclr_response_ci) against the oracle (dense algebra at config 1) and against the closed-form two-level golden, where the whole
chain integrals -> cclr_ccsd -> cclr_create -> cclr_response_ci runs without any oracle input."""
import numpy as np
import pytest
import torch

import synth
from oracle import ccsd, cclr, packing
from oracle.packing import flat
from test_golden_closed_form import GOLD, two_level_system

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cfg1():
    import paper_2307_14296_b200 as cc
    o, v = 4, 20
    eri = synth.eri_packed(o, v, seed=0, scale=0.05)
    f = synth.fock(o, v, seed=0)
    ints = ccsd.Integrals(o, v, f.numpy(), **packing.unpack_eri(o, v, {k: x.numpy() for k, x in eri.items()}))
    t1, t2, info = ccsd.solve_ground_state(ints, tol=1e-10)
    assert info["converged"]
    c = cclr.CCLR(ints, t1, t2)
    A = c.dense_jacobian()
    l1, l2 = c.solve_lambda_dense(A)
    t1p, t2p = packing.pack_amplitudes(t1, t2)
    ctx = cc.cclr_create(o, v, f.cuda(), {k: x.cuda() for k, x in eri.items()}, torch.from_numpy(t1p).cuda(),
                         torch.from_numpy(t2p).cuda())
    ops = [synth.hermitian_operator(o + v, 0, comp) for comp in range(3)]
    ops.append(synth.hermitian_operator(o + v, 0, 3, imaginary_antisymmetric=True))
    dev = dict(f=f.cuda(), eri={k: x.cuda() for k, x in eri.items()}, t1=torch.from_numpy(t1p.reshape(-1).copy()).cuda(),
               t2=torch.from_numpy(t2p.reshape(-1).copy()).cuda())
    yield dict(cc=cc, o=o, v=v, c=c, A=A, lam=(l1, l2), ctx=ctx, ops=ops, dev=dev)
    ctx.close()


def _dev(x):
    return torch.from_numpy(np.ascontiguousarray(x).reshape(-1).copy()).cuda()


def test_lambda_matches_dense_oracle(cfg1):
    s = cfg1
    g1, g2, info = s["cc"].cclr_lambda(s["ctx"], tol=1e-11, maxiter=200)
    assert info.converged == 1
    got = flat(*packing.unpack_amplitudes(g1.cpu().numpy(), g2.cpu().numpy(), s["o"], s["v"]))
    want = flat(*s["lam"])
    assert np.linalg.norm(got - want) <= 1e-8 * np.linalg.norm(want)


@pytest.mark.parametrize("eom", [False, True])
def test_eta_matches_oracle(cfg1, eom):
    s = cfg1
    l1p, l2p = packing.pack_amplitudes(*s["lam"])
    for X in s["ops"]:
        g1, g2 = s["cc"].cclr_eta(s["ctx"], _dev(X), _dev(l1p), _dev(l2p), eom=eom)
        torch.cuda.synchronize()
        w1, w2 = packing.pack_amplitudes(*(s["c"].eta_eom(X, *s["lam"]) if eom else s["c"].eta(X, *s["lam"])))
        assert np.linalg.norm(g1.cpu().numpy() - w1.reshape(-1)) <= 1e-11 * np.linalg.norm(w1)
        assert np.linalg.norm(g2.cpu().numpy() - w2.reshape(-1)) <= 1e-11 * np.linalg.norm(w2)


def test_left_response_equations_match_dense_transpose_solve(cfg1):
    s = cfg1
    e1, e2 = s["c"].eta(s["ops"][0], *s["lam"])
    a, b = packing.pack_amplitudes(e1, e2)
    z = 0.0773 + 0.0045j
    l1, l2, info = s["cc"].cclr_solve_left(s["ctx"], _dev(a)[None], _dev(b)[None], [z.real], z.imag, tol=1e-10)
    assert info.converged == 1
    want = np.linalg.solve((s["A"] - z * np.eye(s["A"].shape[0])).T, -flat(e1, e2))
    got = flat(*packing.unpack_amplitudes(l1[0, 0].cpu().numpy(), l2[0, 0].cpu().numpy(), s["o"], s["v"]))
    assert np.linalg.norm(got - want) <= 1e-8 * np.linalg.norm(want)


@pytest.mark.parametrize("z", [0.0, 0.0773, 0.0773 + 0.0045j])
def test_cc_ci_response_function_end_to_end(cfg1, z):
    s = cfg1
    c, A, (l1, l2), ops = s["c"], s["A"], s["lam"], s["ops"]
    dense = lambda a, b, zz: c.solve_dense(A, a, b, zz)
    for (P, Q) in [(ops[0], ops[0]), (ops[0], ops[1]), (ops[2], ops[3])]:
        want = c.response_cc_ci(dense, P, Q, z, l1, l2)
        got, info = s["cc"].cclr_response_ci(s["ctx"], _dev(P), _dev(Q), complex(z).real, complex(z).imag, tol=1e-11)
        assert info.converged == 1
        assert abs(got - want) <= 1e-8 * abs(want), (z, got, want)


def test_two_level_closed_form_from_integrals_only():
    """integrals -> cclr_ccsd -> cclr_create -> cclr_response_ci, no oracle input anywhere; CCSD is exact for two electrons, so
    the CC-CI response function equals the closed-form sum over states of tests/golden/two_level_closed_form.json."""
    import paper_2307_14296_b200 as cc
    f, V, o, X = two_level_system()
    ints = ccsd.Integrals.from_full(f, V, o)                     # (only used to pack the integral classes)
    full = dict(oooo=ints.oooo, ooov=ints.ooov, oovv=ints.oovv, ovvo=ints.ovvo, ovvv=ints.ovvv, vvvv=ints.vvvv)
    eri = {k: _dev(x) for k, x in packing.pack_eri(full).items()}
    fd = _dev(f)
    t1, t2, info = cc.cclr_ccsd(o, 2, fd, eri, tol=1e-13, maxiter=60)
    assert info.converged == 1 and abs(info.energy_re - GOLD["E_corr"]) < 1e-11
    ctx = cc.cclr_create(o, 2, fd, eri, t1, t2)
    for rec in GOLD["response"]:
        z, want = complex(*rec["z"]), complex(*rec["XX"])
        got, rinfo = cc.cclr_response_ci(ctx, _dev(X), _dev(X), z.real, z.imag, tol=1e-12, maxiter=50)
        assert rinfo.converged == 1
        assert abs(got - want) <= 1e-8 * abs(want), (z, got, want)
    ctx.close()


def test_hessian_contraction_matches_oracle(cfg1):
    """x . F . y (cclr_xfy: exact derivative of the left transform along x) against the oracle's Richardson second derivative
    of the Lagrangian (pinned by the explicit determinant-space F)."""
    s = cfg1
    d = s["dev"]
    l1p, l2p = packing.pack_amplitudes(*s["lam"])
    x1, x2 = synth.amplitudes(s["o"], s["v"], seed=21, cls1="x1", cls2="x2", nvec=2)
    got = s["cc"].cclr_xfy(s["o"], s["v"], d["f"], d["eri"], d["t1"], d["t2"], _dev(l1p), _dev(l2p), x1[0].cuda(), x2[0].cuda(),
                           x1[1].cuda(), x2[1].cuda())
    ux = packing.unpack_amplitudes(x1[0].numpy(), x2[0].numpy(), s["o"], s["v"])
    uy = packing.unpack_amplitudes(x1[1].numpy(), x2[1].numpy(), s["o"], s["v"])
    want = s["c"].xFy(*s["lam"], *ux, *uy)
    assert abs(got - want) <= 1e-9 * abs(want), (got, want)


def test_f_transform_matches_oracle_and_the_stencil_route(cfg1):
    """cclr_f_transform (the direct plan CCLR_PLAN_FY) element by element against oracle.cclr.CCLR.F_transform (pinned by the
    determinant-space F), two vectors in one call; and x . (F y) against cclr_xfy, the library's independent stencil route."""
    s = cfg1
    cc, d, o, v = s["cc"], s["dev"], s["o"], s["v"]
    l1p, l2p = packing.pack_amplitudes(*s["lam"])
    y1, y2 = synth.amplitudes(o, v, seed=23, cls1="x1", cls2="x2", nvec=2)
    g1, g2 = cc.cclr_f_transform(s["ctx"], d["eri"], _dev(l1p), _dev(l2p), y1.cuda(), y2.cuda())
    torch.cuda.synchronize()
    for k in range(2):
        w1, w2 = packing.pack_amplitudes(*s["c"].F_transform(*s["lam"], *packing.unpack_amplitudes(y1[k].numpy(), y2[k].numpy(), o, v)))
        assert np.linalg.norm(g1[k].cpu().numpy() - w1.reshape(-1)) <= 1e-10 * np.linalg.norm(w1)
        assert np.linalg.norm(g2[k].cpu().numpy() - w2.reshape(-1)) <= 1e-10 * np.linalg.norm(w2)
    x1, x2 = synth.amplitudes(o, v, seed=24, cls1="x1", cls2="x2")
    direct = cc.cclr_property(s["ctx"], x1[0].cuda(), x2[0].cuda(), g1[:1].contiguous(), g2[:1].contiguous())[0]
    stencil = cc.cclr_xfy(o, v, d["f"], d["eri"], d["t1"], d["t2"], _dev(l1p), _dev(l2p), x1[0].cuda(), x2[0].cuda(),
                          y1[0].cuda(), y2[0].cuda())
    assert abs(direct - stencil) <= 1e-9 * abs(stencil), (direct, stencil)


@pytest.mark.parametrize("z", [0.0, 0.0773 + 0.0045j])
def test_cc_cc_response_function_end_to_end(cfg1, z):
    s = cfg1
    c, A, (l1, l2), ops, d = s["c"], s["A"], s["lam"], s["ops"], s["dev"]
    dense = lambda a, b, zz: c.solve_dense(A, a, b, zz)
    for (P, Q) in [(ops[0], ops[1]), (ops[2], ops[3])]:
        want = c.response_cc_cc(dense, P, Q, z, l1, l2)
        got, info = s["cc"].cclr_response_cc(s["ctx"], d["eri"], _dev(P), _dev(Q), complex(z).real, complex(z).imag, tol=1e-11)
        assert info.converged == 1
        assert abs(got - want) <= 1e-8 * abs(want), (z, got, want)


def test_cc_cc_response_function_on_an_inplace_context(cfg1):
    """The F contraction reads W_vvvv only through the dressed block, so the symmetric form works on a context created with
    ERI_INPLACE (the caller's vvvv array is overwritten by W_abef; its other classes are read again by cclr_response_cc)."""
    s = cfg1
    cc, c, A, (l1, l2), ops, d = s["cc"], s["c"], s["A"], s["lam"], s["ops"], s["dev"]
    eri = {k: x.clone() for k, x in d["eri"].items()}
    ctx = cc.cclr_create(s["o"], s["v"], d["f"], eri, d["t1"], d["t2"], cc.ERI_INPLACE)
    z = 0.0773 + 0.0045j
    want = c.response_cc_cc(lambda a, b, zz: c.solve_dense(A, a, b, zz), ops[0], ops[2], z, l1, l2)
    got, info = cc.cclr_response_cc(ctx, eri, _dev(ops[0]), _dev(ops[2]), z.real, z.imag, tol=1e-11)
    ctx.close()
    assert info.converged == 1
    assert abs(got - want) <= 1e-8 * abs(want), (got, want)


@pytest.mark.parametrize("gamma", [0.0, 0.0045])
def test_response_tensor_in_one_call_matches_the_oracle_and_the_pairwise_entry_point(cfg1, gamma):
    """cclr_response_ci_tensor (all operator pairs and frequencies from two shared-subspace solves) against the all-oracle
    CC-CI value of Eq. 16-17 (dense solves) for every pair incl. the imaginary-antisymmetric operator, 1e-8."""
    s = cfg1
    cc, c, A = s["cc"], s["c"], s["A"]
    ops = s["ops"]
    omegas = [0.0, 0.0773]
    X = torch.from_numpy(np.stack(ops)).cuda().contiguous()
    got, info = cc.cclr_response_ci_tensor(s["ctx"], X, omegas, gamma, tol=1e-11, maxiter=300)
    assert info.converged == 1
    solve = lambda x1, x2, z: c.solve_dense(A, x1, x2, z)
    for k, w in enumerate(omegas):
        for r in range(len(ops)):
            for q in (r, (r + 1) % len(ops)):
                want = c.response_cc_ci(solve, ops[r], ops[q], complex(w, gamma), *s["lam"])
                assert abs(got[k][r][q] - want) <= 1e-8 * max(abs(want), 1e-4), (k, r, q, got[k][r][q], want)
