"""cclr_eom (EOM-EE eigen-solver on the shared sigma routine) against the oracle's dense
Jacobian spectrum at config 1, the closed-form two-level golden, and the paper's own check: the poles of the linear
response function coincide with the EOM-EE energies."""
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
    t1p, t2p = packing.pack_amplitudes(t1, t2)
    ctx = cc.cclr_create(o, v, f.cuda(), {k: x.cuda() for k, x in eri.items()}, torch.from_numpy(t1p).cuda(),
                         torch.from_numpy(t2p).cuda())
    yield dict(cc=cc, o=o, v=v, c=c, ctx=ctx)
    ctx.close()


def test_lowest_roots_match_dense_oracle_spectrum(cfg1):
    s = cfg1
    A = s["c"].dense_jacobian()
    ref = np.linalg.eigvals(A)
    ref = ref[np.argsort(ref.real)]
    eig, r1, r2, info = s["cc"].cclr_eom(s["ctx"], 5, tol=1e-9, maxiter=200)
    assert info.converged == 1 and info.max_residual <= 1e-9
    for k in range(5):
        assert abs(eig[k] - ref[k]) <= 1e-8 * abs(ref[k]), (k, eig[k], ref[k])
        x1, x2 = packing.unpack_amplitudes(r1[k].cpu().numpy(), r2[k].cpu().numpy(), s["o"], s["v"])
        x = flat(x1, x2)
        assert abs(np.linalg.norm(x) - 1.0) < 1e-10
        q = flat(*s["c"].sigma(x1, x2))                      # A x by the oracle
        assert np.linalg.norm(q - eig[k] * x) <= 1e-8


def test_small_trial_space_collapses_and_still_converges(cfg1):
    s = cfg1
    ref = np.linalg.eigvals(s["c"].dense_jacobian())
    ref = ref[np.argsort(ref.real)]
    s["ctx"].set_max_subspace(8)
    try:
        eig, r1, r2, info = s["cc"].cclr_eom(s["ctx"], 2, tol=1e-8, maxiter=300)
    finally:
        s["ctx"].set_max_subspace(0)
    assert info.converged == 1 and info.subspace <= 8
    assert abs(eig[0] - ref[0]) < 1e-7 and abs(eig[1] - ref[1]) < 1e-7


def test_response_pole_sits_at_the_first_eom_energy(cfg1):
    """t(z) = -(A - z)^-1 xi ~ -x_1 (l_1 . xi) / (theta_1 - z) next to the first pole.  A is not Hermitian
    and the synthetic integrals have no time-reversal symmetry, so theta_1 is complex (Im ~ 1e-3 here, reading 17):
    the pole is approached along z = theta_1 - delta with the damping gamma = Im theta_1 (Eq. 20-21)."""
    s = cfg1
    cc = s["cc"]
    eig, r1, r2, info = cc.cclr_eom(s["ctx"], 1, tol=1e-9, maxiter=200)
    assert info.converged == 1
    th = eig[0].real
    xi = s["c"].xi(synth.hermitian_operator(s["o"] + s["v"], 0, 0))
    a, b = packing.pack_amplitudes(*xi)
    xi1, xi2 = torch.from_numpy(a.reshape(1, -1)).cuda(), torch.from_numpy(b.reshape(1, -1)).cuda()
    t1, t2, sinfo = cc.cclr_solve(s["ctx"], xi1, xi2, [th - 0.002, th - 0.004], eig[0].imag, tol=1e-9, maxiter=400)
    assert sinfo.converged == 1
    T = torch.cat([t1[0], t2[0]], dim=1)                                   # [2, n]
    norms = T.abs().pow(2).sum(dim=1).sqrt()
    assert abs(float(norms[0] / norms[1]) - 2.0) < 0.06                     # 1/(theta - w) growth
    x = torch.cat([r1[0], r2[0]])
    overlap = abs(complex(torch.dot(x.conj(), T[0]))) / float(norms[0])
    assert overlap > 0.99                                                   # and it grows along the eigenvector


def test_two_level_closed_form_spectrum():
    import paper_2307_14296_b200 as cc
    f, V, o, _ = two_level_system()
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2, _ = ccsd.solve_ground_state(ints, tol=1e-13)
    full = dict(oooo=ints.oooo, ooov=ints.ooov, oovv=ints.oovv, ovvo=ints.ovvo, ovvv=ints.ovvv, vvvv=ints.vvvv)
    eri = {k: torch.from_numpy(x.reshape(-1).copy()).cuda() for k, x in packing.pack_eri(full).items()}
    t1p, t2p = packing.pack_amplitudes(t1, t2)
    ctx = cc.cclr_create(o, 2, torch.from_numpy(f).cuda(), eri, torch.from_numpy(t1p.reshape(-1).copy()).cuda(),
                         torch.from_numpy(t2p.reshape(-1).copy()).cuda())
    eig, r1, r2, info = cc.cclr_eom(ctx, 5, tol=1e-10, maxiter=20)
    assert info.converged == 1
    got = np.sort(np.array(eig).real)
    assert np.abs(got - np.sort(GOLD["jacobian_eigenvalues"])).max() < 1e-10
    assert np.abs(np.array(eig).imag).max() < 1e-10
    ctx.close()
