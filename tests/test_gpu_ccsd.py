"""cclr_ccsd (GPU ground state) against the oracle's DIIS solver (oracle/ccsd.py, pinned by the determinant
space): amplitudes, energy, and the residual of the GPU amplitudes re-evaluated by the oracle."""
import numpy as np
import pytest
import torch

import synth
from oracle import ccsd, packing
from test_golden_closed_form import GOLD, two_level_system

pytestmark = pytest.mark.gpu


def _run(o, v, f, eri, tol=1e-10):
    import paper_2307_14296_b200 as cc
    return cc.cclr_ccsd(o, v, f.contiguous().cuda(), {k: x.cuda() for k, x in eri.items()}, tol=tol, maxiter=80)


@pytest.mark.parametrize("o,v,scale,diag", [(4, 20, 0.05, True), (3, 7, 0.08, False), (6, 30, None, True)])
def test_ground_state_matches_oracle(o, v, scale, diag):
    eri = synth.eri_packed(o, v, seed=0, scale=scale)
    f = synth.fock(o, v, seed=0)
    if not diag:
        f = f + 0.03 * torch.from_numpy(synth.hermitian_operator(o + v, 0, 7))
    ints = ccsd.Integrals(o, v, f.numpy(), **packing.unpack_eri(o, v, {k: x.numpy() for k, x in eri.items()}))
    w1, w2, winfo = ccsd.solve_ground_state(ints, tol=1e-11)
    assert winfo["converged"]
    t1, t2, info = _run(o, v, f, eri)
    assert info.converged == 1 and info.residual <= 1e-10
    g1, g2 = packing.unpack_amplitudes(t1.cpu().numpy(), t2.cpu().numpy(), o, v)
    nrm = np.sqrt(np.linalg.norm(w1) ** 2 + np.linalg.norm(w2) ** 2)
    assert np.sqrt(np.linalg.norm(g1 - w1) ** 2 + np.linalg.norm(g2 - w2) ** 2) <= 1e-9 * nrm
    o1, o2 = ccsd.residual(ints, g1, g2)                         # oracle's residual of the GPU amplitudes
    assert np.sqrt(np.linalg.norm(o1) ** 2 + np.linalg.norm(o2) ** 2) <= 2e-10
    e = ccsd.energy(ints, w1, w2)
    assert abs(complex(info.energy_re, info.energy_im) - e) <= 1e-10 * max(1.0, abs(e))


def test_two_level_closed_form_energy():
    f, V, o, _ = two_level_system()
    ints = ccsd.Integrals.from_full(f, V, o)
    full = dict(oooo=ints.oooo, ooov=ints.ooov, oovv=ints.oovv, ovvo=ints.ovvo, ovvv=ints.ovvv, vvvv=ints.vvvv)
    eri = {k: torch.from_numpy(x.reshape(-1).copy()) for k, x in packing.pack_eri(full).items()}
    t1, t2, info = _run(o, 2, torch.from_numpy(f), eri, tol=1e-12)
    assert info.converged == 1
    assert abs(info.energy_re - GOLD["E_corr"]) < 1e-11 and abs(info.energy_im) < 1e-11
    assert abs(complex(t2.cpu().numpy()[0]) - complex(*GOLD["t2_23_01"])) < 1e-11
    assert t1.abs().max().item() < 1e-11


def test_divergent_input_reports_not_converged():
    """The literal sigma_V = 0.05 at a config-2-like size diverges; the call must say so, not hang or throw."""
    import paper_2307_14296_b200 as cc
    o, v = 6, 40
    eri = synth.eri_packed(o, v, seed=0, scale=0.25)
    f = synth.fock(o, v, seed=0)
    t1, t2, info = cc.cclr_ccsd(o, v, f.cuda(), {k: x.cuda() for k, x in eri.items()}, tol=1e-10, maxiter=6)
    assert info.converged == 0 and info.residual > 1e-10


@pytest.mark.parametrize("o,v,diag", [(3, 7, False), (6, 30, True)])
def test_both_residual_routes_match_the_oracle(o, v, diag):
    """cclr_ccsd_residual mode 0 (direct plan) and mode 1 (quadrature of the Jacobian) against oracle.ccsd.residual at random
    unconverged amplitudes."""
    import paper_2307_14296_b200 as cc
    eri = synth.eri_packed(o, v, seed=3, scale=0.1)
    f = synth.fock(o, v, seed=3)
    if not diag:
        f = f + 0.05 * torch.from_numpy(synth.hermitian_operator(o + v, 3, 7))
    t1, t2 = synth.amplitudes(o, v, seed=4, scale=0.05)
    ints = ccsd.Integrals(o, v, f.numpy(), **packing.unpack_eri(o, v, {k: x.numpy() for k, x in eri.items()}))
    w1, w2 = packing.pack_amplitudes(*ccsd.residual(ints, *packing.unpack_amplitudes(t1[0].numpy(), t2[0].numpy(), o, v)))
    dev = {k: x.cuda() for k, x in eri.items()}
    for mode in (0, 1):
        g1, g2 = cc.cclr_ccsd_residual(o, v, f.contiguous().cuda(), dev, t1[0].cuda(), t2[0].cuda(), mode)
        torch.cuda.synchronize()
        assert np.linalg.norm(g1.cpu().numpy() - w1.reshape(-1)) <= 1e-11 * np.linalg.norm(w1), mode
        assert np.linalg.norm(g2.cpu().numpy() - w2.reshape(-1)) <= 1e-11 * np.linalg.norm(w2), mode


def test_residual_routes_agree_at_config5_size():
    """At a size the oracle cannot reach in seconds (o=18, v=150) the two device routes -- which share no residual code --
    must agree with each other."""
    import paper_2307_14296_b200 as cc
    o, v = 18, 150
    eri = {k: synth.eri_class(k, o, v, seed=0, device="cuda") for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv", "vvvv")}
    f = synth.fock(o, v, seed=0).cuda()
    t1, t2 = synth.first_order_amplitudes(o, v, f, eri["oovv"])
    t1 = t1 + synth.amplitudes(o, v, seed=5, scale=1e-3, device="cuda")[0][0]
    a1, a2 = cc.cclr_ccsd_residual(o, v, f, eri, t1, t2, 0)
    b1, b2 = cc.cclr_ccsd_residual(o, v, f, eri, t1, t2, 1)
    rel = lambda x, y: float((x - y).abs().pow(2).sum().sqrt() / y.abs().pow(2).sum().sqrt())
    assert rel(a1, b1) < 1e-11 and rel(a2, b2) < 1e-11
    del eri
    torch.cuda.empty_cache()
