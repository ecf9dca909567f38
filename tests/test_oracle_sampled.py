"""Pins for oracle/sampled.py (the element-by-element definitions used by the full-size GPU parity tests): every element
against oracle.cclr.CCLR (pinned by the determinant-space definitions) at small sizes."""
import numpy as np
import pytest

import synth
from oracle import ccsd, cclr, packing, sampled


@pytest.mark.parametrize("o,v", [(3, 5), (4, 7)])
def test_sigma_T0_elements_match_full_oracle(o, v):
    eri = {k: x.numpy() for k, x in synth.eri_packed(o, v, seed=o + v, scale=0.3).items()}
    f = synth.fock(o, v, seed=1).numpy() + 0.1 * synth.hermitian_operator(o + v, 2, 5)     # f_ov != 0 on purpose
    ints = ccsd.Integrals(o, v, f, **packing.unpack_eri(o, v, eri))
    c = cclr.CCLR(ints, np.zeros((v, o), complex), np.zeros((v, v, o, o), complex))
    x1, x2 = synth.amplitudes(o, v, seed=3, cls1="x1", cls2="x2")
    x1, x2 = x1[0].numpy(), x2[0].numpy()
    z = 0.0773 + 0.0045j
    w1, w2 = c.sigma(*packing.unpack_amplitudes(x1, x2, o, v), z=z)
    vvvv = eri["vvvv"].reshape(packing.npair(v), -1)
    singles = [(a, i) for a in range(v) for i in range(o)]
    doubles = [(a, b, i, j) for b in range(v) for a in range(b) for j in range(o) for i in range(j)]
    g1, g2 = sampled.sigma_T0_elements(o, v, f, eri, lambda ab: vvvv[ab], x1, x2, singles, doubles, z=z)
    assert np.abs(np.array(g1) - np.array([w1[a, i] for a, i in singles])).max() < 1e-13
    assert np.abs(np.array(g2) - np.array([w2[a, b, i, j] for a, b, i, j in doubles])).max() < 1e-13


def test_ladder_rows_is_term_T11():
    o, v = 3, 6
    eri = {k: x.numpy() for k, x in synth.eri_packed(o, v, seed=4, scale=0.3).items()}
    _, x2 = synth.amplitudes(o, v, seed=5, cls1="x1", cls2="x2")
    x2p = x2[0].numpy().reshape(packing.npair(v), packing.npair(o))
    full = packing.unpack_eri(o, v, eri)
    r2 = packing.unpack_pair_axis(packing.unpack_pair_axis(x2p, o, 1), v, 0)
    want = 0.5 * np.einsum("abef,efij->abij", full["vvvv"], r2)                       # T11 as printed
    want = packing.pack_pair_axes(packing.pack_pair_axes(want, 2), 0)
    rows = [0, 3, 14]
    got = sampled.ladder_rows(eri["vvvv"].reshape(15, 15)[rows], x2p)
    assert np.abs(got - want[rows]).max() < 1e-14


def _small_system_with_T(o, v):
    eri = {k: x.numpy() for k, x in synth.eri_packed(o, v, seed=o + 3 * v, scale=0.3).items()}
    f = synth.fock(o, v, seed=2).numpy() + 0.1 * synth.hermitian_operator(o + v, 3, 5)      # f_ov != 0 on purpose
    t1, t2 = synth.amplitudes(o, v, seed=4, scale=0.4)
    t1, t2 = t1[0].numpy(), t2[0].numpy()
    ints = ccsd.Integrals(o, v, f, **packing.unpack_eri(o, v, eri))
    c = cclr.CCLR(ints, *packing.unpack_amplitudes(t1, t2, o, v))
    vvvv = eri["vvvv"].reshape(packing.npair(v), -1)
    s = sampled.SampledCCLR(o, v, f, eri, lambda ab: vvvv[ab], t1, t2)
    return c, s


@pytest.mark.parametrize("o,v", [(3, 5), (4, 6)])
def test_dressed_intermediate_slices_match_full_oracle(o, v):
    """Every slice method of SampledCCLR against the full-tensor intermediates of oracle.cclr.CCLR (pinned by the
    determinant-space definitions), all slices, random complex T: a wrong sign, index or symmetry relation fails here."""
    c, s = _small_system_with_T(o, v)
    tol = 1e-13
    assert np.abs(s.Fme() - c.Fme).max() < tol
    assert np.abs(s.Fmi() - c.Fmi).max() < tol
    for a in range(v):
        assert np.abs(s.Fae_row(a) - c.Fae[a]).max() < tol
        assert np.abs(s.Wamef_a(a) - c.Wamef[a]).max() < tol
    for i in range(o):
        assert np.abs(s.Wmnie_i(i) - c.Wmnie[:, :, i, :]).max() < tol
        for j in range(o):
            assert np.abs(s.Wmnij_col(i, j) - c.Wmnij[:, :, i, j]).max() < tol
    for b in range(v):
        for j in range(o):
            assert np.abs(s.Wbar_bj(b, j) - c.Wbar[:, b, :, j]).max() < tol
            assert np.abs(s.Wmbej_bj(b, j) - c.Wmbej[:, b, :, j]).max() < tol
            for i in range(o):
                assert np.abs(s.Wmbij_bij(b, i, j) - c.Wmbij[:, b, i, j]).max() < tol
    for b in range(v):
        for a in range(b):
            assert np.abs(s.Wabef_row(a, b) - c.Wabef[a, b]).max() < tol
            for j in range(o):
                assert np.abs(s.Wabej_abj(a, b, j) - c.Wabej[a, b, :, j]).max() < tol


@pytest.mark.parametrize("o,v", [(3, 5), (4, 6)])
def test_sigma_elements_with_T_match_full_oracle(o, v):
    c, s = _small_system_with_T(o, v)
    x1, x2 = synth.amplitudes(o, v, seed=6, cls1="x1", cls2="x2")
    x1, x2 = x1[0].numpy(), x2[0].numpy()
    z = 0.0773 + 0.0045j
    w1, w2 = c.sigma(*packing.unpack_amplitudes(x1, x2, o, v), z=z)
    singles = [(a, i) for a in range(v) for i in range(o)]
    doubles = [(a, b, i, j) for b in range(v) for a in range(b) for j in range(o) for i in range(j)]
    g1, g2 = s.sigma_elements(x1, x2, singles, doubles, z=z)
    assert np.abs(np.array(g1) - np.array([w1[a, i] for a, i in singles])).max() < 1e-12
    assert np.abs(np.array(g2) - np.array([w2[a, b, i, j] for a, b, i, j in doubles])).max() < 1e-12
    # and at T = 0 it reduces to the bare-integral definition above
    eri = {k: x.numpy() for k, x in synth.eri_packed(o, v, seed=o + 3 * v, scale=0.3).items()}
    vvvv = eri["vvvv"].reshape(packing.npair(v), -1)
    f = synth.fock(o, v, seed=2).numpy() + 0.1 * synth.hermitian_operator(o + v, 3, 5)
    s0 = sampled.SampledCCLR(o, v, f, eri, lambda ab: vvvv[ab], np.zeros((v, o), complex),
                             np.zeros((packing.npair(v), packing.npair(o)), complex))
    h1, h2 = s0.sigma_elements(x1, x2, singles[:7], doubles[:9], z=z)
    k1, k2 = sampled.sigma_T0_elements(o, v, f, eri, lambda ab: vvvv[ab], x1, x2, singles[:7], doubles[:9], z=z)
    assert np.abs(np.array(h1) - np.array(k1)).max() < 1e-13 and np.abs(np.array(h2) - np.array(k2)).max() < 1e-13


@pytest.mark.parametrize("o,v", [(3, 5), (4, 6)])
def test_left_transform_slices_and_elements_match_full_oracle(o, v):
    """The second family of slices (fixed e / fixed m / columns) and every element of l (A - z) against oracle.cclr.CCLR
    (whose sigma_left is pinned against the transpose of the determinant-space Jacobian)."""
    c, s = _small_system_with_T(o, v)
    tol = 1e-13
    for e in range(v):
        assert np.abs(s.Fae_col(e) - c.Fae[:, e]).max() < tol
        assert np.abs(s.Wabej_e(e) - c.Wabej[:, :, e, :]).max() < tol
        assert np.abs(s.Wabef_e(e) - c.Wabef[:, :, e, :]).max() < tol
        assert np.abs(s.Wbar_e(e) - c.Wbar[:, :, e, :]).max() < tol
        for m in range(o):
            assert np.abs(s.Wmbej_me(m, e) - c.Wmbej[m, :, e, :]).max() < tol
            assert np.abs(s.Wamef_me(m, e) - c.Wamef[:, m, :, e]).max() < tol
            assert np.abs(s.Wmnie_me(m, e) - c.Wmnie[:, m, :, e]).max() < tol
            for f in range(e + 1, v):
                assert np.abs(s.Wamef_mef(m, e, f) - c.Wamef[:, m, e, f]).max() < tol
        for f in range(e + 1, v):
            assert np.abs(s.Wabef_col(e, f) - c.Wabef[:, :, e, f]).max() < tol
    for m in range(o):
        assert np.abs(s.Wmbij_m(m) - c.Wmbij[m]).max() < tol
        assert np.abs(s.Wbar_m(m) - c.Wbar[m]).max() < tol
        for n in range(o):
            assert np.abs(s.Wmnij_row(m, n) - c.Wmnij[m, n]).max() < tol
    y1, y2 = synth.amplitudes(o, v, seed=8, cls1="x1", cls2="x2")
    y1, y2 = y1[0].numpy(), y2[0].numpy()
    z = -0.0773 + 0.0045j
    w1, w2 = c.sigma_left(*packing.unpack_amplitudes(y1, y2, o, v), z=z)
    singles = [(a, i) for a in range(v) for i in range(o)]
    doubles = [(a, b, i, j) for b in range(v) for a in range(b) for j in range(o) for i in range(j)]
    g1, g2 = s.sigma_left_elements(y1, y2, singles, doubles, z=z)
    assert np.abs(np.array(g1) - np.array([w1[a, i] for a, i in singles])).max() < 1e-12
    assert np.abs(np.array(g2) - np.array([w2[a, b, i, j] for a, b, i, j in doubles])).max() < 1e-12
    e1, e2 = c.eta0()
    h1, h2 = s.eta0_elements(singles, doubles)
    assert np.abs(np.array(h1) - np.array([e1[a, i] for a, i in singles])).max() < tol
    assert np.abs(np.array(h2) - np.array([e2[a, b, i, j] for a, b, i, j in doubles])).max() < tol


@pytest.mark.parametrize("o,v", [(3, 5), (4, 6)])
def test_xi_eta_and_omega_elements_match_full_oracle(o, v):
    c, s = _small_system_with_T(o, v)
    singles = [(a, i) for a in range(v) for i in range(o)]
    doubles = [(a, b, i, j) for b in range(v) for a in range(b) for j in range(o) for i in range(j)]
    pick = lambda w1, w2: (np.array([w1[a, i] for a, i in singles]), np.array([w2[a, b, i, j] for a, b, i, j in doubles]))
    lam1, lam2 = synth.amplitudes(o, v, seed=9, cls1="x1", cls2="x2")
    lam1, lam2 = lam1[0].numpy(), lam2[0].numpy()
    L1, L2 = packing.unpack_amplitudes(lam1, lam2, o, v)
    for X in (synth.hermitian_operator(o + v, 1, 0), synth.hermitian_operator(o + v, 1, 1, imaginary_antisymmetric=True)):
        w1, w2 = pick(*c.xi(X))                          # = Omega[f := X, V := 0](t), the definition (pinned)
        g1, g2 = s.xi_elements(X, singles, doubles)
        assert np.abs(np.array(g1) - w1).max() < 1e-13 and np.abs(np.array(g2) - w2).max() < 1e-13
        for eom in (False, True):
            w1, w2 = pick(*(c.eta_eom(X, L1, L2) if eom else c.eta(X, L1, L2)))
            g1, g2 = s.eta_elements(X, lam1, lam2, singles, doubles, eom=eom)
            assert np.abs(np.array(g1) - w1).max() < 1e-12 and np.abs(np.array(g2) - w2).max() < 1e-12
    w1, w2 = pick(*ccsd.residual(c.I, c.t1, c.t2))
    g1, g2 = s.omega_elements(singles, doubles)
    assert np.abs(np.array(g1) - w1).max() < 1e-12 and np.abs(np.array(g2) - w2).max() < 1e-12
