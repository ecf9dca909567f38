"""Host-logic check of the contraction plans (csrc/plans.inc): the plan text the GPU library executes is run by a
numpy interpreter (tests/plan_interp.py) and compared with the oracle -- every intermediate of S-Eq. 15-28
 and the sigma vector of S-Eq. 11-12.  A wrong sign, index order, pair
unpacking or GEMM shape anywhere in the plan fails here, on the CPU, before any kernel runs."""
import numpy as np
import pytest
from conftest import random_system, random_amplitudes
from oracle import ccsd, cclr, packing
import plan_interp


def _setup(o, v, seed, chunk_override=None):
    f, V = random_system(o, v, seed=seed, diag_fock=False)
    t1, t2 = random_amplitudes(o, v, seed=seed + 1)
    ints = ccsd.Integrals.from_full(f, V, o)
    full = dict(oooo=ints.oooo, ooov=ints.ooov, oovv=ints.oovv, ovvo=ints.ovvo, ovvv=ints.ovvv, vvvv=ints.vvvv)
    packed = packing.pack_eri(full)
    t1p, t2p = packing.pack_amplitudes(t1, t2)
    it = plan_interp.run_create(o, v, f, packed, t1p, t2p, chunk_override)
    return it, cclr.CCLR(ints, t1, t2)


def _close(a, b, tol=1e-12):
    return np.abs(a - b).max() <= tol * max(1.0, np.abs(b).max())


@pytest.mark.parametrize("o,v,chunk", [(3, 5, None), (4, 6, 2), (2, 7, 3)])
def test_create_plan_reproduces_oracle_intermediates(o, v, chunk):
    it, c = _setup(o, v, seed=40 + v, chunk_override=chunk)
    P = packing
    assert _close(it.get("Fme"), c.Fme)
    assert _close(it.get("FmeT"), c.Fme.T)
    assert _close(it.get("Fmi"), c.Fmi)
    assert _close(it.get("Fae"), c.Fae)
    assert _close(it.get("Wmnij"), P.pack_pair_axes(P.pack_pair_axes(c.Wmnij, 2), 0))
    assert _close(it.get("Wabef"), P.pack_pair_axes(P.pack_pair_axes(c.Wabef, 2), 0))
    assert _close(it.get("Wring"), c.Wmbej.transpose(1, 3, 2, 0))                    # [b j e m]
    assert _close(it.get("Wie"), P.pack_pair_axes(c.Wmnie, 0).transpose(1, 2, 0))    # [i e (mn)]
    assert _close(it.get("Wnjem"), c.Wmnie.transpose(0, 2, 3, 1))                    # [n j e m] = W[nm,je]
    assert _close(it.get("Wamef"), P.pack_pair_axes(c.Wamef, 2))                     # [a m (ef)]
    assert _close(it.get("Wx"), c.Wamef.transpose(0, 2, 3, 1))                       # [b f e m] = W[bm,fe]
    assert _close(it.get("Wmbij"), P.pack_pair_axes(c.Wmbij, 2))
    assert _close(it.get("Wabej"), P.pack_pair_axes(c.Wabej, 0).transpose(0, 2, 1))  # [(ab) j e]
    assert _close(it.get("Vnm"), P.pack_pair_axes(c.I.oovv, 2))
    assert _close(it.get("Vx"), P.pack_pair_axes(c.I.oovv, 0).transpose(1, 2, 0))    # [f e (mn)]
    assert _close(it.get("Ut"), P.pack_pair_axes(c.t2, 2))
    assert _close(it.get("To"), P.pack_pair_axes(c.t2, 0))


@pytest.mark.parametrize("o,v,chunk", [(3, 5, None), (4, 6, 2)])
def test_sigma_plan_reproduces_oracle_sigma(o, v, chunk):
    it, c = _setup(o, v, seed=50 + v, chunk_override=chunk)
    for k, z in enumerate([0.0, 0.0773 + 0.0045j]):
        x1, x2 = random_amplitudes(o, v, seed=60 + k, scale=1.0)
        x1p, x2p = packing.pack_amplitudes(x1, x2)
        s1, s2 = plan_interp.run_sigma(it, x1p, x2p, z)
        r1, r2 = packing.pack_amplitudes(*c.sigma(x1, x2, z))
        assert np.linalg.norm(s1 - r1) <= 1e-12 * np.linalg.norm(r1)
        assert np.linalg.norm(s2 - r2) <= 1e-12 * np.linalg.norm(r2)


@pytest.mark.parametrize("o,v", [(3, 5), (4, 6)])
def test_xi_plan_reproduces_oracle_xi(o, v):
    from conftest import random_hermitian
    it, c = _setup(o, v, seed=70 + v)
    x1, x2 = random_amplitudes(o, v, seed=71, scale=1.0)
    plan_interp.run_sigma(it, *packing.pack_amplitudes(x1, x2), 0.0)          # declares the shared work buffers
    X = random_hermitian(o + v, 72) + 0.3j * np.random.default_rng(73).normal(size=(o + v, o + v))   # not even Hermitian
    s1, s2 = plan_interp.run_xi(it, X)
    r1, r2 = packing.pack_amplitudes(*c.xi(X))
    assert np.linalg.norm(s1.reshape(-1) - r1.reshape(-1)) <= 1e-12 * np.linalg.norm(r1)
    assert np.linalg.norm(s2.reshape(-1) - r2.reshape(-1)) <= 1e-12 * np.linalg.norm(r2)


@pytest.mark.parametrize("o,v,chunk", [(3, 5, None), (4, 6, 2)])
def test_left_sigma_plan_reproduces_oracle_left_sigma(o, v, chunk):
    it, c = _setup(o, v, seed=80 + v, chunk_override=chunk)
    x1, x2 = random_amplitudes(o, v, seed=81, scale=1.0)
    plan_interp.run_sigma(it, *packing.pack_amplitudes(x1, x2), 0.0)          # declares the shared work buffers
    for k, z in enumerate([0.0, 0.0773 + 0.0045j]):
        l1, l2 = random_amplitudes(o, v, seed=82 + k, scale=1.0)
        s1, s2 = plan_interp.run_sigma_left(it, *packing.pack_amplitudes(l1, l2), z)
        r1, r2 = packing.pack_amplitudes(*c.sigma_left(l1, l2, z))
        assert np.linalg.norm(s1.reshape(-1) - r1.reshape(-1)) <= 1e-12 * np.linalg.norm(r1)
        assert np.linalg.norm(s2.reshape(-1) - r2.reshape(-1)) <= 1e-12 * np.linalg.norm(r2)


@pytest.mark.parametrize("o,v,eom", [(3, 5, False), (4, 6, True)])
def test_eta_plan_reproduces_oracle_eta(o, v, eom):
    from conftest import random_hermitian
    it, c = _setup(o, v, seed=90 + v)
    x1, x2 = random_amplitudes(o, v, seed=91, scale=1.0)
    plan_interp.run_sigma(it, *packing.pack_amplitudes(x1, x2), 0.0)          # declares the shared work buffers
    l1, l2 = random_amplitudes(o, v, seed=92, scale=1.0)
    plan_interp.run_xi(it, random_hermitian(o + v, 1))                         # (xi / left plans declare FX, HX, GLh, GOh ...)
    plan_interp.run_sigma_left(it, *packing.pack_amplitudes(l1, l2), 0.0)
    X = random_hermitian(o + v, 93) + 0.2j * np.random.default_rng(94).normal(size=(o + v, o + v))
    s1, s2 = plan_interp.run_eta(it, X, *packing.pack_amplitudes(l1, l2), eom)
    r1, r2 = packing.pack_amplitudes(*(c.eta_eom(X, l1, l2) if eom else c.eta(X, l1, l2)))
    assert np.linalg.norm(s1.reshape(-1) - r1.reshape(-1)) <= 1e-12 * np.linalg.norm(r1)
    assert np.linalg.norm(s2.reshape(-1) - r2.reshape(-1)) <= 1e-12 * np.linalg.norm(r2)


@pytest.mark.parametrize("o,v,chunk", [(3, 5, None), (4, 6, 2), (2, 7, 3)])
def test_omega_plan_reproduces_oracle_residual(o, v, chunk):
    """The direct CCSD residual plan of cclr_ccsd against oracle.ccsd.residual (pinned by the determinant space), at random
    unconverged complex t and a non-diagonal Fock matrix."""
    f, V = random_system(o, v, seed=100 + v, diag_fock=False)
    t1, t2 = random_amplitudes(o, v, seed=101)
    ints = ccsd.Integrals.from_full(f, V, o)
    full = dict(oooo=ints.oooo, ooov=ints.ooov, oovv=ints.oovv, ovvo=ints.ovvo, ovvv=ints.ovvv, vvvv=ints.vvvv)
    packed = packing.pack_eri(full)
    t1p, t2p = packing.pack_amplitudes(t1, t2)
    s1, s2 = plan_interp.run_omega(o, v, f, packed, t1p, t2p, chunk)
    r1, r2 = packing.pack_amplitudes(*ccsd.residual(ints, t1, t2))
    assert np.abs(s1.reshape(-1) - r1.reshape(-1)).max() <= 1e-12 * max(1.0, np.abs(r1).max())
    assert np.abs(s2.reshape(-1) - r2.reshape(-1)).max() <= 1e-12 * max(1.0, np.abs(r2).max())


@pytest.mark.parametrize("o,v,chunk", [(3, 5, None), (4, 6, 2), (2, 7, 3)])
def test_fy_plan_reproduces_oracle_F_transform(o, v, chunk):
    """The direct F-contraction plan (CCLR_PLAN_FY: derivative of the left transform along y, the two o^2 v^4-sized derivative
    intermediates contracted from the lambda side) against oracle.cclr.CCLR.F_transform, which is pinned by the determinant-space F
    (tests/test_oracle_cclr.py); random unconverged t, random lambda, non-diagonal Fock matrix, every element."""
    f, V = random_system(o, v, seed=110 + v, diag_fock=False)
    t1, t2 = random_amplitudes(o, v, seed=111)
    ints = ccsd.Integrals.from_full(f, V, o)
    full = dict(oooo=ints.oooo, ooov=ints.ooov, oovv=ints.oovv, ovvo=ints.ovvo, ovvv=ints.ovvv, vvvv=ints.vvvv)
    packed = packing.pack_eri(full)
    it = plan_interp.run_create(o, v, f, packed, *packing.pack_amplitudes(t1, t2), chunk)
    c = cclr.CCLR(ints, t1, t2)
    l1, l2 = random_amplitudes(o, v, seed=112, scale=1.0)
    lp = packing.pack_amplitudes(l1, l2)
    plan_interp.run_sigma(it, *lp, 0.0)               # declare the shared work buffers
    plan_interp.run_sigma_left(it, *lp, 0.0)
    for seed in (113, 114):
        y1, y2 = random_amplitudes(o, v, seed=seed, scale=1.0)
        s1, s2 = plan_interp.run_fy(it, packed, *lp, *packing.pack_amplitudes(y1, y2))
        r1, r2 = packing.pack_amplitudes(*c.F_transform(l1, l2, y1, y2))
        assert np.linalg.norm(s1.reshape(-1) - r1.reshape(-1)) <= 1e-12 * np.linalg.norm(r1)
        assert np.linalg.norm(s2.reshape(-1) - r2.reshape(-1)) <= 1e-12 * np.linalg.norm(r2)
