"""Pins for oracle/ccsd.py: brute-force determinant algebra (oracle/bruteforce.py = the definitions of
PAPER.md:131 Eq. 14 and Table 1), FCI for two electrons, packing round trips."""
import numpy as np
import pytest
from conftest import random_system, random_amplitudes
from oracle import bruteforce, ccsd, packing


@pytest.mark.parametrize("o,v", [(2, 4), (3, 4), (4, 4), (2, 5)])
def test_residual_and_energy_match_determinant_space(o, v):
    # non-diagonal complex Fock, random complex (unconverged) amplitudes: every term of Omega is exercised
    f, V = random_system(o, v, seed=11 + o, diag_fock=False)
    t1, t2 = random_amplitudes(o, v, seed=3)
    bf = bruteforce.BruteForce(f, V, o)
    e_bf, o1_bf, o2_bf = bf.energy_and_residual(t1, t2)
    ints = ccsd.Integrals.from_full(f, V, o)
    assert abs(ccsd.energy(ints, t1, t2) - e_bf) < 1e-12
    o1, o2 = ccsd.residual(ints, t1, t2)
    assert np.abs(o1 - o1_bf).max() < 1e-12
    assert np.abs(o2 - o2_bf).max() < 1e-12
    assert np.abs(o2_bf).max() > 0.1            # the comparison is not vacuous


def test_residual_is_holomorphic_in_t():
    # no conjugation of amplitudes anywhere: Omega(t) at complex t equals its Taylor polynomial along i*x
    o, v = 2, 4
    f, V = random_system(o, v, seed=5, diag_fock=False)
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2 = random_amplitudes(o, v, seed=1)
    x1, x2 = random_amplitudes(o, v, seed=2)
    # Cauchy-Riemann: d/d(eps) along x times i == d/d(eps) along i*x
    h = 1e-3
    d_re = [(a - b) / (2 * h) for a, b in zip(ccsd.residual(ints, t1 + h * x1, t2 + h * x2),
                                              ccsd.residual(ints, t1 - h * x1, t2 - h * x2))]
    d_im = [(a - b) / (2 * h) for a, b in zip(ccsd.residual(ints, t1 + 1j * h * x1, t2 + 1j * h * x2),
                                              ccsd.residual(ints, t1 - 1j * h * x1, t2 - 1j * h * x2))]
    for a, b in zip(d_re, d_im):
        assert np.abs(1j * a - b).max() < 1e-5


def test_two_electron_ccsd_is_fci():
    o, v = 2, 4
    f, V = random_system(o, v, seed=1)
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2, info = ccsd.solve_ground_state(ints, tol=1e-12)
    assert info["converged"]
    bf = bruteforce.BruteForce(f, V, o)
    w, _ = bf.fci()
    e_ref = (bf.sp.ref @ bf.H @ bf.sp.ref).real
    assert abs(e_ref + ccsd.energy(ints, t1, t2).real - w[0]) < 1e-11
    assert abs(ccsd.energy(ints, t1, t2).imag) < 1e-11


def test_ground_state_residual_certified_by_determinant_space():
    o, v = 3, 4
    f, V = random_system(o, v, seed=2)
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2, info = ccsd.solve_ground_state(ints, tol=1e-11)
    assert info["converged"]
    _, o1, o2 = bruteforce.BruteForce(f, V, o).energy_and_residual(t1, t2)
    assert np.abs(o1).max() < 1e-10 and np.abs(o2).max() < 1e-10


def test_packing_roundtrip_and_pair_index():
    o, v = 3, 5
    p, q = packing.pairs(v)
    assert np.array_equal(q * (q - 1) // 2 + p, np.arange(v * (v - 1) // 2))
    x1, x2 = random_amplitudes(o, v, seed=4)
    a, b = packing.pack_amplitudes(x1, x2)
    assert b.shape == (10, 3)
    assert b[packing.npair(v) - 1, 0] == x2[v - 2, v - 1, 0, 1]
    y1, y2 = packing.unpack_amplitudes(a, b, o, v)
    assert np.array_equal(x1, y1) and np.array_equal(x2, y2)
    f, V = random_system(o, v, seed=6)
    ints = ccsd.Integrals.from_full(f, V, o)
    full = {k: getattr(ints, k) for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv", "vvvv")}
    back = packing.unpack_eri(o, v, packing.pack_eri(full))
    for k in full:
        assert np.array_equal(full[k], back[k]), k
    z1, z2 = packing.unflat(packing.flat(x1, x2), o, v)
    assert np.array_equal(z1, x1) and np.array_equal(z2, x2)
