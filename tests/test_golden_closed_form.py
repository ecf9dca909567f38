"""The oracle against tests/golden/two_level_closed_form.json: a 2-electron, 4-spinor system whose CCSD energy, amplitude,
Jacobian spectrum and response function have closed forms (written by tests/golden/make_golden.py from the formulas alone)."""
import json
import os

import numpy as np
import pytest

from oracle import ccsd, cclr

GOLD = json.load(open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "two_level_closed_form.json")))


def two_level_system():
    g = GOLD
    K = complex(*g["K"])
    n, o = 4, 2
    f = np.diag([g["eps_o"], g["eps_o"], g["eps_v"], g["eps_v"]]).astype(complex)
    V = np.zeros((n,) * 4, complex)
    for (p, q, sp) in ((2, 3, 1), (3, 2, -1)):
        for (r, s, sr) in ((0, 1, 1), (1, 0, -1)):
            V[p, q, r, s] = sp * sr * K                  # <23||01> = K
            V[r, s, p, q] = sp * sr * np.conj(K)         # <01||23> = conj K
    X = np.zeros((n, n), complex)
    X[2, 0] = X[0, 2] = g["d"]
    return f, V, o, X


def test_ground_state_energy_and_amplitude():
    f, V, o, _ = two_level_system()
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2, info = ccsd.solve_ground_state(ints, tol=1e-13)
    assert info["converged"]
    assert abs(ccsd.energy(ints, t1, t2) - GOLD["E_corr"]) < 1e-12
    assert np.abs(t1).max() < 1e-12
    assert abs(t2[0, 1, 0, 1] - complex(*GOLD["t2_23_01"])) < 1e-12


def test_jacobian_spectrum():
    f, V, o, _ = two_level_system()
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2, _ = ccsd.solve_ground_state(ints, tol=1e-13)
    ev = np.sort(np.linalg.eigvals(cclr.CCLR(ints, t1, t2).dense_jacobian()).real)
    assert np.abs(ev - np.sort(GOLD["jacobian_eigenvalues"])).max() < 1e-10


@pytest.mark.parametrize("k", range(len(GOLD["response"])))
def test_response_function(k):
    f, V, o, X = two_level_system()
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2, _ = ccsd.solve_ground_state(ints, tol=1e-13)
    c = cclr.CCLR(ints, t1, t2)
    A = c.dense_jacobian()
    l1, l2 = c.solve_lambda_dense(A)
    z = complex(*GOLD["response"][k]["z"])
    want = complex(*GOLD["response"][k]["XX"])
    solve = lambda a, b, zz: c.solve_dense(A, a, b, zz)
    assert abs(c.response_cc_cc(solve, X, X, z, l1, l2) - want) < 1e-10 * abs(want)
    assert abs(c.response_cc_ci(solve, X, X, z, l1, l2) - want) < 1e-10 * abs(want)
