"""Pins for oracle/cclr.py.  Independent references: the determinant-space definitions of Table 1
 via oracle/bruteforce.py, the exact finite-difference Jacobian of the (separately pinned)
CCSD residual, closed-form special cases (V = 0, T = 0), FCI excitation energies and exact sum-over-states
response functions for two electrons (Eq. 23-24), and the finite-field static limit."""
import numpy as np
import pytest
from conftest import random_system, random_amplitudes, random_hermitian
from oracle import bruteforce, ccsd, cclr
from oracle.packing import flat, unflat


def _rel(a, b):
    return np.linalg.norm(a - b) / np.linalg.norm(b)


@pytest.mark.parametrize("o,v", [(2, 4), (3, 4), (4, 4)])
def test_sigma_matches_commutator_definition(o, v):
    f, V = random_system(o, v, seed=20 + v, diag_fock=False)
    t1, t2 = random_amplitudes(o, v, seed=1)          # random, unconverged T: sigma = dOmega/dt . x at any t
    x1, x2 = random_amplitudes(o, v, seed=2)
    bf = bruteforce.BruteForce(f, V, o)
    s1_bf, s2_bf = bf.sigma(t1, t2, x1, x2)
    ints = ccsd.Integrals.from_full(f, V, o)
    s1, s2 = cclr.CCLR(ints, t1, t2).sigma(x1, x2)
    assert np.abs(s1 - s1_bf).max() < 1e-12 and np.abs(s2 - s2_bf).max() < 1e-12
    g1, g2 = cclr.sigma_fd(ints, t1, t2, x1, x2)
    assert np.abs(g1 - s1_bf).max() < 1e-12 and np.abs(g2 - s2_bf).max() < 1e-12
    assert np.abs(s2_bf).max() > 1.0


@pytest.mark.parametrize("term", ["S-Eq.20 sign", "S-Eq.21 sign"])
def test_printed_misprints_are_detected(term):
    """DESIGN.md readings 3, 4: the printed variants must FAIL the determinant-space pin (so the pin has teeth)."""
    o, v = 3, 4
    f, V = random_system(o, v, seed=31, diag_fock=False)
    t1, t2 = random_amplitudes(o, v, seed=1)
    x1, x2 = random_amplitudes(o, v, seed=2)
    ints = ccsd.Integrals.from_full(f, V, o)
    c = cclr.CCLR(ints, t1, t2)
    s1_ok, s2_ok = c.sigma(x1, x2)
    if term == "S-Eq.20 sign":       # PAPER.md:919 prints +F t2
        c.Wmbij = c.Wmbij + 2 * np.einsum("me,beij->mbij", c.Fme, t2)
    else:                            # PAPER.md:924 prints + P V t2
        tmp = np.einsum("mbef,afmj->abej", ints.ovvv, t2)
        c.Wabej = c.Wabej + 2 * (tmp - tmp.transpose(1, 0, 2, 3))
    s1, s2 = c.sigma(x1, x2)
    assert max(np.abs(s1 - s1_ok).max(), np.abs(s2 - s2_ok).max()) > 1e-3


def test_sigma_matches_exact_fd_at_config1_size():
    o, v = 4, 20
    rng = np.random.default_rng(7)
    n = o + v
    # full antisymmetric Hermitian V from a random 4-index tensor (tests-only recipe)
    G = (rng.normal(size=(n,) * 4) + 1j * rng.normal(size=(n,) * 4)) * 0.02
    G = G - G.transpose(1, 0, 2, 3)
    G = G - G.transpose(0, 1, 3, 2)
    V = G + G.transpose(2, 3, 0, 1).conj()
    f = np.diag(np.concatenate([np.sort(rng.uniform(-2, -0.5, o)), np.sort(rng.uniform(0.2, 5, v))])).astype(complex)
    K = (rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))) * 0.02
    f = f + K + K.conj().T
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2 = random_amplitudes(o, v, seed=5, scale=0.05)
    x1, x2 = random_amplitudes(o, v, seed=6, scale=1.0)
    s1, s2 = cclr.CCLR(ints, t1, t2).sigma(x1, x2)
    g1, g2 = cclr.sigma_fd(ints, t1, t2, x1, x2)
    assert _rel(s1, g1) < 1e-12 and _rel(s2, g2) < 1e-12


def test_linearity_and_shift_identity():
    o, v = 3, 5
    f, V = random_system(o, v, seed=3)
    ints = ccsd.Integrals.from_full(f, V, o)
    c = cclr.CCLR(ints, *random_amplitudes(o, v, seed=1))
    x = random_amplitudes(o, v, seed=2)
    y = random_amplitudes(o, v, seed=3)
    al, be = 0.3 - 1.1j, -0.7 + 0.2j
    lhs = c.sigma(al * x[0] + be * y[0], al * x[1] + be * y[1])
    sx, sy = c.sigma(*x), c.sigma(*y)
    for k in range(2):
        assert np.abs(lhs[k] - (al * sx[k] + be * sy[k])).max() < 1e-12
    z = 0.0773 + 0.0045j
    sz = c.sigma(*x, z=z)
    for k in range(2):
        assert np.abs(sz[k] - (sx[k] - z * x[k])).max() < 1e-14


def test_special_case_V_zero_gives_orbital_energy_diagonal():
    o, v = 3, 5
    f, V = random_system(o, v, seed=4)
    ints = ccsd.Integrals.from_full(f, 0 * V, o)
    c = cclr.CCLR(ints, *random_amplitudes(o, v, seed=1))       # arbitrary t
    x1, x2 = random_amplitudes(o, v, seed=2)
    s1, s2 = c.sigma(x1, x2)
    D1, D2 = ccsd.denominators(ints)
    assert np.abs(s1 - D1 * x1).max() < 1e-13 and np.abs(s2 - D2 * x2).max() < 1e-13


def test_special_case_T_zero_is_hermitian_cisd_block():
    o, v = 3, 4
    f, V = random_system(o, v, seed=5)       # f_ov = 0 (Brillouin), else <mu|tau_nu H|R> spoils Hermiticity
    ints = ccsd.Integrals.from_full(f, V, o)
    z1, z2 = np.zeros((v, o), complex), np.zeros((v, v, o, o), complex)
    c = cclr.CCLR(ints, z1, z2)
    A = c.dense_jacobian()
    assert np.abs(A - A.conj().T).max() < 1e-13
    # and it IS the CISD block <mu|H|nu> - E_ref delta
    bf = bruteforce.BruteForce(f, V, o)
    Hmu = bf.bra @ bf.H @ bf.bra.T - (bf.sp.ref @ bf.H @ bf.sp.ref) * np.eye(bf.nmu)
    assert np.abs(A - Hmu).max() < 1e-13


def test_two_electron_spectrum_is_fci():
    o, v = 2, 4
    f, V = random_system(o, v, seed=1)
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2, _ = ccsd.solve_ground_state(ints, tol=1e-12)
    ev = np.sort(np.linalg.eigvals(cclr.CCLR(ints, t1, t2).dense_jacobian()).real)
    w, _ = bruteforce.BruteForce(f, V, o).fci()
    assert np.abs(ev - (w[1:] - w[0])).max() < 1e-9


@pytest.fixture(scope="module")
def small_lr():
    out = {}
    for (o, v) in [(2, 4), (3, 4)]:
        f, V = random_system(o, v, seed=1)
        ints = ccsd.Integrals.from_full(f, V, o)
        t1, t2, info = ccsd.solve_ground_state(ints, tol=1e-12)
        c = cclr.CCLR(ints, t1, t2)
        A = c.dense_jacobian()
        l1, l2 = c.solve_lambda_dense(A)
        out[(o, v)] = dict(f=f, V=V, ints=ints, t1=t1, t2=t2, c=c, A=A, l1=l1, l2=l2,
                           bf=bruteforce.BruteForce(f, V, o))
    return out


@pytest.mark.parametrize("o,v", [(2, 4), (3, 4)])
def test_xi_eta_lambda_F_match_definitions(small_lr, o, v):
    s = small_lr[(o, v)]
    c, bf, t1, t2, l1, l2 = s["c"], s["bf"], s["t1"], s["t2"], s["l1"], s["l2"]
    assert np.abs(s["A"] - bf.jacobian(t1, t2)).max() < 1e-12
    lam = bf.lam(t1, t2)
    assert np.abs(flat(l1, l2) - lam).max() < 1e-12
    X = random_hermitian(o + v, 5)
    assert np.abs(flat(*c.xi(X)) - bf.xi(X, t1, t2)).max() < 1e-12
    assert np.abs(flat(*c.xi_printed(X)) - bf.xi(X, t1, t2)).max() < 1e-12
    assert np.abs(flat(*c.eta(X, l1, l2)) - bf.eta(X, t1, t2, lam)).max() < 1e-12
    F = bf.F(t1, t2, lam)
    assert np.abs(F - F.T).max() < 1e-12
    x, y = random_amplitudes(o, v, 7), random_amplitudes(o, v, 8)
    assert abs(flat(*x) @ F @ flat(*y) - c.xFy(l1, l2, *x, *y)) < 1e-11


@pytest.mark.parametrize("o,v", [(2, 4), (3, 4), (2, 5)])
def test_F_transform_is_the_determinant_space_F_times_y(o, v):
    """oracle.cclr.CCLR.F_transform (differentiated intermediates) against the literal F_mu,nu = <Lambda|[[Hbar,tau_mu],tau_nu]|R>
    of Table 1 built in the determinant space, at random UNCONVERGED complex t and lambda and a non-diagonal Fock
    matrix (the identity F y = d/db [eta0 + lambda A](t + b y) holds for any t, lambda), every element; plus symmetry
    x.(F y) = y.(F x) and agreement with the Richardson second derivative of the Lagrangian (xFy)."""
    f, V = random_system(o, v, seed=31 + v, diag_fock=False)
    t1, t2 = random_amplitudes(o, v, seed=32)
    l1, l2 = random_amplitudes(o, v, seed=33, scale=1.0)
    ints = ccsd.Integrals.from_full(f, V, o)
    c = cclr.CCLR(ints, t1, t2)
    bf = bruteforce.BruteForce(f, V, o)
    F = bf.F(t1, t2, flat(l1, l2))
    for seed in (34, 35):
        y = random_amplitudes(o, v, seed, scale=1.0)
        got = flat(*c.F_transform(l1, l2, *y))
        want = F @ flat(*y)
        assert np.abs(got - want).max() < 1e-11 * max(1.0, np.abs(want).max())
    x, y = random_amplitudes(o, v, 36, scale=1.0), random_amplitudes(o, v, 37, scale=1.0)
    xFy = cclr.dot(*x, *c.F_transform(l1, l2, *y))
    assert abs(xFy - cclr.dot(*y, *c.F_transform(l1, l2, *x))) < 1e-11 * abs(xFy)
    assert abs(xFy - c.xFy(l1, l2, *x, *y)) < 1e-10 * abs(xFy)


@pytest.mark.parametrize("z", [0.0, 0.0773, 0.0773 + 0.0045j, 0.83 + 0.0045j])
def test_two_electron_response_functions_equal_exact_sum_over_states(small_lr, z):
    """CCSD is FCI for two electrons: CC-CC (Eq. 15), CC-CI (Eq. 16) and the exact SOS (Eq. 23-24) coincide;
    z = 0.83+0.0045i sits next to the first pole (0.827)."""
    s = small_lr[(2, 4)]
    c, bf, A, l1, l2 = s["c"], s["bf"], s["A"], s["l1"], s["l2"]
    n = 6
    X, Y = random_hermitian(n, 5), random_hermitian(n, 6)
    Kr = np.random.default_rng(9).normal(size=(n, n))
    M = 1j * (Kr - Kr.T)                                   # Hermitian, imaginary antisymmetric (magnetic-dipole type)
    solve = lambda a, b, zz: c.solve_dense(A, a, b, zz)
    for (P, Q) in [(X, X), (X, Y), (X, M)]:
        exact = bf.sos_response(P, Q, z)
        assert abs(c.response_cc_cc(solve, P, Q, z, l1, l2) - exact) < 1e-9 * max(1, abs(exact))
        assert abs(c.response_cc_ci(solve, P, Q, z, l1, l2) - exact) < 1e-9 * max(1, abs(exact))


def test_three_electron_cc_cc_and_cc_ci_are_close_but_distinct(small_lr):
    s = small_lr[(3, 4)]
    c, A, l1, l2 = s["c"], s["A"], s["l1"], s["l2"]
    X = random_hermitian(7, 5)
    solve = lambda a, b, zz: c.solve_dense(A, a, b, zz)
    a = c.response_cc_cc(solve, X, X, 0.0773, l1, l2)
    b = c.response_cc_ci(solve, X, X, 0.0773, l1, l2)
    exact = s["bf"].sos_response(X, X, 0.0773)
    assert 1e-9 < abs(a - b) / abs(a) < 1e-3
    assert abs(a - exact) / abs(exact) < 1e-3


def test_static_limit_equals_finite_field_second_derivative(small_lr):
    """<<X;X>>_0 = Re d2 E_CCSD / d eps2 for H + eps X with unrelaxed orbitals."""
    s = small_lr[(3, 4)]
    c, A, l1, l2, f, V = s["c"], s["A"], s["l1"], s["l2"], s["f"], s["V"]
    o = 3
    X = random_hermitian(7, 5) * 0.5
    solve = lambda a, b, zz: c.solve_dense(A, a, b, zz)
    lr = c.response_cc_cc(solve, X, X, 0.0, l1, l2)
    h = 0.02
    e = {}
    for k in (-2, -1, 0, 1, 2):
        ints = ccsd.Integrals.from_full(f + k * h * X, V, o)
        t1, t2, info = ccsd.solve_ground_state(ints, tol=1e-13)
        assert info["converged"]
        e[k] = ccsd.energy(ints, t1, t2) + np.einsum("ii->", (k * h * X)[:o, :o])
    d2 = (-e[-2] + 16 * e[-1] - 30 * e[0] + 16 * e[1] - e[2]) / (12 * h * h)
    assert abs(lr.real - d2.real) < 2e-6 * abs(d2.real)


def test_iterative_solver_reaches_dense_solution(small_lr):
    s = small_lr[(3, 4)]
    c, A = s["c"], s["A"]
    X = random_hermitian(7, 5)
    z = 0.0773 + 0.0045j
    ti, info = c.solve_iterative(*c.xi(X), z, tol=1e-11)
    td = c.solve_dense(A, *c.xi(X), z)
    assert info["residual"] < 1e-11
    assert np.abs(flat(*ti) - flat(*td)).max() < 1e-9
    # true residual recomputed from sigma
    r = flat(*c.sigma(*ti, z=z)) + flat(*c.xi(X))
    assert np.linalg.norm(r) < 1e-10 * np.linalg.norm(flat(*c.xi(X)))


def test_residual_is_the_gauss_quadrature_of_the_jacobian_along_the_ray():
    """Omega(t) = Omega(0) + 1/2 sum_k A(s_k t) . t, s_k = 1/2 -+ 1/(2 sqrt 3), exactly (Omega is a quartic, A = dOmega/dt);
    E(t) = eta0(t/2) . t.  cclr_ccsd (GPU ground state) rests on these identities."""
    o, v = 3, 4
    f, V = random_system(o, v, seed=21, diag_fock=False)
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2 = random_amplitudes(o, v, 22, scale=0.2)
    z1, z2 = np.zeros_like(t1), np.zeros_like(t2)
    acc1, acc2 = ccsd.residual(ints, z1, z2)
    assert np.abs(acc1 - ints.fvo).max() < 1e-15 and np.abs(acc2 - ints.vvoo).max() < 1e-15
    for s in (0.5 - 0.5 / np.sqrt(3.0), 0.5 + 0.5 / np.sqrt(3.0)):
        s1, s2 = cclr.CCLR(ints, s * t1, s * t2).sigma(t1, t2)
        acc1, acc2 = acc1 + 0.5 * s1, acc2 + 0.5 * s2
    w1, w2 = ccsd.residual(ints, t1, t2)
    assert np.abs(acc1 - w1).max() < 1e-13 and np.abs(acc2 - w2).max() < 1e-13
    e = cclr.dot(*cclr.CCLR(ints, 0.5 * t1, 0.5 * t2).eta0(), t1, t2)
    assert abs(e - ccsd.energy(ints, t1, t2)) < 1e-13


@pytest.mark.parametrize("o,v", [(3, 4), (2, 5), (4, 4)])
def test_sigma_left_is_the_transpose_of_the_pinned_jacobian(o, v):
    """l A through sigma_left equals A^T l with A the dense Jacobian built from sigma() (pinned by the determinant space),
    at random unconverged t, complex shift included."""
    f, V = random_system(o, v, seed=31 + o, diag_fock=False)
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2 = random_amplitudes(o, v, 32, scale=0.2)
    c = cclr.CCLR(ints, t1, t2)
    A = c.dense_jacobian()
    l1, l2 = random_amplitudes(o, v, 33, scale=1.0)
    z = 0.0773 + 0.0045j
    got = flat(*c.sigma_left(l1, l2, z))
    want = A.T @ flat(l1, l2) - z * flat(l1, l2)
    assert np.abs(got - want).max() < 1e-12 * max(1.0, np.abs(want).max())


def test_iterative_lambda_matches_dense_lambda(small_lr):
    s = small_lr[(3, 4)]
    c = s["c"]
    w1, w2 = c.solve_lambda_iterative()
    assert np.abs(flat(w1, w2) - flat(s["l1"], s["l2"])).max() < 1e-9
