"""Host logic of cclr_solve's reduced-space step (csrc/small_dense.h through the C ABI): shifted solves
(G - z_k) beta = rhs via one Hessenberg reduction, against numpy.linalg.solve."""
import ctypes as C
import numpy as np
import pytest


@pytest.mark.parametrize("L", [1, 2, 3, 17, 64])
def test_shifted_hessenberg_solves_match_numpy(L):
    from paper_2307_14296_b200 import _lib
    lib = _lib.load()
    rng = np.random.default_rng(L)
    G = rng.normal(size=(L, L)) + 1j * rng.normal(size=(L, L)) + np.diag(np.linspace(1, 6, L))
    rhs = rng.normal(size=L) + 1j * rng.normal(size=L)
    z = np.array([0.0, 0.0773, 0.0773 + 0.0045j, -0.3 - 0.0045j, 2.5 + 0.1j])
    beta = np.zeros((len(z), L), complex)
    rc = lib.cclr_host_shifted_solve(L, G.ctypes.data_as(C.c_void_p), rhs.ctypes.data_as(C.c_void_p), len(z),
                                     z.ctypes.data_as(C.c_void_p), beta.ctypes.data_as(C.c_void_p))
    assert rc == 0
    for k, zz in enumerate(z):
        want = np.linalg.solve(G - zz * np.eye(L), rhs)
        assert np.abs(beta[k] - want).max() < 1e-11 * max(1.0, np.abs(want).max())


def test_structured_matrices():
    """Already-Hessenberg, diagonal and zero-subdiagonal inputs (Householder steps that degenerate)."""
    from paper_2307_14296_b200 import _lib
    lib = _lib.load()
    for G in (np.diag([1.0, 2.0, 3.0, 4.0]).astype(complex), np.triu(np.ones((5, 5)), -1).astype(complex) + 3 * np.eye(5),
              np.array([[2, 1, 0], [0, 3, 1], [0, 0, 4]], complex)):
        L = G.shape[0]
        rhs = np.arange(1, L + 1).astype(complex)
        z = np.array([0.5 + 0.25j])
        beta = np.zeros((1, L), complex)
        G = np.ascontiguousarray(G)
        assert lib.cclr_host_shifted_solve(L, G.ctypes.data_as(C.c_void_p), rhs.ctypes.data_as(C.c_void_p), 1,
                                           z.ctypes.data_as(C.c_void_p), beta.ctypes.data_as(C.c_void_p)) == 0
        assert np.abs(beta[0] - np.linalg.solve(G - z[0] * np.eye(L), rhs)).max() < 1e-12


@pytest.mark.parametrize("L", [1, 2, 3, 7, 40, 90])
def test_host_eigen_matches_numpy(L):
    """The reduced eigenproblem of cclr_eom (small_dense::eigen: Hessenberg + complex QR + back-substitution)."""
    import ctypes as C
    from paper_2307_14296_b200 import _lib
    lib = _lib.load()
    rng = np.random.default_rng(L)
    G = rng.normal(size=(L, L)) + 1j * rng.normal(size=(L, L))
    if L == 7:
        G = np.diag(np.arange(7.0)).astype(complex) + np.triu(G, 1) * 1e-3      # nearly triangular, tiny couplings
    if L == 40:
        G = G + G.conj().T                                                      # Hermitian
    G = np.ascontiguousarray(G)
    w = np.zeros(L, complex)
    V = np.zeros((L, L), complex)
    rc = lib.cclr_host_eigen(L, G.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p), V.ctypes.data_as(C.c_void_p))
    assert rc == 0
    ref = np.linalg.eigvals(G)
    assert np.abs(np.sort_complex(w) - np.sort_complex(ref)).max() < 1e-10 * max(1.0, np.abs(ref).max())
    for k in range(L):
        assert abs(np.linalg.norm(V[:, k]) - 1.0) < 1e-12
        assert np.linalg.norm(G @ V[:, k] - w[k] * V[:, k]) < 1e-9 * max(1.0, np.abs(ref).max())
