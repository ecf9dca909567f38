import os
import sys
import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))


def pytest_configure(config):
    config.addinivalue_line("markers", "gpu: needs a CUDA device (run on the B200 box)")


def random_system(o, v, seed, sigma_v=0.05, diag_fock=True):
    """Small full-tensor test system (tests only): GUE-like antisymmetric Hermitian <pq||rs> over all pairs of
    n = o+v spinors, Fock diagonal from the config-1 distributions (or a Hermitian perturbation of it)."""
    rng = np.random.default_rng(seed)
    n = o + v
    npair = n * (n - 1) // 2
    M = (rng.normal(size=(npair, npair)) + 1j * rng.normal(size=(npair, npair))) * sigma_v / np.sqrt(2)
    M = (M + M.conj().T) / np.sqrt(2)
    V = np.zeros((n, n, n, n), complex)
    prs = [(p, q) for q in range(n) for p in range(q)]
    for I, (p, q) in enumerate(prs):
        for J, (r, s) in enumerate(prs):
            V[p, q, r, s] = V[q, p, s, r] = M[I, J]
            V[q, p, r, s] = V[p, q, s, r] = -M[I, J]
    eo = np.sort(rng.uniform(-2.0, -0.5, o))
    ev = np.sort(rng.uniform(0.2, 5.0, v))
    f = np.diag(np.concatenate([eo, ev])).astype(complex)
    if not diag_fock:
        K = (rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))) * 0.05
        f = f + K + K.conj().T
    return f, V


def random_amplitudes(o, v, seed, scale=0.3):
    rng = np.random.default_rng(seed + 1000)
    x1 = (rng.normal(size=(v, o)) + 1j * rng.normal(size=(v, o))) * scale
    x2 = (rng.normal(size=(v, v, o, o)) + 1j * rng.normal(size=(v, v, o, o))) * scale
    x2 = x2 - x2.transpose(1, 0, 2, 3)
    x2 = x2 - x2.transpose(0, 1, 3, 2)
    return x1, x2


def random_hermitian(n, seed):
    rng = np.random.default_rng(seed + 2000)
    K = rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))
    return (K + K.conj().T) / 2


@pytest.fixture(scope="session")
def helpers():
    class H:
        pass
    H.random_system = staticmethod(random_system)
    H.random_amplitudes = staticmethod(random_amplitudes)
    H.random_hermitian = staticmethod(random_hermitian)
    return H
