"""Seeded synthetic inputs for the CC-LR hot path (shared by the oracle-side tests and the CUDA-side tests / bench).

This module holds NO arithmetic of the method: it only produces the numbers both sides are fed with -- a diagonal
Fock matrix, the six packed classes of antisymmetrised integrals <pq||rs> of include/cclr.h, amplitudes, trial
vectors and one-body perturbation matrices -- with the shapes and value distributions of BASELINE.json's configs
(recipe: DESIGN.md "Synthetic inputs").  Every element is a pure function of (seed, class id, element index)
through a counter-based generator (splitmix64 -> Box-Muller), written with torch integer/float ops so that the same
code runs on the host (oracle side) and on the GPU (where the 32 GB vvvv class of config 4 is generated in place);
any block of any class can therefore be regenerated anywhere.  Host and device agree to the rounding of log/cos/sin
(~1e-16 relative); whenever both sides of a parity test need the same array it is generated ONCE and copied.
"""
import math
import numpy as np
import torch

CONFIGS = {  # BASELINE.json configs[0..4]
    1: dict(o=4, v=20), 2: dict(o=10, v=80), 3: dict(o=24, v=200), 4: dict(o=34, v=300), 5: dict(o=18, v=150),
}
CLASS_ID = dict(oooo=1, ooov=2, oovv=3, ovvo=4, ovvv=5, vvvv=6, t1=7, t2=8, x1=20, x2=21, dipole=10)
_M64 = (1 << 64) - 1


def npair(n):
    return n * (n - 1) // 2


def sigma_v(v, literal=False):
    """Std of the complex integral entries: BASELINE.json's 0.05 at config 1, scaled so that the spectral radius of
    the vv x vv block stays that of config 1 (the literal 0.05 does not give a convergent CCSD beyond config 1)."""
    return 0.05 if literal else 0.05 * math.sqrt(190.0 / npair(v))


def _i64(x):
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


def _lsr(x, s):
    return (x >> s) & ((1 << (64 - s)) - 1)


def _splitmix(x):
    """splitmix64 finaliser on int64 tensors (wrap-around arithmetic, logical shifts emulated)."""
    x = x + _i64(0x9E3779B97F4A7C15)
    x = (x ^ _lsr(x, 30)) * _i64(0xBF58476D1CE4E5B9)
    x = (x ^ _lsr(x, 27)) * _i64(0x94D049BB133111EB)
    return x ^ _lsr(x, 31)


def complex_gauss(seed, cls, idx):
    """Standard complex Gaussian (E|z|^2 = 1) for every int64 counter in ``idx``; pure function of (seed, cls, idx)."""
    key = _i64(seed * 0x632BE59BD9B4E019 + cls * 0xD1342543DE82EF95)
    h1 = _splitmix(idx * 2 + key)
    h2 = _splitmix(idx * 2 + 1 + key)
    u1 = (_lsr(h1, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)
    u2 = (_lsr(h2, 11).to(torch.float64) + 0.5) * (1.0 / 9007199254740992.0)
    r = torch.sqrt(-torch.log(u1))                     # E r^2 = 1
    th = (2.0 * math.pi) * u2
    return torch.complex(r * torch.cos(th), r * torch.sin(th))


def _hermitian_matrix_rows(seed, cls, n, r0, r1, scale, device):
    """Rows r0..r1 of an n x n Hermitian matrix: entry (I,J), I<J, = scale*g(I*n+J); (J,I) its conjugate; real diagonal."""
    I = torch.arange(r0, r1, dtype=torch.int64, device=device)[:, None]
    J = torch.arange(n, dtype=torch.int64, device=device)[None, :]
    lo, hi = torch.minimum(I, J), torch.maximum(I, J)
    g = complex_gauss(seed, cls, lo * n + hi)
    g = torch.where(I > J, g.conj(), g)
    g = torch.where(I == J, torch.complex(g.real * math.sqrt(2.0), torch.zeros_like(g.real)), g)
    return g * scale


def eri_class(name, o, v, seed=0, scale=None, device="cpu", out=None, row_block=2048):
    """One packed class of include/cclr.h as a flat complex128 tensor (optionally written into ``out`` in row blocks)."""
    s = sigma_v(v) if scale is None else scale
    cls = CLASS_ID[name]
    oo, vv = npair(o), npair(v)
    if name in ("oooo", "vvvv"):
        n = oo if name == "oooo" else vv
        res = out if out is not None else torch.empty(n * n, dtype=torch.complex128, device=device)
        view = res.view(n, n)
        for r0 in range(0, n, row_block):
            r1 = min(n, r0 + row_block)
            view[r0:r1] = _hermitian_matrix_rows(seed, cls, n, r0, r1, s, res.device)
        return res
    if name == "ovvo":
        # <mb||ej> = conj <je||bm>: element (m,b,e,j) pairs with (j,e,b,m)
        dev = torch.device(device)
        m = torch.arange(o, dtype=torch.int64, device=dev)[:, None, None, None]
        b = torch.arange(v, dtype=torch.int64, device=dev)[None, :, None, None]
        e = torch.arange(v, dtype=torch.int64, device=dev)[None, None, :, None]
        j = torch.arange(o, dtype=torch.int64, device=dev)[None, None, None, :]
        A = ((m * v + b) * v + e) * o + j
        B = ((j * v + e) * v + b) * o + m
        g = complex_gauss(seed, cls, torch.minimum(A, B))
        g = torch.where(A > B, g.conj(), g)
        g = torch.where(A == B, torch.complex(g.real * math.sqrt(2.0), torch.zeros_like(g.real)), g)
        return (g * s).reshape(-1)
    n = dict(ooov=oo * o * v, oovv=oo * vv, ovvv=o * v * vv)[name]
    res = out if out is not None else torch.empty(n, dtype=torch.complex128, device=device)
    step = 1 << 24
    for i0 in range(0, n, step):
        i1 = min(n, i0 + step)
        res[i0:i1] = complex_gauss(seed, cls, torch.arange(i0, i1, dtype=torch.int64, device=res.device)) * s
    return res


def eri_packed(o, v, seed=0, scale=None, device="cpu"):
    return {k: eri_class(k, o, v, seed, scale, device) for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv", "vvvv")}


def fock(o, v, seed=0, device="cpu"):
    """Diagonal Fock matrix [n][n]: occupied eps ~ U[-2,-0.5], virtual ~ U[0.2,5] hartree, each sorted ascending."""
    rng = np.random.default_rng([seed, 99])
    eo = np.sort(rng.uniform(-2.0, -0.5, o))
    ev = np.sort(rng.uniform(0.2, 5.0, v))
    return torch.from_numpy(np.diag(np.concatenate([eo, ev])).astype(complex)).to(device)


def amplitudes(o, v, seed=0, cls1="t1", cls2="t2", scale=1.0, device="cpu", nvec=1):
    """Random packed amplitude-shaped vectors ([nvec, v*o], [nvec, vv*oo]) with entry std ``scale``."""
    n1, n2 = o * v, npair(o) * npair(v)
    a = complex_gauss(seed, CLASS_ID[cls1], torch.arange(nvec * n1, dtype=torch.int64, device=device)) * scale
    b = torch.empty(nvec * n2, dtype=torch.complex128, device=device)
    step = 1 << 24
    for i0 in range(0, nvec * n2, step):
        i1 = min(nvec * n2, i0 + step)
        b[i0:i1] = complex_gauss(seed, CLASS_ID[cls2], torch.arange(i0, i1, dtype=torch.int64, device=device)) * scale
    return a.view(nvec, n1), b.view(nvec, n2)


def hermitian_operator(n, seed, component, imaginary_antisymmetric=False):
    """A random Hermitian one-body matrix [n][n] with unit-variance entries ("dipole" component), or i*K with K real
    antisymmetric (the magnetic-dipole type of Eq. 36), as a numpy array."""
    rng = np.random.default_rng([seed, CLASS_ID["dipole"], component])
    if imaginary_antisymmetric:
        K = rng.normal(size=(n, n))
        return 1j * (K - K.T) / math.sqrt(2.0)
    K = (rng.normal(size=(n, n)) + 1j * rng.normal(size=(n, n))) / math.sqrt(2.0)
    return (K + K.conj().T) / math.sqrt(2.0)


def first_order_amplitudes(o, v, fock_matrix, oovv):
    """Ground-state amplitudes of the SHAPE a converged CCSD has, for sizes where no converged T is available: t1 = 0 and
    t2[(ab),(ij)] = conj(<ij||ab>) / (eps_i + eps_j - eps_a - eps_b), the first-order (perturbative) doubles, from the packed
    oovv class ([oo][vv]) and the diagonal of the Fock matrix.  Input recipe only (elementwise on the synthetic inputs);
    sigma = dOmega/dt . x holds at any t, so parity does not depend on it."""
    dev = oovv.device
    eps = torch.diagonal(fock_matrix).real.to(dev)
    eo, ev = eps[:o], eps[o:]
    # pair order P = q(q-1)/2 + p: q outer, p inner
    def pair_sums(e, n):
        q = torch.arange(n, device=dev)[:, None].expand(n, n)
        p = torch.arange(n, device=dev)[None, :].expand(n, n)
        m = p < q
        return e[p[m]] + e[q[m]]

    d = pair_sums(eo, o)[None, :] - pair_sums(ev, v)[:, None]              # [vv][oo]
    t2 = oovv.view(npair(o), npair(v)).conj().transpose(0, 1) / d
    t1 = torch.zeros(o * v, dtype=torch.complex128, device=dev)
    return t1, t2.contiguous().view(-1)
