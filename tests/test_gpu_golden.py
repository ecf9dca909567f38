"""The CUDA path on the closed-form two-level system of tests/golden/two_level_closed_form.json (o = 2, v = 2: the smallest
sizes the library accepts, every GEMM has M, N or K of 1-4): response amplitudes from cclr_solve, contracted by the
oracle's Eq. 15 / Eq. 16 assembly, must reproduce the closed-form <<X;X>>_z to 1e-8 (north_star tolerance)."""
import numpy as np
import pytest
import torch

from oracle import ccsd, cclr, packing
from test_golden_closed_form import GOLD, two_level_system

pytestmark = pytest.mark.gpu


def test_two_level_response_through_the_gpu_solver():
    import paper_2307_14296_b200 as cc
    f, V, o, X = two_level_system()
    v = 2
    ints = ccsd.Integrals.from_full(f, V, o)
    t1, t2, _ = ccsd.solve_ground_state(ints, tol=1e-13)
    c = cclr.CCLR(ints, t1, t2)
    l1, l2 = c.solve_lambda_dense()
    full = dict(oooo=ints.oooo, ooov=ints.ooov, oovv=ints.oovv, ovvo=ints.ovvo, ovvv=ints.ovvv, vvvv=ints.vvvv)
    eri = {k: torch.from_numpy(x.reshape(-1).copy()).cuda() for k, x in packing.pack_eri(full).items()}
    t1p, t2p = packing.pack_amplitudes(t1, t2)
    ctx = cc.cclr_create(o, v, torch.from_numpy(f).cuda(), eri, torch.from_numpy(t1p.reshape(-1).copy()).cuda(),
                         torch.from_numpy(t2p.reshape(-1).copy()).cuda())
    # Jacobian spectrum through cclr_sigma on unit vectors
    n1, n2 = o * v, 1
    eye = np.eye(n1 + n2, dtype=complex)
    s1, s2 = cc.cclr_sigma(ctx, torch.from_numpy(eye[:, :n1].copy()).cuda(), torch.from_numpy(eye[:, n1:].copy()).cuda())
    A = torch.cat([s1, s2], dim=1).cpu().numpy().T
    ev = np.sort(np.linalg.eigvals(A).real)
    assert np.abs(ev - np.sort(GOLD["jacobian_eigenvalues"])).max() < 1e-10

    def gpu_solve(x1, x2, zz):
        a, b = packing.pack_amplitudes(x1, x2)
        r1, r2, info = cc.cclr_solve(ctx, torch.from_numpy(a.reshape(1, -1).copy()).cuda(),
                                     torch.from_numpy(b.reshape(1, -1).copy()).cuda(), [complex(zz).real],
                                     complex(zz).imag, tol=1e-12, maxiter=50)
        assert info.converged == 1
        return packing.unpack_amplitudes(r1[0, 0].cpu().numpy(), r2[0, 0].cpu().numpy(), o, v)

    for rec in GOLD["response"]:
        z, want = complex(*rec["z"]), complex(*rec["XX"])
        assert abs(c.response_cc_cc(gpu_solve, X, X, z, l1, l2) - want) <= 1e-8 * abs(want)
        assert abs(c.response_cc_ci(gpu_solve, X, X, z, l1, l2) - want) <= 1e-8 * abs(want)
    ctx.close()
