"""Full-size GPU parity (BASELINE.json configs 3, 4, 5 — the shapes and launch configuration bench.py times): outputs the
oracle can compute one by one (oracle/sampled.py), plus properties that hold at any size.

Inputs are generated on the device by synth/ (counter-based: any block can be regenerated on the host), so the oracle side
regenerates exactly the integral rows it needs.  oracle.sampled.SampledCCLR evaluates slices of every dressed intermediate of
S-Eq. 15-28 and single elements of sigma (S-Eq. 11-12) at T != 0 from the packed inputs, so the full-size cclr_create (chunked
o^2 v^4 builds, W_vvvv dressed in place over the 32 GB buffer) and the whole sigma vector (all 17 terms' kernels, full size)
are compared with the oracle where it can afford to look: first / last rows, the last chunk, corners and random elements.
Tolerances: intermediates max-norm 1e-11 relative per slice; sigma |gpu - oracle| <= 1e-10 * rms(sigma) per sampled element
(north_star's 1e-10 is norm-wise; rms is the per-element scale of that norm)."""
import numpy as np
import pytest
import torch

import synth
from oracle import packing, sampled

pytestmark = pytest.mark.gpu


def _device_inputs(o, v, t_scale):
    eri = {k: synth.eri_class(k, o, v, seed=0, device="cuda") for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv", "vvvv")}
    f = synth.fock(o, v, seed=0) + 0.05 * torch.from_numpy(synth.hermitian_operator(o + v, 0, 7))
    t1, t2 = synth.amplitudes(o, v, seed=0, scale=t_scale, device="cuda")
    return eri, f, t1[0].contiguous(), t2[0].contiguous()


def _samples(o, v, rng, n):
    vv, oo = synth.npair(v), synth.npair(o)
    doubles = [(0, 1, 0, 1), (v - 2, v - 1, o - 2, o - 1), (0, v - 1, 0, o - 1)]      # first, last, corner
    while len(doubles) < n:
        a, b = sorted(rng.choice(v, 2, replace=False))
        i, j = sorted(rng.choice(o, 2, replace=False))
        doubles.append((int(a), int(b), int(i), int(j)))
    singles = [(0, 0), (v - 1, o - 1)] + [(int(rng.integers(v)), int(rng.integers(o))) for _ in range(n - 2)]
    return singles, doubles


def _index_sets(o, v, rng, na, ni):
    """Small sets of virtual / occupied indices: first, second, last two, plus random ones (sorted, distinct)."""
    A = {0, 1, v - 2, v - 1}
    while len(A) < na:
        A.add(int(rng.integers(v)))
    I = {0, o - 1}
    while len(I) < ni:
        I.add(int(rng.integers(o)))
    return sorted(A), sorted(I)


def _close(got, want, tol, what):
    got, want = np.asarray(got), np.asarray(want)
    err = np.abs(got - want).max()
    assert err <= tol * np.abs(want).max(), (what, err, np.abs(want).max())


@pytest.mark.parametrize("cfg", [5, 3, 4])
def test_dressed_intermediates_and_sigma_with_T_at_full_size(cfg):
    """T != 0 (entry std 2 sigma_V), CCLR_ERI_INPLACE, damped z: (i) slices of every persistent intermediate of cclr_create
    against SampledCCLR incl. the first and last rows and the last chunk of every chunked build, (ii) >= 20 singles and 60
    doubles elements of sigma per vector."""
    import paper_2307_14296_b200 as cc
    o, v = synth.CONFIGS[cfg]["o"], synth.CONFIGS[cfg]["v"]
    nvec = 3 if cfg == 5 else 1
    vv, oo = synth.npair(v), synth.npair(o)
    scale = synth.sigma_v(v)
    eri, f, t1, t2 = _device_inputs(o, v, 2 * scale)
    host = {k: eri[k].cpu().numpy() for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv")}
    ctx = cc.cclr_create(o, v, f.cuda(), eri, t1, t2, cc.ERI_INPLACE)
    del eri
    row = lambda ab: synth._hermitian_matrix_rows(0, synth.CLASS_ID["vvvv"], vv, ab, ab + 1, scale, "cpu")[0].numpy()
    S = sampled.SampledCCLR(o, v, f.numpy(), host, row, t1.cpu().numpy(), t2.cpu().numpy())
    rng = np.random.default_rng(100 + cfg)
    A, I = _index_sets(o, v, rng, 5, 4)
    P = sampled.pair_index
    get = lambda name, off, cnt: ctx.get_intermediate_slice(name, off, cnt).cpu().numpy()
    pack_ef = lambda x, axis: packing.pack_pair_axes(x, axis)
    tol = 1e-11

    # ---- (i) intermediates (layouts: DESIGN.md "Data layout") ----
    _close(ctx.get_intermediate("Fme").cpu().numpy().reshape(o, v), S.Fme(), tol, "Fme")
    _close(ctx.get_intermediate("Fmi").cpu().numpy().reshape(o, o), S.Fmi(), tol, "Fmi")
    Fae = ctx.get_intermediate("Fae").cpu().numpy().reshape(v, v)
    Wmnij = ctx.get_intermediate("Wmnij").cpu().numpy().reshape(oo, oo)
    for a in A:
        _close(Fae[a], S.Fae_row(a), tol, ("Fae", a))
        w = S.Wamef_a(a)                                                            # [m,e,f]
        _close(get("Wamef", a * o * vv, o * vv).reshape(o, vv), pack_ef(w, 1), tol, ("Wamef", a))
        _close(get("Wx", a * v * v * o, v * v * o).reshape(v, v, o), w.transpose(1, 2, 0), tol, ("Wx", a))
    for i in I:
        w = S.Wmnie_i(i)                                                            # [m,n,e]
        _close(get("Wie", i * v * oo, v * oo).reshape(v, oo), packing.pack_pair_axes(w, 0).T, tol, ("Wie", i))
        for n in (0, o - 1):                                                        # Wnjem[n][j][e][m] = W_mnie[nm,je]
            _close(get("Wnjem", (n * o + i) * v * o, v * o).reshape(v, o), w[n].T, tol, ("Wnjem", n, i))
    for ji, j in enumerate(I):
        for i in I[:ji]:
            _close(Wmnij[:, P(i, j)], packing.pack_pair_axes(S.Wmnij_col(i, j), 0), tol, ("Wmnij", i, j))
    for b in A:
        for j in I[:2] + I[-1:]:                                                    # Wring[b][j][e][m] = W_mbej[mb,ej]
            _close(get("Wring", (b * o + j) * v * o, v * o).reshape(v, o), S.Wmbej_bj(b, j).T, tol, ("Wring", b, j))
    Wmbij_rows = {(m, b): get("Wmbij", (m * v + b) * oo, oo) for m in (0, o - 1) for b in (A[0], A[-1])}
    for (m, b), g in Wmbij_rows.items():
        for (i, j) in ((I[0], I[1]), (I[0], I[-1]), (I[-2], I[-1])):
            w = S.Wmbij_bij(b, i, j)[m]
            assert abs(g[P(i, j)] - w) <= tol * max(abs(w), np.abs(g).max()), ("Wmbij", m, b, i, j, g[P(i, j)], w)
    pairs_ab = [(A[0], A[1]), (A[-2], A[-1]), (A[0], A[-1]), (A[1], A[2])]            # first row, last row, corner, middle
    for (a, b) in pairs_ab:
        _close(get("Wabef", P(a, b) * vv, vv), pack_ef(S.Wabef_row(a, b), 0), tol, ("Wabef", a, b))
        g = get("Wabej", P(a, b) * o * v, o * v).reshape(o, v)                      # Wabej[(ab)][j][e]
        for j in (I[0], I[-1]):
            _close(g[j], S.Wabej_abj(a, b, j), tol, ("Wabej", a, b, j))

    # ---- (ii) sigma elements at a damped frequency ----
    x1, x2 = synth.amplitudes(o, v, seed=7, cls1="x1", cls2="x2", device="cuda", nvec=nvec)
    z = 0.0773 + 0.0045j
    s1, s2 = cc.cclr_sigma(ctx, x1, x2, z.real, z.imag)
    torch.cuda.synchronize()
    singles = [(a, i) for a in A for i in I]
    doubles = [(a, b, i, j) for bi, b in enumerate(A) for a in A[:bi] for ji, j in enumerate(I) for i in I[:ji]]
    assert len(singles) >= 20 and len(doubles) >= 60
    for k in range(nvec):
        w1, w2 = S.sigma_elements(x1[k].cpu().numpy(), x2[k].cpu().numpy(), singles, doubles, z=z)
        g1 = s1[k].cpu().numpy().reshape(v, o)
        g2 = s2[k].view(vv, oo)
        rms1 = float(s1[k].abs().pow(2).mean().sqrt())
        rms2 = float(s2[k].abs().pow(2).mean().sqrt())
        for (a, i), w in zip(singles, w1):
            assert abs(g1[a, i] - w) <= 1e-10 * rms1, ("sigma1", cfg, k, a, i, g1[a, i], w)
        for (a, b, i, j), w in zip(doubles, w2):
            g = complex(g2[P(a, b), P(i, j)].item())
            assert abs(g - w) <= 1e-10 * rms2, ("sigma2", cfg, k, a, b, i, j, g, w)
    ctx.close()
    del ctx, s1, s2, x1, x2, S
    torch.cuda.empty_cache()


@pytest.mark.parametrize("cfg", [5])
def test_sigma_T0_sampled_elements_at_full_size(cfg):
    import paper_2307_14296_b200 as cc
    o, v = synth.CONFIGS[cfg]["o"], synth.CONFIGS[cfg]["v"]
    nvec = 3 if cfg == 5 else 1
    vv, oo = synth.npair(v), synth.npair(o)
    eri, f, t1, t2 = _device_inputs(o, v, 0.0)
    host = {k: eri[k].cpu().numpy() for k in ("oooo", "ooov", "ovvo", "ovvv")}
    ctx = cc.cclr_create(o, v, f.cuda(), eri, t1, t2, cc.ERI_INPLACE)
    del eri
    x1, x2 = synth.amplitudes(o, v, seed=7, cls1="x1", cls2="x2", device="cuda", nvec=nvec)
    z = 0.0773 + 0.0045j
    s1, s2 = cc.cclr_sigma(ctx, x1, x2, z.real, z.imag)
    torch.cuda.synchronize()
    assert torch.isfinite(s2.abs().sum()).item()
    rng = np.random.default_rng(cfg)
    singles, doubles = _samples(o, v, rng, 12)
    scale = synth.sigma_v(v)
    row = lambda ab: synth._hermitian_matrix_rows(0, synth.CLASS_ID["vvvv"], vv, ab, ab + 1, scale, "cpu")[0].numpy()
    for k in range(nvec):
        w1, w2 = sampled.sigma_T0_elements(o, v, f.numpy(), host, row, x1[k].cpu().numpy(), x2[k].cpu().numpy(),
                                           singles, doubles, z=z)
        g1 = s1[k].cpu().numpy().reshape(v, o)
        g2 = s2[k].view(vv, oo)
        rms1 = float(s1[k].abs().pow(2).mean().sqrt())
        rms2 = float(s2[k].abs().pow(2).mean().sqrt())
        for (a, i), w in zip(singles, w1):
            assert abs(g1[a, i] - w) <= 1e-10 * rms1, ("sigma1", cfg, k, a, i, g1[a, i], w)
        for (a, b, i, j), w in zip(doubles, w2):
            g = complex(g2[sampled.pair_index(a, b), sampled.pair_index(i, j)].item())
            assert abs(g - w) <= 1e-10 * rms2, ("sigma2", cfg, k, a, b, i, j, g, w)
    # the ladder entry point alone, whole sampled rows incl. the first and the last (ragged last tile)
    lad = cc.cclr_ladder(ctx, x2[:1].contiguous())
    torch.cuda.synchronize()
    rows = [0, 1, vv // 2 + 3, vv - 1]
    w_rows = np.stack([row(r) for r in rows])
    want = sampled.ladder_rows(w_rows, x2[0].cpu().numpy().reshape(vv, oo))
    got = lad[0].view(vv, oo)[rows].cpu().numpy()
    # default path at this size: 6 integer slices on the INT8 tensor path, operands truncated 41 bits below their row maxima ->
    # 2^-35 norm-wise (measured 6e-12); the FP64 tensor-core (DMMA) path of the same context: rounding level
    assert ctx.set_gemm_path(1) == 1
    assert np.linalg.norm(got - want) <= 2.0 ** -35 * np.linalg.norm(want)
    assert ctx.set_gemm_path(0) == 0
    lad = cc.cclr_ladder(ctx, x2[:1].contiguous())
    torch.cuda.synchronize()
    got = lad[0].view(vv, oo)[rows].cpu().numpy()
    assert np.linalg.norm(got - want) <= 1e-12 * np.linalg.norm(want)
    ctx.close()
    del ctx, lad, s1, s2, x1, x2
    torch.cuda.empty_cache()


@pytest.mark.parametrize("cfg", [3])
def test_properties_at_full_size_with_T(cfg):
    """T != 0 at full size: linearity, the shift identity and x^H (A y) computed two ways (sigma then dot vs dot of sigmas)
    hold at any size; here they exercise the dressed intermediates in bench.py's launch configuration."""
    import paper_2307_14296_b200 as cc
    o, v = synth.CONFIGS[cfg]["o"], synth.CONFIGS[cfg]["v"]
    eri, f, t1, t2 = _device_inputs(o, v, 2 * synth.sigma_v(v))
    ctx = cc.cclr_create(o, v, f.cuda(), eri, t1, t2, cc.ERI_INPLACE)
    del eri
    x1, x2 = synth.amplitudes(o, v, seed=8, cls1="x1", cls2="x2", device="cuda", nvec=2)
    a, b = 0.3 - 1.1j, -0.7 + 0.2j
    y1 = (a * x1[0] + b * x1[1])[None].contiguous()
    y2 = (a * x2[0] + b * x2[1])[None].contiguous()
    rel = lambda u, w: float((u - w).abs().pow(2).sum().sqrt() / w.abs().pow(2).sum().sqrt())
    # path 1 (default at this size): ladder and ring as integer-slice products -- the slicing of the trial vector is not a linear
    # map, so linearity holds to the truncation level (sigma tolerance 1e-10); path 0: DMMA, rounding level
    for path, tol in ((1, 1e-10), (0, 1e-12)):
        assert ctx.set_gemm_path(path) == path
        o1, o2 = cc.cclr_sigma(ctx, x1, x2)
        p1, p2 = cc.cclr_sigma(ctx, y1, y2)
        assert rel(p2[0], a * o2[0] + b * o2[1]) < tol, path
        assert rel(p1[0], a * o1[0] + b * o1[1]) < tol, path
        zz = 0.0773 + 0.0045j
        q1, q2 = cc.cclr_sigma(ctx, x1, x2, zz.real, zz.imag)
        assert rel(q2, o2 - zz * x2) < 1e-14 and rel(q1, o1 - zz * x1) < 1e-14
        # the host-buffer entry (x2 copied on a second stream under the x1-only statements at this size) returns the same bits
        h1, h2 = torch.empty_like(x1, device="cpu").pin_memory(), torch.empty_like(x2, device="cpu").pin_memory()
        cc.cclr_sigma_host(ctx, x1.cpu().pin_memory(), x2.cpu().pin_memory(), zz.real, zz.imag, h1, h2)
        assert torch.equal(h1, q1.cpu()) and torch.equal(h2, q2.cpu())
    ctx.close()
    torch.cuda.empty_cache()


@pytest.mark.parametrize("cfg", [3])
def test_precision_on_demand_keeps_the_true_residual(cfg):
    """cclr_solve on the integer-slice path forms the sigma vectors of late trial vectors with fewer slices (subspace.cuh: their
    coefficients in the solutions are of the size of the residual at the time they were added).  The converged solutions are
    checked here with the OTHER arithmetic: the residual (A - z) t + xi recomputed whole-vector by cclr_sigma on the FP64 tensor
    cores (cclr_set_gemm_path 0) must sit at the solver's tolerance, for a real and a damped shift pair, and for the left solver."""
    import paper_2307_14296_b200 as cc
    o, v = synth.CONFIGS[cfg]["o"], synth.CONFIGS[cfg]["v"]
    eri = {k: synth.eri_class(k, o, v, seed=0, device="cuda") for k in ("oooo", "ooov", "oovv", "ovvo", "ovvv", "vvvv")}
    f = synth.fock(o, v, seed=0).cuda()
    t1, t2 = synth.first_order_amplitudes(o, v, f, eri["oovv"])      # a well-conditioned Jacobian (random T is not, at this size)
    ctx = cc.cclr_create(o, v, f, eri, t1, t2, cc.ERI_INPLACE)
    del eri
    assert ctx.gemm_slices() == 6
    xi1, xi2 = synth.amplitudes(o, v, seed=21, cls1="x1", cls2="x2", device="cuda", nvec=1)
    tol = 1e-10
    nxi = float(torch.sqrt(xi1.abs().pow(2).sum() + xi2.abs().pow(2).sum()))
    for gamma, solve, sig in ((0.0, cc.cclr_solve, cc.cclr_sigma), (0.0045, cc.cclr_solve, cc.cclr_sigma),
                              (0.0, cc.cclr_solve_left, cc.cclr_sigma_left)):
        omegas = [0.0773, -0.0773]
        s1, s2, info = solve(ctx, xi1, xi2, omegas, gamma, tol=tol, maxiter=200)
        assert info.converged == 1
        assert ctx.set_gemm_path(0) == 0
        for k, w in enumerate(omegas):
            q1, q2 = sig(ctx, s1[0, k][None].contiguous(), s2[0, k][None].contiguous(), w, gamma)
            r = float(torch.sqrt((q1[0] + xi1[0]).abs().pow(2).sum() + (q2[0] + xi2[0]).abs().pow(2).sum()))
            assert r <= 1.2 * tol * nxi, (gamma, w, r / nxi)
        assert ctx.set_gemm_path(1) == 1
    ctx.close()
    torch.cuda.empty_cache()
