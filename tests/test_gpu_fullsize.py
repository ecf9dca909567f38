"""Full-size GPU parity (BASELINE.json configs 3, 4, 5 — the shapes and launch configuration bench.py times): outputs the
oracle can compute one by one (oracle/sampled.py), plus properties that hold at any size.

Inputs are generated on the device by synth/ (counter-based: any block can be regenerated on the host), so the oracle side
regenerates exactly the integral rows it needs.  At T = 0 every intermediate equals the bare block of the same name, which
makes sampled elements of the WHOLE sigma vector (all 17 terms' kernels run, at full size) checkable against the definition.
Tolerance: |gpu - oracle| <= 1e-10 * rms(sigma) per sampled element (north_star's 1e-10 is norm-wise; rms is the per-element
scale of that norm)."""
import numpy as np
import pytest
import torch

import synth
from oracle import sampled

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


@pytest.mark.parametrize("cfg", [5, 3, 4])
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
    o1, o2 = cc.cclr_sigma(ctx, x1, x2)
    p1, p2 = cc.cclr_sigma(ctx, y1, y2)
    rel = lambda u, w: float((u - w).abs().pow(2).sum().sqrt() / w.abs().pow(2).sum().sqrt())
    assert rel(p2[0], a * o2[0] + b * o2[1]) < 1e-12
    assert rel(p1[0], a * o1[0] + b * o1[1]) < 1e-12
    zz = 0.0773 + 0.0045j
    q1, q2 = cc.cclr_sigma(ctx, x1, x2, zz.real, zz.imag)
    assert rel(q2, o2 - zz * x2) < 1e-14 and rel(q1, o1 - zz * x1) < 1e-14
    ctx.close()
    torch.cuda.empty_cache()
