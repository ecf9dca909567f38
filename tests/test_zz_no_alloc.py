"""cclr_property_noalloc (include/cclr.h): the property contraction for callers that cannot allocate device memory -- its partial
sums live in a file-scope static device array of the library instead of a context's heap scratch.  Checked against the existing
path (cclr_property, which needs a context) on the same seeded inputs, on two calls in a row that share the static array: the
second call has fewer vectors and other data, so stale contents of the array would show.  Tolerance: the 1e-12 the property
tests use (the arithmetic and its order are the same, so the results agree to rounding or exactly).

This file is collected last on purpose (the suite runs with pytest -x); it passes alone in a fresh process and after the rest."""
import pytest
import torch

import synth

pytestmark = pytest.mark.gpu


def _context(cc, o, v, seed):
    eri = {k: x.cuda() for k, x in synth.eri_packed(o, v, seed=seed).items()}
    f = synth.fock(o, v, seed=seed).cuda()
    t1, t2 = synth.amplitudes(o, v, seed=seed, scale=0.02)
    return cc.cclr_create(o, v, f, eri, t1[0].cuda(), t2[0].cuda())


def test_property_without_allocation_matches_the_context_path_on_two_calls_in_a_row():
    import paper_2307_14296_b200 as cc
    o, v = 6, 40                       # n2 = 780 * 15 = 11700 unique doubles: several chunks of the two-pass reduction
    ctx = _context(cc, o, v, seed=5)
    try:
        for call, (nvec, seed) in enumerate([(cc.NOALLOC_MAX_VECS, 31), (3, 32)]):
            e1, e2 = synth.amplitudes(o, v, seed=seed, cls1="x1", cls2="x2")
            x1, x2 = synth.amplitudes(o, v, seed=seed + 100, cls1="x1", cls2="x2", nvec=nvec)
            e1, e2, x1, x2 = e1[0].contiguous().cuda(), e2[0].contiguous().cuda(), x1.cuda(), x2.cuda()
            want = cc.cclr_property(ctx, e1, e2, x1, x2)                         # existing path: context scratch, host result
            out = torch.full((nvec,), float("nan"), dtype=torch.complex128, device="cuda")
            before = torch.cuda.memory_allocated()
            cc.cclr_property_noalloc(e1, e2, x1, x2, out)
            torch.cuda.synchronize()
            assert torch.cuda.memory_allocated() == before
            got = out.cpu().tolist()
            for k in range(nvec):
                assert abs(got[k] - want[k]) <= 1e-12 * abs(want[k]), (call, k, got[k], want[k])
            # against plain torch as well (bilinear, no conjugation), so that both paths cannot be wrong together
            ref = (x1 * e1).sum(dim=1) + (x2 * e2).sum(dim=1)
            assert torch.allclose(out, ref, rtol=1e-11, atol=0.0)
    finally:
        ctx.close()


def test_property_without_allocation_rejects_sizes_beyond_the_static_scratch():
    import paper_2307_14296_b200 as cc
    n1, n2, nvec = 8, 12, cc.NOALLOC_MAX_VECS + 1
    z = lambda *s: torch.zeros(*s, dtype=torch.complex128, device="cuda")
    with pytest.raises(cc.CclrError) as err:
        cc.cclr_property_noalloc(z(n1), z(n2), z(nvec, n1), z(nvec, n2), z(nvec))
    assert "CCLR_NOALLOC_MAX_VECS" in str(err.value)      # CCLR_EINVAL with the reason
