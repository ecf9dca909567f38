"""The oracle's own pack / unpack between the C-ABI's packed layouts (include/cclr.h) and full tensors
(TEST INFRASTRUCTURE).  Pair index P(p<q) = q(q-1)/2 + p.  No method arithmetic here, only index bookkeeping:
antisymmetry V[pq,rs] = -V[qp,rs] = -V[pq,sr] of the integrals / amplitudes."""
import numpy as np


def pairs(n):
    """Arrays (p, q) with p<q ordered by P = q(q-1)/2 + p."""
    q, p = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
    m = p < q
    return p[m], q[m]


def npair(n):
    return n * (n - 1) // 2


def unpack_pair_axis(x, n, axis):
    """Expand one packed antisymmetric pair axis of length n(n-1)/2 into two axes (n, n) at ``axis``."""
    p, q = pairs(n)
    x = np.moveaxis(x, axis, 0)
    full = np.zeros((n, n) + x.shape[1:], x.dtype)
    full[p, q] = x
    full[q, p] = -x
    return np.moveaxis(full.reshape((n, n) + x.shape[1:]), [0, 1], [axis, axis + 1])


def pack_pair_axes(x, axis):
    """Take the p<q elements of the two axes (axis, axis+1) -> one packed axis."""
    n = x.shape[axis]
    p, q = pairs(n)
    x = np.moveaxis(x, [axis, axis + 1], [0, 1])
    return np.moveaxis(x[p, q], 0, axis)


def pack_amplitudes(x1, x2):
    """(x1[a,i], x2[a,b,i,j]) -> (x1[v][o], x2p[vv][oo])."""
    return np.ascontiguousarray(x1), np.ascontiguousarray(pack_pair_axes(pack_pair_axes(x2, 2), 0))


def unpack_amplitudes(x1, x2p, o, v):
    return x1.reshape(v, o), unpack_pair_axis(unpack_pair_axis(x2p.reshape(npair(v), npair(o)), o, 1), v, 0)


def flat(x1, x2):
    """Unique-element flat vector: singles row-major then packed doubles row-major."""
    a, b = pack_amplitudes(x1, x2)
    return np.concatenate([a.ravel(), b.ravel()])


def unflat(x, o, v):
    return unpack_amplitudes(x[: o * v], x[o * v:], o, v)


def unpack_eri(o, v, packed):
    """The six packed classes of include/cclr.h (dict of arrays) -> dict of full blocks.
    oooo[oo][oo], ooov[oo][o][v], oovv[oo][vv], ovvo[o][v][v][o], ovvv[o][v][vv], vvvv[vv][vv]."""
    oo, vv = npair(o), npair(v)
    full = {}
    full["oooo"] = unpack_pair_axis(unpack_pair_axis(packed["oooo"].reshape(oo, oo), o, 1), o, 0)
    full["ooov"] = unpack_pair_axis(packed["ooov"].reshape(oo, o, v), o, 0)
    full["oovv"] = unpack_pair_axis(unpack_pair_axis(packed["oovv"].reshape(oo, vv), v, 1), o, 0)
    full["ovvo"] = packed["ovvo"].reshape(o, v, v, o)
    full["ovvv"] = unpack_pair_axis(packed["ovvv"].reshape(o, v, vv), v, 2)
    full["vvvv"] = unpack_pair_axis(unpack_pair_axis(packed["vvvv"].reshape(vv, vv), v, 1), v, 0)
    return full


def pack_eri(full):
    """Inverse of unpack_eri (used to feed the GPU path from a full antisymmetrised V in tests)."""
    out = {}
    out["oooo"] = pack_pair_axes(pack_pair_axes(full["oooo"], 2), 0)
    out["ooov"] = pack_pair_axes(full["ooov"], 0)
    out["oovv"] = pack_pair_axes(pack_pair_axes(full["oovv"], 2), 0)
    out["ovvo"] = full["ovvo"]
    out["ovvv"] = pack_pair_axes(full["ovvv"], 2)
    out["vvvv"] = pack_pair_axes(pack_pair_axes(full["vvvv"], 2), 0)
    return {k: np.ascontiguousarray(val) for k, val in out.items()}
