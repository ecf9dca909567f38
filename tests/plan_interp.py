"""numpy interpreter of the contraction plans in paper_2307_14296_b200/csrc/plans.inc (TEST INFRASTRUCTURE).

The CUDA library executes the plan text with its own parser (csrc/plan.cu), its gather kernel and its DMMA GEMM.
This file re-implements the *semantics* of the three plan operations (gemm / perm / scat) with numpy fancy
indexing and ``@`` so that the plan text itself -- every index permutation, antisymmetry sign, chunk loop and
GEMM shape the GPU will run -- can be checked against the oracle on the CPU (tests/test_plan_host.py).
It shares no code with the product and none with the oracle.
"""
import os
import re
import numpy as np

PLANS_INC = os.path.join(os.path.dirname(os.path.dirname(os.path.abspath(__file__))), "paper_2307_14296_b200",
                         "csrc", "plans.inc")
OCC, VIR = "ijklmn", "abcdefgh"


def load_plan(name):
    text = open(PLANS_INC).read()
    m = re.search(name + r'\s*=\s*R"PLAN\((.*?)\)PLAN"', text, re.S)
    assert m, name
    return m.group(1)


def parse_spec(s):
    """'(ab)E;j' -> [[('P','a','b'), ('L','E')], [('L','j')]]"""
    groups = []
    for g in s.split(";"):
        axes, k = [], 0
        while k < len(g):
            c = g[k]
            if c == "(":
                axes.append(("P", g[k + 1], g[k + 2]))
                assert g[k + 3] == ")"
                k += 4
            elif c == "1":
                axes.append(("1",))
                k += 1
            else:
                axes.append(("L", c))
                k += 1
        groups.append(axes)
    return groups


def npair(n):
    return n * (n - 1) // 2


class Interp:
    def __init__(self, o, v, chunk_override=None):
        self.o, self.v = o, v
        self.bufs = {}       # name -> [flat array, declared axes]
        self.chunk = {}      # upper-case letter -> (offset, length)
        self.scalars = {}
        self.chunk_override = chunk_override
        self.peak_elems = 0

    # ---- extents -----------------------------------------------------------------------------------------
    def full_extent(self, letter):
        l = letter.lower()
        return self.o if l in OCC else self.v

    def extent(self, letter):
        if letter.isupper():
            return self.chunk[letter][1]
        return self.full_extent(letter)

    def axis_extent(self, ax):
        if ax[0] == "1":
            return 1
        if ax[0] == "L":
            return self.extent(ax[1])
        assert ax[1].islower() and ax[2].islower()
        assert self.full_extent(ax[1]) == self.full_extent(ax[2])
        return npair(self.full_extent(ax[1]))

    def max_axis_extent(self, ax, chunk_max):
        if ax[0] == "L" and ax[1].isupper():
            return chunk_max[ax[1]]
        return self.axis_extent(ax)

    # ---- buffers -------------------------------------------------------------------------------------------
    def bind(self, name, spec, array):
        axes = parse_spec(spec)[0]
        n = int(np.prod([self.axis_extent(a) for a in axes]))
        flat = np.ascontiguousarray(array, dtype=complex).reshape(-1)
        assert flat.size == n, (name, flat.size, n)
        self.bufs[name] = [flat, axes]

    def get(self, name, shape=None):
        flat, axes = self.bufs[name]
        n = int(np.prod([self.axis_extent(a) for a in axes]))
        out = flat[:n]
        return out.reshape(shape) if shape is not None else out.reshape([self.axis_extent(a) for a in axes])

    # ---- index evaluation -----------------------------------------------------------------------------------
    def iteration(self, axes):
        """letter -> global value arrays broadcast over the iteration shape; returns (values, shape)."""
        shape = [self.axis_extent(a) for a in axes]
        vals = {}
        for k, ax in enumerate(axes):
            bshape = [1] * len(axes)
            bshape[k] = shape[k]
            if ax[0] == "1":
                continue
            if ax[0] == "L":
                off = self.chunk[ax[1]][0] if ax[1].isupper() else 0
                assert ax[1] not in vals
                vals[ax[1]] = (off + np.arange(shape[k])).reshape(bshape)
            else:
                n = self.full_extent(ax[1])
                q, p = np.meshgrid(np.arange(n), np.arange(n), indexing="ij")
                m = p < q
                assert ax[1] not in vals and ax[2] not in vals
                vals[ax[1]] = p[m].reshape(bshape)
                vals[ax[2]] = q[m].reshape(bshape)
        return vals, shape

    def offsets(self, name, access_axes, vals, shape):
        """flat offset and sign (0 = structurally zero) of buffer ``name`` accessed with ``access_axes``."""
        flat, decl = self.bufs[name]
        assert len(decl) == len(access_axes), (name, decl, access_axes)
        ext = [self.axis_extent(a) for a in decl]
        strides = [int(np.prod(ext[k + 1:])) for k in range(len(ext))]
        off = np.zeros(shape, dtype=np.int64)
        sign = np.ones(shape, dtype=np.int64)
        for d, a, st, ex in zip(decl, access_axes, strides, ext):
            if d[0] == "1":
                assert a[0] == "1"
                continue
            if d[0] == "L":
                assert a[0] == "L", (name, d, a)
                assert self.full_extent(d[1]) == self.full_extent(a[1]), (name, d, a)
                idx = vals[a[1]] - (self.chunk[d[1]][0] if d[1].isupper() else 0)
                assert idx.min() >= 0 and idx.max() < ex, (name, d, a)
                off = off + idx * st
            else:
                assert a[0] == "P", (name, d, a)
                assert self.full_extent(d[1]) == self.full_extent(a[1]) == self.full_extent(a[2])
                p, q = np.broadcast_arrays(vals[a[1]], vals[a[2]])
                lo, hi = np.minimum(p, q), np.maximum(p, q)
                sign = sign * np.sign(q - p)
                off = off + (hi * (hi - 1) // 2 + lo) * (p != q) * st
        return np.broadcast_to(off, shape), np.broadcast_to(sign, shape)

    def gemm_view(self, name, spec):
        """Dense [R][C] view of a buffer for a gemm operand 'rows;cols'."""
        flat, decl = self.bufs[name]
        rows, cols = parse_spec(spec)
        acc = [a for a in rows + cols if a[0] != "1"]
        decl = [d for d in decl if d[0] != "1"]
        assert len(acc) == len(decl), (name, spec, decl)
        base = 0
        for k, (d, a) in enumerate(zip(decl, acc)):
            if d == a:
                continue
            if d[0] == "L" and a[0] == "L" and self.full_extent(d[1]) == self.full_extent(a[1]):
                if k == 0 and a[1].isupper() and d[1].islower():
                    rest = int(np.prod([self.axis_extent(x) for x in decl[1:]]))
                    base = self.chunk[a[1]][0] * rest
                    continue
                if d[1].islower() and a[1].islower():
                    continue                                       # renamed letter of the same range
            if d[0] == "P" and a[0] == "P" and self.full_extent(d[1]) == self.full_extent(a[1]):
                continue
            raise AssertionError("gemm view mismatch %s[%s] vs declared %s" % (name, spec, decl))
        R = int(np.prod([self.axis_extent(a) for a in rows]))
        Cc = int(np.prod([self.axis_extent(a) for a in cols]))
        assert base + R * Cc <= flat.size, (name, spec)
        return flat[base:base + R * Cc].reshape(R, Cc)

    # ---- execution ----------------------------------------------------------------------------------------
    def coef(self, tok):
        return self.scalars[tok] if tok.startswith("$") else complex(float(tok))

    @staticmethod
    def split_ref(tok):
        m = re.match(r"(\w+)\[(.*)\]$", tok)
        assert m, tok
        return m.group(1), m.group(2)

    def run(self, text, chunk_max_default=None):
        lines = [l.split("#")[0].strip() for l in text.splitlines()]
        lines = [l for l in lines if l]
        self._exec(lines)

    def _exec(self, lines):
        k = 0
        while k < len(lines):
            t = lines[k].split()
            op = t[0]
            if op == "chunk":
                depth, e = 1, k + 1
                while depth:
                    w = lines[e].split()[0]
                    depth += (w == "chunk") - (w == "end")
                    e += 1
                body = lines[k + 1:e - 1]
                letter, clen = t[1], int(t[2])
                if self.chunk_override:
                    clen = self.chunk_override
                full = self.full_extent(letter)
                clen = min(clen, full)
                self._chunk_max = getattr(self, "_chunk_max", {})
                self._chunk_max[letter] = clen
                created = [l.split()[1] for l in body if l.split()[0] == "buf"]
                for off in range(0, full, clen):
                    self.chunk[letter] = (off, min(clen, full - off))
                    self._exec(body)
                del self.chunk[letter]
                for nme in created:
                    self.bufs.pop(nme, None)
                k = e
                continue
            if op.startswith("@"):
                pass
            elif op == "buf":
                name, spec = t[1], t[2]
                if name not in self.bufs:
                    axes = parse_spec(spec)[0]
                    cm = getattr(self, "_chunk_max", {})
                    n = int(np.prod([self.max_axis_extent(a, cm) for a in axes]))
                    self.bufs[name] = [np.full(n, np.nan + 0j), axes]
                    self.peak_elems = max(self.peak_elems, sum(b[0].size for b in self.bufs.values()))
            elif op == "free":
                del self.bufs[t[1]]
            elif op == "gemm":
                cname, cspec = self.split_ref(t[1])
                acc = t[2]
                alpha = self.coef(t[3])
                r = t[4:]
                conj_a = r[0] == "conj"
                r = r[1:] if conj_a else r
                aname, aspec = self.split_ref(r[0])
                r = r[1:]
                conj_b = r[0] == "conj"
                r = r[1:] if conj_b else r
                bname, bspec = self.split_ref(r[0])
                mode = r[1]
                Cv, Av, Bv = self.gemm_view(cname, cspec), self.gemm_view(aname, aspec), self.gemm_view(bname, bspec)
                A = Av.conj() if conj_a else Av
                B = Bv.conj() if conj_b else Bv
                if mode == "nk":
                    B = B.T
                assert A.shape[1] == B.shape[0] and Cv.shape == (A.shape[0], B.shape[1]), (lines[k], A.shape, B.shape, Cv.shape)
                res = alpha * (A @ B)
                if acc == "+=":
                    Cv += res
                else:
                    Cv[...] = res
            elif op in ("perm", "scat"):
                dname, dspec = self.split_ref(t[1])
                acc = t[2]
                r = t[3:]
                cond = "all"
                if op == "scat":
                    ci = r.index("cond")
                    cond = r[ci + 1]
                    ii = r.index("iter")
                    it_axes = parse_spec(r[ii + 1])[0]
                    r = r[:ii]
                else:
                    it_axes = parse_spec(dspec)[0]
                vals, shape = self.iteration(it_axes)
                doff, dsign = self.offsets(dname, parse_spec(dspec)[0], vals, shape)
                total = np.zeros(shape, complex)
                while r:
                    c = self.coef(r[0])
                    r = r[1:]
                    cj = r[0] == "conj"
                    r = r[1:] if cj else r
                    sname, sspec = self.split_ref(r[0])
                    r = r[1:]
                    soff, ssign = self.offsets(sname, parse_spec(sspec)[0], vals, shape)
                    val = self.bufs[sname][0][soff]
                    val = val.conj() if cj else val
                    total = total + c * ssign * val
                mask = dsign != 0
                if op == "perm":
                    assert mask.all()
                    flat_off = doff.reshape(-1)
                    assert (flat_off - flat_off[0] == np.arange(flat_off.size)).all(), ("gather dst not linear", lines[k])
                else:
                    assert acc == "+="
                    dpair = [a for a in parse_spec(dspec)[0] if a[0] == "P"]
                    if cond != "all":
                        p, q = np.broadcast_arrays(vals[dpair[0][1]], vals[dpair[0][2]])
                        mask = mask & np.broadcast_to((p < q) if cond == "lt" else (p > q), shape)
                    sel = doff[mask]
                    assert np.unique(sel).size == sel.size, ("scatter race", lines[k])
                dst = self.bufs[dname][0]
                if acc == "+=":
                    dst[doff[mask]] += (dsign * total)[mask]
                else:
                    dst[doff[mask]] = (dsign * total)[mask]
            else:
                raise AssertionError("unknown op " + lines[k])
            k += 1


def run_create(o, v, fock, packed, t1, t2p, chunk_override=None):
    """Execute CCLR_PLAN_CREATE on numpy arrays; returns the interpreter holding every persist buffer."""
    it = Interp(o, v, chunk_override)
    for name, spec in (("oooo", "(mn)(ij)"), ("ooov", "(mn)ie"), ("oovv", "(mn)(ef)"), ("ovvo", "mbej"),
                       ("ovvv", "mb(ef)")):
        it.bind(name, spec, packed[name])
    it.bind("Wabef", "(ab)(ef)", packed["vvvv"].copy())
    it.bind("t1", "ai", t1)
    it.bind("t2", "(ab)(ij)", t2p)
    it.bind("foo", "mi", fock[:o, :o])
    it.bind("fov", "me", fock[:o, o:])
    it.bind("fvv", "ae", fock[o:, o:])
    it.run(load_plan("CCLR_PLAN_CREATE"))
    return it


def run_sigma(it, x1, x2p, z):
    o, v = it.o, it.v
    it.scalars["$nz"] = -complex(z)
    it.bind("x1", "ai", x1)
    it.bind("x2", "(ab)(ij)", x2p)
    it.bind("out1", "ai", np.zeros(v * o, complex))
    it.bind("out2", "(ab)(ij)", np.zeros(npair(v) * npair(o), complex))
    it.run(load_plan("CCLR_PLAN_SIGMA"))
    return it.get("out1").copy(), it.get("out2").copy()


def run_xi(it, X):
    """Execute CCLR_PLAN_XI (after run_sigma has declared the work buffers it reuses) for the one-body matrix X [n][n]."""
    o, v = it.o, it.v
    it.bind("xoo", "mi", np.ascontiguousarray(X[:o, :o]).reshape(-1))
    it.bind("xov", "me", np.ascontiguousarray(X[:o, o:]).reshape(-1))
    it.bind("xvo", "ai", np.ascontiguousarray(X[o:, :o]).reshape(-1))
    it.bind("xvv", "ae", np.ascontiguousarray(X[o:, o:]).reshape(-1))
    it.bind("out1", "ai", np.zeros(v * o, complex))
    it.bind("out2", "(ab)(ij)", np.zeros(npair(v) * npair(o), complex))
    it.run(load_plan("CCLR_PLAN_XI"))
    return it.get("out1").copy(), it.get("out2").copy()


def run_sigma_left(it, l1, l2p, z):
    """Execute CCLR_PLAN_SIGMA_LEFT (after run_sigma has declared the shared work buffers)."""
    o, v = it.o, it.v
    it.scalars["$nz"] = -complex(z)
    it.bind("x1", "ai", l1)
    it.bind("x2", "(ab)(ij)", l2p)
    it.bind("out1", "ai", np.zeros(v * o, complex))
    it.bind("out2", "(ab)(ij)", np.zeros(npair(v) * npair(o), complex))
    it.run(load_plan("CCLR_PLAN_SIGMA_LEFT"))
    return it.get("out1").copy(), it.get("out2").copy()


def run_eta(it, X, l1, l2p, eom):
    """Execute CCLR_PLAN_XI (into xiw1 / xiw2), CCLR_PLAN_ETA and optionally CCLR_PLAN_ETA_EOM for operator X and multipliers."""
    o, v = it.o, it.v
    it.bind("xoo", "mi", np.ascontiguousarray(X[:o, :o]).reshape(-1))
    it.bind("xov", "me", np.ascontiguousarray(X[:o, o:]).reshape(-1))
    it.bind("xvo", "ai", np.ascontiguousarray(X[o:, :o]).reshape(-1))
    it.bind("xvv", "ae", np.ascontiguousarray(X[o:, o:]).reshape(-1))
    it.bind("x1", "ai", l1)
    it.bind("x2", "(ab)(ij)", l2p)
    xi1, xi2 = np.zeros(v * o, complex), np.zeros(npair(v) * npair(o), complex)
    if eom:
        it.bind("out1", "ai", xi1)
        it.bind("out2", "(ab)(ij)", xi2)
        it.run(load_plan("CCLR_PLAN_XI"))
        xi1 = it.get("out1").copy()
    it.bind("out1", "ai", np.zeros(v * o, complex))
    it.bind("out2", "(ab)(ij)", np.zeros(npair(v) * npair(o), complex))
    it.run(load_plan("CCLR_PLAN_ETA"))
    if eom:
        it.get("xiw1")[...] = xi1.reshape(it.get("xiw1").shape)
        it.run(load_plan("CCLR_PLAN_ETA_EOM"))
    return it.get("out1").copy(), it.get("out2").copy()


def run_omega(o, v, fock, packed, t1, t2p, chunk_override=None):
    """Execute CCLR_PLAN_OMEGA (the direct CCSD residual of cclr_ccsd) on numpy arrays; returns (om1, om2)."""
    it = Interp(o, v, chunk_override)
    for name, spec in (("oooo", "(mn)(ij)"), ("ooov", "(mn)ie"), ("oovv", "(mn)(ef)"), ("ovvo", "mbej"),
                       ("ovvv", "mb(ef)"), ("vvvv", "(ab)(ef)")):
        it.bind(name, spec, packed[name])
    it.bind("t1", "ai", t1)
    it.bind("t2", "(ab)(ij)", t2p)
    it.bind("foo", "mi", fock[:o, :o])
    it.bind("fov", "me", fock[:o, o:])
    it.bind("fvo", "ai", fock[o:, :o])
    it.bind("fvv", "ae", fock[o:, o:])
    it.run(load_plan("CCLR_PLAN_OMEGA"))
    return it.get("om1").copy(), it.get("om2").copy()


def run_fy(it, packed, l1, l2p, y1, y2p):
    """Execute CCLR_PLAN_FY (after run_sigma and run_sigma_left have declared the shared work buffers): out = F y for the
    multipliers (l1, l2) and the vector (y1, y2), with the caller's bare ooov / oovv / ovvo / ovvv bound again (vvvv is not)."""
    o, v = it.o, it.v
    for name, spec in (("ooov", "(mn)ie"), ("oovv", "(mn)(ef)"), ("ovvo", "mbej"), ("ovvv", "mb(ef)")):
        it.bind(name, spec, packed[name])
    it.bind("x1", "ai", l1)
    it.bind("x2", "(ab)(ij)", l2p)
    it.bind("y1", "ai", y1)
    it.bind("y2", "(ab)(ij)", y2p)
    it.bind("out1", "ai", np.zeros(v * o, complex))
    it.bind("out2", "(ab)(ij)", np.zeros(npair(v) * npair(o), complex))
    it.run(load_plan("CCLR_PLAN_FY_M"))       # the lambda-only ladder, once per set of multipliers
    it.run(load_plan("CCLR_PLAN_FY"))
    return it.get("out1").copy(), it.get("out2").copy()
