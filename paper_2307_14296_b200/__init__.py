"""paper_2307_14296_b200 — thin Python binding of the B200-native CC-LR hot-path library (include/cclr.h).

Same names as the C ABI; this layer only marshals arguments (torch tensors -> device pointers, the current CUDA
stream).  Every step of the path runs in the library's own sm_100a kernels; PyTorch supplies device memory and
streams only.  There is no CPU fallback: a missing ``libcclr.so`` or a non-CUDA tensor raises.
"""
import ctypes as C

import torch

from . import _lib
from ._lib import CclrError, SolveInfo  # noqa: F401

__all__ = ["Context", "cclr_create", "cclr_ccsd", "cclr_response_ci", "cclr_response_ci_tensor", "cclr_response_cc", "cclr_f_transform", "cclr_xfy", "cclr_eom", "cclr_xi", "cclr_eta", "cclr_lambda", "cclr_solve_left", "cclr_sigma_left", "cclr_sigma", "cclr_solve", "cclr_property", "cclr_zgemm", "cclr_ladder",
           "cclr_ring", "cclr_fp64_tensor_peak", "cclr_hbm_copy_peak", "CclrError"]


def _dev(t, name, shape_numel=None):
    if not isinstance(t, torch.Tensor) or not t.is_cuda or t.dtype != torch.complex128 or not t.is_contiguous():
        raise TypeError("%s must be a contiguous complex128 CUDA tensor" % name)
    if shape_numel is not None and t.numel() != shape_numel:
        raise ValueError("%s has %d elements, expected %d" % (name, t.numel(), shape_numel))
    return C.c_void_p(t.data_ptr())


def _host(t, name, shape_numel=None):
    if not isinstance(t, torch.Tensor) or t.is_cuda or t.dtype != torch.complex128 or not t.is_contiguous():
        raise TypeError("%s must be a contiguous complex128 host tensor" % name)
    if shape_numel is not None and t.numel() != shape_numel:
        raise ValueError("%s has %d elements, expected %d" % (name, t.numel(), shape_numel))
    return C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


ERI_INPLACE = 1
SMALL_CHUNKS = 2
GEMM_4M = 4
NO_GRAPH = 8
NO_SUM_PLANES = 16
GEMM_DMMA = 32
GEMM_INT8_ANY_SIZE = 64
NO_LEFT_SLICES = 128


class Context:
    """Owner of a ``cclr_ctx*``; created by :func:`cclr_create`."""

    def __init__(self, handle, o, v, keep):
        self.handle, self.o, self.v = handle, o, v
        self._keep = keep  # buffers the C context may still reference (vvvv with ERI_INPLACE)
        self.oo, self.vv = o * (o - 1) // 2, v * (v - 1) // 2
        self.n1, self.n2 = o * v, self.oo * self.vv

    def close(self):
        if self.handle is not None:
            _lib.load().cclr_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def bytes(self):
        return int(_lib.load().cclr_ctx_bytes(self.handle))

    def get_intermediate(self, name):
        lib = _lib.load()
        n = lib.cclr_get_intermediate(self.handle, name.encode(), None, 0)
        if n < 0:
            raise CclrError(int(n), "cclr_get_intermediate(%s)" % name)
        out = torch.empty(int(n), dtype=torch.complex128, device="cuda")
        m = lib.cclr_get_intermediate(self.handle, name.encode(), _dev(out, "out"), n)
        if m < 0:
            raise CclrError(int(m), "cclr_get_intermediate(%s)" % name)
        torch.cuda.current_stream().synchronize()
        return out

    def get_intermediate_slice(self, name, offset, count):
        """``count`` consecutive elements of the named intermediate starting at element ``offset`` (device tensor)."""
        out = torch.empty(int(count), dtype=torch.complex128, device="cuda")
        m = _lib.load().cclr_get_intermediate_slice(self.handle, name.encode(), int(offset), int(count), _dev(out, "out"))
        if m < 0:
            raise CclrError(int(m), "cclr_get_intermediate_slice(%s)" % name)
        torch.cuda.current_stream().synchronize()
        return out

    def set_max_subspace(self, dim):
        _lib.check(_lib.load().cclr_set_max_subspace(self.handle, int(dim)), "cclr_set_max_subspace")

    def set_gemm_path(self, path):
        """1: ladder / ring as integer-slice products on the INT8 tensor path (if the context holds the slices), 0: DMMA.
        Returns the path now in use."""
        return int(_lib.load().cclr_set_gemm_path(self.handle, int(path)))

    def gemm_slices(self):
        """Integer slices per operand of the INT8 tensor path in use (0: ladder and ring on the FP64 tensor cores)."""
        return int(_lib.load().cclr_gemm_slices(self.handle))

    def set_profiling(self, on):
        _lib.check(_lib.load().cclr_set_profiling(self.handle, int(bool(on))), "cclr_set_profiling")

    def last_sigma_ms(self):
        ms = (C.c_double * 5)()
        _lib.check(_lib.load().cclr_last_sigma_ms(self.handle, ms), "cclr_last_sigma_ms")
        return dict(zip(("total", "ladder", "ring", "other_gemm", "layout"), list(ms)))


    def last_sigma_ops(self):
        """[(plan statement, ms)] of the last profiled cclr_sigma call."""
        lib = _lib.load()
        n = lib.cclr_sigma_op_count(self.handle)
        ms = (C.c_double * n)()
        _lib.check(min(lib.cclr_last_sigma_op_ms(self.handle, ms, n), 0), "cclr_last_sigma_op_ms")
        return [(lib.cclr_sigma_op_text(self.handle, k).decode(), ms[k]) for k in range(n)]


def cclr_create(o, v, fock, eri, t1, t2, flags=0):
    """eri: dict with the six packed classes of include/cclr.h (device tensors)."""
    lib = _lib.load()
    oo, vv, n = o * (o - 1) // 2, v * (v - 1) // 2, o + v
    sizes = dict(oooo=oo * oo, ooov=oo * o * v, oovv=oo * vv, ovvo=o * v * v * o, ovvv=o * v * vv, vvvv=vv * vv)
    e = _lib.EriPacked()
    for k, sz in sizes.items():
        setattr(e, k, _dev(eri[k], "eri." + k, sz))
    h = C.c_void_p()
    rc = lib.cclr_create(o, v, _dev(fock, "fock", n * n), C.byref(e), _dev(t1, "t1", o * v), _dev(t2, "t2", vv * oo),
                         flags, _stream(), C.byref(h))
    _lib.check(rc, "cclr_create")
    return Context(h, o, v, keep=[eri["vvvv"]] if flags & ERI_INPLACE else [])


def _eri_struct(o, v, eri):
    oo, vv = o * (o - 1) // 2, v * (v - 1) // 2
    sizes = dict(oooo=oo * oo, ooov=oo * o * v, oovv=oo * vv, ovvo=o * v * v * o, ovvv=o * v * vv, vvvv=vv * vv)
    e = _lib.EriPacked()
    for k, sz in sizes.items():
        setattr(e, k, _dev(eri[k], "eri." + k, sz))
    return e


def cclr_ccsd(o, v, fock, eri, t1=None, t2=None, tol=1e-10, maxiter=100):
    """Ground-state CCSD amplitudes on the device; returns (t1 [v*o], t2 [vv*oo], info).  t1/t2: start amplitudes (updated
    in place) or None for zeros."""
    oo, vv, n = o * (o - 1) // 2, v * (v - 1) // 2, o + v
    if t1 is None:
        t1 = torch.zeros(o * v, dtype=torch.complex128, device="cuda")
    if t2 is None:
        t2 = torch.zeros(vv * oo, dtype=torch.complex128, device="cuda")
    e = _eri_struct(o, v, eri)
    info = _lib.CcsdInfo()
    rc = _lib.load().cclr_ccsd(o, v, _dev(fock, "fock", n * n), C.byref(e), _dev(t1, "t1", o * v), _dev(t2, "t2", vv * oo),
                               float(tol), int(maxiter), _stream(), C.byref(info))
    if rc not in (0, -4):
        _lib.check(rc, "cclr_ccsd")
    return t1, t2, info


def cclr_ccsd_residual(o, v, fock, eri, t1, t2, mode=0):
    """Omega(t) on the device: mode 0 = direct residual plan, mode 1 = quadrature of the Jacobian.  Returns (om1, om2)."""
    oo, vv, n = o * (o - 1) // 2, v * (v - 1) // 2, o + v
    e = _eri_struct(o, v, eri)
    om1 = torch.empty(o * v, dtype=torch.complex128, device="cuda")
    om2 = torch.empty(vv * oo, dtype=torch.complex128, device="cuda")
    rc = _lib.load().cclr_ccsd_residual(o, v, _dev(fock, "fock", n * n), C.byref(e), _dev(t1, "t1", o * v),
                                        _dev(t2, "t2", vv * oo), int(mode), _stream(), _dev(om1, "om1"), _dev(om2, "om2"))
    _lib.check(rc, "cclr_ccsd_residual")
    return om1, om2


def cclr_sigma(ctx, x1, x2, omega=0.0, gamma=0.0, out1=None, out2=None):
    """out = A x - (omega + i gamma) x.  x1: [nvec, v*o] (or [v*o]), x2: [nvec, vv*oo]."""
    nvec = x1.numel() // ctx.n1
    if out1 is None:
        out1 = torch.empty_like(x1)
    if out2 is None:
        out2 = torch.empty_like(x2)
    rc = _lib.load().cclr_sigma(ctx.handle, _dev(x1, "x1", nvec * ctx.n1), _dev(x2, "x2", nvec * ctx.n2), nvec,
                                float(omega), float(gamma), _dev(out1, "out1", nvec * ctx.n1),
                                _dev(out2, "out2", nvec * ctx.n2))
    _lib.check(rc, "cclr_sigma")
    return out1, out2


def cclr_sigma_left(ctx, l1, l2, omega=0.0, gamma=0.0, out1=None, out2=None):
    """out = l (A - (omega + i gamma)): the left Jacobian transform.  l1: [nvec, v*o] (or [v*o]), l2: [nvec, vv*oo]."""
    nvec = l1.numel() // ctx.n1
    if out1 is None:
        out1 = torch.empty_like(l1)
    if out2 is None:
        out2 = torch.empty_like(l2)
    rc = _lib.load().cclr_sigma_left(ctx.handle, _dev(l1, "l1", nvec * ctx.n1), _dev(l2, "l2", nvec * ctx.n2), nvec,
                                     float(omega), float(gamma), _dev(out1, "out1", nvec * ctx.n1),
                                     _dev(out2, "out2", nvec * ctx.n2))
    _lib.check(rc, "cclr_sigma_left")
    return out1, out2


def cclr_sigma_host(ctx, x1, x2, omega, gamma, out1, out2):
    """Same through HOST tensors (copies inside the call)."""
    nvec = x1.numel() // ctx.n1
    rc = _lib.load().cclr_sigma_host(ctx.handle, _host(x1, "x1", nvec * ctx.n1), _host(x2, "x2", nvec * ctx.n2), nvec,
                                     float(omega), float(gamma), _host(out1, "out1", nvec * ctx.n1),
                                     _host(out2, "out2", nvec * ctx.n2))
    _lib.check(rc, "cclr_sigma_host")
    return out1, out2


def cclr_solve(ctx, xi1, xi2, omegas, gamma=0.0, tol=1e-10, maxiter=200):
    """Solve (A - (omega_k + i gamma)) t = -xi_r.  Returns t1 [nrhs, nomega, v*o], t2 [nrhs, nomega, vv*oo], info."""
    nrhs = xi1.numel() // ctx.n1
    om = (C.c_double * len(omegas))(*[float(w) for w in omegas])
    t1 = torch.empty((nrhs, len(omegas), ctx.n1), dtype=torch.complex128, device="cuda")
    t2 = torch.empty((nrhs, len(omegas), ctx.n2), dtype=torch.complex128, device="cuda")
    info = SolveInfo()
    rc = _lib.load().cclr_solve(ctx.handle, _dev(xi1, "xi1", nrhs * ctx.n1), _dev(xi2, "xi2", nrhs * ctx.n2), nrhs, om,
                                len(omegas), float(gamma), float(tol), int(maxiter), _dev(t1, "t1"), _dev(t2, "t2"),
                                C.byref(info))
    if rc not in (0, -4):
        _lib.check(rc, "cclr_solve")
    return t1, t2, info


def cclr_eom(ctx, nroots, tol=1e-8, maxiter=200):
    """Lowest nroots eigenpairs of the Jacobian: (list of complex eigenvalues, r1 [nroots, v*o], r2 [nroots, vv*oo], info)."""
    eig = (_lib.Complex * nroots)()
    r1 = torch.empty((nroots, ctx.n1), dtype=torch.complex128, device="cuda")
    r2 = torch.empty((nroots, ctx.n2), dtype=torch.complex128, device="cuda")
    info = _lib.EomInfo()
    rc = _lib.load().cclr_eom(ctx.handle, int(nroots), float(tol), int(maxiter), eig, _dev(r1, "r1"), _dev(r2, "r2"),
                              C.byref(info))
    if rc not in (0, -4):
        _lib.check(rc, "cclr_eom")
    return [complex(e.re, e.im) for e in eig], r1, r2, info


def cclr_xi(ctx, X):
    """xi^X for a one-body operator X ([n, n] complex128 CUDA tensor): returns (xi1 [v*o], xi2 [vv*oo])."""
    n = ctx.o + ctx.v
    xi1 = torch.empty(ctx.n1, dtype=torch.complex128, device="cuda")
    xi2 = torch.empty(ctx.n2, dtype=torch.complex128, device="cuda")
    _lib.check(_lib.load().cclr_xi(ctx.handle, _dev(X, "X", n * n), _dev(xi1, "xi1"), _dev(xi2, "xi2")), "cclr_xi")
    return xi1, xi2


def cclr_solve_left(ctx, eta1, eta2, omegas, gamma=0.0, tol=1e-10, maxiter=200):
    """Solve l (A - (omega_k + i gamma)) = -eta_r.  Returns l1 [nrhs, nomega, v*o], l2 [nrhs, nomega, vv*oo], info."""
    nrhs = eta1.numel() // ctx.n1
    om = (C.c_double * len(omegas))(*[float(w) for w in omegas])
    l1 = torch.empty((nrhs, len(omegas), ctx.n1), dtype=torch.complex128, device="cuda")
    l2 = torch.empty((nrhs, len(omegas), ctx.n2), dtype=torch.complex128, device="cuda")
    info = SolveInfo()
    rc = _lib.load().cclr_solve_left(ctx.handle, _dev(eta1, "eta1", nrhs * ctx.n1), _dev(eta2, "eta2", nrhs * ctx.n2), nrhs,
                                     om, len(omegas), float(gamma), float(tol), int(maxiter), _dev(l1, "l1"), _dev(l2, "l2"),
                                     C.byref(info))
    if rc not in (0, -4):
        _lib.check(rc, "cclr_solve_left")
    return l1, l2, info


def cclr_lambda(ctx, tol=1e-10, maxiter=200):
    """Ground-state multipliers: lambda A = -eta0.  Returns (lam1 [v*o], lam2 [vv*oo], info)."""
    lam1 = torch.empty(ctx.n1, dtype=torch.complex128, device="cuda")
    lam2 = torch.empty(ctx.n2, dtype=torch.complex128, device="cuda")
    info = SolveInfo()
    rc = _lib.load().cclr_lambda(ctx.handle, float(tol), int(maxiter), _dev(lam1, "lam1"), _dev(lam2, "lam2"), C.byref(info))
    if rc not in (0, -4):
        _lib.check(rc, "cclr_lambda")
    return lam1, lam2, info


def cclr_eta(ctx, X, lam1, lam2, eom=False):
    """eta^X (eom=False, S-Eq. 5-6) or EOM-eta^X (eom=True, S-Eq. 7) for operator X [n, n] and multipliers lam1, lam2."""
    n = ctx.o + ctx.v
    e1 = torch.empty(ctx.n1, dtype=torch.complex128, device="cuda")
    e2 = torch.empty(ctx.n2, dtype=torch.complex128, device="cuda")
    _lib.check(_lib.load().cclr_eta(ctx.handle, _dev(X, "X", n * n), _dev(lam1, "lam1", ctx.n1), _dev(lam2, "lam2", ctx.n2),
                                    int(bool(eom)), _dev(e1, "eta1"), _dev(e2, "eta2")), "cclr_eta")
    return e1, e2


def cclr_response_ci(ctx, X, Y, omega, gamma=0.0, tol=1e-10, maxiter=200):
    """<<X;Y>>_{omega + i gamma} (CC-CI form, Eq. 16-17) computed end to end on the device; returns (complex, info)."""
    n = ctx.o + ctx.v
    res = _lib.Complex()
    info = SolveInfo()
    rc = _lib.load().cclr_response_ci(ctx.handle, _dev(X, "X", n * n), _dev(Y, "Y", n * n), float(omega), float(gamma),
                                      float(tol), int(maxiter), C.byref(res), C.byref(info))
    if rc not in (0, -4):
        _lib.check(rc, "cclr_response_ci")
    return complex(res.re, res.im), info


def cclr_response_ci_tensor(ctx, X, omegas, gamma=0.0, tol=1e-10, maxiter=200):
    """<<X_r;X_s>>_{omega_k + i gamma} for all operator pairs and frequencies (CC-CI, Eq. 16-17) in one call.
    X: [nop, n, n] complex128 CUDA tensor.  Returns (list [nomega][nop][nop] of complex, info)."""
    n = ctx.o + ctx.v
    nop = X.numel() // (n * n)
    om = (C.c_double * len(omegas))(*[float(w) for w in omegas])
    res = (_lib.Complex * (len(omegas) * nop * nop))()
    info = SolveInfo()
    rc = _lib.load().cclr_response_ci_tensor(ctx.handle, _dev(X, "X", nop * n * n), nop, om, len(omegas), float(gamma),
                                             float(tol), int(maxiter), res, C.byref(info))
    if rc not in (0, -4):
        _lib.check(rc, "cclr_response_ci_tensor")
    flat = [complex(r.re, r.im) for r in res]
    out = [[[flat[(k * nop + r) * nop + s] for s in range(nop)] for r in range(nop)] for k in range(len(omegas))]
    return out, info


def cclr_xfy(o, v, fock, eri, t1, t2, lam1, lam2, x1, x2, y1, y2):
    """x . F . y (CC Hessian contraction) as an exact derivative of the left transform; returns a complex."""
    e = _eri_struct(o, v, eri)
    res = _lib.Complex()
    n1, n2 = o * v, (o * (o - 1) // 2) * (v * (v - 1) // 2)
    rc = _lib.load().cclr_xfy(o, v, _dev(fock, "fock", (o + v) ** 2), C.byref(e), _dev(t1, "t1", n1), _dev(t2, "t2", n2),
                              _dev(lam1, "lam1", n1), _dev(lam2, "lam2", n2), _dev(x1, "x1", n1), _dev(x2, "x2", n2),
                              _dev(y1, "y1", n1), _dev(y2, "y2", n2), _stream(), C.byref(res))
    _lib.check(rc, "cclr_xfy")
    return complex(res.re, res.im)


def _eri_struct_partial(o, v, eri, names):
    """EriPacked with only the classes in `names` set (the others stay NULL: the callee documents which ones it reads)."""
    oo, vv = o * (o - 1) // 2, v * (v - 1) // 2
    sizes = dict(oooo=oo * oo, ooov=oo * o * v, oovv=oo * vv, ovvo=o * v * v * o, ovvv=o * v * vv, vvvv=vv * vv)
    e = _lib.EriPacked()
    for k in names:
        setattr(e, k, _dev(eri[k], "eri." + k, sizes[k]))
    return e


def cclr_f_transform(ctx, eri, lam1, lam2, y1, y2):
    """F y_k for every vector y_k (y1 [nvec, v*o], y2 [nvec, vv*oo]) and the multipliers lam1, lam2; eri: dict holding at
    least ooov, oovv, ovvo, ovvv of the integrals the context was created from.  Returns (out1, out2) shaped like y."""
    nvec = y1.numel() // ctx.n1
    e = _eri_struct_partial(ctx.o, ctx.v, eri, ("ooov", "oovv", "ovvo", "ovvv"))
    out1, out2 = torch.empty_like(y1), torch.empty_like(y2)
    _lib.check(_lib.load().cclr_f_transform(ctx.handle, C.byref(e), _dev(lam1, "lam1", ctx.n1), _dev(lam2, "lam2", ctx.n2),
                                            _dev(y1, "y1", nvec * ctx.n1), _dev(y2, "y2", nvec * ctx.n2), nvec,
                                            _dev(out1, "out1"), _dev(out2, "out2")), "cclr_f_transform")
    return out1, out2


def cclr_response_cc(ctx, eri, X, Y, omega, gamma=0.0, tol=1e-10, maxiter=200):
    """<<X;Y>>_{omega + i gamma} in the symmetric CC-CC form (Eq. 15, 17) on the device; eri as for cclr_f_transform.
    Returns (complex, info)."""
    n = ctx.o + ctx.v
    e = _eri_struct_partial(ctx.o, ctx.v, eri, ("ooov", "oovv", "ovvo", "ovvv"))
    res = _lib.Complex()
    info = SolveInfo()
    rc = _lib.load().cclr_response_cc(ctx.handle, C.byref(e), _dev(X, "X", n * n), _dev(Y, "Y", n * n), float(omega),
                                      float(gamma), float(tol), int(maxiter), C.byref(res), C.byref(info))
    if rc not in (0, -4):
        _lib.check(rc, "cclr_response_cc")
    return complex(res.re, res.im), info


def cclr_property(ctx, eta1, eta2, x1, x2):
    """Bilinear eta . x_k for every vector k; returns a Python list of complex."""
    nvec = x1.numel() // ctx.n1
    res = (_lib.Complex * nvec)()
    rc = _lib.load().cclr_property(ctx.handle, _dev(eta1, "eta1", ctx.n1), _dev(eta2, "eta2", ctx.n2),
                                   _dev(x1, "x1", nvec * ctx.n1), _dev(x2, "x2", nvec * ctx.n2), nvec, res)
    _lib.check(rc, "cclr_property")
    return [complex(r.re, r.im) for r in res]


NOALLOC_MAX_VECS = 16


def cclr_property_noalloc(eta1, eta2, x1, x2, out):
    """Bilinear eta . x_k for every vector k WITHOUT any device allocation inside the library (include/cclr.h:
    cclr_property_noalloc): eta1 [n1], eta2 [n2], x1 [nvec, n1], x2 [nvec, n2] and out [nvec] are CUDA tensors of the caller;
    nvec <= NOALLOC_MAX_VECS.  The result stays on the device (no synchronisation).  Calls that overlap on the GPU race."""
    n1, n2 = eta1.numel(), eta2.numel()
    nvec = x1.numel() // n1
    rc = _lib.load().cclr_property_noalloc(_stream(), _dev(eta1, "eta1", n1), _dev(eta2, "eta2", n2), _dev(x1, "x1", nvec * n1),
                                           _dev(x2, "x2", nvec * n2), n1, n2, nvec, _dev(out, "out", nvec))
    _lib.check(rc, "cclr_property_noalloc")
    return out


def cclr_ladder(ctx, x2, out2=None):
    nvec = x2.numel() // ctx.n2
    if out2 is None:
        out2 = torch.empty_like(x2)
    _lib.check(_lib.load().cclr_ladder(ctx.handle, _dev(x2, "x2", nvec * ctx.n2), nvec, _dev(out2, "out2")),
               "cclr_ladder")
    return out2


def cclr_ring(ctx, x2, out2=None):
    if out2 is None:
        out2 = torch.empty_like(x2)
    _lib.check(_lib.load().cclr_ring(ctx.handle, _dev(x2, "x2", ctx.n2), _dev(out2, "out2", ctx.n2)), "cclr_ring")
    return out2


def cclr_zgemm(A, B, C_out, alpha=1.0, beta=0.0, conj_a=False, conj_b=False, b_is_kn=False, M=None, N=None, K=None,
               lda=None, ldb=None, ldc=None, batch=1, sa=0, sb=0, sc=0, three_m=True):
    """C = alpha opA(A) opB(B) + beta C on 2-D (or batched 3-D) row-major tensors; see include/cclr.h.
    three_m: large shapes use the 3M complex product (False: 4M everywhere)."""
    if M is None:
        M, K = A.shape[-2], A.shape[-1]
        N = B.shape[-1] if b_is_kn else B.shape[-2]
        lda, ldb, ldc = A.shape[-1], B.shape[-1], C_out.shape[-1]
        if A.dim() == 3:
            batch = A.shape[0]
            sa, sb, sc = A.shape[1] * A.shape[2], B.shape[1] * B.shape[2], C_out.shape[1] * C_out.shape[2]
    al, be = _lib.Complex(complex(alpha).real, complex(alpha).imag), _lib.Complex(complex(beta).real, complex(beta).imag)
    rc = _lib.load().cclr_zgemm(_stream(), M, N, K, C.byref(al), _dev(A, "A"), lda, int(conj_a), _dev(B, "B"), ldb,
                                int(b_is_kn), int(conj_b), C.byref(be), _dev(C_out, "C"), ldc, batch, sa, sb, sc,
                                int(bool(three_m)))
    _lib.check(rc, "cclr_zgemm")
    return C_out


def cclr_zgemm_oz_eligible(M, N, K):
    """Whether the integer-slice product takes this shape (include/cclr.h: cclr_zgemm_oz)."""
    return M >= 512 and N >= 32 and 512 <= K < (1 << 17) and ((M + 255) // 256) * ((2 * N + 255) // 256) >= 64


def cclr_zgemm_oz(A, B, C_out, alpha=1.0, beta=0.0, conj_a=False, conj_b=False, b_is_kn=False, slices=6, bn=0, reps=1, b_side=False):
    """C = alpha opA(A) opB(B) + beta C on 2-D row-major tensors through the integer-slice product on the INT8 tensor path
    (include/cclr.h: cclr_zgemm_oz).  b_side: B ([K][N]) is the constant operand whose transpose is sliced once (C^T = B^T A^T route).
    Returns (C_out, [ms slicing the constant operand, ms per product incl. slicing the other one, ms of that slicing])."""
    M, K = A.shape
    N = B.shape[1] if b_is_kn else B.shape[0]
    al, be = _lib.Complex(complex(alpha).real, complex(alpha).imag), _lib.Complex(complex(beta).real, complex(beta).imag)
    ms = (C.c_double * 3)()
    rc = _lib.load().cclr_zgemm_oz(_stream(), M, N, K, C.byref(al), _dev(A, "A"), A.shape[1], int(conj_a), _dev(B, "B"), B.shape[1],
                                   int(b_is_kn), int(conj_b), C.byref(be), _dev(C_out, "C"), C_out.shape[1], slices + (100 if b_side else 0), bn, reps, ms)
    _lib.check(rc, "cclr_zgemm_oz")
    return C_out, [ms[0], ms[1], ms[2]]


def cclr_vec_block_lincomb(ctx, Y, X, coef, V, nrm2=None, z=None, P=None):
    """Y[r] = X[r] + sum_j coef[r][j] V[j] for R <= 8 rows in one pass (Y [R, n], X [R, n] / [n] shared / None, coef [R, m],
    V [m, n]); optional nrm2 (float64 CUDA tensor [R]) and P [R, n] = Y / (z - D) with z [R] complex."""
    R, n = Y.shape
    m = V.shape[0]
    ldx = 0 if X is None or X.dim() == 1 else X.shape[1]
    null = C.c_void_p(None)
    rc = _lib.load().cclr_vec_block_lincomb(ctx.handle, R, _dev(Y, "Y"), n, null if X is None else _dev(X, "X"), ldx, _dev(coef, "coef", R * m),
                                            _dev(V, "V"), V.shape[1], m, n, null if nrm2 is None else C.c_void_p(nrm2.data_ptr()),
                                            null if z is None else _dev(z, "z"), null if P is None else _dev(P, "P"), n)
    _lib.check(rc, "cclr_vec_block_lincomb")
    return Y


def cclr_vec_dots(ctx, A, B):
    """out[ia][ib] = <A_ia | B_ib> (sesquilinear) for A [na, n], B [nb, n]; returns a list of lists of complex."""
    na, n = A.shape
    nb = B.shape[0]
    res = (_lib.Complex * (na * nb))()
    _lib.check(_lib.load().cclr_vec_dots(ctx.handle, _dev(A, "A"), na, _dev(B, "B"), nb, n, n, res), "cclr_vec_dots")
    return [[complex(res[i * nb + j].re, res[i * nb + j].im) for j in range(nb)] for i in range(na)]


def cclr_kernel_launches():
    return int(_lib.load().cclr_kernel_launches())


def cclr_fp64_tensor_peak(iters=20000):
    out = C.c_double()
    _lib.check(_lib.load().cclr_fp64_tensor_peak(_stream(), iters, C.byref(out)), "cclr_fp64_tensor_peak")
    return out.value


def cclr_fp64_pipe_probe(mode, iters=20000):
    out = C.c_double()
    _lib.check(_lib.load().cclr_fp64_pipe_probe(_stream(), int(mode), iters, C.byref(out)), "cclr_fp64_pipe_probe")
    return out.value


def cclr_hbm_copy_peak(nbytes=4 << 30):
    out = C.c_double()
    _lib.check(_lib.load().cclr_hbm_copy_peak(_stream(), nbytes, C.byref(out)), "cclr_hbm_copy_peak")
    return out.value
