"""O4-O9 — CC-LR on the CPU (TEST INFRASTRUCTURE; see oracle/__init__.py).

sigma = A x, A = CCSD Jacobian (Eq. 14; Table 1), two ways:
  * sigma_fd      : the definition A x = d/de Omega(t + e x)|0 by a 5-point stencil, exact because Omega is a
                    polynomial of degree <= 4 in t;
  * CCLR.sigma    : hand-coded from S-Eq. 11-12 with the intermediates S-Eq. 15-28
                     in the readings listed in DESIGN.md ("Readings of the paper").
Response equations (A - z) t = -xi, z = w + i*gamma (Eq. 19, 183-187 Eq. 20-21), xi / eta
(S-Eq. 2-6), Lambda (Eq. 13), the F.x.y contraction as the second derivative of
the Lagrangian, and the response functions Eq. 15-17.

Conventions: V[p,q,r,s] = <pq||rs>, upper index = bra; t1[a,i], t2[a,b,i,j]; lam1[a,i] =
lambda^i_a, lam2[a,b,i,j] = lambda^ij_ab; all tensors full (unpacked) complex128; dots over UNIQUE elements
(singles + a<b,i<j).  P(pq) g = g - g(p<->q) (the minus sign is lost in the extracted text).
"""
import numpy as np
from . import ccsd
from .packing import flat, unflat


def _Pab(x):
    return x - x.transpose(1, 0, 2, 3)


def _Pij(x):
    return x - x.transpose(0, 1, 3, 2)


# ------------------------------------------------------------------------------------------------------------
# O4: sigma by the definition
# ------------------------------------------------------------------------------------------------------------
def sigma_fd(ints, t1, t2, x1, x2, h=None):
    """A x = [Omega(t-2hx) - 8 Omega(t-hx) + 8 Omega(t+hx) - Omega(t+2hx)] / (12h); exact for a quartic."""
    if h is None:
        nx = np.sqrt(np.linalg.norm(x1) ** 2 + np.linalg.norm(x2) ** 2)
        nt = np.sqrt(np.linalg.norm(t1) ** 2 + np.linalg.norm(t2) ** 2)
        h = max(nt, 1e-1) / max(nx, 1e-300)
    acc1 = acc2 = 0.0
    for c, s in ((1.0, -2.0), (-8.0, -1.0), (8.0, 1.0), (-1.0, 2.0)):
        o1, o2 = ccsd.residual(ints, t1 + s * h * x1, t2 + s * h * x2)
        acc1 = acc1 + c * o1
        acc2 = acc2 + c * o2
    return acc1 / (12 * h), acc2 / (12 * h)


# ------------------------------------------------------------------------------------------------------------
# O5: intermediates and hand-coded sigma
# ------------------------------------------------------------------------------------------------------------
class CCLR:
    """Intermediates of S-Eq. 15-28 for given integrals and ground-state amplitudes, and A x from S-Eq. 11-12."""

    def __init__(self, ints, t1, t2):
        I = self.I = ints
        self.o, self.v = ints.o, ints.v
        self.t1, self.t2 = t1, t2
        tau = self.tau = ccsd.tau(t1, t2)                                          # S-Eq. 28
        vovv = -I.ovvv.transpose(1, 0, 2, 3)                                       # <am||ef> = -<ma||ef>
        oovo = -I.ooov.transpose(0, 1, 3, 2)                                       # <mn||ej> = -<mn||je>
        # S-Eq. 17, 15, 16 (16 read as F^a_e with a = bra, DESIGN reading 2)
        self.Fme = I.fov + np.einsum("mnef,fn->me", I.oovv, t1)
        self.Fmi = (I.foo + np.einsum("me,ei->mi", I.fov, t1) + np.einsum("mnie,en->mi", I.ooov, t1)
                    + 0.5 * np.einsum("mnef,efin->mi", I.oovv, tau))
        self.Fae = (I.fvv - np.einsum("am,me->ae", t1, I.fov) + np.einsum("fm,amef->ae", t1, vovv)
                    - 0.5 * np.einsum("afmn,mnef->ae", tau, I.oovv))
        # S-Eq. 18
        self.Wmnij = (I.oooo + _Pij(np.einsum("ej,mnie->mnij", t1, I.ooov))
                      + 0.5 * np.einsum("efij,mnef->mnij", tau, I.oovv))
        # S-Eq. 22
        self.Wabef = (I.vvvv - _Pab(np.einsum("bm,amef->abef", t1, vovv))
                      + 0.5 * np.einsum("abmn,mnef->abef", tau, I.oovv))
        # S-Eq. 23, 19
        self.Wbar = I.ovvo - np.einsum("bfnj,mnef->mbej", t2, I.oovv)
        self.Wmbej = (I.ovvo + np.einsum("fj,mbef->mbej", t1, I.ovvv) - np.einsum("bn,mnej->mbej", t1, oovo)
                      - np.einsum("fbjn,mnef->mbej", t2 + np.einsum("fj,bn->fbjn", t1, t1), I.oovv))
        # S-Eq. 24, 25
        self.Wmnie = I.ooov + np.einsum("fi,mnfe->mnie", t1, I.oovv)
        self.Wamef = vovv - np.einsum("an,nmef->amef", t1, I.oovv)
        # S-Eq. 20 (sign of the F.t2 term: reading 3)
        self.Wmbij = (I.ovoo - np.einsum("me,beij->mbij", self.Fme, t2)
                      - np.einsum("bn,mnij->mbij", t1, self.Wmnij)
                      + 0.5 * np.einsum("mbef,efij->mbij", I.ovvv, tau)
                      + _Pij(np.einsum("mnie,bejn->mbij", I.ooov, t2))
                      + _Pij(np.einsum("ei,mbej->mbij", t1, self.Wbar)))
        # S-Eq. 21 (sign of the P V t2 term and q -> g: reading 4)
        self.Wabej = (I.vvvo - np.einsum("me,abmj->abej", self.Fme, t2)
                      + np.einsum("fj,abef->abej", t1, self.Wabef)
                      + 0.5 * np.einsum("mnej,abmn->abej", oovo, tau)
                      - _Pab(np.einsum("mbef,afmj->abej", I.ovvv, t2))
                      - _Pab(np.einsum("am,mbej->abej", t1, self.Wbar)))
        self.D1, self.D2 = ccsd.denominators(ints)

    # ---- S-Eq. 11-12 -------------------------------------------------------------------------------------
    def sigma(self, r1, r2, z=0.0):
        """(A - z) r for r1[a,i], r2[a,b,i,j] antisymmetric; z = omega + i*gamma."""
        I, t2 = self.I, self.t2
        s1 = (np.einsum("ae,ei->ai", self.Fae, r1) - np.einsum("mi,am->ai", self.Fmi, r1)      # S1-S2
              + np.einsum("me,aeim->ai", self.Fme, r2)                                          # S3
              + np.einsum("maei,em->ai", self.Wmbej, r1)                                        # S4 (reading 1)
              + 0.5 * np.einsum("amef,efim->ai", self.Wamef, r2)                                # S5
              - 0.5 * np.einsum("mnie,aemn->ai", self.Wmnie, r2))                               # S6
        s2 = -_Pab(np.einsum("mbij,am->abij", self.Wmbij, r1))                                  # T1
        s2 += _Pij(np.einsum("abej,ei->abij", self.Wabej, r1))                                  # T2
        s2 += _Pab(np.einsum("bf,afij->abij", np.einsum("bmfe,em->bf", self.Wamef, r1), t2))    # T3
        s2 -= _Pij(np.einsum("nj,abin->abij", np.einsum("nmje,em->nj", self.Wmnie, r1), t2))    # T4
        s2 += _Pab(np.einsum("be,aeij->abij", self.Fae, r2))                                    # T5
        s2 -= _Pij(np.einsum("mj,abim->abij", self.Fmi, r2))                                    # T6
        s2 += 0.5 * np.einsum("mnij,abmn->abij", self.Wmnij, r2)                                # T7
        ring = np.einsum("mbej,aeim->abij", self.Wmbej, r2)                                     # T8
        s2 += _Pab(_Pij(ring))
        s2 -= 0.5 * _Pab(np.einsum("fa,fbij->abij", np.einsum("nmfe,eamn->fa", I.oovv, r2), t2))   # T9
        s2 -= 0.5 * _Pij(np.einsum("ni,bajn->abij", np.einsum("nmfe,feim->ni", I.oovv, r2), t2))   # T10
        s2 += 0.5 * np.einsum("abef,efij->abij", self.Wabef, r2)                                # T11
        return s1 - z * r1, s2 - z * r2

    # ---- left transform l A (adjoint of S-Eq. 11-12 term by term) ------------------------------------------
    def sigma_left(self, l1, l2, z=0.0):
        """l (A - z) for l1[a,i] = l^i_a, l2[a,b,i,j] = l^ij_ab: the left Jacobian transform of the Lambda / left response
        equations (Eq. 13; S-Eq. 13, whose printed form has three misprints, DESIGN.md
        reading 5).  Written here as the adjoint of sigma(): every term of S-Eq. 11-12 is bilinear in an intermediate and r,
        so with <l, s> = sum l1 s1 + 1/4 sum l2 s2 each term  s[out] += W . r[in]  gives  L[in] += W . l[out]; the three-index
        terms T3, T4, T9, T10 produce the one-index intermediates G of S-Eq. 26-27."""
        I, t2 = self.I, self.t2
        GL = np.einsum("abij,afij->bf", l2, t2)            # = -2 G^f_b of S-Eq. 26
        GO = np.einsum("abij,abin->jn", l2, t2)            # =  2 G^j_n of S-Eq. 27
        L1 = (np.einsum("ai,ae->ei", l1, self.Fae) - np.einsum("ai,mi->am", l1, self.Fmi)            # S1, S2
              + np.einsum("ai,maei->em", l1, self.Wmbej)                                            # S4
              - 0.5 * np.einsum("abij,mbij->am", l2, self.Wmbij)                                    # T1
              + 0.5 * np.einsum("abij,abej->ei", l2, self.Wabej)                                    # T2
              + 0.5 * np.einsum("bf,bmfe->em", GL, self.Wamef)                                      # T3
              - 0.5 * np.einsum("jn,nmje->em", GO, self.Wmnie))                                     # T4
        L2 = _Pab(_Pij(np.einsum("ai,me->aeim", l1, self.Fme)))                                     # S3
        L2 += _Pij(np.einsum("ai,amef->efim", l1, self.Wamef))                                      # S5
        L2 -= _Pab(np.einsum("ai,mnie->aemn", l1, self.Wmnie))                                      # S6
        L2 += _Pab(np.einsum("abij,be->aeij", l2, self.Fae))                                        # T5
        L2 -= _Pij(np.einsum("abij,mj->abim", l2, self.Fmi))                                        # T6
        L2 += 0.5 * np.einsum("abij,mnij->abmn", l2, self.Wmnij)                                    # T7
        L2 += _Pab(_Pij(np.einsum("abij,mbej->aeim", l2, self.Wmbej)))                              # T8
        L2 -= 0.5 * _Pab(np.einsum("af,nmfe->eamn", GL, I.oovv))                                    # T9
        L2 -= 0.5 * _Pij(np.einsum("in,nmfe->feim", GO, I.oovv))                                    # T10
        L2 += 0.5 * np.einsum("abij,abef->efij", l2, self.Wabef)                                    # T11
        return L1 - z * l1, L2 - z * l2

    def solve_lambda_iterative(self, tol=1e-11, maxiter=200):
        """lambda A = -eta0 by a plain preconditioned Krylov iteration on sigma_left (same scheme as solve_iterative)."""
        o, v = self.o, self.v
        d = flat(self.D1 + 0j, self.D2 + 0j)
        rhs = flat(*self.eta0())
        B, S = [], []
        new = -rhs / d
        for it in range(maxiter):
            for _ in range(2):
                for bj in B:
                    new = new - bj * np.vdot(bj, new)
            new = new / np.linalg.norm(new)
            B.append(new)
            S.append(flat(*self.sigma_left(*unflat(new, o, v))))
            Bm, Sm = np.array(B).T, np.array(S).T
            beta = np.linalg.solve(Bm.conj().T @ Sm, -Bm.conj().T @ rhs)
            r = Sm @ beta + rhs
            if np.linalg.norm(r) <= tol * np.linalg.norm(rhs):
                break
            new = -r / d
        return unflat(Bm @ beta, o, v)

    # ---- dense algebra over unique elements (small sizes) ---------------------------------------------------
    def dim(self):
        o, v = self.o, self.v
        return o * v + (o * (o - 1) // 2) * (v * (v - 1) // 2)

    def dense_jacobian(self):
        n = self.dim()
        A = np.zeros((n, n), complex)
        e = np.zeros(n, complex)
        for k in range(n):
            e[k] = 1.0
            A[:, k] = flat(*self.sigma(*unflat(e, self.o, self.v)))
            e[k] = 0.0
        return A

    # ---- Lambda, xi, eta -----------------------------------------------------------------------------------
    def eta0(self):
        """eta0_nu = <R|[Hbar,tau_nu]|R> = (Fme[i,a], <ij||ab>)."""
        return self.Fme.T.copy(), self.I.oovv.transpose(2, 3, 0, 1).copy()

    def solve_lambda_dense(self, A=None):
        """lambda A = -eta0 (Eq. 13) by dense LU over unique elements."""
        A = self.dense_jacobian() if A is None else A
        lam = np.linalg.solve(A.T, -flat(*self.eta0()))
        return unflat(lam, self.o, self.v)

    def xi(self, X):
        """xi^X_mu = <mu|Xbar|R> = Omega[f := X, V := 0](t)  (S-Eq. 1)."""
        return ccsd.residual(self.I.one_body_only(X), self.t1, self.t2)

    def xi_printed(self, X):
        """S-Eq. 2-3 as printed."""
        o = self.o
        t1, t2 = self.t1, self.t2
        Xoo, Xov, Xvo, Xvv = X[:o, :o], X[:o, o:], X[o:, :o], X[o:, o:]
        x1 = (Xvo + Xvv @ t1 - t1 @ Xoo - t1 @ (Xov @ t1) + np.einsum("me,aeim->ai", Xov, t2))
        x2 = (_Pab(np.einsum("bf,afij->abij", Xvv, t2)) - _Pij(np.einsum("mj,abim->abij", Xoo, t2))
              - _Pij(np.einsum("mi,abmj->abij", Xov @ t1, t2))
              - _Pab(np.einsum("af,fbij->abij", t1 @ Xov, t2)))
        return x1, x2

    def eta(self, X, lam1, lam2):
        """S-Eq. 5-6 as printed; X^p_q = X[p,q]; result laid out like amplitudes [a,i], [a,b,i,j]."""
        o = self.o
        t1, t2 = self.t1, self.t2
        Xoo, Xov, Xvo, Xvv = X[:o, :o], X[:o, o:], X[o:, :o], X[o:, o:]
        e1 = (Xov.T + np.einsum("ea,ei->ai", Xvv, lam1) - np.einsum("im,am->ai", Xoo, lam1)
              - np.einsum("ma,em,ei->ai", Xov, t1, lam1) - np.einsum("ie,em,am->ai", Xov, t1, lam1)
              - 0.5 * np.einsum("ni,na->ai", np.einsum("femn,femi->ni", t2, lam2), Xov)
              - 0.5 * np.einsum("ea,ie->ai", np.einsum("fenm,fanm->ea", t2, lam2), Xov))
        e2 = (_Pij(_Pab(np.einsum("ai,jb->abij", lam1, Xov)))
              + _Pab(np.einsum("aeij,eb->abij", lam2, Xvv))
              - _Pij(np.einsum("abim,jm->abij", lam2, Xoo))
              - _Pab(np.einsum("aeij,em,mb->abij", lam2, t1, Xov))
              - _Pij(np.einsum("abim,em,je->abij", lam2, t1, Xov)))
        return e1, e2

    def eta_eom(self, X, lam1, lam2):
        """EOM-eta = eta + (lambda_2 . xi_1 on singles)  (S-Eq. 7)."""
        e1, e2 = self.eta(X, lam1, lam2)
        x1, _ = self.xi(X)
        return e1 + np.einsum("abij,bj->ai", lam2, x1), e2

    # ---- F.x.y as the second derivative of the Lagrangian (PAPER.md:861-879 is unusable) ----
    def lagrangian(self, lam1, lam2, t1, t2):
        e = ccsd.energy(self.I, t1, t2)
        o1, o2 = ccsd.residual(self.I, t1, t2)
        return e + dot(lam1, lam2, o1, o2)

    def xFy(self, lam1, lam2, x1, x2, y1, y2):
        """x.F.y = d2/da db [E + lambda.Omega](t + a x + b y)|0: mixed 4-point stencil + one Richardson step,
        exact for a quartic."""
        nt = max(np.sqrt(np.linalg.norm(self.t1) ** 2 + np.linalg.norm(self.t2) ** 2), 0.1)
        hx = nt / max(np.sqrt(np.linalg.norm(x1) ** 2 + np.linalg.norm(x2) ** 2), 1e-300)
        hy = nt / max(np.sqrt(np.linalg.norm(y1) ** 2 + np.linalg.norm(y2) ** 2), 1e-300)

        def L(a, b):
            return self.lagrangian(lam1, lam2, self.t1 + a * hx * x1 + b * hy * y1,
                                   self.t2 + a * hx * x2 + b * hy * y2)

        def D(h):
            return (L(h, h) - L(h, -h) - L(-h, h) + L(-h, -h)) / (4 * h * h)

        return (4 * D(0.5) - D(1.0)) / 3 / (hx * hy)

    def F_transform(self, lam1, lam2, y1, y2):
        """(F y)_nu = <Lambda|[[Hbar, tau_nu], Y]|R> (F of Table 1; "only t.F is formed") as the
        derivative of the left transform along y:  F y = d/db [eta0 + lambda A](t + b y)|0.  eta0 and every term of sigma_left
        are linear in the intermediates of S-Eq. 15-28, so this is sigma_left with each intermediate replaced by its derivative
        (product rule on S-Eq. 15-28, term by term in the order of __init__), plus the terms in which t2 appears explicitly
        (GL, GO of T3, T4, T9, T10).  The printed S-Eq. 8 ff. are unusable (reading 6); pinned
        against the determinant-space F and against xFy.  Result laid out like amplitudes."""
        I, t1, t2 = self.I, self.t1, self.t2
        E = np.einsum
        vovv = -I.ovvv.transpose(1, 0, 2, 3)
        oovo = -I.ooov.transpose(0, 1, 3, 2)
        yt = E("ai,bj->abij", y1, t1) + E("ai,bj->abij", t1, y1)
        dtau = y2 + yt - yt.transpose(1, 0, 2, 3)                                              # d S-Eq. 28
        dFme = E("mnef,fn->me", I.oovv, y1)                                                     # d S-Eq. 17
        dFmi = E("me,ei->mi", I.fov, y1) + E("mnie,en->mi", I.ooov, y1) + 0.5 * E("mnef,efin->mi", I.oovv, dtau)
        dFae = -E("am,me->ae", y1, I.fov) + E("fm,amef->ae", y1, vovv) - 0.5 * E("afmn,mnef->ae", dtau, I.oovv)
        dWmnij = _Pij(E("ej,mnie->mnij", y1, I.ooov)) + 0.5 * E("efij,mnef->mnij", dtau, I.oovv)
        dWabef = -_Pab(E("bm,amef->abef", y1, vovv)) + 0.5 * E("abmn,mnef->abef", dtau, I.oovv)
        dWbar = -E("bfnj,mnef->mbej", y2, I.oovv)
        dWmbej = (E("fj,mbef->mbej", y1, I.ovvv) - E("bn,mnej->mbej", y1, oovo)
                  - E("fbjn,mnef->mbej", y2 + E("fj,bn->fbjn", y1, t1) + E("fj,bn->fbjn", t1, y1), I.oovv))
        dWmnie = E("fi,mnfe->mnie", y1, I.oovv)
        dWamef = -E("an,nmef->amef", y1, I.oovv)
        dWmbij = (-E("me,beij->mbij", dFme, t2) - E("me,beij->mbij", self.Fme, y2)
                  - E("bn,mnij->mbij", y1, self.Wmnij) - E("bn,mnij->mbij", t1, dWmnij)
                  + 0.5 * E("mbef,efij->mbij", I.ovvv, dtau)
                  + _Pij(E("mnie,bejn->mbij", I.ooov, y2))
                  + _Pij(E("ei,mbej->mbij", y1, self.Wbar)) + _Pij(E("ei,mbej->mbij", t1, dWbar)))
        dWabej = (-E("me,abmj->abej", dFme, t2) - E("me,abmj->abej", self.Fme, y2)
                  + E("fj,abef->abej", y1, self.Wabef) + E("fj,abef->abej", t1, dWabef)
                  + 0.5 * E("mnej,abmn->abej", oovo, dtau)
                  - _Pab(E("mbef,afmj->abej", I.ovvv, y2))
                  - _Pab(E("am,mbej->abej", y1, self.Wbar)) - _Pab(E("am,mbej->abej", t1, dWbar)))
        GL, GO = E("abij,afij->bf", lam2, t2), E("abij,abin->jn", lam2, t2)
        dGL, dGO = E("abij,afij->bf", lam2, y2), E("abij,abin->jn", lam2, y2)
        L1 = (dFme.T                                                                              # d eta0
              + E("ai,ae->ei", lam1, dFae) - E("ai,mi->am", lam1, dFmi) + E("ai,maei->em", lam1, dWmbej)
              - 0.5 * E("abij,mbij->am", lam2, dWmbij) + 0.5 * E("abij,abej->ei", lam2, dWabej)
              + 0.5 * E("bf,bmfe->em", GL, dWamef) - 0.5 * E("jn,nmje->em", GO, dWmnie)
              + 0.5 * E("bf,bmfe->em", dGL, self.Wamef) - 0.5 * E("jn,nmje->em", dGO, self.Wmnie))
        L2 = _Pab(_Pij(E("ai,me->aeim", lam1, dFme)))
        L2 += _Pij(E("ai,amef->efim", lam1, dWamef))
        L2 -= _Pab(E("ai,mnie->aemn", lam1, dWmnie))
        L2 += _Pab(E("abij,be->aeij", lam2, dFae))
        L2 -= _Pij(E("abij,mj->abim", lam2, dFmi))
        L2 += 0.5 * E("abij,mnij->abmn", lam2, dWmnij)
        L2 += _Pab(_Pij(E("abij,mbej->aeim", lam2, dWmbej)))
        L2 -= 0.5 * _Pab(E("af,nmfe->eamn", dGL, I.oovv))
        L2 -= 0.5 * _Pij(E("in,nmfe->feim", dGO, I.oovv))
        L2 += 0.5 * E("abij,abef->efij", lam2, dWabef)
        return L1, L2

    # ---- response equations and functions ---------------------------------------------------------------------
    def solve_dense(self, A, xi1, xi2, z):
        """t(z) = -(A - z)^-1 xi  (Eq. 19-21) by dense LU."""
        n = A.shape[0]
        t = np.linalg.solve(A - z * np.eye(n), -flat(xi1, xi2))
        return unflat(t, self.o, self.v)

    def solve_iterative(self, xi1, xi2, z, tol=1e-10, maxiter=200):
        """Same by a plain preconditioned Krylov subspace method on CCLR.sigma (steps 1-5 of PAPER.md:952-967,
        in the readings of DESIGN.md): trial space b, sigma_j = A b_j, reduced system
        (b^H sigma - z b^H b) beta = -b^H xi, residual r = (sigma - z b) beta + xi, correction r/(z - D)."""
        o, v = self.o, self.v
        d = flat(self.D1 + 0j, self.D2 + 0j)
        rhs = flat(xi1, xi2)
        nrm_rhs = np.linalg.norm(rhs)
        B, S = [], []
        new = -rhs / (d - z)
        for it in range(maxiter):
            for _ in range(2):
                for bj in B:
                    new = new - bj * np.vdot(bj, new)
            new = new / np.linalg.norm(new)
            B.append(new)
            S.append(flat(*self.sigma(*unflat(new, o, v))))
            Bm, Sm = np.array(B).T, np.array(S).T
            G = Bm.conj().T @ Sm - z * (Bm.conj().T @ Bm)
            beta = np.linalg.solve(G, -Bm.conj().T @ rhs)
            r = (Sm - z * Bm) @ beta + rhs
            if np.linalg.norm(r) <= tol * nrm_rhs:
                break
            new = r / (z - d)
        return unflat(Bm @ beta, o, v), dict(iterations=it + 1, residual=np.linalg.norm(r) / nrm_rhs)

    def response_cc_cc(self, solve, X, Y, z, lam1, lam2):
        """<<X;Y>>_z, symmetric CC-CC form, Eq. 15 + Eq. 17 in readings 7-8:
        g(z) = eta^X.t^Y(z) + eta^Y.t^X(-z) + t^X(-z).F.t^Y(z);  <<X;Y>>_z = 1/2 [ g(z) + conj g(-conj z) ].
        ``solve(xi1, xi2, z)`` returns t(z)."""
        def g(zz):
            tY = solve(*self.xi(Y), zz)
            tX = solve(*self.xi(X), -zz)
            return (dot(*self.eta(X, lam1, lam2), *tY) + dot(*self.eta(Y, lam1, lam2), *tX)
                    + self.xFy(lam1, lam2, *tX, *tY))
        return 0.5 * (g(z) + np.conj(g(-np.conj(z))))

    def response_cc_ci(self, solve, X, Y, z, lam1, lam2):
        """CC-CI (EOM-CC) form, Eq. 16: g(z) = EOMeta^X.t^Y(z) - (lam.t^X(-z))(lam.xi^Y) + (X<->Y, z<->-z)."""
        xiX, xiY = self.xi(X), self.xi(Y)
        zc = -np.conj(z)
        return cc_ci_from_vectors(lambda u, w: dot(*u, *w), self.eta_eom(X, lam1, lam2), self.eta_eom(Y, lam1, lam2),
                                  (lam1, lam2), xiX, xiY, solve(*xiY, z), solve(*xiX, -z), solve(*xiY, zc), solve(*xiX, -zc))


def cc_ci_from_vectors(d, etaX, etaY, lam, xiX, xiY, tY_z, tX_mz, tY_zc, tX_mzc):
    """<<X;Y>>_z of Eq. 16 with the symmetriser of Eq. 17 (readings 7-8) from the vectors it is made of:
    g(w) = EOMeta^X.t^Y(w) - (lam.t^X(-w))(lam.xi^Y) + EOMeta^Y.t^X(-w) - (lam.t^Y(w))(lam.xi^X),
    <<X;Y>>_z = 1/2 [ g(z) + conj g(zc) ],  zc = -conj(z).  ``d(u, w)`` is the bilinear dot over unique elements; the vectors
    may be in any representation d understands (full tensors here, packed arrays in the full-size tests)."""
    def g(tY, tX):
        return d(etaX, tY) - d(lam, tX) * d(lam, xiY) + d(etaY, tX) - d(lam, tY) * d(lam, xiX)
    return 0.5 * (g(tY_z, tX_mz) + np.conj(g(tY_zc, tX_mzc)))


def dot(a1, a2, b1, b2):
    """Bilinear (no conjugation) dot over unique elements: sum_ai a1 b1 + sum_{a<b,i<j} a2 b2 = ... + 1/4 full sum."""
    return np.sum(a1 * b1) + 0.25 * np.sum(a2 * b2)

