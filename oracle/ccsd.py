"""O2/O3 — tensor-level CCSD energy E(t), residual Omega(t) and ground state (TEST INFRASTRUCTURE).

The paper does not print the ground-state equations; it cites its ref. 47 for the Kramers-unrestricted CCSD
(PAPER.md:205).  These are the textbook spin-orbital CCSD equations (Stanton, Gauss, Watts, Bartlett,
J. Chem. Phys. 94, 4334 (1991)) written as a residual (no division by denominators, full Fock matrix, so a
non-diagonal f is fine) and with the bra/ket placement needed for complex integrals: amplitudes are never
conjugated (Omega is holomorphic in t).  Pinned by tests/test_oracle_ccsd.py against oracle/bruteforce.py.

Conventions: V[p,q,r,s] = <pq||rs> (upper = bra), f[p,q] = <p|f|q>, t1[a,i], t2[a,b,i,j].
``ints`` is an ``Integrals`` holding full (unpacked) blocks named by their index spaces.
"""
import numpy as np


class Integrals:
    """Full blocks of f and <pq||rs> with o occupied / v virtual spinors.

    Stored: foo, fov, fvo, fvv and oooo, ooov, oovv, ovvo, ovvv, vvvv, vvoo, ovoo, vvvo (the last three are
    the Hermitian conjugates of oovv, ooov, ovvv: V[pq,rs] = conj(V[rs,pq])).  Index order = the block name.
    """

    def __init__(self, o, v, f, oooo, ooov, oovv, ovvo, ovvv, vvvv):
        self.o, self.v = o, v
        self.f = f
        self.foo, self.fov, self.fvo, self.fvv = f[:o, :o], f[:o, o:], f[o:, :o], f[o:, o:]
        self.oooo, self.ooov, self.oovv, self.ovvo, self.ovvv, self.vvvv = oooo, ooov, oovv, ovvo, ovvv, vvvv
        self.vvoo = oovv.transpose(2, 3, 0, 1).conj()     # <ab||ij> = conj <ij||ab>
        self.ovoo = ooov.transpose(2, 3, 0, 1).conj()     # <mb||ij> = conj <ij||mb>
        self.vvvo = -ovvv.transpose(2, 3, 1, 0).conj()    # <ab||ej> = conj <ej||ab> = -conj <je||ab>

    @classmethod
    def from_full(cls, f, V, o):
        O, Vv = slice(0, o), slice(o, None)
        return cls(o, f.shape[0] - o, f, V[O, O, O, O], V[O, O, O, Vv], V[O, O, Vv, Vv], V[O, Vv, Vv, O],
                   V[O, Vv, Vv, Vv], V[Vv, Vv, Vv, Vv])

    def one_body_only(self, X):
        """Integrals with f := X and V := 0 (used for xi^X = Omega[f:=X, V:=0])."""
        o, v = self.o, self.v
        z = lambda *s: np.zeros(s, complex)
        return Integrals(o, v, X, z(o, o, o, o), z(o, o, o, v), z(o, o, v, v), z(o, v, v, o), z(o, v, v, v),
                         z(v, v, v, v))


def tau(t1, t2, fac=1.0):
    """tau = t2 + fac * (t1[a,i]t1[b,j] - t1[b,i]t1[a,j])   (S-Eq. 28, for fac = 1)."""
    tt = np.einsum("ai,bj->abij", t1, t1)
    return t2 + fac * (tt - tt.transpose(1, 0, 2, 3))


def energy(ints, t1, t2):
    """Correlation energy  E = f[i,a] t1[a,i] + 1/4 <ij||ab> tau[a,b,i,j]."""
    return np.einsum("ia,ai->", ints.fov, t1) + 0.25 * np.einsum("ijab,abij->", ints.oovv, tau(t1, t2))


def residual(ints, t1, t2):
    """Omega1[a,i] = <a i|Hbar|R>, Omega2[a,b,i,j] = <ab ij|Hbar|R>  (Stanton et al. 1991, Eqs. 1-13)."""
    I = ints
    ttil = tau(t1, t2, 0.5)
    ta = tau(t1, t2, 1.0)
    # one-particle intermediates (full f: no (1-delta) factors because nothing is divided out)
    Fae = (I.fvv - 0.5 * np.einsum("me,am->ae", I.fov, t1)
           + np.einsum("fm,mafe->ae", t1, I.ovvv)
           - 0.5 * np.einsum("afmn,mnef->ae", ttil, I.oovv))
    Fmi = (I.foo + 0.5 * np.einsum("ei,me->mi", t1, I.fov)
           + np.einsum("en,mnie->mi", t1, I.ooov)
           + 0.5 * np.einsum("efin,mnef->mi", ttil, I.oovv))
    Fme = I.fov + np.einsum("fn,mnef->me", t1, I.oovv)
    # two-particle intermediates (Stanton's CCSD ones, 1/4 factors)
    tmp = np.einsum("ej,mnie->mnij", t1, I.ooov)
    Wmnij = I.oooo + tmp - tmp.transpose(0, 1, 3, 2) + 0.25 * np.einsum("efij,mnef->mnij", ta, I.oovv)
    # <am||ef> = -<ma||ef>
    tmp = -np.einsum("bm,maef->abef", t1, I.ovvv)                    # sum_m t1[b,m] <am||ef>
    Wabef = I.vvvv - (tmp - tmp.transpose(1, 0, 2, 3)) + 0.25 * np.einsum("abmn,mnef->abef", ta, I.oovv)
    # <mn||ej> = -<mn||je>
    Wmbej = (I.ovvo + np.einsum("fj,mbef->mbej", t1, I.ovvv)
             + np.einsum("bn,mnje->mbej", t1, I.ooov)
             - np.einsum("fbjn,mnef->mbej", 0.5 * t2 + np.einsum("fj,bn->fbjn", t1, t1), I.oovv))

    # ---- singles
    O1 = (I.fvo + np.einsum("ei,ae->ai", t1, Fae) - np.einsum("am,mi->ai", t1, Fmi)
          + np.einsum("aeim,me->ai", t2, Fme)
          - np.einsum("fn,naif->ai", t1, -I.ovvo.transpose(0, 1, 3, 2))   # <na||if> = -<na||fi>
          - 0.5 * np.einsum("efim,maef->ai", t2, I.ovvv)
          - 0.5 * np.einsum("aemn,nmei->ai", t2, -I.ooov.transpose(0, 1, 3, 2)))  # <nm||ei> = -<nm||ie>
    # ---- doubles
    O2 = I.vvoo.copy()
    tmp = np.einsum("aeij,be->abij", t2, Fae - 0.5 * np.einsum("bm,me->be", t1, Fme))
    O2 += tmp - tmp.transpose(1, 0, 2, 3)
    tmp = np.einsum("abim,mj->abij", t2, Fmi + 0.5 * np.einsum("ej,me->mj", t1, Fme))
    O2 -= tmp - tmp.transpose(0, 1, 3, 2)
    O2 += 0.5 * np.einsum("abmn,mnij->abij", ta, Wmnij)
    O2 += 0.5 * np.einsum("efij,abef->abij", ta, Wabef)
    tmp = (np.einsum("aeim,mbej->abij", t2, Wmbej)
           - np.einsum("ei,am,mbej->abij", t1, t1, I.ovvo))
    O2 += tmp - tmp.transpose(1, 0, 2, 3) - tmp.transpose(0, 1, 3, 2) + tmp.transpose(1, 0, 3, 2)
    tmp = np.einsum("ei,abej->abij", t1, I.vvvo)
    O2 += tmp - tmp.transpose(0, 1, 3, 2)
    tmp = np.einsum("am,mbij->abij", t1, I.ovoo)
    O2 -= tmp - tmp.transpose(1, 0, 2, 3)
    return O1, O2


def denominators(ints):
    """D1[a,i] = eps_a - eps_i, D2[a,b,i,j] = eps_a + eps_b - eps_i - eps_j from diag(f)."""
    eo = np.real(np.diag(ints.foo))
    ev = np.real(np.diag(ints.fvv))
    D1 = ev[:, None] - eo[None, :]
    D2 = ev[:, None, None, None] + ev[None, :, None, None] - eo[None, None, :, None] - eo[None, None, None, :]
    return D1, D2


def solve_ground_state(ints, tol=1e-10, maxiter=200, ndiis=8, verbose=False):
    """O3: Omega(t) = 0 by quasi-Newton steps t -= Omega/D with DIIS; converged when ||Omega||_2 <= tol
    (2-norm over all elements of Omega1 and the full antisymmetric Omega2)."""
    o, v = ints.o, ints.v
    D1, D2 = denominators(ints)
    t1 = np.zeros((v, o), complex)
    t2 = np.zeros((v, v, o, o), complex)
    hist_t, hist_e = [], []
    for it in range(maxiter):
        O1, O2 = residual(ints, t1, t2)
        nrm = np.sqrt(np.linalg.norm(O1) ** 2 + np.linalg.norm(O2) ** 2)
        if verbose:
            print(f"ccsd it {it:3d} |Omega| = {nrm:.3e}  E = {energy(ints, t1, t2):.12f}")
        if nrm <= tol:
            return t1, t2, dict(iterations=it, residual=nrm, converged=True)
        if not np.isfinite(nrm) or nrm > 1e6:
            break
        t1 = t1 - O1 / D1
        t2 = t2 - O2 / D2
        hist_t.append(np.concatenate([t1.ravel(), t2.ravel()]))
        hist_e.append(np.concatenate([(O1 / D1).ravel(), (O2 / D2).ravel()]))
        hist_t, hist_e = hist_t[-ndiis:], hist_e[-ndiis:]
        m = len(hist_t)
        if m >= 2:
            B = np.zeros((m + 1, m + 1), complex)
            for p in range(m):
                for q in range(m):
                    B[p, q] = np.vdot(hist_e[p], hist_e[q])
            B[m, :m] = B[:m, m] = -1.0
            rhs = np.zeros(m + 1, complex)
            rhs[m] = -1.0
            try:
                c = np.linalg.solve(B, rhs)[:m]
                tn = sum(ci * ti for ci, ti in zip(c, hist_t))
                t1 = tn[: v * o].reshape(v, o)
                t2 = tn[v * o:].reshape(v, v, o, o)
            except np.linalg.LinAlgError:
                pass
    return t1, t2, dict(iterations=maxiter, residual=nrm, converged=False)
