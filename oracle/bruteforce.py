"""O1 — brute force on an explicit determinant space (TEST INFRASTRUCTURE; see oracle/__init__.py).

Everything here is the literal definition, nothing is factorised:

  H      = sum_pq h_pq a+_p a_q + 1/4 sum_pqrs <pq||rs> a+_p a+_q a_s a_r ,  h = f - sum_i <pi||qi>
  T      = sum_ai t1[a,i] tau^a_i + 1/4 sum_abij t2[a,b,i,j] tau^ab_ij          (Eq. 8-11)
  Hbar   = exp(-T) H exp(T)                                                      (Eq. 14)
  Omega_mu = <mu|Hbar|R>,  E = <R|Hbar|R>
  A_mu,nu  = <mu|[Hbar, tau_nu]|R>                                               (Table 1)
  xi^X_mu  = <mu|Xbar|R>,  eta^X_nu = <Lambda|[Xbar, tau_nu]|R>,
  F_mu,nu  = <Lambda|[[Hbar, tau_mu], tau_nu]|R>,  <Lambda| = <R| + sum_mu lambda_mu <mu|
  lambda A = -eta0,  eta0_nu = <R|[Hbar, tau_nu]|R>                              (Eq. 13)

Spinors 0..o-1 are occupied in the reference |R>, o..n-1 virtual.  Unique excitations: singles (a,i),
doubles (a<b, i<j); flat order = singles [a,i] row-major, then doubles [(a<b),(i<j)] row-major with the pair
index P(p<q) = q(q-1)/2 + p (the C-ABI's convention, include/cclr.h).
Usable for n = o+v <= ~10.
"""
import itertools
import numpy as np


def pair_list(n):
    """Pairs (p,q), p<q, ordered by P = q(q-1)/2 + p."""
    return [(p, q) for q in range(n) for p in range(q)]


class DetSpace:
    """N-electron determinant space of n spinors with a+_p a_q and a_s a_r as dense matrices."""

    def __init__(self, n, nelec):
        self.n, self.nelec = n, nelec
        masks = [m for m in range(1 << n) if bin(m).count("1") == nelec]
        masks2 = [m for m in range(1 << n) if bin(m).count("1") == nelec - 2]
        self.index = {m: k for k, m in enumerate(masks)}
        index2 = {m: k for k, m in enumerate(masks2)}
        self.dim = d = len(masks)
        d2 = len(masks2)

        def annihilate(mask, p):
            if not (mask >> p) & 1:
                return 0, 0
            sign = -1 if bin(mask & ((1 << p) - 1)).count("1") % 2 else 1
            return sign, mask & ~(1 << p)

        # A[r,s] = a_s a_r : N -> N-2 sector
        self.A = np.zeros((n, n, d2, d))
        for col, m in enumerate(masks):
            for r in range(n):
                s1, m1 = annihilate(m, r)
                if not s1:
                    continue
                for s in range(n):
                    s2, m2 = annihilate(m1, s)
                    if s2:
                        self.A[r, s, index2[m2], col] = s1 * s2
        # E[p,q] = a+_p a_q within the N sector
        self.E = np.zeros((n, n, d, d))
        for col, m in enumerate(masks):
            for q in range(n):
                s1, m1 = annihilate(m, q)
                if not s1:
                    continue
                for p in range(n):
                    if (m1 >> p) & 1:
                        continue
                    sign = -1 if bin(m1 & ((1 << p) - 1)).count("1") % 2 else 1
                    self.E[p, q, self.index[m1 | (1 << p)], col] = s1 * sign
        self.ref = np.zeros(d)
        self.ref[self.index[(1 << nelec) - 1]] = 1.0

    def one_body(self, X):
        return np.tensordot(X, self.E, axes=([0, 1], [0, 1]))

    def two_body(self, V):
        """1/4 sum V[p,q,r,s] a+_p a+_q a_s a_r  (a+_p a+_q = (a_q a_p)^T = A[p,q]^T)."""
        M = np.tensordot(V, self.A, axes=([2, 3], [0, 1]))           # M[p,q] = sum_rs V[pq,rs] a_s a_r
        return 0.25 * np.einsum("pqxy,pqxz->yz", self.A, M)


class BruteForce:
    """Definitions of PAPER.md Table 1 for given f[n,n], V[n,n,n,n] (= <pq||rs>), o occupied spinors."""

    def __init__(self, f, V, o):
        n = f.shape[0]
        self.n, self.o, self.v = n, o, n - o
        self.sp = sp = DetSpace(n, o)
        h = f - np.einsum("piqi->pq", V[:, :o, :, :o])
        self.H = sp.one_body(h) + sp.two_body(V)
        o_, v_ = self.o, self.v
        self.singles = [(a, i) for a in range(v_) for i in range(o_)]
        self.doubles = [(a, b, i, j) for (a, b) in pair_list(v_) for (i, j) in pair_list(o_)]
        # excitation operators tau_mu (dense d x d) for unique mu
        self.tau = []
        for a, i in self.singles:
            self.tau.append(sp.E[o_ + a, i])
        for a, b, i, j in self.doubles:
            self.tau.append(sp.A[o_ + a, o_ + b].T @ sp.A[i, j])
        self.nmu = len(self.tau)
        self.bra = np.array([t @ sp.ref for t in self.tau])          # rows <mu| (real, +-1 entries)

    # ---- amplitude containers -------------------------------------------------------------------------
    def flatten(self, x1, x2):
        """(x1[a,i], x2[a,b,i,j] antisymmetric) -> unique flat vector."""
        out = [x1[a, i] for a, i in self.singles] + [x2[a, b, i, j] for a, b, i, j in self.doubles]
        return np.array(out, dtype=complex)

    def unflatten(self, x):
        o_, v_ = self.o, self.v
        x1 = np.zeros((v_, o_), complex)
        x2 = np.zeros((v_, v_, o_, o_), complex)
        for k, (a, i) in enumerate(self.singles):
            x1[a, i] = x[k]
        for k, (a, b, i, j) in enumerate(self.doubles):
            val = x[len(self.singles) + k]
            x2[a, b, i, j] = x2[b, a, j, i] = val
            x2[b, a, i, j] = x2[a, b, j, i] = -val
        return x1, x2

    def excitation_operator(self, x1, x2):
        """sum_unique x_mu tau_mu  (= sum x1 tau + 1/4 sum x2 tau over all index values)."""
        x = self.flatten(x1, x2)
        return np.tensordot(x, np.array(self.tau), axes=(0, 0))

    # ---- similarity transformation -------------------------------------------------------------------
    @staticmethod
    def _exp_nilpotent(T):
        out = np.eye(T.shape[0], dtype=complex)
        term = np.eye(T.shape[0], dtype=complex)
        for k in range(1, 64):
            term = term @ T / k
            if not np.any(term):
                break
            out = out + term
        return out

    def bar(self, Op, t1, t2):
        T = self.excitation_operator(t1, t2)
        return self._exp_nilpotent(-T) @ Op @ self._exp_nilpotent(T)

    def project(self, vec):
        """<mu|vec> for all unique mu -> (c1, c2)."""
        return self.unflatten(self.bra @ vec)

    # ---- Table 1 ---------------------------------------------------------------------------------------
    def energy_and_residual(self, t1, t2):
        Hb = self.bar(self.H, t1, t2)
        v = Hb @ self.sp.ref
        e = self.sp.ref @ v - self.sp.ref @ self.H @ self.sp.ref
        return e, *self.project(v)                                   # correlation energy, Omega1, Omega2

    def sigma(self, t1, t2, x1, x2):
        Hb = self.bar(self.H, t1, t2)
        R = self.excitation_operator(x1, x2)
        return self.project((Hb @ R - R @ Hb) @ self.sp.ref)

    def jacobian(self, t1, t2):
        """Dense A over unique excitations, A[mu,nu] = <mu|[Hbar,tau_nu]|R>."""
        Hb = self.bar(self.H, t1, t2)
        A = np.zeros((self.nmu, self.nmu), complex)
        for nu, tau in enumerate(self.tau):
            A[:, nu] = self.bra @ ((Hb @ tau - tau @ Hb) @ self.sp.ref)
        return A

    def xi(self, X, t1, t2):
        Xb = self.bar(self.sp.one_body(X), t1, t2)
        return self.bra @ (Xb @ self.sp.ref)

    def eta0(self, t1, t2):
        Hb = self.bar(self.H, t1, t2)
        return np.array([self.sp.ref @ ((Hb @ tau - tau @ Hb) @ self.sp.ref) for tau in self.tau])

    def lam(self, t1, t2):
        """lambda A = -eta0 (Eq. 13), flat unique vector."""
        return np.linalg.solve(self.jacobian(t1, t2).T, -self.eta0(t1, t2))

    def eta(self, X, t1, t2, lam):
        Xb = self.bar(self.sp.one_body(X), t1, t2)
        Lam = self.sp.ref + lam @ self.bra
        return np.array([Lam @ ((Xb @ tau - tau @ Xb) @ self.sp.ref) for tau in self.tau])

    def F(self, t1, t2, lam):
        Hb = self.bar(self.H, t1, t2)
        Lam = self.sp.ref + lam @ self.bra
        Fm = np.zeros((self.nmu, self.nmu), complex)
        comm = [Hb @ tau - tau @ Hb for tau in self.tau]
        for mu in range(self.nmu):
            for nu, tau in enumerate(self.tau):
                Fm[mu, nu] = Lam @ ((comm[mu] @ tau - tau @ comm[mu]) @ self.sp.ref)
        return Fm

    # ---- exact (FCI) references -------------------------------------------------------------------------
    def fci(self):
        """Eigenvalues/vectors of H in the N-electron space (H Hermitian)."""
        return np.linalg.eigh(self.H)

    def sos_response(self, X, Y, z):
        """Exact <<X;Y>>_z by sum over states, Eq. 23/24 with complex z = w + i*gamma:
        sum_n [ <0|X|n><n|Y|0> / (z - w_n) - <0|Y|n><n|X|0> / (z + w_n) ]  (the quantity whose negative is alpha)."""
        w, U = self.fci()
        Xm = U.conj().T @ self.sp.one_body(X) @ U
        Ym = U.conj().T @ self.sp.one_body(Y) @ U
        tot = 0.0
        for k in range(1, len(w)):
            wk = w[k] - w[0]
            tot += Xm[0, k] * Ym[k, 0] / (z - wk) - Ym[0, k] * Xm[k, 0] / (z + wk)
        return tot
