"""Element-by-element definitions for FULL-SIZE parity checks (TEST INFRASTRUCTURE; see oracle/__init__.py).

At the sizes of BASELINE.json's configs 3-5 the full-tensor oracle (oracle/cclr.py) does not fit host memory, but single
output elements do have plain definitions that can be evaluated one by one from the packed inputs:

  ladder_rows        : the particle-particle ladder T11 of S-Eq. 12 for chosen rows (ab),
                       out[(ab),(ij)] = 1/2 sum_ef W[ab,ef] r2[ef,ij] = sum_{e<f} W[(ab),(ef)] r2[(ef),(ij)];
  sigma_T0_elements  : chosen elements of sigma = A x at T = 0, where every intermediate of S-Eq. 15-28
                        reduces to the bare integral / Fock block of the same name and A is the CISD
                       block <mu|H_N|nu> (Table 1): S-Eq. 11-12 with t1 = t2 = 0.

  SampledCCLR        : the same at T != 0 -- slices of every dressed intermediate of S-Eq. 15-28 (rows of W_abef, (b,j)
                       slices of W_mbej / Wbar, rows of W_abej, ...) and chosen elements of sigma = (A - z) x built on them,
                       and (sigma_left_elements) of the left transform l (A - z).

Pins (tests/test_oracle_sampled.py): all against oracle.cclr.CCLR (itself pinned by the determinant-space definitions) at
small sizes, all elements, random complex T.
"""
import numpy as np

from .packing import npair, pack_pair_axes, pairs, unpack_pair_axis


def pair_index(p, q):
    """P(p<q) = q(q-1)/2 + p."""
    return q * (q - 1) // 2 + p


def ladder_rows(w_rows, x2p):
    """w_rows: [nrows][vv] rows (ab) of the packed W_vvvv; x2p: [vv][oo] packed trial doubles -> [nrows][oo]."""
    return np.asarray(w_rows) @ np.asarray(x2p)


def sigma_T0_elements(o, v, f, packed, vvvv_row, x1, x2p, singles, doubles, z=0.0):
    """sigma at T = 0 for the sampled elements.

    f        : [n][n] Fock matrix, n = o + v
    packed   : dict of the packed classes oooo, ooov, oovv (unused at T = 0), ovvo, ovvv as numpy arrays (include/cclr.h)
    vvvv_row : callable P(a<b) -> row [vv] of the packed <ab||ef>  (rows are regenerated on demand by the caller)
    x1, x2p  : trial vector, [v][o] and packed [vv][oo]
    singles  : list of (a, i);  doubles : list of (a, b, i, j) with a < b, i < j
    Returns (list of sigma1 values, list of sigma2 values), each (A x - z x) element.
    """
    oo, vv = npair(o), npair(v)
    foo, fov, fvv = f[:o, :o], f[:o, o:], f[o:, o:]
    r1 = np.asarray(x1).reshape(v, o)
    x2p = np.asarray(x2p).reshape(vv, oo)
    r2 = unpack_pair_axis(unpack_pair_axis(x2p, o, 1), v, 0)               # r2[a,b,i,j], antisymmetric
    oooo = np.asarray(packed["oooo"]).reshape(oo, oo)
    ooov = np.asarray(packed["ooov"]).reshape(oo, o, v)
    ovvo = np.asarray(packed["ovvo"]).reshape(o, v, v, o)
    ovvv = np.asarray(packed["ovvv"]).reshape(o, v, vv)
    ooov_full = unpack_pair_axis(ooov, o, 0)                                # <mn||ie> [m,n,i,e]
    pe, pf = pairs(v)
    pm, pn = pairs(o)

    out1 = []
    for (a, i) in singles:
        s = fvv[a, :] @ r1[:, i] - foo[:, i] @ r1[a, :]                                    # S1, S2
        s += np.einsum("me,em->", fov, r2[a, :, i, :])                                      # S3: f[m,e] r2[a,e,i,m]
        s += np.einsum("me,em->", ovvo[:, a, :, i], r1)                                     # S4: <ma||ei> r1[e,m]
        # S5: 1/2 sum_mef <am||ef> r2[ef,im] = sum_m sum_{e<f} (-<ma||ef>) r2[(ef),i,m]
        s += -np.einsum("mp,pm->", ovvv[:, a, :], r2[pe, pf, i, :])
        # S6: -1/2 sum_mne <mn||ie> r2[ae,mn] = -sum_{m<n} sum_e <mn||ie> r2[a,e,(mn)]
        s += -np.einsum("pe,ep->", ooov[:, i, :], r2[a][:, pm, pn])
        out1.append(s - z * r1[a, i])

    out2 = []
    for (a, b, i, j) in doubles:
        ab, ij = pair_index(a, b), pair_index(i, j)
        s = 0.0 + 0.0j
        # T1: -P(ab) sum_m <mb||ij> r1[a,m],  <mb||ij> = conj <ij||mb>
        s -= np.conj(ooov[ij, :, b]) @ r1[a, :] - np.conj(ooov[ij, :, a]) @ r1[b, :]
        # T2: P(ij) sum_e <ab||ej> r1[e,i],  <ab||ej> = conj <ej||ab> = -conj <je||ab>
        s += -np.conj(ovvv[j, :, ab]) @ r1[:, i] + np.conj(ovvv[i, :, ab]) @ r1[:, j]
        # T5: P(ab) sum_e f[b,e] r2[ae,ij]
        s += fvv[b, :] @ r2[a, :, i, j] - fvv[a, :] @ r2[b, :, i, j]
        # T6: -P(ij) sum_m f[m,j] r2[ab,im]
        s -= foo[:, j] @ r2[a, b, i, :] - foo[:, i] @ r2[a, b, j, :]
        # T7: 1/2 sum_mn <mn||ij> r2[ab,mn] = sum_{m<n}
        s += oooo[:, ij] @ x2p[ab, :]
        # T8: P(ab) P(ij) sum_me <mb||ej> r2[ae,im]
        for (aa, bb, sab) in ((a, b, 1.0), (b, a, -1.0)):
            for (ii, jj, sij) in ((i, j, 1.0), (j, i, -1.0)):
                s += sab * sij * np.einsum("me,em->", ovvo[:, bb, :, jj], r2[aa, :, ii, :])
        # T11: 1/2 sum_ef <ab||ef> r2[ef,ij] = sum_{e<f}
        s += np.asarray(vvvv_row(ab)) @ x2p[:, ij]
        out2.append(s - z * x2p[ab, ij])
    return out1, out2


# ------------------------------------------------------------------------------------------------------------
# T != 0: slices of the dressed intermediates and elements of sigma, from the packed inputs
# ------------------------------------------------------------------------------------------------------------
def _Pij2(fn, i, j):
    """P(ij) g(i, j) = g(i, j) - g(j, i)  (the minus sign is lost in the extracted text)."""
    return fn(i, j) - fn(j, i)


class SampledCCLR:
    """The intermediates of S-Eq. 15-28 one slice at a time, and sigma = (A - z) x of S-Eq. 11-12
     one element at a time, at arbitrary amplitudes T, in the readings of DESIGN.md (the same ones as
    oracle.cclr.CCLR).  Every method is the printed expression with the free indices it names held fixed and every summed
    index running over its FULL range (factors 1/2 as printed; no packed sums), written with numpy contractions over
    slices of the unpacked blocks.  The O(v^4) block <ab||ef> is never held: ``vvvv_row(P(a<b))`` returns one packed row.

    Index conventions as in oracle/cclr.py: V[pq,rs] = <pq||rs>, upper = bra; t1[a,i], t2[a,b,i,j]; r1[a,i], r2[a,b,i,j].
    Blocks held unpacked: oooo[m,n,i,j], ooov[m,n,i,e], oovv[m,n,e,f] (and the same numbers once more as
    oovv_menf[m,e,n,f], a pure copy in another index order), ovvo[m,b,e,j], t2, tau; ovvv stays packed over (e<f) and is
    unpacked per fixed b.  Blocks not stored come from the symmetries of include/cclr.h:
    <am||ef> = -<ma||ef>, <mn||ej> = -<mn||je>, <mb||ij> = conj<ij||mb>, <ab||ej> = conj<ej||ab> = -conj<je||ab>.

    Pins (tests/test_oracle_sampled.py): every slice and every sigma element against oracle.cclr.CCLR at two small sizes
    with random complex T and a non-diagonal Fock matrix.
    """

    def __init__(self, o, v, f, packed, vvvv_row, t1, t2p):
        self.o, self.v = o, v
        oo, vv = npair(o), npair(v)
        f = np.asarray(f)
        self.foo, self.fov, self.fvo, self.fvv = f[:o, :o], f[:o, o:], f[o:, :o], f[o:, o:]
        self.t1 = np.asarray(t1).reshape(v, o)
        self.t2 = unpack_pair_axis(unpack_pair_axis(np.asarray(t2p).reshape(vv, oo), o, 1), v, 0)
        tt = np.einsum("ai,bj->abij", self.t1, self.t1)
        self.tau = self.t2 + tt - tt.transpose(1, 0, 2, 3)                           # S-Eq. 28
        del tt
        self.oooo = unpack_pair_axis(unpack_pair_axis(np.asarray(packed["oooo"]).reshape(oo, oo), o, 1), o, 0)
        self.ooov = unpack_pair_axis(np.asarray(packed["ooov"]).reshape(oo, o, v), o, 0)
        self.oovv = unpack_pair_axis(unpack_pair_axis(np.asarray(packed["oovv"]).reshape(oo, vv), v, 1), o, 0)
        self.oovv_menf = np.ascontiguousarray(self.oovv.transpose(0, 2, 1, 3))       # same numbers, [m,e,n,f]
        self.ovvo = np.asarray(packed["ovvo"]).reshape(o, v, v, o)
        self.ovvv_packed = np.asarray(packed["ovvv"]).reshape(o, v, vv)
        self.vvvv_row = vvvv_row
        self._cache = {}
        self._Fme = self._Fmi = None

    # ---- bare blocks by symmetry -------------------------------------------------------------------------
    def ovvv_b(self, b):
        """<mb||ef> for fixed b -> [m,e,f]."""
        return self._memo(("ovvv", b), lambda: unpack_pair_axis(self.ovvv_packed[:, b, :], self.v, 1))

    def vovv_a(self, a):
        """<am||ef> = -<ma||ef> for fixed a -> [m,e,f]."""
        return -self.ovvv_b(a)

    def vvvv_ab(self, a, b):
        """<ab||ef> for fixed a < b -> [e,f]."""
        return unpack_pair_axis(np.asarray(self.vvvv_row(pair_index(a, b))), self.v, 0)

    def vvvo_ab(self, a, b):
        """<ab||ej> = -conj<je||ab> for fixed a < b -> [e,j]."""
        return -np.conj(self.ovvv_packed[:, :, pair_index(a, b)]).T

    def oovo_j(self, j):
        """<mn||ej> = -<mn||je> for fixed j -> [m,n,e]."""
        return -self.ooov[:, :, j, :]

    def ovoo_b(self, b):
        """<mb||ij> = conj<ij||mb> for fixed b -> [m,i,j]."""
        return np.conj(self.ooov[:, :, :, b]).transpose(2, 0, 1)

    def _memo(self, key, fn):
        if key not in self._cache:
            self._cache[key] = fn()
        return self._cache[key]

    # ---- one-particle intermediates, S-Eq. 15-17 ---------------------------------------
    def Fme(self):
        """F_me[m,e] = f[m,e] + sum_nf <mn||ef> t1[f,n]   (S-Eq. 17) -> [m,e]."""
        if self._Fme is None:
            self._Fme = self.fov + np.einsum("menf,fn->me", self.oovv_menf, self.t1, optimize=True)
        return self._Fme

    def Fmi(self):
        """F_mi[m,i] = f[m,i] + sum_e f[m,e] t1[e,i] + sum_en <mn||ie> t1[e,n] + 1/2 sum_nef <mn||ef> tau[ef,in]  (S-Eq. 15)."""
        if self._Fmi is None:
            self._Fmi = (self.foo + self.fov @ self.t1 + np.einsum("mnie,en->mi", self.ooov, self.t1)
                         + 0.5 * np.einsum("mnef,efin->mi", self.oovv, self.tau, optimize=True))
        return self._Fmi

    def Fae_row(self, a):
        """F_ae[a,e] = f[a,e] - sum_m t1[a,m] f[m,e] + sum_fm t1[f,m] <am||ef> - 1/2 sum_fmn tau[af,mn] <mn||ef>
        (S-Eq. 16 in reading 2) for fixed a -> [e]."""
        return self._memo(("Fae", a), lambda: (
            self.fvv[a] - self.t1[a] @ self.fov + np.einsum("fm,mef->e", self.t1, self.vovv_a(a))
            - 0.5 * np.einsum("fmn,mnef->e", self.tau[a], self.oovv, optimize=True)))

    # ---- two-particle intermediates ----------------------------------------------------------------------
    def Wmnij_col(self, i, j):
        """W_mnij[mn,ij] = <mn||ij> + P(ij) sum_e t1[e,j] <mn||ie> + 1/2 sum_ef tau[ef,ij] <mn||ef>  (S-Eq. 18) -> [m,n]."""
        return self._memo(("Wmnij", i, j), lambda: (
            self.oooo[:, :, i, j]
            + _Pij2(lambda p, q: np.einsum("e,mne->mn", self.t1[:, q], self.ooov[:, :, p, :]), i, j)
            + 0.5 * np.einsum("ef,mnef->mn", self.tau[:, :, i, j], self.oovv, optimize=True)))

    def Wabef_row(self, a, b):
        """W_abef[ab,ef] = <ab||ef> - P(ab) sum_m t1[b,m] <am||ef> + 1/2 sum_mn tau[ab,mn] <mn||ef>  (S-Eq. 22) -> [e,f]."""
        return self._memo(("Wabef", a, b), lambda: (
            self.vvvv_ab(a, b)
            - _Pij2(lambda p, q: np.einsum("m,mef->ef", self.t1[q], self.vovv_a(p)), a, b)
            + 0.5 * np.einsum("mn,mnef->ef", self.tau[a, b], self.oovv, optimize=True)))

    def Wbar_bj(self, b, j):
        """Wbar[mb,ej] = <mb||ej> - sum_nf t2[bf,nj] <mn||ef>  (S-Eq. 23) for fixed (b,j) -> [m,e]."""
        return self._memo(("Wbar", b, j), lambda: (
            self.ovvo[:, b, :, j] - np.einsum("fn,menf->me", self.t2[b, :, :, j], self.oovv_menf, optimize=True)))

    def Wmbej_bj(self, b, j):
        """W_mbej[mb,ej] = <mb||ej> + sum_f t1[f,j] <mb||ef> - sum_n t1[b,n] <mn||ej>
        - sum_nf (t2[fb,jn] + t1[f,j] t1[b,n]) <mn||ef>  (S-Eq. 19) for fixed (b,j) -> [m,e]."""
        return self._memo(("Wmbej", b, j), lambda: (
            self.ovvo[:, b, :, j] + np.einsum("f,mef->me", self.t1[:, j], self.ovvv_b(b))
            - np.einsum("n,mne->me", self.t1[b], self.oovo_j(j))
            - np.einsum("fn,menf->me", self.t2[:, b, j, :] + np.outer(self.t1[:, j], self.t1[b]), self.oovv_menf,
                        optimize=True)))

    def Wmnie_i(self, i):
        """W_mnie[mn,ie] = <mn||ie> + sum_f t1[f,i] <mn||fe>  (S-Eq. 24) for fixed i -> [m,n,e]."""
        return self._memo(("Wmnie", i), lambda: (
            self.ooov[:, :, i, :] + np.einsum("f,mnfe->mne", self.t1[:, i], self.oovv, optimize=True)))

    def Wamef_a(self, a):
        """W_amef[am,ef] = <am||ef> - sum_n t1[a,n] <nm||ef>  (S-Eq. 25) for fixed a -> [m,e,f]."""
        return self._memo(("Wamef", a), lambda: (
            self.vovv_a(a) - np.einsum("n,nmef->mef", self.t1[a], self.oovv, optimize=True)))

    def Wmbij_bij(self, b, i, j):
        """W_mbij[mb,ij] (S-Eq. 20 with the sign of reading 3) for fixed (b,i,j) -> [m]:
        <mb||ij> - sum_e F_me t2[be,ij] - sum_n t1[b,n] W_mnij[mn,ij] + 1/2 sum_ef <mb||ef> tau[ef,ij]
        + P(ij) sum_ne <mn||ie> t2[be,jn] + P(ij) sum_e t1[e,i] Wbar[mb,ej]."""
        return self._memo(("Wmbij", b, i, j), lambda: (
            self.ovoo_b(b)[:, i, j] - self.Fme() @ self.t2[b, :, i, j]
            - np.einsum("n,mn->m", self.t1[b], self.Wmnij_col(i, j))
            + 0.5 * np.einsum("mef,ef->m", self.ovvv_b(b), self.tau[:, :, i, j])
            + _Pij2(lambda p, q: np.einsum("mne,en->m", self.ooov[:, :, p, :], self.t2[b, :, q, :]), i, j)
            + _Pij2(lambda p, q: np.einsum("e,me->m", self.t1[:, p], self.Wbar_bj(b, q)), i, j)))

    def Wabej_abj(self, a, b, j):
        """W_abej[ab,ej] (S-Eq. 21 in reading 4) for fixed (a<b, j) -> [e]:
        <ab||ej> - sum_m F_me t2[ab,mj] + sum_f t1[f,j] W_abef[ab,ef] + 1/2 sum_mn <mn||ej> tau[ab,mn]
        - P(ab) sum_mf <mb||ef> t2[af,mj] - P(ab) sum_m t1[a,m] Wbar[mb,ej]."""
        return self._memo(("Wabej", a, b, j), lambda: (
            self.vvvo_ab(a, b)[:, j] - self.t2[a, b, :, j] @ self.Fme()
            + np.einsum("f,ef->e", self.t1[:, j], self.Wabef_row(a, b))
            + 0.5 * np.einsum("mne,mn->e", self.oovo_j(j), self.tau[a, b])
            - _Pij2(lambda p, q: np.einsum("mef,fm->e", self.ovvv_b(q), self.t2[p, :, :, j]), a, b)
            - _Pij2(lambda p, q: np.einsum("m,me->e", self.t1[p], self.Wbar_bj(q, j)), a, b)))

    # ---- sigma = (A - z) r, S-Eq. 11-12, element by element ------------------------------
    def sigma_elements(self, x1, x2p, singles, doubles, z=0.0):
        """x1 [v][o], x2p packed [vv][oo]; singles: list of (a,i); doubles: list of (a,b,i,j), a<b, i<j.
        Returns (list of sigma1[a,i], list of sigma2[a,b,i,j])."""
        o, v = self.o, self.v
        r1 = np.asarray(x1).reshape(v, o)
        r2 = unpack_pair_axis(unpack_pair_axis(np.asarray(x2p).reshape(npair(v), npair(o)), o, 1), v, 0)
        t2 = self.t2
        rc = {}                                                     # r-dependent one-index intermediates

        def memo(key, fn):
            if key not in rc:
                rc[key] = fn()
            return rc[key]

        def G3(b):   # sum_em W_amef[bm,fe] r1[e,m] -> [f]                                   (inner sum of T3)
            return memo(("G3", b), lambda: np.einsum("mfe,em->f", self.Wamef_a(b), r1))

        def G4(j):   # sum_em W_mnie[nm,je] r1[e,m] -> [n]                                   (inner sum of T4)
            return memo(("G4", j), lambda: np.einsum("nme,em->n", self.Wmnie_i(j), r1))

        def Z9(a):   # sum_nme <nm||fe> r2[ea,mn] -> [f]                                     (inner sum of T9)
            return memo(("Z9", a), lambda: np.einsum("nmfe,emn->f", self.oovv, r2[:, a, :, :], optimize=True))

        def Z10(i):  # sum_mfe <nm||fe> r2[fe,im] -> [n]                                     (inner sum of T10)
            return memo(("Z10", i), lambda: np.einsum("nmfe,fem->n", self.oovv, r2[:, :, i, :], optimize=True))

        out1 = []
        for (a, i) in singles:
            s = self.Fae_row(a) @ r1[:, i] - self.Fmi()[:, i] @ r1[a, :]                        # S1, S2
            s += np.einsum("me,em->", self.Fme(), r2[a, :, i, :])                               # S3
            s += np.einsum("me,em->", self.Wmbej_bj(a, i), r1)                                  # S4 (reading 1)
            s += 0.5 * np.einsum("mef,efm->", self.Wamef_a(a), r2[:, :, i, :])                  # S5
            s -= 0.5 * np.einsum("mne,emn->", self.Wmnie_i(i), r2[a])                           # S6
            out1.append(s - z * r1[a, i])

        out2 = []
        for (a, b, i, j) in doubles:
            s = -_Pij2(lambda p, q: self.Wmbij_bij(q, i, j) @ r1[p, :], a, b)                   # T1
            s += _Pij2(lambda p, q: self.Wabej_abj(a, b, q) @ r1[:, p], i, j)                   # T2
            s += _Pij2(lambda p, q: G3(q) @ t2[p, :, i, j], a, b)                               # T3
            s -= _Pij2(lambda p, q: G4(q) @ t2[a, b, p, :], i, j)                               # T4
            s += _Pij2(lambda p, q: self.Fae_row(q) @ r2[p, :, i, j], a, b)                     # T5
            s -= _Pij2(lambda p, q: self.Fmi()[:, q] @ r2[a, b, p, :], i, j)                    # T6
            s += 0.5 * np.einsum("mn,mn->", self.Wmnij_col(i, j), r2[a, b])                     # T7
            s += _Pij2(lambda p, q: _Pij2(lambda k, l: np.einsum("me,em->", self.Wmbej_bj(q, l), r2[p, :, k, :]),
                                          i, j), a, b)                                          # T8
            s -= 0.5 * _Pij2(lambda p, q: Z9(p) @ t2[:, q, i, j], a, b)                         # T9
            s -= 0.5 * _Pij2(lambda p, q: Z10(p) @ t2[b, a, q, :], i, j)                        # T10
            s += 0.5 * np.einsum("ef,ef->", self.Wabef_row(a, b), r2[:, :, i, j])               # T11
            out2.append(s - z * r2[a, b, i, j])
        return out1, out2

    # ========================================================================================================
    # More slices (other fixed indices) for the left transform, then l (A - z), xi, eta and Omega by elements
    # ========================================================================================================
    def with_amplitudes(self, t1, t2p):
        """A second SampledCCLR on the SAME integrals (shared arrays, nothing copied) at other amplitudes."""
        import copy
        s = copy.copy(self)
        o, v = self.o, self.v
        s.t1 = np.asarray(t1).reshape(v, o)
        s.t2 = unpack_pair_axis(unpack_pair_axis(np.asarray(t2p).reshape(npair(v), npair(o)), o, 1), v, 0)
        tt = np.einsum("ai,bj->abij", s.t1, s.t1)
        s.tau = s.t2 + tt - tt.transpose(1, 0, 2, 3)
        s._cache = {k: val for k, val in self._cache.items() if k[0] == "ovvv"}     # bare-integral slices only
        s._Fme = s._Fmi = None
        return s

    def ovvv_e(self, e):
        """<mb||ef> for fixed e -> [m,b,f] (packed over e<f: sign of the pair, zero for f = e)."""
        def build():
            v = self.v
            fidx = np.arange(v)
            lo, hi = np.minimum(e, fidx), np.maximum(e, fidx)
            sign = np.where(fidx > e, 1.0, np.where(fidx < e, -1.0, 0.0))
            idx = np.where(fidx == e, 0, hi * (hi - 1) // 2 + lo)
            return self.ovvv_packed[:, :, idx] * sign
        return self._memo(("ovvv_e", e), build)

    def vvvv_ef_col(self, e, f):
        """<ab||ef> for fixed e < f, all a,b -> [a,b]:  <ab||ef> = conj<ef||ab>."""
        return np.conj(self.vvvv_ab(e, f))

    def vvvv_e(self, e):
        """<ab||ef> for fixed e, all a,b,f -> [a,b,f] (v rows of the packed block)."""
        def build():
            v = self.v
            out = np.zeros((v, v, v), complex)
            for f in range(v):
                if f != e:
                    out[:, :, f] = self.vvvv_ef_col(min(e, f), max(e, f)) * (1.0 if e < f else -1.0)
            return out
        return self._memo(("vvvv_e", e), build)

    def Fae_col(self, e):
        """F_ae[a,e] (S-Eq. 16, reading 2) for fixed e -> [a]."""
        return self._memo(("Fae_col", e), lambda: (
            self.fvv[:, e] - self.t1 @ self.fov[:, e] - np.einsum("fm,maf->a", self.t1, self.ovvv_e(e))
            - 0.5 * np.einsum("afmn,mnf->a", self.tau, self.oovv[:, :, e, :], optimize=True)))

    def Wmnij_row(self, m, n):
        """W_mnij[mn,ij] (S-Eq. 18) for fixed (m,n) -> [i,j]."""
        def build():
            q = np.einsum("ej,ie->ij", self.t1, self.ooov[m, n])
            return (self.oooo[m, n] + q - q.T + 0.5 * np.einsum("efij,ef->ij", self.tau, self.oovv[m, n], optimize=True))
        return self._memo(("Wmnij_row", m, n), build)

    def Wabef_col(self, e, f):
        """W_abef[ab,ef] (S-Eq. 22) for fixed (e<f), all a,b -> [a,b]."""
        def build():
            q = np.einsum("bm,ma->ab", self.t1, -self.ovvv_packed[:, :, pair_index(e, f)])     # sum_m t1[b,m] <am||ef>
            return (self.vvvv_ef_col(e, f) - (q - q.T)
                    + 0.5 * np.einsum("abmn,mn->ab", self.tau, self.oovv[:, :, e, f], optimize=True))
        return self._memo(("Wabef_col", e, f), build)

    def Wabef_e(self, e):
        """W_abef[ab,ef] (S-Eq. 22) for fixed e, all a,b,f -> [a,b,f]."""
        def build():
            q = np.einsum("bm,maf->abf", self.t1, -self.ovvv_e(e), optimize=True)              # sum_m t1[b,m] <am||ef>
            return (self.vvvv_e(e) - (q - q.transpose(1, 0, 2))
                    + 0.5 * np.einsum("abmn,mnf->abf", self.tau, self.oovv[:, :, e, :], optimize=True))
        return self._memo(("Wabef_e", e), build)

    def Wbar_e(self, e):
        """Wbar[mb,ej] (S-Eq. 23) for fixed e -> [m,b,j]."""
        return self._memo(("Wbar_e", e), lambda: (
            self.ovvo[:, :, e, :] - np.einsum("bfnj,mnf->mbj", self.t2, self.oovv[:, :, e, :], optimize=True)))

    def Wbar_m(self, m):
        """Wbar[mb,ej] (S-Eq. 23) for fixed m -> [b,e,j]."""
        return self._memo(("Wbar_m", m), lambda: (
            self.ovvo[m] - np.einsum("bfnj,nef->bej", self.t2, self.oovv[m], optimize=True)))

    def Wmbej_me(self, m, e):
        """W_mbej[mb,ej] (S-Eq. 19) for fixed (m,e) -> [b,j]."""
        return self._memo(("Wmbej_me", m, e), lambda: (
            self.ovvo[m, :, e, :] + np.einsum("fj,bf->bj", self.t1, self.ovvv_e(e)[m])
            - np.einsum("bn,nj->bj", self.t1, -self.ooov[m, :, :, e])
            - np.einsum("fbjn,nf->bj", self.t2, self.oovv[m, :, e, :], optimize=True)
            - np.einsum("fj,bn,nf->bj", self.t1, self.t1, self.oovv[m, :, e, :], optimize=True)))

    def Wamef_me(self, m, e):
        """W_amef[am,fe] (S-Eq. 25) for fixed m and fixed LAST index e -> [a,f]  (<am||fe> = -<ma||fe> = <ma||ef>)."""
        return self.ovvv_e(e)[m] - np.einsum("an,nf->af", self.t1, self.oovv[:, m, :, e])

    def Wamef_mef(self, m, e, f):
        """W_amef[am,ef] (S-Eq. 25) for fixed (m, e<f) -> [a]."""
        return -self.ovvv_packed[m, :, pair_index(e, f)] - self.t1 @ self.oovv[:, m, e, f]

    def Wmnie_me(self, m, e):
        """W_mnie[nm,je] (S-Eq. 24) as a function of (n,j) for fixed second index m and fixed e -> [n,j]."""
        return self.ooov[:, m, :, e] + np.einsum("fj,nf->nj", self.t1, self.oovv[:, m, :, e])

    def Wmbij_m(self, m):
        """W_mbij[mb,ij] (S-Eq. 20, reading 3) for fixed m -> [b,i,j]."""
        def build():
            o, v = self.o, self.v
            ovvv_m = unpack_pair_axis(self.ovvv_packed[m], v, 1)                                   # <mb||ef> [b,e,f]
            wmnij_m = np.stack([self.Wmnij_row(m, n) if n != m else np.zeros((o, o), complex) for n in range(o)])
            c6 = np.einsum("nie,bejn->bij", self.ooov[m], self.t2, optimize=True)
            c7 = np.einsum("ei,bej->bij", self.t1, self.Wbar_m(m), optimize=True)
            return (np.conj(self.ooov[:, :, m, :]).transpose(2, 0, 1)
                    - np.einsum("e,beij->bij", self.Fme()[m], self.t2, optimize=True)
                    - np.einsum("bn,nij->bij", self.t1, wmnij_m)
                    + 0.5 * np.einsum("bef,efij->bij", ovvv_m, self.tau, optimize=True)
                    + (c6 - c6.transpose(0, 2, 1)) + (c7 - c7.transpose(0, 2, 1)))
        return self._memo(("Wmbij_m", m), build)

    def Wabej_e(self, e):
        """W_abej[ab,ej] (S-Eq. 21, reading 4) for fixed e -> [a,b,j]."""
        def build():
            o, v = self.o, self.v
            vvvo_e = -np.conj(self.ovvv_b(e)).transpose(1, 2, 0)                                   # <ab||ej> [a,b,j]
            c1 = np.einsum("mbf,afmj->abj", self.ovvv_e(e), self.t2, optimize=True)
            c2 = np.einsum("am,mbj->abj", self.t1, self.Wbar_e(e), optimize=True)
            return (vvvo_e - np.einsum("m,abmj->abj", self.Fme()[:, e], self.t2, optimize=True)
                    + np.einsum("fj,abf->abj", self.t1, self.Wabef_e(e), optimize=True)
                    + 0.5 * np.einsum("mnj,abmn->abj", -self.ooov[:, :, :, e], self.tau, optimize=True)
                    - (c1 - c1.transpose(1, 0, 2)) - (c2 - c2.transpose(1, 0, 2)))
        return self._memo(("Wabej_e", e), build)

    def sigma_left_elements(self, y1, y2p, singles, doubles, z=0.0):
        """Elements of the left transform L = l (A - z) for l1[a,i] = l^i_a, l2 packed [vv][oo] (Eq. 13; S-Eq. 13,
        PAPER.md:895-901 in reading 5 of DESIGN.md: the term-by-term adjoint of S-Eq. 11-12 -- each  s[out] += W . r[in]  gives
        L[in] += W . l[out] under <l,s> = sum l1 s1 + 1/4 sum l2 s2, exactly as oracle.cclr.CCLR.sigma_left).
        singles: list of (e,m); doubles: list of (c,d,k,l) with c<d, k<l."""
        o, v = self.o, self.v
        l1 = np.asarray(y1).reshape(v, o)
        l2 = unpack_pair_axis(unpack_pair_axis(np.asarray(y2p).reshape(npair(v), npair(o)), o, 1), v, 0)
        GL = np.einsum("abij,afij->bf", l2, self.t2, optimize=True)          # = -2 G^f_b of S-Eq. 26
        GO = np.einsum("abij,abin->jn", l2, self.t2, optimize=True)          # =  2 G^j_n of S-Eq. 27
        Fme, Fmi = self.Fme(), self.Fmi()
        out1 = []
        for (e, m) in singles:
            s = l1[:, m] @ self.Fae_col(e) - l1[e, :] @ Fmi[m, :]                                   # S1, S2
            s += np.einsum("ai,ai->", l1, self.Wmbej_me(m, e))                                      # S4
            s -= 0.5 * np.einsum("bij,bij->", l2[e], self.Wmbij_m(m))                               # T1
            s += 0.5 * np.einsum("abj,abj->", l2[:, :, m, :], self.Wabej_e(e))                      # T2
            s += 0.5 * np.einsum("bf,bf->", GL, self.Wamef_me(m, e))                                # T3
            s -= 0.5 * np.einsum("jn,nj->", GO, self.Wmnie_me(m, e))                                # T4
            out1.append(s - z * l1[e, m])
        out2 = []
        for (c, d, k, l) in doubles:
            s = _Pij2(lambda p, q: _Pij2(lambda r, t: l1[p, r] * Fme[t, q], k, l), c, d)            # S3
            s += _Pij2(lambda r, t: l1[:, r] @ self.Wamef_mef(t, c, d), k, l)                       # S5
            s -= _Pij2(lambda p, q: l1[p, :] @ (self.ooov[k, l, :, q] + self.t1.T @ self.oovv[k, l, :, q]), c, d)   # S6
            s += _Pij2(lambda p, q: l2[p, :, k, l] @ self.Fae_col(q), c, d)                         # T5
            s -= _Pij2(lambda r, t: l2[c, d, r, :] @ Fmi[t, :], k, l)                               # T6
            s += 0.5 * np.einsum("ij,ij->", l2[c, d], self.Wmnij_row(k, l))                         # T7
            s += _Pij2(lambda p, q: _Pij2(lambda r, t: np.einsum("bj,bj->", l2[p, :, r, :], self.Wmbej_me(t, q)),
                                          k, l), c, d)                                              # T8
            s -= 0.5 * _Pij2(lambda p, q: GL[q, :] @ self.oovv[l, k, :, p], c, d)                   # T9
            s -= 0.5 * _Pij2(lambda r, t: GO[r, :] @ self.oovv[:, t, c, d], k, l)                   # T10
            s += 0.5 * np.einsum("ab,ab->", l2[:, :, k, l], self.Wabef_col(c, d))                   # T11
            out2.append(s - z * l2[c, d, k, l])
        return out1, out2

    def eta0_elements(self, singles, doubles):
        """eta0_nu = <R|[Hbar,tau_nu]|R> = (F_me[i,a], <ij||ab>) (right-hand side of lambda A = -eta0, Eq. 13)."""
        return ([self.Fme()[i, a] for (a, i) in singles], [self.oovv[i, j, a, b] for (a, b, i, j) in doubles])

    # ---- xi^X, S-Eq. 2-3 as printed -----------------------------------------------------
    def xi_elements(self, X, singles, doubles):
        o = self.o
        t1, t2 = self.t1, self.t2
        Xoo, Xov, Xvo, Xvv = X[:o, :o], X[:o, o:], X[o:, :o], X[o:, o:]
        Xt = Xov @ t1                                                     # [m,i]
        tX = t1 @ Xov                                                     # [a,f]
        out1 = [Xvo[a, i] + Xvv[a] @ t1[:, i] - t1[a] @ Xoo[:, i] - t1[a] @ Xt[:, i] + np.einsum("me,em->", Xov, t2[a, :, i, :])
                for (a, i) in singles]
        out2 = []
        for (a, b, i, j) in doubles:
            s = _Pij2(lambda p, q: Xvv[q] @ t2[p, :, i, j], a, b)
            s -= _Pij2(lambda p, q: Xoo[:, q] @ t2[a, b, p, :], i, j)
            s -= _Pij2(lambda p, q: Xt[:, p] @ t2[a, b, :, q], i, j)
            s -= _Pij2(lambda p, q: tX[p] @ t2[:, q, i, j], a, b)
            out2.append(s)
        return out1, out2

    # ---- eta^X, S-Eq. 5-6 as printed, EOM term S-Eq. 7 ---------------------
    def eta_elements(self, X, y1, y2p, singles, doubles, eom=False):
        """lam1[a,i] = lambda^i_a, lam2 packed; X^p_q = X[p,q].  eom: add sum_bj lam2[ab,ij] xi1[b,j] to the singles."""
        o, v = self.o, self.v
        t1, t2 = self.t1, self.t2
        lam1 = np.asarray(y1).reshape(v, o)
        lam2 = unpack_pair_axis(unpack_pair_axis(np.asarray(y2p).reshape(npair(v), npair(o)), o, 1), v, 0)
        Xoo, Xov, Xvv = X[:o, :o], X[:o, o:], X[o:, o:]
        Goo = np.einsum("femn,femi->ni", t2, lam2, optimize=True)
        Gvv = np.einsum("fenm,fanm->ea", t2, lam2, optimize=True)
        tl = t1.T @ lam1                                                  # sum_e t1[e,m] lam1[e,i] -> [m,i]
        lt = lam1 @ t1.T                                                  # sum_m lam1[a,m] t1[e,m] -> [a,e]
        if eom:
            xi1 = np.array(self.xi_elements(X, [(b, j) for b in range(v) for j in range(o)], [])[0]).reshape(v, o)
        out1 = []
        for (a, i) in singles:
            s = (Xov[i, a] + Xvv[:, a] @ lam1[:, i] - Xoo[i] @ lam1[a] - Xov[:, a] @ tl[:, i] - Xov[i] @ lt[a]
                 - 0.5 * Goo[:, i] @ Xov[:, a] - 0.5 * Gvv[:, a] @ Xov[i])
            if eom:
                s += np.einsum("bj,bj->", lam2[a, :, i, :], xi1)
            out1.append(s)
        tXov = t1 @ Xov                                                   # sum_m t1[e,m] Xov[m,b] -> [e,b]
        Xovt = Xov @ t1                                                   # sum_e Xov[j,e] t1[e,m] -> [j,m]
        out2 = []
        for (a, b, i, j) in doubles:
            s = _Pij2(lambda k, l: _Pij2(lambda p, q: lam1[p, k] * Xov[l, q], a, b), i, j)
            s += _Pij2(lambda p, q: lam2[p, :, i, j] @ Xvv[:, q], a, b)
            s -= _Pij2(lambda k, l: lam2[a, b, k, :] @ Xoo[l], i, j)
            s -= _Pij2(lambda p, q: lam2[p, :, i, j] @ tXov[:, q], a, b)
            s -= _Pij2(lambda k, l: lam2[a, b, k, :] @ Xovt[l], i, j)
            out2.append(s)
        return out1, out2

    # ---- Omega(t) by the Gauss quadrature of the Jacobian along the ray ----------------------
    def omega_elements(self, singles, doubles):
        """CCSD residual elements: Omega(t) = Omega(0) + int_0^1 A(s t) . t ds = Omega(0) + 1/2 [A(s1 t).t + A(s2 t).t],
        s = 1/2 -+ 1/(2 sqrt 3) (2-point Gauss-Legendre is exact: s -> A(s t).t is a cubic), Omega(0) = (f[a,i], <ab||ij>).
        Uses sigma_elements at the two scaled amplitude sets; <ab||ij> = conj<ij||ab>."""
        t2p = pack_pair_axes(pack_pair_axes(self.t2, 2), 0)
        acc1 = np.array([self.fvo[a, i] for (a, i) in singles], complex)
        acc2 = np.array([np.conj(self.oovv[i, j, a, b]) for (a, b, i, j) in doubles], complex)
        for s in (0.5 - 0.5 / np.sqrt(3.0), 0.5 + 0.5 / np.sqrt(3.0)):
            g1, g2 = self.with_amplitudes(s * self.t1, s * t2p).sigma_elements(self.t1, t2p, singles, doubles)
            acc1 = acc1 + 0.5 * np.array(g1, complex).reshape(acc1.shape)
            acc2 = acc2 + 0.5 * np.array(g2, complex).reshape(acc2.shape)
        return list(acc1), list(acc2)
