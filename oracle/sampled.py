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

from .packing import npair, pairs, unpack_pair_axis


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
        self.foo, self.fov, self.fvv = f[:o, :o], f[:o, o:], f[o:, o:]
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
