"""Element-by-element definitions for FULL-SIZE parity checks (TEST INFRASTRUCTURE; see oracle/__init__.py).

At the sizes of BASELINE.json's configs 3-5 the full-tensor oracle (oracle/cclr.py) does not fit host memory, but single
output elements do have plain definitions that can be evaluated one by one from the packed inputs:

  ladder_rows        : the particle-particle ladder T11 of S-Eq. 12 for chosen rows (ab),
                       out[(ab),(ij)] = 1/2 sum_ef W[ab,ef] r2[ef,ij] = sum_{e<f} W[(ab),(ef)] r2[(ef),(ij)];
  sigma_T0_elements  : chosen elements of sigma = A x at T = 0, where every intermediate of S-Eq. 15-28
                        reduces to the bare integral / Fock block of the same name and A is the CISD
                       block <mu|H_N|nu> (Table 1): S-Eq. 11-12 with t1 = t2 = 0.

Pins (tests/test_oracle_sampled.py): both against oracle.cclr.CCLR (itself pinned by the determinant-space definitions) at
small sizes, all elements.
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
