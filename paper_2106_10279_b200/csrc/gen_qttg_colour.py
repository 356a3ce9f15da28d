"""Colour matrix of the five diagrams of (light quark line) + t tbar + gluon (mf_me_qttg.cuh), product side.

Prints CC[d][e] = sum over all colours of conj(C_d) C_e for
  C_0 = (T^b T^a)_{ji} T^b_{kl},  C_1 = (T^a T^b)_{ji} T^b_{kl},  C_2 = T^b_{ji} (T^a T^b)_{kl},
  C_3 = T^b_{ji} (T^b T^a)_{kl},  C_4 = f^{bca} T^b_{ji} T^c_{kl}
from the Gell-Mann matrices, as exact multiples of 1/9 (the entries are rational; C_4 is imaginary relative to the rest).
Run: python gen_qttg_colour.py   (the values are typed into mf_me_qttg.cuh; this script documents where they come from)
"""
import itertools
from fractions import Fraction

import numpy as np


def gell_mann():
    l = np.zeros((8, 3, 3), dtype=complex)
    l[0][0, 1] = l[0][1, 0] = 1
    l[1][0, 1], l[1][1, 0] = -1j, 1j
    l[2][0, 0], l[2][1, 1] = 1, -1
    l[3][0, 2] = l[3][2, 0] = 1
    l[4][0, 2], l[4][2, 0] = -1j, 1j
    l[5][1, 2] = l[5][2, 1] = 1
    l[6][1, 2], l[6][2, 1] = -1j, 1j
    l[7] = np.diag([1, 1, -2]) / np.sqrt(3)
    return l / 2


def main():
    T = gell_mann()
    f = np.zeros((8, 8, 8))
    for a, b, c in itertools.product(range(8), repeat=3):
        f[a, b, c] = (-2j * np.trace((T[a] @ T[b] - T[b] @ T[a]) @ T[c])).real
    TT = np.einsum("bjm,ami->baji", T, T)                     # (T^b T^a)_{ji}
    C = np.zeros((5, 8, 3, 3, 3, 3), dtype=complex)           # [d][a][j][i][k][l]
    C[0] = np.einsum("baji,bkl->ajikl", TT, T)
    C[1] = np.einsum("abji,bkl->ajikl", TT, T)
    C[2] = np.einsum("bji,abkl->ajikl", T, TT)
    C[3] = np.einsum("bji,bakl->ajikl", T, TT)
    C[4] = np.einsum("bca,bji,ckl->ajikl", f, T, T)
    CC = np.einsum("dajikl,eajikl->de", C.conj(), C)
    for d in range(5):
        row = []
        for e in range(5):
            v = CC[d, e]
            re, im = Fraction(v.real * 9).limit_denominator(1000), Fraction(v.imag * 9).limit_denominator(1000)
            row.append("(%s%s)/9" % (re, (" %+si" % im) if im else ""))
        print("  ".join(row))


if __name__ == "__main__":
    main()
