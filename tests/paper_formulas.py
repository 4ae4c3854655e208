"""The paper's closed forms, transcribed as printed, for tests only.

eqs. (3.7)-(3.9) and the cubic case (B.1)-(B.3) with z1 = 0, roots from
numpy.roots (the "companion matrix" route of PAPER.md:163), complex principal square roots, and the ORACLE's
independent scalar Carlson functions (oracle.rf/rc/rd/rj).  Used to pin (a) that the oracle's quadrature and the
paper's formulae agree (so DESIGN.md's readings of the printed equations are right) and (b) the permutation
invariance stated at PAPER.md:225.  Shares nothing with the CUDA path.
"""
import cmath
import itertools

import numpy as np

import oracle


def _roots_z(Om, OL, Or):
    Ok = 1.0 - Om - OL - Or
    if Or != 0.0:
        rho = np.roots([Or, Om, Ok, 0.0, OL])
    else:
        rho = np.roots([Om, Ok, 0.0, OL])
    # polish on the original polynomial (root accuracy matters)
    c = [Or, Om, Ok, 0.0, OL] if Or != 0.0 else [Om, Ok, 0.0, OL]
    p = np.poly1d(c)
    dp = p.deriv()
    for _ in range(3):
        rho = rho - p(rho) / dp(rho)
    return [complex(r) - 1.0 for r in rho]      # roots of E^2(z): z = x - 1


def quartic(z, Om, OL, Or, perm=(0, 1, 2, 3)):
    """(I0, T, A) by eqs. (3.7), (3.8), (3.9); perm = (i, j, k, l) indexes into the root list."""
    r = _roots_z(Om, OL, Or)
    i, j, k, l = perm
    z1, z2, dz = 0.0, z, z
    X = [cmath.sqrt(z2 - rn) for rn in r]
    Y = [cmath.sqrt(z1 - rn) for rn in r]
    d = lambda a, b: r[b] - r[a]
    d5 = lambda a: -(1.0 + r[a])

    def u(a, b):
        c, e = [m for m in range(4) if m not in (a, b)]
        return X[a] * X[b] * Y[c] * Y[e] + Y[a] * Y[b] * X[c] * X[e]

    uij, uik, uil = u(i, j), u(i, k), u(i, l)
    alpha = Or
    RF = oracle.rf(uij ** 2, uik ** 2, uil ** 2)
    I0 = alpha ** -0.5 * 2 * dz * RF
    # (3.8)
    ui5sq = uij ** 2 - dz ** 2 * d(i, k) * d(i, l) * d5(j) / d5(i)
    qi5sq = (z1 + 1) * (z2 + 1) / ((z1 - r[i]) * (z2 - r[i])) * ui5sq
    si5sq = qi5sq + dz ** 2 * d5(k) * d5(l) * d5(j) / d5(i)
    RJ5 = oracle.rj(uij ** 2, uik ** 2, uil ** 2, ui5sq)
    RC5 = oracle.rc(si5sq, qi5sq)
    T = alpha ** -0.5 * (2 * dz / (r[i] + 1)) * (RF - (dz ** 2 / 3 * d(i, j) * d(i, k) * d(i, l) / d5(i) * RJ5 + RC5))
    # (3.9)
    ui0sq = uij ** 2 - dz ** 2 * d(i, k) * d(i, l)
    qi0sq = ui0sq / ((z1 - r[i]) * (z2 - r[i]))
    si0sq = qi0sq + dz ** 2
    RJ0 = oracle.rj(uij ** 2, uik ** 2, uil ** 2, ui0sq)
    RC0 = oracle.rc(si0sq, qi0sq)
    RD = oracle.rd(uij ** 2, uik ** 2, uil ** 2)
    bnd = X[i] * X[j] * X[k] / X[l] - Y[i] * Y[j] * Y[k] / Y[l]
    A = alpha ** -0.5 * dz * (
        bnd / dz
        + (2 * (r[i] + 1) ** 2 - d(i, j) * d(i, k)) * RF
        + d(j, l) * d(k, l) * (dz ** 2 / 3 * d(i, j) * d(i, k) * RD + X[i] * Y[i] / (X[l] * Y[l] * uil))
        + (sum(r) + 4) * (dz ** 2 / 3 * d(i, j) * d(i, k) * d(i, l) / (-1.0) * RJ0 + RC0))
    return complex(I0), complex(T), complex(A)


def cubic(z, Om, OL, perm=(0, 1, 2)):
    """(I0, T, A) by eqs. (B.1), (B.2), (B.3)  (Or = 0)."""
    r = _roots_z(Om, OL, 0.0)
    i, j, k = perm
    z1, z2, dz = 0.0, z, z
    X = [cmath.sqrt(z2 - rn) for rn in r]
    Y = [cmath.sqrt(z1 - rn) for rn in r]
    d = lambda a, b: r[b] - r[a]

    def u(a):
        b, c = [m for m in range(3) if m != a]
        return X[a] * Y[b] * Y[c] + Y[a] * X[b] * X[c]

    ui, uj, uk = u(i), u(j), u(k)
    alpha = Om
    RF = oracle.rf(ui ** 2, uj ** 2, uk ** 2)
    I0 = alpha ** -0.5 * 2 * dz * RF
    ui5sq = ui ** 2 + dz ** 2 * (r[i] + 1)
    s5 = Y[0] * Y[1] * Y[2] * (z2 + 1) + X[0] * X[1] * X[2] * (z1 + 1)
    qi5sq = (z1 + 1) * (z2 + 1) * ui5sq
    T = alpha ** -0.5 * 2 * dz * (dz ** 2 / 3 * oracle.rj(ui ** 2, uj ** 2, uk ** 2, ui5sq) + oracle.rc(s5 ** 2, qi5sq))
    RD = oracle.rd(uj ** 2, uk ** 2, ui ** 2)
    A = alpha ** -0.5 * (2 * dz / 3) * (
        (X[0] * X[1] * X[2] - Y[0] * Y[1] * Y[2]) / dz
        + (3 * (r[i] + 1) ** 2 - d(i, j) * d(i, k)) * RF
        + 2 * (sum(r) + 3) * (dz ** 2 / 3 * d(i, j) * d(i, k) * RD + X[i] * Y[i] / ui))
    return complex(I0), complex(T), complex(A)


def all_perms(m):
    return list(itertools.permutations(range(m)))
