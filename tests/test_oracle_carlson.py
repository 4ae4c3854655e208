"""Pins of the oracle's independent scalar Carlson functions (oracle/cosmo_oracle.c part (4)) and, through them, of
the reading of the paper's closed forms (3.7)-(3.9), (B.1)-(B.3) against the quadrature.  CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest
from scipy import special as sp

import oracle
import paper_formulas as pf


def cx(p):
    return complex(p[0], p[1])


def test_special_values():
    for x in (0.3, 1.0, 7.5):
        lx = np.longdouble(x)
        assert abs(oracle.rf(x, x, x) * np.sqrt(lx) - 1) < 1e-18
        assert abs(oracle.rc(x, x) * np.sqrt(lx) - 1) < 1e-18
        assert abs(oracle.rd(x, x, x) * lx * np.sqrt(lx) - 1) < 1e-18
        assert abs(oracle.rj(x, x, x, x) * lx * np.sqrt(lx) - 1) < 1e-18
    assert abs(float(oracle.rc(0, 0.25)) - math.pi) < 1e-15
    assert abs(float(oracle.rc(2.25, 2)) - math.log(2)) < 1e-16
    assert abs(float(oracle.rc(0.25, -2)) - math.log(2) / 3) < 1e-16          # Cauchy principal value
    # R_F(0,1,2) is the lemniscate constant: Gamma(1/4)^2 / (4 sqrt(2 pi))
    assert abs(float(oracle.rf(0, 1, 2)) - math.gamma(0.25) ** 2 / (4 * math.sqrt(2 * math.pi))) < 1e-15


def test_survey_values(goldens):
    c = goldens["carlson"]
    for a, b, d, v in c["RF"]:
        assert abs(oracle.rf(cx(a), cx(b), cx(d)) - float(v)) < 2e-15
    for a, b, d, p, v in c["RJ"]:
        assert abs(oracle.rj(cx(a), cx(b), cx(d), cx(p)) - float(v)) < 2e-15
    for a, b, d, v in c["RD"]:
        assert abs(oracle.rd(cx(a), cx(b), cx(d)) - float(v)) < 2e-15


def test_homogeneity_and_identities():
    rng = np.random.default_rng(11)
    for _ in range(20):
        x, y, z, p = rng.uniform(0.1, 5, 4)
        lam = rng.uniform(0.2, 9)
        assert abs(oracle.rf(lam * x, lam * y, lam * z) / oracle.rf(x, y, z) - lam ** -0.5) < 1e-15
        assert abs(oracle.rj(lam * x, lam * y, lam * z, lam * p) / oracle.rj(x, y, z, p) - lam ** -1.5) < 1e-15
        # R_D(y,z,x) + R_D(z,x,y) + R_D(x,y,z) = 3/sqrt(xyz)
        s = oracle.rd(y, z, x) + oracle.rd(z, x, y) + oracle.rd(x, y, z)
        assert abs(float(s) * math.sqrt(x * y * z) / 3 - 1) < 1e-15   # (double arithmetic in the test)
        # eq. (2.9): R_D(x,y,z) = R_J(x,y,z,z);  eq. (2.8): R_C(x,y) = R_F(x,y,y)
        assert abs(oracle.rd(x, y, z) / oracle.rj(x, y, z, z) - 1) < 1e-16
        assert abs(oracle.rc(x, y) / oracle.rf(x, y, y) - 1) < 1e-16
        # eq. (2.10): dR_F/dz = -R_D/6, by central differences
        h = 1e-4
        fd = (8 * (oracle.rf(x, y, z + h / 2) - oracle.rf(x, y, z - h / 2)) - (oracle.rf(x, y, z + h) - oracle.rf(x, y, z - h))) / (6 * h)
        assert abs(float(fd) / float(-oracle.rd(x, y, z) / 6) - 1) < 1e-11


def test_against_scipy_and_mpmath():
    rng = np.random.default_rng(12)
    mp.mp.dps = 30
    for n in range(40):
        x, y, z, p = rng.uniform(0.01, 20, 4)
        assert abs(float(oracle.rf(x, y, z)) / sp.elliprf(x, y, z) - 1) < 1e-15
        assert abs(float(oracle.rd(x, y, z)) / sp.elliprd(x, y, z) - 1) < 2e-15
        assert abs(float(oracle.rj(x, y, z, p)) / sp.elliprj(x, y, z, p) - 1) < 4e-15
        assert abs(float(oracle.rc(x, y)) / sp.elliprc(x, y) - 1) < 1e-15
        # conjugate pair + real (the argument pattern of the cosmography formulae)
        w = complex(rng.uniform(-3, 3), rng.uniform(0.1, 3))
        got = oracle.rf(x, w, w.conjugate())
        ref = mp.elliprf(x, mp.mpc(w), mp.mpc(w.conjugate()))
        assert abs(mp.mpf(float(np.real(got))) - mp.re(ref)) / abs(ref) < 1e-15 and abs(np.imag(got)) < 1e-15
        got = oracle.rj(x, w, w.conjugate(), p)
        ref = mp.elliprj(x, mp.mpc(w), mp.mpc(w.conjugate()), p)
        assert abs(mp.mpf(float(np.real(got))) - mp.re(ref)) / abs(ref) < 1e-14
        got = oracle.rd(w, w.conjugate(), x)
        ref = mp.elliprd(mp.mpc(w), mp.mpc(w.conjugate()), x)
        assert abs(mp.mpf(float(np.real(got))) - mp.re(ref)) / abs(ref) < 1e-14


CASES = [(1.0, 0.3, 0.7, 9e-5), (2.5, 0.25, 0.6, 9e-5), (4.0, 0.5, 1.0, 1e-3), (0.05, 0.3, 0.7, 1e-5)]


@pytest.mark.parametrize("z,Om,OL,Or", CASES)
def test_paper_quartic_formulae_equal_quadrature(z, Om, OL, Or):
    """eqs. (3.7)-(3.9) as printed == quadrature of (2.3)-(2.5); (3.7) for every permutation, (3.8) and
    (3.9) for the labellings DESIGN.md uses (i = 'big' for t; (i,..,l) = ('neg', pair, 'big') for d_abs)."""
    ref = oracle.integrals(z, Om, OL, Or, False)[:3].astype(float)
    r = np.array(pf._roots_z(Om, OL, Or))
    real = [n for n in range(4) if abs(r[n].imag) < 1e-9]
    pair = [n for n in range(4) if n not in real]
    big = min(real, key=lambda n: r[n].real)
    neg = [n for n in real if n != big][0]
    for perm in pf.all_perms(4):
        I0 = pf.quartic(z, Om, OL, Or, perm)[0]
        assert abs(I0 - ref[0]) / ref[0] < 1e-14
    T = pf.quartic(z, Om, OL, Or, (big, neg, pair[0], pair[1]))[1]
    assert abs(T - ref[1]) / ref[1] < 1e-14
    A = pf.quartic(z, Om, OL, Or, (neg, pair[0], pair[1], big))[2]
    assert abs(A - ref[2]) / ref[2] < 2e-10          # "prone to small roundoff errors" (double complex here)


@pytest.mark.parametrize("z,Om,OL", [(1.0, 0.3, 0.7), (0.2, 0.25, 0.6), (6.0, 1.3, 0.2), (3.0, 0.1, 1.1)])
def test_paper_cubic_formulae_equal_quadrature(z, Om, OL):
    ref = oracle.integrals(z, Om, OL, 0.0, False)[:3].astype(float)
    for perm in pf.all_perms(3):
        I0, T, A = pf.cubic(z, Om, OL, perm)
        assert abs(I0 - ref[0]) / ref[0] < 1e-14
        assert abs(T - ref[1]) / ref[1] < 1e-13, perm
        assert abs(A - ref[2]) / ref[2] < 1e-11, perm
