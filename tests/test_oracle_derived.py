"""Pins of the oracle's further derived observables (oracle.derived_batch: D_A, comoving volume, age; SURVEY NEXT-1,
PAPER.md:95): closed forms (Einstein-de Sitter, flat LCDM, Milne), the defining integral of the volume by brute force on
the oracle's own D_M (which is pinned elsewhere), lookback <-> age, and central finite differences of every gradient."""
import math

import numpy as np
import pytest

import oracle

C_KM_S, HUBBLE_GYR = 299792.458, 977.7922216807891
one = lambda v: np.array([float(v)])


def rel(a, b):
    return abs(float(a) - float(b)) / abs(float(b))


def test_einstein_de_sitter():
    z = np.array([0.0, 0.1, 1.0, 7.0, 1100.0])
    val, _, st = oracle.derived_batch(z, one(1.0), one(0.0), one(0.0), one(70.0), with_grad=False)
    dH, tH = C_KM_S / 70, HUBBLE_GYR / 70
    for i, zz in enumerate(z):
        DM = 2 * dH * (1 - 1 / math.sqrt(1 + zz))
        assert rel(val[i, 2], tH * 2 / 3 * (1 + zz) ** -1.5) < 5e-15
        if zz > 0:
            assert rel(val[i, 0], DM / (1 + zz)) < 5e-15      # the reference itself is float64
            assert rel(val[i, 1], 4 * math.pi / 3 * DM ** 3) < 1e-14


@pytest.mark.parametrize("Om", [0.2, 0.3, 0.45])
def test_flat_lcdm_age_and_volume(Om):
    OL = 1 - Om
    z = np.array([0.0, 0.5, 2.0, 20.0])
    val, _, _ = oracle.derived_batch(z, one(Om), one(OL), one(0.0), one(67.0), with_grad=False)
    base, _, _ = oracle.observables_batch(z, one(Om), one(OL), one(0.0), one(67.0), with_grad=False)
    tH = HUBBLE_GYR / 67
    for i, zz in enumerate(z):
        age = tH * 2 / (3 * math.sqrt(OL)) * math.asinh(math.sqrt(OL / Om) * (1 + zz) ** -1.5)
        assert rel(val[i, 2], age) < 5e-15
        # lookback + age(z) = age(0)
        assert rel(float(base[i, 4]) + float(val[i, 2]), val[0, 2]) < 5e-15
        if zz > 0:
            assert rel(val[i, 1], 4 * math.pi / 3 * float(base[i, 1]) ** 3) < 1e-14


def test_milne_volume_closed_form():
    """Om = OL = Or = 0 is outside the method but inside the oracle: Ok = 1, I0 = ln(1+z), D_M = d_H sinh(I0)"""
    z = np.array([0.3, 2.0])
    val, _, st = oracle.derived_batch(z, one(0.0), one(0.0), one(0.0), one(70.0), with_grad=False)
    dH = C_KM_S / 70
    for i, zz in enumerate(z):
        I0 = math.log1p(zz)
        assert rel(val[i, 1], 4 * math.pi * dH ** 3 * (math.sinh(2 * I0) / 2 - I0) / 2) < 1e-14


@pytest.mark.parametrize("Om,OL,Or", [(0.3, 0.5, 9e-5), (0.5, 1.0, 1e-3), (0.3, 0.7003, 0.0)])
def test_volume_is_the_integral_of_DM_squared(Om, OL, Or):
    """V_C = 4 pi int_0^z D_M(z')^2 (c/H0)/E(z') dz' by composite Simpson on the oracle's D_M (open, closed, nearly flat)"""
    zmax, n = 3.0, 2001
    z = np.linspace(0.0, zmax, n)
    z[0] = 1e-12
    base, _, _ = oracle.observables_batch(z, one(Om), one(OL), one(Or), one(70.0), with_grad=False)
    Ok = 1 - Om - OL - Or
    E = np.sqrt(Or * (1 + z) ** 4 + Om * (1 + z) ** 3 + Ok * (1 + z) ** 2 + OL)
    f = 4 * math.pi * base[:, 1].astype(float) ** 2 * (C_KM_S / 70) / E
    h = zmax / (n - 1)
    simpson = h / 3 * (f[0] + f[-1] + 4 * f[1:-1:2].sum() + 2 * f[2:-1:2].sum())
    val, _, _ = oracle.derived_batch(np.array([zmax]), one(Om), one(OL), one(Or), one(70.0), with_grad=False)
    assert rel(val[0, 1], simpson) < 1e-9


@pytest.mark.parametrize("p", [dict(z=1.3, Om=0.3, OL=0.5, Or=9e-5, H0=68.0), dict(z=0.4, Om=0.5, OL=1.0, Or=1e-3, H0=75.0),
                               dict(z=2.5, Om=0.3, OL=0.7, Or=0.0, H0=70.0)])
def test_gradients_by_finite_differences(p):
    def f(**kw):
        q = dict(p); q.update(kw)
        v, _, _ = oracle.derived_batch(np.array([q["z"]]), one(q["Om"]), one(q["OL"]), one(q["Or"]), one(q["H0"]), with_grad=False)
        return v[0].astype(np.float64)
    _, g, _ = oracle.derived_batch(np.array([p["z"]]), one(p["Om"]), one(p["OL"]), one(p["Or"]), one(p["H0"]))
    for k, (nm, h) in enumerate((("z", 1e-5), ("Om", 1e-5), ("OL", 1e-5), ("Or", 1e-7), ("H0", 1e-3))):
        if nm == "Or" and p["Or"] == 0.0:
            fd = (-f(Or=2 * h) + 4 * f(Or=h) - 3 * f(Or=0.0)) / (2 * h)      # one-sided, second order
            tol = 3e-3       # d(age)/dOr is finite at Or = 0 but its next derivative is not: the one-sided difference converges like sqrt(h)
        else:
            fd = (f(**{nm: p[nm] + h}) - f(**{nm: p[nm] - h})) / (2 * h)
            tol = 2e-7
        for i in range(3):
            assert abs(fd[i] - float(g[0, i, k])) <= tol * abs(float(g[0, i, k])), (nm, oracle.DERIVED[i])
