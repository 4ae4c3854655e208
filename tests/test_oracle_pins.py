"""Pins of the oracle's quadrature path (oracle/cosmo_oracle.c parts (1)-(3),(5)) to things other than itself:
closed forms, the flat-LCDM hypergeometric/asinh/elementary expressions, Mattig's formula, 40-digit mpmath
goldens (tests/golden/survey_goldens.json), mpmath quadrature at 30 digits, finite differences, lookback<->age.
CPU only."""
import math

import mpmath as mp
import numpy as np
import pytest

import oracle

LD = np.longdouble
C_KM_S = np.longdouble('299792.458')
HUBBLE_GYR = np.longdouble('977.7922216807891')


def rel(a, b):
    return abs(float((LD(a) - LD(b)) / LD(b)))


# ---------------------------------------------------------------- the quadrature rule itself
def test_gk21_rule_exactness():
    x, wk, wg = oracle.gk21_rule()
    assert abs(float(wk.sum() - 2)) < 1e-18 and abs(float(wg.sum() - 2)) < 1e-18
    for k in range(0, 32):
        exact = LD(0) if k % 2 else LD(2) / LD(k + 1)
        assert abs(float((wk * x ** k).sum() - exact)) < 5e-18, k            # Kronrod: degree 3n+1 = 31
        if k <= 19:
            assert abs(float((wg * x ** k).sum() - exact)) < 5e-18, k        # Gauss: degree 2n-1 = 19
    assert abs(float((wk * x ** 32).sum() - LD(2) / 33)) > 1e-12              # and not more
    gx, gw = np.polynomial.legendre.leggauss(10)
    np.testing.assert_allclose(x[1::2].astype(float), gx, rtol=0, atol=1e-15)
    np.testing.assert_allclose(wg[1::2].astype(float), gw, rtol=0, atol=1e-15)


# ---------------------------------------------------------------- closed forms (single-component universes)
ZS = [1e-4, 0.01, 0.3, 1.0, 2.5, 30.0, 1100.0]


@pytest.mark.parametrize("z", ZS)
def test_einstein_de_sitter(z):     # Om = 1: E = x^(3/2)
    x = LD(1) + LD(z)
    I0, T, A = oracle.integrals(z, 1.0, 0.0, 0.0, False)[:3]
    assert rel(I0, 2 * (1 - 1 / np.sqrt(x))) < 2e-18 / min(z, 1)   # D_C = 2(1 - 1/sqrt(1+z)) c/H0
    assert rel(T, LD(2) / 3 * (1 - x ** LD(-1.5))) < 2e-18 / min(z, 1)
    assert rel(A, LD(2) / 3 * (x ** LD(1.5) - 1)) < 2e-18 / min(z, 1)


@pytest.mark.parametrize("z", ZS)
def test_de_sitter(z):              # OL = 1: E = 1
    x = LD(1) + LD(z)
    I0, T, A = oracle.integrals(z, 0.0, 1.0, 0.0, False)[:3]
    assert rel(I0, LD(z)) < 1e-18
    assert rel(T, np.log1p(LD(z))) < 1e-18
    assert rel(A, (x ** 3 - 1) / 3) < 2e-18 / min(z, 1)


@pytest.mark.parametrize("z", ZS)
def test_milne_and_radiation_only(z):
    x = LD(1) + LD(z)
    I0, T, A = oracle.integrals(z, 0.0, 0.0, 0.0, False)[:3]     # Ok = 1: E = x
    assert rel(I0, np.log1p(LD(z))) < 1e-18
    assert rel(T, LD(z) / x) < 1e-18
    assert rel(A, LD(z) * (x + 1) / 2) < 1e-18
    val, _, rc = oracle.observables(z, 0.0, 0.0, 0.0, 70.0, with_grad=False)
    assert rc == 0 and rel(val[1], C_KM_S / 70 * LD(z) * (x + 1) / (2 * x)) < 1e-17   # D_M = d_H sinh(ln x) = d_H (x - 1/x)/2
    I0, T, A = oracle.integrals(z, 0.0, 0.0, 1.0, False)[:3]     # Or = 1: E = x^2
    assert rel(I0, LD(z) / x) < 1e-18
    assert rel(T, LD(z) * (x + 1) / (2 * x * x)) < 1e-18
    assert rel(A, LD(z)) < 1e-18


# ---------------------------------------------------------------- flat LCDM (Om + OL = 1, Or = 0)
@pytest.mark.parametrize("Om", [0.25, 0.0625, 0.875])      # binary fractions: Om + OL == 1 exactly, so Ok == 0 exactly
@pytest.mark.parametrize("z", [0.01, 0.5, 2.0, 50.0])
def test_flat_lcdm_closed_forms(Om, z):
    OL = 1.0 - Om
    I0, T, A = oracle.integrals(z, Om, OL, 0.0, False)[:3]
    mp.mp.dps = 30
    x = mp.mpf(1) + mp.mpf(z)
    m, l = mp.mpf(Om), mp.mpf(OL)
    G = lambda xx: 2 / mp.sqrt(m * xx) * mp.hyp2f1(mp.mpf(1) / 6, mp.mpf(1) / 2, mp.mpf(7) / 6, -l / (m * xx ** 3))
    chi = G(1) - G(x)                                            # hypergeometric form (ref. [2] of the paper)
    tl = 2 / (3 * mp.sqrt(l)) * (mp.asinh(mp.sqrt(l / m)) - mp.asinh(mp.sqrt(l / m) * x ** mp.mpf(-1.5)))
    ab = 2 / (3 * m) * (mp.sqrt(m * x ** 3 + l) - 1)
    assert abs(mp.mpf(float(I0)) - chi) / chi < 1e-15
    assert abs(mp.mpf(float(T)) - tl) / tl < 1e-15
    assert abs(mp.mpf(float(A)) - ab) / ab < 1e-15


@pytest.mark.parametrize("Om", [0.3, 1.6])
@pytest.mark.parametrize("z", [0.1, 1.0, 4.0])
def test_mattig(Om, z):             # OL = Or = 0: open (0.3) and closed (1.6) curvature transform
    val, _, rc = oracle.observables(z, Om, 0.0, 0.0, 70.0, with_grad=False)
    Om_, z_ = LD(Om), LD(z)
    dm = 2 * (Om_ * z_ + (Om_ - 2) * (np.sqrt(1 + Om_ * z_) - 1)) / (Om_ ** 2 * (1 + z_)) * C_KM_S / 70
    assert rc == 0 and rel(val[1], dm) < 5e-17


@pytest.mark.parametrize("Om,OL,Or", [(0.3, 0.7, 0.0), (0.3, 0.7, 9e-5), (0.25, 0.6, 1e-3), (1.2, 0.1, 0.0)])
def test_lookback_plus_age_is_age_today(Om, OL, Or):
    age0 = oracle.age_dimless(0.0, Om, OL, Or)
    for z in (0.1, 1.0, 7.0, 300.0):
        T = oracle.integrals(z, Om, OL, Or, False)[1]
        assert rel(T + oracle.age_dimless(z, Om, OL, Or), age0) < 1e-16
    if Or == 0.0 and abs(Om + OL - 1) < 1e-15:
        assert rel(age0, 2 / (3 * math.sqrt(OL)) * math.asinh(math.sqrt(OL / Om))) < 1e-15


# ---------------------------------------------------------------- goldens from SURVEY.md section 8(c)
def test_goldens_values(goldens):
    c = goldens["config1_cosmology"]
    for row in goldens["config1_table"]:
        val, _, rc = oracle.observables(row["z"], c["Om"], c["OL"], c["Or"], c["H0"], with_grad=False)
        assert rc == 0
        assert rel(val[0], LD(row["DC"])) < 1e-16 and rel(val[3], LD(row["MU"])) < 3e-17   # (one D_C is printed to 17 digits)
        assert rel(val[4] * LD(c["H0"]) / HUBBLE_GYR, LD(row["H0tL"])) < 1e-16
        assert rel(val[5], LD(row["DABS"])) < 1e-16
    for row in goldens["general"]:
        val, _, rc = oracle.observables(row["z"], row["Om"], row["OL"], row["Or"], row["H0"], with_grad=False)
        assert rc == 0
        for name, idx in (("DC", 0), ("DM", 1), ("MU", 3), ("DABS", 5)):
            assert rel(val[idx], LD(row[name])) < 2e-15, (row, name)       # survey printed 15-18 digits
        assert rel(val[4] * LD(row["H0"]) / HUBBLE_GYR, LD(row["H0tL"])) < 2e-15
    # SURVEY.md 8(c)-O3's "non-guaranteed R_J" case (c.c. pair with Re > 0, large z).  The survey printed its inputs
    # rounded, so its 16-digit value is not reproducible from them; the reference is recomputed here with mpmath.
    g = goldens["rj_nonguaranteed"]
    T = oracle.integrals(g["z"], g["Om"], g["OL"], g["Or"], False)[1]
    mp.mp.dps = 30
    m, l = mp.mpf(g["Om"]), mp.mpf(g["OL"])
    ref = mp.quad(lambda x: 1 / (x * mp.sqrt(m * x ** 3 + (1 - m - l) * x ** 2 + l)),
                  [1, 1.5, 2, 2.5, 3, 4, 6, 10, 30, mp.mpf(g["z"]) + 1])
    assert abs(mp.mpf(float(T)) - ref) / ref < 3e-16


def test_goldens_gradients(goldens):
    for row in goldens["gradients"]:
        val, grad, rc = oracle.observables(row["z"], row["Om"], row["OL"], row["Or"], row["H0"])
        assert rc == 0
        for name, idx in (("DC", 0), ("DM", 1), ("MU", 3)):
            for w, wname in enumerate(oracle.WRT):
                assert rel(grad[idx, w], LD(row[name][wname])) < 5e-13, (row["z"], name, wname)


# ---------------------------------------------------------------- independent 30-digit quadrature (mpmath), incl. t and d_abs gradients
@pytest.mark.parametrize("z,Om,OL,Or", [(0.7, 0.31, 0.65, 2.3e-4), (4.2, 0.12, 1.1, 1e-5), (800.0, 0.3, 0.7, 9e-5),
                                        (2.0, 1.3, 0.05, 0.0), (1e-3, 0.3, 0.7, 9e-5)])
def test_against_mpmath_quadrature(z, Om, OL, Or):
    mp.mp.dps = 30
    m, l, r = mp.mpf(Om), mp.mpf(OL), mp.mpf(Or)
    k = 1 - m - l - r
    E2 = lambda x: r * x ** 4 + m * x ** 3 + k * x ** 2 + l
    dE2 = [lambda x: x ** 3 - x ** 2, lambda x: 1 - x ** 2, lambda x: x ** 4 - x ** 2]
    pts = [mp.mpf(1)] + [mp.mpf(p) for p in (2, 10, 100) if p < 1 + z] + [mp.mpf(1) + mp.mpf(z)]
    got = oracle.integrals(z, Om, OL, Or, True)
    for n, power in enumerate((0, -1, 2)):
        ref = mp.quad(lambda x: x ** power / mp.sqrt(E2(x)), pts)
        assert abs(mp.mpf(float(got[n])) - ref) / abs(ref) < 3e-16
        for p in range(3):
            ref = mp.quad(lambda x: -dE2[p](x) * x ** power / (2 * E2(x) ** mp.mpf(1.5)), pts)
            assert abs(mp.mpf(float(got[3 + 3 * n + p])) - ref) / abs(ref) < 3e-16, (n, p)


# ---------------------------------------------------------------- every gradient against central finite differences (long double, Richardson)
@pytest.mark.parametrize("z,Om,OL,Or,H0", [(1.0, 0.3, 0.7, 9e-5, 70.0), (0.05, 0.3, 0.7, 0.0, 70.0),
                                           (3.0, 0.2, 0.9, 1e-3, 65.0), (6.0, 0.9, 0.05, 9e-5, 75.0),
                                           (0.8, 0.3, 0.7 - 9e-5, 9e-5, 70.0)])
def test_gradients_by_finite_differences(z, Om, OL, Or, H0):
    p0 = [LD(v) for v in (z, Om, OL, Or, H0)]
    _, grad, rc = oracle.observables(*p0)
    assert rc == 0

    def f(p):
        return oracle.observables(*p, with_grad=False)[0]

    for w in range(5):
        if w == 3 and Or == 0.0:
            continue                         # one-sided at Or = 0: covered by the golden cubic row
        h = LD(1e-3) * max(abs(p0[w]), LD(1e-2))

        def cd(hh):
            a, b = list(p0), list(p0)
            a[w] += hh
            b[w] -= hh
            return (f(a) - f(b)) / (2 * hh)

        fd = (4 * cd(h / 2) - cd(h)) / 3     # O(h^4)
        for o in range(6):
            scale = max(abs(grad[o, w]), abs(f(p0)[o]) * LD(1e-3))
            assert abs(float((fd[o] - grad[o, w]) / scale)) < 1e-10, (oracle.OBS[o], oracle.WRT[w])


def test_small_curvature_series_matches_closed_form():
    # |Ok| I0^2 just below / above the series switch of sinn_transform must agree
    for Ok in (1e-3, -1e-3, 3e-2, -3e-2):
        a = oracle.observables(1.0, 0.3, 0.7 - Ok, 0.0, 70.0)
        b = oracle.observables(1.0, 0.3 * (1 + 1e-15), 0.7 - Ok, 0.0, 70.0)
        assert rel(a[0][1], b[0][1]) < 1e-14


# ---------------------------------------------------------------- status path and batch API
def test_invalid_and_antipode_status():
    val, _, rc = oracle.observables(8.0, 0.05, 1.5, 0.0, 70.0, with_grad=False)
    assert rc == -1 and np.isnan(float(val[0]))
    val, _, rc = oracle.observables(1.9397181621475743, 1.1668523881503172, 2.7772502139506177, 0.0, 70.0,
                                    with_grad=False)     # closed, loitering: sqrt|Ok| I0 = 9.69 in (3 pi, 4 pi)... sin < 0
    assert rc == 1 and float(val[1]) < 0 and np.isnan(float(val[3]))


def test_batch_matches_scalar():
    rng = np.random.default_rng(0)
    z = rng.uniform(0.01, 3, 50)
    Om = rng.uniform(0.1, 0.5, 50)
    val, grad, st = oracle.observables_batch(z, Om, 0.7, 9e-5, 70.0 * np.ones(1)) if False else \
        oracle.observables_batch(z, Om, np.full(50, 0.7), np.full(50, 9e-5), np.full(50, 70.0))
    for i in (0, 17, 49):
        v, g, rc = oracle.observables(z[i], Om[i], 0.7, 9e-5, 70.0)
        assert rc == st[i] == 0 and np.array_equal(v, val[i]) and np.array_equal(g, grad[i])


# ---------------------------------------------------------------- likelihood
def test_loglike_special_cases_and_brute_force():
    rng = np.random.default_rng(7)
    z = rng.uniform(0.05, 1.4, 10)
    sig = rng.uniform(0.05, 0.2, 10)
    cos = (0.28, 0.69, 9e-5, 68.0)
    val, grad, _ = oracle.observables_batch(z, *cos)
    mu = val[:, 3]
    out = oracle.snia_loglike(z, mu.astype(np.float64), sig, *cos)
    # mu_obs = mu (to double rounding): logL = -sum(ln sigma + 1/2 ln 2pi), gradient ~ 0
    assert abs(float(out[0]) + float(np.sum(np.log(sig)) + 5 * math.log(2 * math.pi))) < 1e-12
    assert np.all(np.abs(out[1:].astype(float)) < 1e-9)
    mu_obs = mu.astype(np.float64) + rng.normal(0, 0.1, 10)
    out = oracle.snia_loglike(z, mu_obs, sig, *cos)
    mp.mp.dps = 30
    ll = mp.mpf(0)
    gr = [mp.mpf(0)] * 4
    for n in range(10):
        r_ = (mp.mpf(mu_obs[n]) - mp.mpf(float(mu[n]))) / mp.mpf(sig[n])
        ll += -r_ * r_ / 2 - mp.log(mp.mpf(sig[n])) - mp.log(2 * mp.pi) / 2
        for p in range(4):
            gr[p] += r_ / mp.mpf(sig[n]) * mp.mpf(float(grad[n, 3, 1 + p]))
    assert abs(mp.mpf(float(out[0])) - ll) < 1e-12
    for p in range(4):
        assert abs(mp.mpf(float(out[1 + p])) - gr[p]) < 1e-10 * max(1, abs(gr[p]))


def test_loglike_against_scipy_density_and_finite_differences():
    """Pins of oracle.snia_loglike that do not retype its formula (mu_obs | mu ~ N(mu, sigma^2)):
    the value against SciPy's normal log-density summed over objects, and all four parameter gradients against Richardson-
    extrapolated central differences of the VALUE (so a wrong sign, a missing 1/sigma^2 or a wrong d mu/d theta fails)."""
    from scipy import stats
    rng = np.random.default_rng(17)
    n = 25
    z = rng.uniform(0.02, 1.5, n)
    sig = rng.uniform(0.05, 0.25, n)
    th = [0.31, 0.66, 9e-5, 68.5]
    one = lambda v: np.array([float(v)])
    mu_of = lambda t: oracle.observables_batch(z, one(t[0]), one(t[1]), one(t[2]), one(t[3]), with_grad=False)[0][:, 3].astype(np.float64)
    mu_obs = mu_of(th) + rng.normal(0, 0.15, n)
    out = oracle.snia_loglike(z, mu_obs, sig, *th)
    ref = stats.norm.logpdf(mu_obs, loc=mu_of(th), scale=sig).sum()
    assert abs(float(out[0]) - ref) <= 1e-12 * abs(ref)
    f = lambda t: oracle.snia_loglike(z, mu_obs, sig, *t, with_grad=False)[0]          # long double
    for p, h in enumerate((2e-4, 2e-4, 2e-5, 2e-2)):
        def cd(hh):
            tp, tm = list(th), list(th)
            tp[p] += hh; tm[p] -= hh
            return (f(tp) - f(tm)) / np.longdouble(2 * hh)
        fd = (4 * cd(h / 2) - cd(h)) / 3                                                # Richardson: O(h^4)
        g = out[1 + p]
        assert abs(float(fd - g)) <= 1e-9 * max(abs(float(g)), 1.0), (p, float(fd), float(g))
    # a single object: the gradient is (residual / sigma^2) * d mu / d theta of the (separately pinned) observables
    o1 = oracle.snia_loglike(z[:1], mu_obs[:1], sig[:1], *th)
    _, g1, _ = oracle.observables(z[0], *th)
    for p in range(4):
        assert abs(float(o1[1 + p]) - (mu_obs[0] - mu_of(th)[0]) / sig[0] ** 2 * float(g1[3, 1 + p])) <= 1e-9 * abs(float(o1[1 + p]))
