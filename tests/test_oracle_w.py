"""Pins for the oracle's chi family with extra constant-w components (oracle.w_chi_batch; PAPER.md:82 fn.4):
E^2 = Or x^4 + Om x^3 + (Ok + Ow13) x^2 + Ow23 x + OL.  Closed forms of single- and two-component universes, reduction to
the pinned LCDM oracle, the curvature convention (Ow13 behaves like curvature in E but not in sinn), a different quadrature
routine on the defining integral, and finite differences of d/dz.
"""
import math

import numpy as np

import oracle

C_KM_S = 299792.458
H0 = 70.0
DH = C_KM_S / H0
Z = np.array([1e-3, 0.1, 0.5, 1.0, 2.5, 9.0, 99.0])
X = 1.0 + Z
OBS = {n: i for i, n in enumerate(oracle.OBSW)}


def rel(a, b):
    a = np.asarray(a, dtype=np.float64); b = np.asarray(b, dtype=np.float64)
    return np.abs(a - b) / np.abs(b)


def test_reduces_to_the_lcdm_oracle():
    for Om, OL, Or in ((0.3, 0.7, 0.0), (0.3, 0.6, 9e-5), (0.2, 0.9, 1e-3)):
        v, d, s = oracle.w_chi_batch(Z, Om, OL, Or, 0.0, 0.0, H0)
        v0, g0, s0 = oracle.observables_batch(Z, [Om], [OL], [Or], [H0], True)
        assert (s == 0).all()
        assert rel(v, v0[:, :4]).max() < 1e-17 and rel(d, g0[:, :4, 0]).max() < 1e-17


def _mp(f):
    """closed form f(z) evaluated with 30 digits on the exact double z (float64 forms like sqrt(x) - 1 cancel at small z)"""
    import mpmath as mp
    mp.mp.dps = 30
    return np.array([float(f(mp, mp.mpf(float(z)))) for z in Z])


def test_pure_w_minus_two_thirds():
    """E^2 = x: I0 = 2 (sqrt(x) - 1), flat."""
    v, d, s = oracle.w_chi_batch(Z, 0.0, 0.0, 0.0, 0.0, 1.0, H0)
    ref = DH * _mp(lambda mp, z: 2 * (mp.sqrt(1 + z) - 1))
    assert rel(v[:, OBS["DC"]], ref).max() < 5e-16
    assert rel(v[:, OBS["DM"]], ref).max() < 5e-16
    assert rel(v[:, OBS["DL"]], X * ref).max() < 5e-16
    assert rel(v[:, OBS["MU"]], 5 * np.log10(X * ref) + 25).max() < 5e-16
    assert rel(d[:, OBS["DC"]], DH / np.sqrt(X)).max() < 5e-16


def test_pure_w_minus_one_third_is_flat_unlike_milne():
    """E^2 = x^2 with Ok = 0: I0 = ln x and D_M = D_C; the Milne universe has the same E but D_M = dH sinh(ln x)."""
    v, d, s = oracle.w_chi_batch(Z, 0.0, 0.0, 0.0, 1.0, 0.0, H0)
    lnx = _mp(lambda mp, z: mp.log1p(z))
    assert rel(v[:, OBS["DC"]], DH * lnx).max() < 5e-16
    assert rel(v[:, OBS["DM"]], DH * lnx).max() < 5e-16
    vm, _, _ = oracle.w_chi_batch(Z, 0.0, 0.0, 0.0, 0.0, 0.0, H0)          # Milne: Ok = 1
    assert rel(vm[:, OBS["DC"]], DH * lnx).max() < 5e-16
    assert rel(vm[:, OBS["DM"]], DH * _mp(lambda mp, z: mp.sinh(mp.log1p(z)))).max() < 5e-16


def test_two_component_closed_forms():
    a = 0.35
    # Ow23 = a, OL = 1 - a: E^2 = a x + 1 - a
    v, _, _ = oracle.w_chi_batch(Z, 0.0, 1.0 - a, 0.0, 0.0, a, H0)
    am = lambda mp: mp.mpf(a)
    assert rel(v[:, 0], DH * _mp(lambda mp, z: (2 / am(mp)) * (mp.sqrt(am(mp) * (1 + z) + (1 - am(mp))) - 1))).max() < 1e-15
    # Ow13 = a, OL = 1 - a: E^2 = a x^2 + 1 - a
    v, _, _ = oracle.w_chi_batch(Z, 0.0, 1.0 - a, 0.0, a, 0.0, H0)
    assert rel(v[:, 0], DH * _mp(lambda mp, z: (mp.asinh(mp.sqrt(am(mp) / (1 - am(mp))) * (1 + z))
                                                 - mp.asinh(mp.sqrt(am(mp) / (1 - am(mp))))) / mp.sqrt(am(mp)))).max() < 1e-15
    # Om = a, Ow13 = 1 - a: the E of an open matter universe (pinned by Mattig's formula in test_oracle_pins), but flat
    v, _, _ = oracle.w_chi_batch(Z, a, 0.0, 0.0, 1.0 - a, 0.0, H0)
    v0, _, _ = oracle.observables_batch(Z, [a], [0.0], [0.0], [H0], False)
    assert rel(v[:, 0], v0[:, 0]).max() < 1e-17
    assert rel(v[:, 1], v0[:, 0]).max() < 1e-17 and (v[:, 1] < v0[:, 1]).all()      # D_M = D_C here, sinh(...) there
    # Om = a, Ow23 = 1 - a: E^2 = x (a x^2 + 1 - a); x = t^2 gives 2 int dt / sqrt(a t^4 + 1 - a), checked by mpmath below


def test_generic_mixture_against_mpmath_quadrature():
    import mpmath as mp
    mp.mp.dps = 30
    Om, OL, Or, O13, O23 = 0.27, 0.55, 8e-5, 0.06, 0.09
    Ok = 1 - Om - OL - Or - O13 - O23
    E = lambda x: mp.sqrt(Or * x ** 4 + Om * x ** 3 + (Ok + O13) * x ** 2 + O23 * x + OL)
    v, d, s = oracle.w_chi_batch(Z, Om, OL, Or, O13, O23, H0)
    for i, z in enumerate(Z):
        I0 = mp.quad(lambda x: 1 / E(x), [1, 1 + mp.mpf(float(z))])
        sk = mp.sqrt(abs(Ok))
        F = mp.sinh(sk * I0) / sk if Ok > 0 else mp.sin(sk * I0) / sk
        assert abs(float(v[i, 0]) / (DH * float(I0)) - 1) < 2e-15
        assert abs(float(v[i, 1]) / (DH * float(F)) - 1) < 2e-15
    # the matter + w = -2/3 flat mixture of the previous test
    a = 0.35
    v, _, _ = oracle.w_chi_batch(Z, a, 0.0, 0.0, 0.0, 1.0 - a, H0)
    for i, z in enumerate(Z):
        I0 = 2 * mp.quad(lambda t: 1 / mp.sqrt(a * t ** 4 + 1 - a), [1, mp.sqrt(1 + mp.mpf(float(z)))])
        assert abs(float(v[i, 0]) / (DH * float(I0)) - 1) < 2e-15


def test_dz_by_finite_differences():
    Om, OL, Or, O13, O23 = 0.27, 0.55, 8e-5, 0.06, 0.09
    h = 1e-5
    z = np.array([0.1, 0.7, 2.0, 8.0])
    v, d, _ = oracle.w_chi_batch(z, Om, OL, Or, O13, O23, H0)
    vp, _, _ = oracle.w_chi_batch(z + h, Om, OL, Or, O13, O23, H0)
    vm, _, _ = oracle.w_chi_batch(z - h, Om, OL, Or, O13, O23, H0)
    fd = (vp - vm) / (2 * h)
    assert rel(d, fd).max() < 1e-8


def test_invalid_path_and_status():
    v, d, s = oracle.w_chi_batch(np.array([5.0]), 0.1, 2.0, 0.0, 0.0, 0.05, H0)      # no Big Bang: E^2 < 0 at x = 2
    assert s[0] == -1 and np.isnan(v).all()


# ---------------------------------------------------------------- all six observables with every gradient (oracle.w_observables_batch)
OBS6 = {n: i for i, n in enumerate(oracle.OBS)}
WRT = {n: i for i, n in enumerate(oracle.WRTW)}
TH = 977.7922216807891 / H0


def test_full_reduces_to_the_lcdm_oracle():
    """no extra components: values and the (z, Om, OL, Or, H0) gradients of all six observables equal the pinned LCDM oracle's"""
    for Om, OL, Or in ((0.3, 0.7, 0.0), (0.3, 0.6, 9e-5), (0.2, 0.9, 1e-3)):
        v, g, s = oracle.w_observables_batch(Z, Om, OL, Or, 0.0, 0.0, H0)
        v0, g0, s0 = oracle.observables_batch(Z, [Om], [OL], [Or], [H0], True)
        assert (s == 0).all()
        assert rel(v, v0).max() < 1e-17
        assert rel(g[:, :, [0, 1, 2, 3, 6]], g0).max() < 1e-15
    # and the chi family agrees with w_chi_batch for a mixture
    p = (0.27, 0.55, 8e-5, 0.06, 0.09, H0)
    v, g, _ = oracle.w_observables_batch(Z, *p)
    vc, dc, _ = oracle.w_chi_batch(Z, *p)
    assert rel(v[:, :4], vc).max() < 1e-17 and rel(g[:, :4, 0], dc).max() < 1e-17


def test_full_single_and_two_component_closed_forms():
    # E^2 = x (pure w = -2/3): T = 2 (1 - x^-1/2), A = (2/5)(x^5/2 - 1)
    v, g, _ = oracle.w_observables_batch(Z, 0.0, 0.0, 0.0, 0.0, 1.0, H0)
    assert rel(v[:, OBS6["TL"]], TH * _mp(lambda mp, z: 2 * (1 - 1 / mp.sqrt(1 + z)))).max() < 5e-16
    assert rel(v[:, OBS6["DABS"]], DH * _mp(lambda mp, z: mp.mpf(2) / 5 * ((1 + z) ** mp.mpf(2.5) - 1))).max() < 5e-16
    # E^2 = x^2 (pure w = -1/3, flat): T = 1 - 1/x, A = (x^2 - 1)/2
    v, g, _ = oracle.w_observables_batch(Z, 0.0, 0.0, 0.0, 1.0, 0.0, H0)
    assert rel(v[:, OBS6["TL"]], TH * _mp(lambda mp, z: z / (1 + z))).max() < 5e-16
    assert rel(v[:, OBS6["DABS"]], DH * _mp(lambda mp, z: z * (2 + z) / 2)).max() < 5e-16
    # E^2 = a x + b, b = 1 - a (w = -2/3 and Lambda): elementary
    a = 0.35
    v, g, _ = oracle.w_observables_batch(Z, 0.0, 1.0 - a, 0.0, 0.0, a, H0)

    def T_ab(mp, z):
        A_, b = mp.mpf(a), 1 - mp.mpf(a)
        s = lambda x: mp.sqrt(A_ * x + b)
        G = lambda x: mp.log((s(x) - mp.sqrt(b)) / (s(x) + mp.sqrt(b))) / mp.sqrt(b)
        return G(1 + z) - G(1)

    def A_ab(mp, z):
        A_, b = mp.mpf(a), 1 - mp.mpf(a)
        G = lambda x: 2 * mp.sqrt(A_ * x + b) * (3 * A_ ** 2 * x ** 2 - 4 * A_ * b * x + 8 * b ** 2) / (15 * A_ ** 3)
        return G(1 + z) - G(1)
    assert rel(v[:, OBS6["TL"]], TH * _mp(T_ab)).max() < 2e-15
    assert rel(v[:, OBS6["DABS"]], DH * _mp(A_ab)).max() < 2e-14          # the closed form itself cancels at small z in 30 digits: ok
    # Leibniz gradient of that case in closed form: d I0 / d Ow23 at fixed sum (OL compensates? no: Ok does): dE^2 = (x - x^2) dOw23
    # checked against mpmath quadrature below for all parameters


def test_full_against_mpmath_quadrature():
    """independent quadrature (mpmath tanh-sinh, 30 digits) of the three integrals and of all twelve Leibniz gradient integrals"""
    import mpmath as mp
    mp.mp.dps = 30
    Om, OL, Or, O13, O23 = 0.27, 0.55, 8e-5, 0.06, 0.09
    Ok = 1 - Om - OL - Or - O13 - O23
    E2 = lambda x: Or * x ** 4 + Om * x ** 3 + (Ok + O13) * x ** 2 + O23 * x + OL
    D = {"Om": lambda x: x ** 3 - x ** 2, "OL": lambda x: 1 - x ** 2, "Or": lambda x: x ** 4 - x ** 2, "Ow23": lambda x: x - x ** 2}
    W = {"DC": (lambda x: mp.mpf(1), DH), "TL": (lambda x: 1 / x, TH), "DABS": (lambda x: x ** 2, DH)}
    zs = np.array([0.05, 0.8, 3.0, 40.0])
    v, g, s = oracle.w_observables_batch(zs, Om, OL, Or, O13, O23, H0)
    for i, z in enumerate(zs):
        for name, (wf, unit) in W.items():
            ref = unit * mp.quad(lambda x: wf(x) / mp.sqrt(E2(x)), [1, 1 + mp.mpf(float(z))])
            assert abs(mp.mpf(float(v[i, OBS6[name]])) - ref) <= 1e-15 * abs(ref), (z, name)
            for th, Df in D.items():
                ref = -unit / 2 * mp.quad(lambda x: wf(x) * Df(x) / E2(x) ** mp.mpf(1.5), [1, 1 + mp.mpf(float(z))])
                got = mp.mpf(float(g[i, OBS6[name], WRT[th]]))
                assert abs(got - ref) <= 1e-14 * abs(ref), (z, name, th)
            assert g[i, OBS6[name], WRT["Ow13"]] == 0          # Ow13 enters E^2 exactly like curvature: no E^2 dependence at fixed sum
    # ... but the transverse distance feels it through Ok alone: d D_M / d Ow13 = -d_H dF/dOk != 0
    assert (np.abs(g[:, OBS6["DM"], WRT["Ow13"]].astype(float)) > 1e-3 * np.abs(v[:, OBS6["DM"]].astype(float)) * zs ** 2 * 0.1).all()


def test_full_gradients_by_finite_differences():
    """Richardson-extrapolated central differences of the VALUES for every observable and every parameter (long double)"""
    th = [0.27, 0.55, 8e-5, 0.06, 0.09, 68.0]
    zs = np.array([0.03, 0.7, 2.2, 15.0])
    v, g, s = oracle.w_observables_batch(zs, *th)
    f = lambda zz, t: oracle.w_observables_batch(zz, *t, with_grad=False)[0]
    hs = {"Om": 2e-4, "OL": 2e-4, "Or": 2e-6, "Ow13": 2e-4, "Ow23": 2e-4, "H0": 2e-2}
    for k, (name, h) in enumerate(hs.items()):
        def cd(hh):
            tp, tm = list(th), list(th)
            tp[k] += hh; tm[k] -= hh
            return (f(zs, tp) - f(zs, tm)) / np.longdouble(2 * hh)
        fd = (4 * cd(h / 2) - cd(h)) / 3
        an = g[:, :, WRT[name]]
        err = np.abs((fd - an).astype(float)) / np.maximum(np.abs(an.astype(float)), 1e-3 * np.abs(v.astype(float)))
        assert err.max() <= 2e-9, (name, err.max())
    h = 1e-4 * (1 + zs)
    fd = (f(zs + h, th) - f(zs - h, th)) / (2 * h[:, None])
    fd2 = (f(zs + h / 2, th) - f(zs - h / 2, th)) / h[:, None]
    fdz = (4 * fd2 - fd) / 3
    assert (np.abs((fdz - g[:, :, 0]).astype(float)) <= 2e-9 * np.abs(g[:, :, 0].astype(float))).all()
