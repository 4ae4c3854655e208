"""CPU checks (-m "not gpu") of the CUDA path's host logic.

(1) tests/hostcheck/hostcheck.cpp compiles the per-element math headers of the CUDA path with plain g++ (test helper
    only; the product never loads it) and the result is compared with the oracle and the survey's mpmath goldens: this
    exercises the root factorisation, the fused Carlson duplication, eqs. (3.7)-(3.9)/(B.1)-(B.3) and the gradient bases
    before any GPU time is spent.
(2) libcosmo_b200.so (nvcc, sm_100a) loads without a GPU and exports every symbol include/cosmo_b200.h declares; its
    argument checking works without launching anything.
"""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

import oracle
from paper_2212_01937_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HC_DIR = os.path.join(ROOT, "tests", "hostcheck")
DP = C.POINTER(C.c_double)


@pytest.fixture(scope="module")
def hc():
    src = os.path.join(HC_DIR, "hostcheck.cpp")
    so = os.path.join(HC_DIR, "libhostcheck.so")
    csrc = os.path.join(ROOT, "paper_2212_01937_b200", "csrc")
    newest = max([os.path.getmtime(src)] + [os.path.getmtime(os.path.join(csrc, f)) for f in os.listdir(csrc)])
    if not os.path.exists(so) or os.path.getmtime(so) < newest:
        subprocess.run(["g++", "-O2", "-std=c++17", "-fPIC", "-shared", "-ffp-contract=off", "-Wno-unknown-pragmas", "-o", so, src],
                       check=True)
    return C.CDLL(so)


ELEM = False


@pytest.fixture(autouse=True, params=["outer-sequence", "elementwise-sequence"])
def sequence(request):
    """every test of the per-element math runs twice: through the OUTER kernels' sequence (gradient bases stored per cosmology) and
    through the ELEMENTWISE kernel's (cosmo_obs.cuh, elem_one: rows solved where consumed, constants re-formed after the loop)"""
    global ELEM
    ELEM = request.param.startswith("elementwise")
    yield


def run(hc, z, Om, OL, Or, H0, which=63, gup=None, f32=False, elem=None):
    elem = ELEM if elem is None else elem
    n = len(z)
    arrs = [np.ascontiguousarray(np.broadcast_to(np.asarray(a, dtype=np.float64), (n,))) for a in (z, Om, OL, Or, H0)]
    out = np.zeros((9, n)); gz = np.zeros(n); gp = np.zeros((4, n)); st = np.zeros(n, dtype=np.uint8)
    dp = lambda a: a.ctypes.data_as(DP) if a is not None else None
    f = (hc.hostcheck_elem_f32 if f32 else hc.hostcheck_elem_f64) if elem else (hc.hostcheck_f32 if f32 else hc.hostcheck_f64)
    f(C.c_int64(n), *[dp(a) for a in arrs], C.c_uint(which), dp(gup), dp(out), dp(gz), dp(gp), st.ctypes.data_as(C.POINTER(C.c_uint8)))
    return out, gz, gp, st


def test_factorisation_reproduces_polynomial(hc):
    rng = np.random.default_rng(0)
    out5 = np.zeros(5)
    for _ in range(300):
        Om, OL = rng.uniform(0.05, 1.5), rng.uniform(0.0, 1.2)
        Or = rng.choice([0.0, 1e-5, 9e-5, 1e-3])
        hc.hostcheck_factor(C.c_double(Om), C.c_double(OL), C.c_double(Or), out5.ctypes.data_as(DP))
        m, rn, b, c, st = out5
        if st != 0:
            continue
        Ok = 1 - Om - OL - Or
        for x in (0.3, 1.0, 2.5, 40.0):
            P = Or * x ** 4 + Om * x ** 3 + Ok * x ** 2 + OL
            F = (Or * x + m) * (x - rn) * (x * x + b * x + c)
            assert abs(F - P) <= 1e-12 * (abs(Or) * x ** 4 + Om * x ** 3 + abs(Ok) * x ** 2 + OL)
        assert rn <= 1e-12 and m > 0


def test_survey_goldens(hc, goldens):
    for r in goldens["general"] + [dict(goldens["config1_cosmology"], **row) for row in goldens["config1_table"]]:
        out, _, _, st = run(hc, [r["z"]], r["Om"], r["OL"], r["Or"], r["H0"])
        assert st[0] == 0
        tH = 977.7922216807891 / r["H0"]
        for i, key, sc, tol in ((0, "DC", 1, 2e-15), (1, "DM", 1, 2e-15), (3, "MU", 1, 2e-15), (4, "H0tL", tH, 3e-15), (5, "DABS", 1, 2e-12)):
            if key in r:
                ref = float(r[key]) * sc
                assert abs(out[i, 0] - ref) <= tol * abs(ref), (r, key)
    for r in goldens["gradients"]:
        for i, key in ((0, "DC"), (1, "DM"), (3, "MU")):
            if key not in r:
                continue
            g1 = np.zeros((6, 1)); g1[i] = 1
            _, gz, gp, _ = run(hc, [r["z"]], r["Om"], r["OL"], r["Or"], r["H0"], 63, g1)
            mine = dict(z=gz[0], Om=gp[0, 0], OL=gp[1, 0], Or=gp[2, 0], H0=gp[3, 0])
            for wrt, v in mine.items():
                if wrt in r[key]:
                    assert abs(v - float(r[key][wrt])) <= 1e-12 * abs(float(r[key][wrt])), (r["z"], key, wrt)


@pytest.mark.parametrize("cfg", ["config1", "config2"])
def test_host_math_matches_oracle(hc, cfg):
    w = W.config1(n=500) if cfg == "config1" else W.config2(n=1500)
    n = w.n_z
    rng = np.random.default_rng(1)
    gup = rng.standard_normal((6, n))
    out, gz, gp, st = run(hc, w.z, w.Om, w.OL, w.Or, w.H0, 63, gup)
    assert (st == 0).all()
    val, grad, sto = oracle.observables_batch(w.z, w.Om, w.OL, w.Or, w.H0, with_grad=True)
    val, grad = val.astype(np.float64), grad.astype(np.float64)
    for i, name in enumerate(oracle.OBS):
        e = np.abs(out[i] - val[:, i]) / np.abs(val[:, i])
        tol = 1e-11
        assert e.max() <= tol, (name, e.max())
        if name != "DABS":
            assert e.max() <= 5e-15, (name, e.max())
    mine = np.vstack([gz[None], gp])
    for p in range(5):
        ref = sum(gup[i] * grad[:, i, p] for i in range(6))
        scale = sum(np.abs(gup[i] * grad[:, i, p]) for i in range(6))
        assert (np.abs(mine[p] - ref) <= 1e-8 * scale).all(), p


def test_dabs_gradient(hc):
    """d(d_abs)/d(Om, OL, Or) on config 2 (the perturbative J' recursion of cosmo_obs.cuh where radiation is small)"""
    w = W.config2(n=1500)
    n = w.n_z
    g1 = np.zeros((6, n)); g1[5] = 1
    _, gz, gp, _ = run(hc, w.z, w.Om, w.OL, w.Or, w.H0, 63, g1)
    val, grad, _ = oracle.observables_batch(w.z, w.Om, w.OL, w.Or, w.H0, with_grad=True)
    val, grad = val.astype(np.float64), grad.astype(np.float64)
    for p, tol in ((1, 1e-8), (2, 1e-9), (3, 1e-8)):
        ref = grad[:, 5, p]
        e = np.abs(gp[p - 1] - ref) / np.maximum(np.abs(ref), 1e-3 * np.abs(val[:, 5]))
        assert e.max() <= tol, (p, e.max())


def test_host_math_stress_blocks(hc):
    w = W.config5(n=4000, n_struct=1500)
    out, _, _, st = run(hc, w.z, w.Om, w.OL, w.Or, w.H0)
    val, _, sto = oracle.observables_batch(w.z, w.Om, w.OL, w.Or, w.H0, with_grad=False)
    val = val.astype(np.float64)
    assert ((st & 3) == 0).all() and (sto >= 0).all()
    assert (((st & 4) != 0) == (sto == 1)).all()
    for i, tol in ((0, 1e-9), (4, 1e-9)):
        e = np.abs(out[i] - val[:, i]) / np.abs(val[:, i])
        assert e.max() <= tol and np.mean(e <= 1e-11) > 0.995, (i, e.max())


def test_two_complex_pairs_slow_path(hc):
    """E^2 without a real negative root (Om^2 < 4 Or Ok): eqs. (3.8)/(3.9) with a complex r_i (cosmo_c4.cuh) against the oracle"""
    rng = np.random.default_rng(7)
    n = 60
    Om = rng.uniform(0.050, 0.056, n); Or = rng.uniform(9.3e-4, 1e-3, n); OL = rng.uniform(0.0, 0.12, n)
    z = rng.uniform(0.001, 5.0, n); H0 = rng.uniform(60, 80, n)
    for i in range(n):   # every row really has no real negative root
        r = np.roots([Or[i], Om[i], 1 - Om[i] - OL[i] - Or[i], 0.0, OL[i]])
        assert not np.any((np.abs(r.imag) < 1e-9 * np.abs(r)) & (r.real < 0))
    out, _, _, st = run(hc, z, Om, OL, Or, H0)
    assert (st == 0).all()
    val, _, sto = oracle.observables_batch(z, Om, OL, Or, H0, with_grad=False)
    val = val.astype(np.float64)
    for i, tol in ((0, 1e-14), (1, 1e-14), (3, 1e-14), (4, 1e-14), (5, 1e-11)):
        assert (np.abs(out[i] - val[:, i]) / np.abs(val[:, i])).max() <= tol, i
    # gradients: the bases of cosmo_prep.cuh with the pair's [+1, -3] integral (cosmo_c4.cuh) as the K column
    _, grad, _ = oracle.observables_batch(z, Om, OL, Or, H0, with_grad=True)
    grad = grad.astype(np.float64)
    for pl, tols in ((0, (1e-14, 1e-9, 1e-9, 1e-8, 1e-14)), (3, (1e-14, 1e-9, 1e-9, 1e-8, 1e-14)), (4, (1e-14, 1e-9, 1e-9, 1e-8, 1e-14)),
                     (5, (1e-14, 1e-8, 1e-8, 1e-8, 1e-11))):       # d_abs: ill-conditioned basis -> quadrature (cosmo_obs.cuh, grad_quad)
        g1 = np.zeros((6, n)); g1[pl] = 1
        _, gz, gp, st = run(hc, z, Om, OL, Or, H0, 63, g1)
        assert (st == 0).all()
        mine = np.vstack([gz[None], gp])
        for p in range(5):
            ref = grad[:, pl, p]
            e = np.abs(mine[p] - ref) / np.maximum(np.abs(ref), 1e-3 * np.abs(val[:, pl]))
            assert e.max() <= tols[p], (pl, p, e.max())
    # D_A, V_C and age(z) (T_inf by the same slow path at x = 1e10) on these rows
    dv, dg, _ = oracle.derived_batch(z, Om, OL, Or, H0)
    dv, dg = dv.astype(np.float64), dg.astype(np.float64)
    for k, pl in enumerate((6, 7, 8)):
        g1 = np.zeros((9, n)); g1[pl] = 1
        out9, gz, gp, st = run(hc, z, Om, OL, Or, H0, 511, g1)
        assert (st == 0).all() and (np.abs(out9[pl] - dv[:, k]) <= 1e-13 * np.abs(dv[:, k])).all(), pl
        mine = np.vstack([gz[None], gp])
        for p in range(5):
            e = np.abs(mine[p] - dg[:, k, p]) / np.maximum(np.abs(dg[:, k, p]), 1e-3 * np.abs(dv[:, k]))
            assert e.max() <= 1e-8, (pl, p, e.max())


def test_derived_observables_host(hc):
    """D_A, comoving volume and age (planes 64, 128, 256) with their gradients against oracle.derived_batch"""
    for w in (W.config1(n=300), W.config2(n=800)):
        n = w.n_z
        bc = lambda a: np.ascontiguousarray(np.broadcast_to(a, (n,)) if a.shape[0] == 1 else a)
        z, Om, OL, Or, H0 = w.z, bc(w.Om), bc(w.OL), bc(w.Or), bc(w.H0)
        val, grad, _ = oracle.derived_batch(z, Om, OL, Or, H0)
        val, grad = val.astype(np.float64), grad.astype(np.float64)
        for i in range(3):
            g1 = np.zeros((9, n)); g1[6 + i] = 1
            out, gz, gp, st = run(hc, z, Om, OL, Or, H0, 511, g1)
            assert (np.abs(out[6 + i] - val[:, i]) / np.abs(val[:, i])).max() <= 1e-12, oracle.DERIVED[i]
            mine = np.vstack([gz[None], gp])
            for k in range(5):
                e = np.abs(mine[k] - grad[:, i, k]) / np.maximum(np.abs(grad[:, i, k]), 1e-3 * np.abs(val[:, i]))
                assert e.max() <= 1e-8, (oracle.DERIVED[i], oracle.WRT[k], e.max())


def test_two_limit_host(hc):
    """chi(z1,z2), D_M12, t(z1,z2), d_abs(z1,z2), D_A12 and their gradients (cosmo_two.cuh) against oracle.observables2_batch"""
    rng = np.random.default_rng(1)
    n = 1200
    z1 = rng.uniform(0, 3, n); z2 = z1 + 10 ** rng.uniform(-3, 0.8, n)
    Om = rng.uniform(.08, .6, n); OL = rng.uniform(0, 1.2, n); Or = rng.choice([0.0, 1e-5, 9e-5, 1e-3], n); H0 = rng.uniform(60, 80, n)
    val = np.zeros((5, n)); g1 = np.zeros((5, n)); g2 = np.zeros((5, n)); gp = np.zeros((5, 4, n)); st = np.zeros(n, dtype=np.uint8)
    dp = lambda a: a.ctypes.data_as(DP)
    hc.hostcheck_two(C.c_int64(n), dp(z1), dp(z2), dp(Om), dp(OL), dp(Or), dp(H0), dp(val), dp(g1), dp(g2), dp(gp),
                     st.ctypes.data_as(C.POINTER(C.c_uint8)))
    v, g, so = oracle.observables2_batch(z1, z2, Om, OL, Or, H0)
    v, g = v.astype(np.float64), g.astype(np.float64)
    assert (so == 0).all() and (st == 0).all()
    for o, nm in enumerate(oracle.OBS2):
        assert (np.abs(val[o] - v[:, o]) / np.abs(v[:, o])).max() <= 1e-11, nm
        mine = [g1[o], g2[o]] + [gp[o, t] for t in range(4)]
        for k in range(6):
            e = np.abs(mine[k] - g[:, o, k]) / np.maximum(np.abs(g[:, o, k]), 1e-3 * np.abs(v[:, o]))
            tol = 1e-8
            assert e.max() <= tol, (nm, oracle.WRT2[k], e.max())


def test_two_limit_two_complex_pairs_host(hc):
    """the two-limit forms on cosmologies without a real negative root (cosmo_c4.cuh between x1 and x2), both orders of the limits"""
    rng = np.random.default_rng(7)
    n = 80
    Om = rng.uniform(0.050, 0.056, n); Or = rng.uniform(9.3e-4, 1e-3, n); OL = rng.uniform(0.01, 0.12, n); H0 = rng.uniform(60, 80, n)
    z1 = rng.uniform(0, 3, n); z2 = z1 + 10 ** rng.uniform(-3, 0.8, n)
    z1[:8], z2[:8] = z2[:8].copy(), z1[:8].copy()
    val = np.zeros((5, n)); g1 = np.zeros((5, n)); g2 = np.zeros((5, n)); gp = np.zeros((5, 4, n)); st = np.zeros(n, dtype=np.uint8)
    dp = lambda a: a.ctypes.data_as(DP)
    hc.hostcheck_two(C.c_int64(n), dp(z1), dp(z2), dp(Om), dp(OL), dp(Or), dp(H0), dp(val), dp(g1), dp(g2), dp(gp),
                     st.ctypes.data_as(C.POINTER(C.c_uint8)))
    v, g, so = oracle.observables2_batch(z1, z2, Om, OL, Or, H0)
    v, g = v.astype(np.float64), g.astype(np.float64)
    assert (so == 0).all() and (st == 0).all()
    for o, nm in enumerate(oracle.OBS2):
        assert (np.abs(val[o] - v[:, o]) / np.abs(v[:, o])).max() <= 1e-11, nm
        mine = [g1[o], g2[o]] + [gp[o, t] for t in range(4)]
        for k in range(6):
            e = np.abs(mine[k] - g[:, o, k]) / np.maximum(np.abs(g[:, o, k]), 1e-3 * np.abs(v[:, o]))
            tol = 1e-8
            assert e.max() <= tol, (nm, oracle.WRT2[k], e.max())


def test_extra_w_components_host(hc):
    """chi family on the general quartic (cosmo_w.cuh; PAPER.md:82 fn.4) against oracle.w_chi_batch"""
    w = W.wmix(n=6000)
    n = len(w["z"])
    val = np.zeros((4, n)); dz = np.zeros((4, n)); st = np.zeros(n, dtype=np.uint8)
    dp = lambda a: np.ascontiguousarray(a).ctypes.data_as(DP)
    hc.hostcheck_w(C.c_int64(n), dp(w["z"]), dp(w["Om"]), dp(w["OL"]), dp(w["Or"]), dp(w["Ow13"]), dp(w["Ow23"]), dp(w["H0"]), dp(val), dp(dz),
                   st.ctypes.data_as(C.POINTER(C.c_uint8)))
    v, d, so = oracle.w_chi_batch(w["z"], w["Om"], w["OL"], w["Or"], w["Ow13"], w["Ow23"], w["H0"])
    v, d = v.astype(np.float64), d.astype(np.float64)
    ok = so == 0
    assert ok.mean() > 0.95 and (st[ok] == 0).all() and (st[so == -1] & 3).all()
    for o, nm in enumerate(oracle.OBSW):
        assert (np.abs(val[o][ok] - v[ok, o]) / np.abs(v[ok, o])).max() <= 1e-11, nm
        assert (np.abs(dz[o][ok] - d[ok, o]) / np.abs(d[ok, o])).max() <= 1e-11, nm
    assert np.isnan(val[:, so == -1]).all()


def test_extra_w_components_full_host(hc):
    """t_L, d_abs and every parameter gradient on the general quartic (cosmo_w.cuh: eqs. (3.8)/(3.9) with complex roots and complex
    Carlson functions; gradient integrals by quadrature) against oracle.w_observables_batch"""
    w = W.wmix(n=3000)
    n = len(w["z"])
    names = ("z", "Om", "OL", "Or", "Ow13", "Ow23", "H0")
    val = np.zeros((6, n)); dz = np.zeros((6, n)); gp = np.zeros((6, 6, n)); st = np.zeros(n, dtype=np.uint8)
    dp = lambda a: np.ascontiguousarray(a).ctypes.data_as(DP)
    hc.hostcheck_w_full(C.c_int64(n), *[dp(w[k]) for k in names], dp(val), dp(dz), dp(gp), st.ctypes.data_as(C.POINTER(C.c_uint8)))
    v, g, so = oracle.w_observables_batch(*[w[k] for k in names])
    v, g = v.astype(np.float64), g.astype(np.float64)
    ok = (so == 0) & ((st & 1) == 0)
    assert ok.mean() > 0.95 and (st[so == -1] & 3).all()
    chi_ok = ok & np.isfinite(val[0])
    for o in range(4):
        assert (np.abs(val[o][chi_ok] - v[chi_ok, o]) / np.abs(v[chi_ok, o])).max() <= 1e-11, oracle.OBS[o]
    # t_L, d_abs: every element of degree 3 or 4 and the monomials; the few of degree <= 2 with distinct roots are marked unsupported
    sup = ok & ((st & 2) == 0)
    assert sup.sum() >= ok.sum() - 8 and np.isnan(val[4][ok & ~sup]).all()
    for o, tol in ((4, 1e-11), (5, 1e-10)):      # d_abs: the Om/Or cancellation of eq. (3.9), up to Om/Or = 5e4 here
        e = np.abs(val[o][sup] - v[sup, o]) / np.abs(v[sup, o])
        assert e.max() <= tol, (oracle.OBS[o], e.max())
        ez = np.abs(dz[o][sup] - g[sup, o, 0]) / np.abs(g[sup, o, 0])
        assert ez.max() <= 1e-11, (oracle.OBS[o], ez.max())
    # parameter gradients (Om, OL, Or, Ow13, Ow23, H0) of all six observables; elements the quadrature cannot serve are flagged
    fl = (st & 16) != 0
    assert fl[ok].mean() < 0.05
    for o in range(6):
        m = (sup if o >= 4 else chi_ok) & ~fl & np.isfinite(v[:, o])
        for t in range(6):
            r = g[:, o, 1 + t]
            e = np.abs(gp[o, t] - r)[m] / np.maximum(np.abs(r[m]), 1e-3 * np.abs(v[m, o]))
            assert e.max() <= (1e-7 if (o == 5 and t == 5) else 1e-8), (oracle.OBS[o], oracle.WRTW[1 + t], e.max())


def test_host_math_fp32(hc):
    w = W.config3(n=3000, S=1)
    z = w.z.astype(np.float32).astype(np.float64)
    out, _, _, st = run(hc, z, w.Om[0], w.OL[0], w.Or[0], w.H0[0], 15, None, f32=True)
    val, _, _ = oracle.observables_batch(z, w.Om[:1], w.OL[:1], w.Or[:1], w.H0[:1], with_grad=False)
    val = val.astype(np.float64)
    for i in range(4):
        assert (np.abs(out[i] - val[:, i]) / np.abs(val[:, i])).max() <= 2e-5, i


def test_vanishing_lambda_gradients(hc):
    """OL -> 0 closes the gap of the pair (+-sqrt(-OL/Ok)) and the gradient bases degenerate (singular at OL = 0, the 1/prod(r_j - r_k)
    of PAPER.md:320-345): such elements take the quadrature of the Leibniz integrals instead (cosmo_obs.cuh, grad_quad; PAPER.md:145
    "limits have to be explicitly implemented when arguments are repeated").  Every gradient of every plane meets the tolerance and
    nothing is flagged -- Einstein-de Sitter (a triple root), open and closed matter models included."""
    rng = np.random.default_rng(3)
    n = 120
    z = rng.uniform(0.01, 5, n); H0 = np.full(n, 70.0)
    cases = [(rng.uniform(0.1, 1.6, n), np.full(n, OLv), np.full(n, Orv)) for OLv in (0.0, 1e-12, 1e-9, 1e-6, 1e-3) for Orv in (0.0, 9e-5)]
    cases.append((np.ones(n), np.zeros(n), np.zeros(n)))                                   # Einstein-de Sitter
    eps = 10.0 ** rng.uniform(-12, -2, n)
    cases.append((1.0 - eps, eps, np.zeros(n)))                                            # flat, OL -> 0: three roots close in on x = 0
    for Om, OL, Or in cases:
        val, grad, _ = oracle.observables_batch(z, Om, OL, Or, H0, with_grad=True)
        val, grad = val.astype(np.float64), grad.astype(np.float64)
        for pl in (0, 1, 3, 4, 5):
            g1 = np.zeros((6, n)); g1[pl] = 1
            out, gz, gp, st = run(hc, z, Om, OL, Or, H0, 63, g1)
            assert (st == 0).all(), (OL[0], Or[0], pl)
            assert (np.abs(out[pl] - val[:, pl]) <= 1e-11 * np.abs(val[:, pl])).all(), (OL[0], Or[0], pl)
            mine = np.vstack([gz[None], gp])
            for p in range(5):
                e = np.abs(mine[p] - grad[:, pl, p]) / np.maximum(np.abs(grad[:, pl, p]), 1e-3 * np.abs(val[:, pl]))
                assert e.max() <= 1e-8, (OL[0], Or[0], pl, p, e.max())
    # closed forms at Einstein-de Sitter (E^2 = x^3): I0 = 2 (1 - x^-1/2), dI0/dOm = -1/2 int (x^3 - x^2) x^-9/2 dx = -(1/x - 1) - (x^-3/2 - 1)/3 ... by hand:
    zz = np.array([0.5, 2.0]); x = 1 + zz
    g1 = np.zeros((6, 2)); g1[0] = 1
    _, _, gp, st = run(hc, zz, 1.0, 0.0, 0.0, 70.0, 63, g1)
    dH = 299792.458 / 70.0
    F = lambda p: (x ** (p - 3.5) - 1) / (p - 3.5)                     # int_1^x t^p t^-9/2 dt
    ref = [-0.5 * dH * (F(3) - F(2)), -0.5 * dH * (F(0) - F(2)), -0.5 * dH * (F(4) - F(2))]
    for p in range(3):
        assert np.allclose(gp[p], ref[p], rtol=1e-12, atol=0), p


def test_gradient_at_z_zero(hc):
    """z = 0: every integral vanishes, D_M = 0 and mu is undefined (status 4), but d/dz of the other planes is the integrand at z = 0
    (d t_L/dz = t_H, d D_C/dz = d_H, E(0) = 1) and their parameter gradients are exactly zero -- no 0 x inf"""
    z = np.array([0.0, 0.0]); Om = np.array([0.3, 0.25]); OL = np.array([0.7, 0.6]); Or = np.array([0.0, 9e-5]); H0 = np.array([70.0, 67.0])
    dH, tH = 299792.458 / H0, 977.7922216807891 / H0
    expect = {0: dH, 1: dH, 2: dH, 4: tH, 5: dH, 6: dH, 8: -tH}        # D_L = (1+z) D_M, D_A = D_M/(1+z): slope d_H at z = 0
    for pl, dz_ref in expect.items():
        g1 = np.zeros((9, 2)); g1[pl] = 1
        out, gz, gp, st = run(hc, z, Om, OL, Or, H0, 511 & ~8, g1)
        assert np.isfinite(gz).all() and np.isfinite(gp).all(), pl
        assert np.allclose(gz, dz_ref, rtol=1e-14), (pl, gz, dz_ref)
        if pl != 8:
            assert (gp[:3] == 0).all() and (out[pl] == 0).all(), pl
    # with the mu plane selected but no upstream gradient on it the others stay finite
    g1 = np.zeros((9, 2)); g1[0] = 1; g1[4] = 1
    out, gz, gp, st = run(hc, z, Om, OL, Or, H0, 511, g1)
    assert np.isfinite(gz).all() and np.isfinite(gp).all() and ((st & 4) != 0).all()
    assert np.allclose(gz, dH + tH, rtol=1e-14)


def test_invalid_rows_status(hc):
    for z, Om, OL, Or, H0, bit in W.invalid_rows():
        out, _, _, st = run(hc, [z], Om, OL, Or, H0)
        assert st[0] & bit, (z, Om, OL, Or, st[0])
        assert np.isnan(out[0, 0])


# ---------------------------------------------------------------- the CUDA library itself (no GPU needed to load it)
def test_library_exports_every_declared_symbol():
    from paper_2212_01937_b200 import binding, build
    build.build()
    L = binding.lib()
    hdr = "".join(open(os.path.join(ROOT, "include", f)).read() for f in sorted(os.listdir(os.path.join(ROOT, "include"))) if f.endswith(".h"))
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cosmo_[a-z0-9_]+)\s*\(", hdr))
    assert declared == set(binding.SYMBOLS), declared ^ set(binding.SYMBOLS)
    for s in declared:
        assert hasattr(L, s), s
    assert b"sm_100a" in L.cosmo_version()


def test_library_argument_errors_without_gpu():
    from paper_2212_01937_b200 import binding
    L = binding.lib()
    P = binding.CosmoParams(0, 0, 0, 0)
    assert L.cosmo_eval(None, -1, P, 1, 0, 1, None, None, None, 0, None) == -2
    assert L.cosmo_eval(None, 4, P, 1, 0, 0, None, None, None, 0, None) == -3
    assert L.cosmo_eval(None, 4, P, 1, 9, 1, None, None, None, 0, None) == -4
    assert L.cosmo_eval(None, 4, P, 3, 0, 1, None, None, None, 0, None) == -2
    assert L.cosmo_eval(None, 4, P, 1, 0, 1, None, None, None, 0, None) == -1
    assert L.cosmo_strerror(-5).decode().startswith("workspace")
    assert binding.workspace_bytes(1_000_000, 64, binding.OUTER, ("MU",), True) > 64 * 600
    assert binding.workspace_bytes(1000, 1000, binding.ELEMENTWISE, ("MU",), False) == 0
    assert binding.workspace_bytes(1000, 1000, binding.ELEMENTWISE, ("MU",), True) >= 4 * 1000      # work list of the VJP's second pass


def test_binding_refuses_cpu():
    import torch
    from paper_2212_01937_b200 import binding
    if torch.cuda.is_available():
        pytest.skip("CUDA present")
    z = torch.zeros(4, dtype=torch.float64)
    with pytest.raises(binding.CosmoError):
        binding.cosmo_eval(z, z, z, z, z)


def test_sinn_quartering_against_mpmath(hc):
    """cosmo_eval.cuh sinn(): S = sin(sqrt(-w))/sqrt(-w) (sinh for w > 0), C = cos / cosh, S' = (C - S)/(2w), by the degree-7 series on the
    quartered argument and the doubling steps back -- against 40-digit values over closed models up to the antipode (w = -pi^2), open
    ones up to w = 200, the series range, zero and the switch points between m and m + 1 quarterings"""
    import mpmath as mp
    mp.mp.dps = 40
    rng = np.random.default_rng(11)
    w = np.concatenate([rng.uniform(-9.8, 0, 300), rng.uniform(0, 200, 300), rng.uniform(-0.5, 0.5, 100), -np.pi ** 2 + 10.0 ** rng.uniform(-8, 0, 50),
                        [0.0, 0.5, -0.5, np.nextafter(0.5, 1), 2.0, np.nextafter(2.0, 3), -2.0, 8.0, np.nextafter(8.0, 9), 1e-300, -1e-12]])
    I0 = rng.uniform(0.05, 3.0, w.size)
    k = w / I0 ** 2
    F, Fi, Fk = np.zeros_like(w), np.zeros_like(w), np.zeros_like(w)
    hc.hostcheck_sinn(C.c_int64(w.size), k.ctypes.data_as(DP), I0.ctypes.data_as(DP), F.ctypes.data_as(DP), Fi.ctypes.data_as(DP), Fk.ctypes.data_as(DP))
    for i in range(w.size):
        ww = mp.mpf(float(k[i])) * mp.mpf(float(I0[i])) ** 2
        if ww < 0:
            y = mp.sqrt(-ww); S, Cc = mp.sin(y) / y, mp.cos(y)
        elif ww > 0:
            y = mp.sqrt(ww); S, Cc = mp.sinh(y) / y, mp.cosh(y)
        else:
            S, Cc = mp.mpf(1), mp.mpf(1)
        Sd = (Cc - S) / (2 * ww) if abs(ww) > 1e-6 else mp.mpf(1) / 6 + ww / 60
        # S -> 0 at the antipode: the error is absolute there (it is the rounding of w that decides, |dS/dw| = 1/2 pi^2)
        assert abs(F[i] / I0[i] - S) <= 4e-15 * max(1.0, abs(S)), (w[i], float(S))
        assert abs(Fi[i] - Cc) <= 4e-15 * max(1.0, abs(Cc)), (w[i], float(Cc))
        assert abs(Fk[i] / I0[i] ** 3 - Sd) <= 2e-14 * max(abs(Sd), 0.05), (w[i], float(Sd))
    # not-a-number and infinite arguments stay what they are
    kk = np.array([np.nan, 1e300, 1.0]); ii = np.array([1.0, 1e10, np.nan]); o = [np.zeros(3) for _ in range(3)]
    hc.hostcheck_sinn(C.c_int64(3), kk.ctypes.data_as(DP), ii.ctypes.data_as(DP), *[a.ctypes.data_as(DP) for a in o])
    assert not np.isfinite(o[0]).any()


def test_band_solve_against_moments(hc):
    """cosmo_eval.cuh band_solve(): the truncated moment recurrences of d_abs against the moments themselves by quadrature --
    value shape: u_j = int_1^x t^j dt/E from u_0, u_1 and b_k = [t^k E]; gradient shape: J'_p = int t^p dt/E^3 from J'_2..J'_4 and
    b_k = [t^k/E].  The returned bound has to cover the truncation error wherever that is visible; outside Om^2 >= 8 Or Ok it is infinite"""
    from scipy.integrate import quad
    rng = np.random.default_rng(5)
    seen_trunc = 0
    for it in range(60):
        if it < 30:      # radiation as a perturbation: the truncation is far below rounding
            Om, OL, Or = rng.uniform(0.05, 1.0), rng.uniform(0, 1.2), 10.0 ** rng.uniform(-6, -3.5)
        else:            # radiation large enough for the truncation to show, so that the bound is really tested
            Om, OL, Or = rng.uniform(0.5, 1.0), rng.uniform(0.3, 0.9), 10.0 ** rng.uniform(-1.8, -1.0)
        Ok = 1 - Om - OL - Or
        x = rng.uniform(1.05, 3.5)
        E = lambda t: np.sqrt(Or * t ** 4 + Om * t ** 3 + Ok * t ** 2 + OL)
        for shape, NR in ((0, 9), (1, 11)):
            if shape == 0:
                mom = [quad(lambda t: t ** j / E(t), 1, x, epsabs=0, epsrel=1e-13)[0] for j in range(NR + 2)]
                b = np.array([x ** k * E(x) - E(1.0) for k in range(NR)])
                km, truth, j0 = (mom[1], mom[0], 0.0), np.array(mom[2:NR + 2]), 0
            else:
                mom = [quad(lambda t: t ** p / E(t) ** 3, 1, x, epsabs=0, epsrel=1e-13)[0] for p in range(NR + 5)]
                b = np.array([x ** k / E(x) - 1.0 / E(1.0) for k in range(3, NR + 3)])
                km, truth, j0 = (mom[4], mom[3], mom[2]), np.array(mom[5:NR + 5]), 1
            v = np.zeros(NR); tr = C.c_double()
            hc.hostcheck_band(shape, C.c_double(Om), C.c_double(OL), C.c_double(Or), C.c_double(Ok), b.ctypes.data_as(DP), C.c_double(km[0]),
                              C.c_double(km[1]), C.c_double(km[2]), C.c_double(x), v.ctypes.data_as(DP), C.byref(tr))
            err = abs(v[j0] - truth[j0])
            if Om * Om >= 8 * Or * Ok:
                assert err <= 1.001 * tr.value + 2e-12 * abs(truth[j0]), (shape, Om, OL, Or, x, err, tr.value)
                seen_trunc += err > 1e-10 * abs(truth[j0])
                if it < 30:
                    assert err <= 2e-12 * abs(truth[j0]) and tr.value <= 1e-15 * abs(truth[j0])
            else:
                assert np.isinf(tr.value)
    assert seen_trunc >= 10        # the bound was exercised where the truncation is visible
    # no real negative root (Om^2 < 4 Or Ok): refused
    v = np.zeros(9); tr = C.c_double(); b = np.ones(10)
    hc.hostcheck_band(0, C.c_double(0.05), C.c_double(0.0), C.c_double(1e-3), C.c_double(0.949), b.ctypes.data_as(DP), C.c_double(1.0), C.c_double(1.0),
                      C.c_double(0.0), C.c_double(2.0), v.ctypes.data_as(DP), C.byref(tr))
    assert np.isinf(tr.value)


def test_two_complex_pairs_tiny_z(hc):
    """the complex slow path (cosmo_c4.cuh) at z = 1e-8 .. 1e-3: the range has to come in as z, not as (1 + z) - 1 (which cost eps/z of
    every integral), and the boundary term of eq. (3.9) has its factor z taken out analytically (subtracted directly it cost d_abs another
    eps/z); found by a wide-prior comparison with the oracle"""
    rng = np.random.default_rng(17)
    n = 80
    Om = rng.uniform(0.050, 0.20, n); Or = rng.uniform(0.03, 0.08, n); OL = rng.uniform(0.0, 0.3, n)
    z = 10.0 ** rng.uniform(-8, -3, n); H0 = rng.uniform(60, 80, n)
    assert (Om ** 2 < 4 * Or * (1 - Om - OL - Or)).all()          # no real negative root: every row takes the slow path
    out, _, _, st = run(hc, z, Om, OL, Or, H0)
    assert (st == 0).all()
    val, grad, sto = oracle.observables_batch(z, Om, OL, Or, H0, with_grad=True)
    val, grad = val.astype(np.float64), grad.astype(np.float64)
    for i, tol in ((0, 2e-14), (1, 2e-14), (4, 2e-14), (5, 1e-12)):
        assert (np.abs(out[i] - val[:, i]) / np.abs(val[:, i])).max() <= tol, (i, (np.abs(out[i] - val[:, i]) / np.abs(val[:, i])).max())
    for pl in (0, 4, 5):
        g1 = np.zeros((6, n)); g1[pl] = 1
        _, gz, gp, st = run(hc, z, Om, OL, Or, H0, 63, g1)
        assert (st == 0).all()
        mine = np.vstack([gz[None], gp])
        for p in range(5):
            ref = grad[:, pl, p]
            e = np.abs(mine[p] - ref) / np.maximum(np.abs(ref), 1e-3 * np.abs(val[:, pl]))
            assert e.max() <= 1e-8, (pl, p, e.max())


def test_ol_zero_with_complex_pair(hc):
    """OL = 0 exactly and Om^2 < 4 Or Ok: E^2 = x^2 (Or x^2 + Om x + Ok) with a complex pair.  The real labelling has no m > 0 for it;
    cosmo_factor hands it to the complex slow path with the double root at 0 as the second pair (the limit OL -> 0+ of two complex
    pairs).  Values and every gradient against the oracle, and continuity in OL."""
    rng = np.random.default_rng(23)
    n = 60
    Om = rng.uniform(0.050, 0.060, n); Or = np.full(n, 1e-3); OL = np.zeros(n)
    z = np.concatenate([10.0 ** rng.uniform(-6, -1, n // 3), rng.uniform(0.1, 14.0, n - n // 3)]); H0 = rng.uniform(60, 80, n)
    assert (Om ** 2 < 4 * Or * (1 - Om - OL - Or)).all()
    out, _, _, st = run(hc, z, Om, OL, Or, H0)
    assert (st == 0).all()
    val, grad, sto = oracle.observables_batch(z, Om, OL, Or, H0, with_grad=True)
    val, grad = val.astype(np.float64), grad.astype(np.float64)
    assert (sto == 0).all()
    for i, tol in ((0, 1e-13), (1, 1e-13), (3, 1e-13), (4, 1e-13), (5, 1e-11)):
        assert (np.abs(out[i] - val[:, i]) / np.abs(val[:, i])).max() <= tol, i
    out_eps, _, _, st_eps = run(hc, z, Om, np.full(n, 1e-300), Or, H0)
    assert (st_eps == 0).all() and np.allclose(out_eps[:6], out[:6], rtol=1e-13, atol=0)
    for pl in (0, 3, 4, 5):
        g1 = np.zeros((6, n)); g1[pl] = 1
        _, gz, gp, st = run(hc, z, Om, OL, Or, H0, 63, g1)
        assert (st == 0).all()
        mine = np.vstack([gz[None], gp])
        for p in range(5):
            ref = grad[:, pl, p]
            e = np.abs(mine[p] - ref) / np.maximum(np.abs(ref), 1e-3 * np.abs(val[:, pl]))
            assert e.max() <= 1e-8, (pl, p, e.max())


def test_w_family_wide_priors(hc):
    """the extra-w family (cosmo_w.cuh) far outside its seeded mix: Om = 0 or OL = 0 in a sixth of the rows each, Or log-uniform down
    to 1e-7 or absent, both extra components from -0.2 to 0.8 or absent, z from 1e-6 to 30, OL up to 1.5 (real root pairs right of the
    path).  What this comparison found and fixed in w_TA: the branch of sqrt(x - r) for real roots right of the path (d_abs wrong by orders
    of magnitude), r_i of eq. (3.8) a member of a conjugate pair where a real root exists (t_L with the wrong sign at Om = 0), the pair
    taken as (r_i, r_l) of eq. (3.9) with two complex pairs, the range formed as (1 + z) - 1 and the boundary terms subtracted directly
    (eps/z).  d_abs is assembled through the hot path's moment recurrence with this family's x^1 term where there is matter; without
    matter it keeps the cancellation of eq. (3.9) as printed, which grows as 1/Or: its tolerance says so."""
    rng = np.random.default_rng(31)
    n = 12000
    u = rng.random(n)
    z = np.where(u < 0.2, 10 ** rng.uniform(-6, -2, n), np.where(u < 0.4, rng.uniform(3, 30, n), rng.uniform(0.01, 3, n)))
    Om = np.where(rng.random(n) < 0.15, 0.0, rng.uniform(0.02, 1.5, n))
    OL = np.where(rng.random(n) < 0.15, 0.0, rng.uniform(0.0, 1.5, n))
    Or = np.where(rng.random(n) < 0.3, 0.0, 10 ** rng.uniform(-7, -1, n))
    Ow13 = np.where(rng.random(n) < 0.3, 0.0, rng.uniform(-0.2, 0.8, n))
    Ow23 = np.where(rng.random(n) < 0.3, 0.0, rng.uniform(-0.2, 0.8, n))
    H0 = rng.uniform(50, 90, n)
    A = [z, Om, OL, Or, Ow13, Ow23, H0]
    val = np.zeros((6, n)); dz = np.zeros((6, n)); gp = np.zeros((6, 6, n)); st = np.zeros(n, dtype=np.uint8)
    dp = lambda a: np.ascontiguousarray(a).ctypes.data_as(DP)
    hc.hostcheck_w_full(C.c_int64(n), *[dp(a) for a in A], dp(val), dp(dz), dp(gp), st.ctypes.data_as(C.POINTER(C.c_uint8)))
    v, g, so = oracle.w_observables_batch(*A)
    v, g = v.astype(np.float64), g.astype(np.float64)
    st = st.astype(np.int64)
    assert (((st & 1) != 0) == (so == -1)).all()                  # a root on the path: the same rows as the oracle
    ok = (so == 0) & ((st & 3) == 0)
    deg_le2 = (Or == 0) & (Om == 0)
    assert (((st & 2) != 0) & (so == 0) <= deg_le2).all()         # refused (t_L, d_abs only): degree <= 2, outside the method
    assert ok.sum() > 0.85 * n
    rel = lambda a, b: np.abs(a - b) / np.abs(b)
    for o in range(4):
        m = ok & np.isfinite(v[:, o])
        assert rel(val[o][m], v[m, o]).max() <= 1e-11, oracle.OBS[o]
    assert rel(val[4][ok], v[ok, 4]).max() <= 1e-11
    tolA = 2e-11 + np.where((Or > 0) & (Om == 0), 1e-15 / np.maximum(Or, 1e-300), 0.0)      # (no matter: no moment recurrence, eq. (3.9) as printed)
    assert (rel(val[5][ok], v[ok, 5]) <= tolA[ok]).all(), float((rel(val[5][ok], v[ok, 5]) / tolA[ok]).max())
    for o in (4, 5):
        assert rel(dz[o][ok], g[ok, o, 0]).max() <= 1e-11
