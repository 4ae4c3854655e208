"""Pins of the oracle's two-limit observables (oracle.observables2_batch; PAPER.md:88-93 define chi(z1,z2), t(z1,z2),
d_abs(z1,z2)): additivity against the (already pinned) one-limit oracle, Einstein-de Sitter closed forms, finite differences."""
import math

import numpy as np

import oracle

one = lambda v: np.array([float(v)])
C_KM_S, HUBBLE_GYR = 299792.458, 977.7922216807891


def test_additivity_with_one_limit_oracle():
    rng = np.random.default_rng(3)
    n = 30
    z1 = rng.uniform(0.0, 2.0, n); z2 = z1 + rng.uniform(0.01, 3.0, n)
    Om, OL, Or, H0 = rng.uniform(0.1, 0.5, n), rng.uniform(0.2, 1.0, n), rng.choice([0.0, 9e-5, 1e-3], n), rng.uniform(60, 80, n)
    v12, _, st = oracle.observables2_batch(z1, z2, Om, OL, Or, H0, with_grad=False)
    a, _, _ = oracle.observables_batch(z1, Om, OL, Or, H0, with_grad=False)
    b, _, _ = oracle.observables_batch(z2, Om, OL, Or, H0, with_grad=False)
    assert (st == 0).all()
    for k12, k in ((0, 0), (2, 4), (3, 5)):          # D_C, t, d_abs are differences of the one-limit values
        ref = (b[:, k] - a[:, k]).astype(np.float64)
        assert (np.abs(v12[:, k12].astype(np.float64) - ref) <= 1e-14 * np.abs(b[:, k].astype(np.float64))).all(), k12


def test_einstein_de_sitter_two_limit():
    z1, z2 = np.array([0.3, 1.0]), np.array([0.9, 4.0])
    v, _, _ = oracle.observables2_batch(z1, z2, one(1.0), one(0.0), one(0.0), one(70.0), with_grad=False)
    dH, tH = C_KM_S / 70, HUBBLE_GYR / 70
    for i in range(2):
        x1, x2 = 1 + z1[i], 1 + z2[i]
        assert abs(float(v[i, 0]) - 2 * dH * (x1 ** -0.5 - x2 ** -0.5)) <= 1e-14 * float(v[i, 0])
        assert abs(float(v[i, 1]) - float(v[i, 0])) <= 1e-15 * float(v[i, 0])                      # flat: D_M12 = D_C12
        assert abs(float(v[i, 2]) - tH * 2 / 3 * (x1 ** -1.5 - x2 ** -1.5)) <= 1e-14 * float(v[i, 2])
        assert abs(float(v[i, 3]) - dH * 2 / 3 * (x2 ** 1.5 - x1 ** 1.5)) <= 1e-14 * float(v[i, 3])
        assert abs(float(v[i, 4]) - float(v[i, 1]) / x2) <= 1e-15 * float(v[i, 4])


def test_gradients_by_finite_differences():
    p = dict(z1=0.4, z2=1.7, Om=0.3, OL=0.55, Or=9e-5, H0=68.0)
    def f(**kw):
        q = dict(p); q.update(kw)
        return oracle.observables2_batch(one(q["z1"]), one(q["z2"]), one(q["Om"]), one(q["OL"]), one(q["Or"]), one(q["H0"]),
                                         with_grad=False)[0][0].astype(np.float64)
    _, g, _ = oracle.observables2_batch(one(p["z1"]), one(p["z2"]), one(p["Om"]), one(p["OL"]), one(p["Or"]), one(p["H0"]))
    for k, (nm, h) in enumerate((("z1", 1e-5), ("z2", 1e-5), ("Om", 1e-5), ("OL", 1e-5), ("Or", 1e-7), ("H0", 1e-3))):
        fd = (f(**{nm: p[nm] + h}) - f(**{nm: p[nm] - h})) / (2 * h)
        for o in range(5):
            assert abs(fd[o] - float(g[0, o, k])) <= 2e-7 * abs(float(g[0, o, k])), (nm, oracle.OBS2[o])
