"""Pins of oracle.snia_logjoint (section-4 toy model with latent redshifts): SciPy's norm / gamma log-densities
on the oracle's own mu (pinned elsewhere), the value at perfect data, and finite differences of every gradient."""
import numpy as np
from scipy import stats

import oracle

MU = oracle.OBS.index("MU")


def _mu(z, Om, OL, Or, H0):
    one = lambda v: np.array([float(v)])
    return oracle.observables_batch(z, one(Om), one(OL), one(Or), one(H0), with_grad=False)[0][:, MU].astype(np.float64)


def test_against_scipy_densities():
    rng = np.random.default_rng(0)
    n = 40
    z = rng.gamma(3.0, 1 / 3.0, n) + 0.01
    th = (0.31, 0.68, 0.0, 69.0)
    mu_obs = _mu(z, *th) + rng.normal(0, 0.14, n)
    z_obs = z + (1 + z) * 0.04 * rng.standard_normal(n)
    sig = np.full(n, 0.14)
    out, gz = oracle.snia_logjoint(z, z_obs, mu_obs, sig, 0.04, 3.0, 3.0, *th)
    ref = (stats.norm.logpdf(mu_obs, _mu(z, *th), sig).sum() + stats.norm.logpdf(z_obs, z, (1 + z) * 0.04).sum()
           + stats.gamma.logpdf(z, a=3.0, scale=1 / 3.0).sum())
    assert abs(float(out[0]) - ref) <= 1e-12 * abs(ref)


def test_perfect_data_value():
    z = np.array([0.1, 0.5, 1.2])
    th = (0.3, 0.7, 0.0, 70.0)
    sig = np.array([0.1, 0.14, 0.2])
    out, _ = oracle.snia_logjoint(z, z, _mu(z, *th), sig, 0.04, 3.0, 3.0, *th)
    ref = (-(np.log(sig) + 0.5 * np.log(2 * np.pi)).sum() - (np.log((1 + z) * 0.04) + 0.5 * np.log(2 * np.pi)).sum()
           + (3 * np.log(3.0) - np.log(2.0) + 2 * np.log(z) - 3 * z).sum())
    assert abs(float(out[0]) - ref) <= 1e-14 * abs(ref)


def test_gradients_by_finite_differences():
    rng = np.random.default_rng(1)
    n = 12
    z = rng.uniform(0.05, 1.5, n)
    th = [0.3, 0.65, 9e-5, 70.0]
    mu_obs = _mu(z, *th) + rng.normal(0, 0.14, n)
    z_obs = z + (1 + z) * 0.04 * rng.standard_normal(n)
    sig = np.full(n, 0.14)
    f = lambda zz, t: float(oracle.snia_logjoint(zz, z_obs, mu_obs, sig, 0.04, 3.0, 3.0, *t, with_grad=False)[0][0])
    out, gz = oracle.snia_logjoint(z, z_obs, mu_obs, sig, 0.04, 3.0, 3.0, *th)
    for p, h in enumerate((1e-6, 1e-6, 1e-8, 1e-4)):
        tp, tm = list(th), list(th)
        tp[p] += h; tm[p] -= h
        fd = (f(z, tp) - f(z, tm)) / (2 * h)
        assert abs(fd - float(out[1 + p])) <= 2e-6 * max(abs(float(out[1 + p])), 1.0), p
    for i in (0, 5, 11):
        zp, zm = z.copy(), z.copy()
        zp[i] += 1e-6; zm[i] -= 1e-6
        fd = (f(zp, th) - f(zm, th)) / 2e-6
        assert abs(fd - float(gz[i])) <= 1e-6 * max(abs(float(gz[i])), 1.0), i
