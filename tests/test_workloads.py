"""The seeded input generators: determinism, shapes, ranges and structure.  CPU only."""
import numpy as np

from paper_2212_01937_b200 import workloads as W


def test_deterministic_and_shapes():
    a, b = W.config2(n=5000), W.config2(n=5000)
    assert np.array_equal(a.z, b.z) and np.array_equal(a.Or, b.Or)
    assert a.mode == "elementwise" and a.n_cosmo == a.n_z == 5000 and a.which == ("DC", "DM", "TL", "DABS")
    assert (a.Or >= 1e-5).all() and (a.Or <= 1e-3).all() and (W.e2_min_on_path(a.z, a.Om, a.OL, a.Or) > 0).all()
    c1 = W.config1()
    assert c1.n_z == 10_000 and c1.n_cosmo == 1 and c1.z.min() >= 0.01 and c1.z.max() <= 2.0
    c3 = W.config3(n=4096, S=8)
    assert c3.mode == "outer" and c3.n_evals == 8 * 4096 and c3.grad_out.shape == (1, 8, 4096)
    assert np.all(np.diff(c3.z) >= 0) and np.all(c3.Or == 9e-5)
    c4 = W.config4(lambda z, *p: 5 * np.log10(z) + 43.0, n=1000, S=16)
    assert c4.extra["mu_obs"].shape == (1000,) and np.all(c4.extra["sigma"] == 0.1) and np.all(c4.Or == 0.0)


def test_config5_structure():
    w = W.config5(n=20_000, n_struct=2_000)
    Ok = 1.0 - w.Om - w.OL - w.Or
    assert w.n_z == 26_000 and np.all(np.abs(Ok) <= 0.5 + 1e-12) and np.all(w.OL >= 0) and np.all(w.Om > 0)
    assert set(np.unique(w.Or)) == {0.0, 9e-5, 1e-3}
    assert (W.e2_min_on_path(w.z, w.Om, w.OL, w.Or) > 0).all()
    a0, a1 = w.extra["blocks"]["a_boundary"]
    x_d, delta = w.extra["info"]["a_boundary"]["x_d"], w.extra["info"]["a_boundary"]["delta"]
    # block a: E^2 at the would-be double root equals -delta (1 - x_d^2) > 0 and small; z is past it
    e2 = w.Or[a0:a1] * x_d ** 4 + w.Om[a0:a1] * x_d ** 3 + Ok[a0:a1] * x_d ** 2 + w.OL[a0:a1]
    np.testing.assert_allclose(e2, delta * (x_d ** 2 - 1), rtol=1e-6, atol=1e-13)
    assert np.all(1 + w.z[a0:a1] > x_d)
    b0, b1 = w.extra["blocks"]["b_real_pair"]
    xc, gap = w.extra["info"]["b_real_pair"]["x_c"], w.extra["info"]["b_real_pair"]["gap"]
    for x in (xc - gap / 2, xc + gap / 2):      # both are roots of E^2, inside (0,1)
        e2 = w.Or[b0:b1] * x ** 4 + w.Om[b0:b1] * x ** 3 + Ok[b0:b1] * x ** 2 + w.OL[b0:b1]
        assert np.all(np.abs(e2) < 1e-11) and np.all((x > 0) & (x < 1))
    c0, c1 = w.extra["blocks"]["c_cc_pair_re_gt_1"]
    rho = w.extra["info"]["c_cc_pair_re_gt_1"]["x_re"] + 1j * w.extra["info"]["c_cc_pair_re_gt_1"]["x_im"]
    e2 = w.Or[c0:c1] * rho ** 4 + w.Om[c0:c1] * rho ** 3 + Ok[c0:c1] * rho ** 2 + w.OL[c0:c1]
    assert np.all(np.abs(e2) < 1e-10) and np.all(rho.real > 1)


def test_invalid_rows_are_invalid():
    for z, Om, OL, Or, H0, bit in W.invalid_rows():
        if bit == 1:
            assert not (W.e2_min_on_path(z, Om, OL, Or) > 0)
