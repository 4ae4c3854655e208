"""The minimal VI loop of the section-4 toy model (paper_2212_01937_b200/vi.py).

The model evaluations are the fused log-joint kernel, whose parity with the oracle is tests/test_gpu_parity.py's job; what is
checked here is the loop around it: the optimiser, the reparameterised ELBO gradient (through its fixed point: the guide must
land on the parameters that generated the mock data, with a width that shrinks like 1/sqrt(N)) and the
shrinkage of the latent redshifts towards their true values.
"""
import math

import numpy as np
import pytest


def test_adam_ascent_reaches_the_maximum_of_a_quadratic():
    import torch
    from paper_2212_01937_b200.vi import _Adam
    x = torch.tensor([3.0, -2.0], dtype=torch.float64)
    target = torch.tensor([0.5, 1.5], dtype=torch.float64)
    opt = _Adam([x], [0.05])
    for it in range(2000):
        opt.step([-(x - target) * torch.tensor([1.0, 1e4], dtype=torch.float64)], scale=0.5 * (1 + math.cos(math.pi * it / 2000)))
    assert torch.allclose(x, target, atol=2e-3)


@pytest.mark.gpu
def test_vi_recovers_the_mock_cosmology_and_shrinks_like_inverse_sqrt_n():
    import torch
    assert torch.cuda.is_available()
    from paper_2212_01937_b200 import vi
    truth = np.array([0.3, 0.7])
    sd = {}
    for N in (2_000, 20_000):
        d = vi.mock_snia(N, Om=truth[0], OL=truth[1], seed=1)
        r = vi.fit_snia_vi(d["z_obs"], d["mu_obs"], d["sigma_mu"], steps=600, n_samples=8, seed=2)
        mean = r["mean"].cpu().numpy()
        cov = r["cov"].cpu().numpy()
        sd[N] = np.sqrt(np.diag(cov))
        elbo = np.array(r["elbo"])
        assert np.isfinite(elbo).all()
        assert elbo[-50:].mean() > elbo[:10].mean() + 0.4 * abs(elbo[:10].mean())          # starts far away (init 0.5, 0.5)
        # the guide ignores part of the posterior correlations, so its width is a lower bound: allow 6 widths + the
        # 1/sqrt(N) statistical scatter of the mock data itself
        assert (np.abs(mean - truth) <= 6 * sd[N] + 3.0 / math.sqrt(N)).all(), (N, mean, sd[N])
        assert np.all(np.linalg.eigvalsh(cov) > 0)
        # latent redshifts: the guide's means are closer to the truth than the photometric estimates they started from
        rms0 = float((d["z_obs"] - d["z_true"]).pow(2).mean().sqrt())
        rms1 = float((r["z_mean"] - d["z_true"]).pow(2).mean().sqrt())
        assert rms1 < 0.7 * rms0, (rms0, rms1)
        assert float(r["z_scale"].min()) > 0
    ratio = sd[20_000] / sd[2_000]
    assert (ratio < 0.5).all() and (ratio > 0.15).all(), ratio          # 1/sqrt(10) = 0.32
