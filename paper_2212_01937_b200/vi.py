"""Minimal variational-inference loop for the section-4 toy model: SURVEY NEXT-2, second half.

Model: latent redshifts z_s ~ Gamma(shape, rate beta), z_obs | z ~ N(z, (1+z)^2 sigma_z^2),
mu_obs | z, theta ~ N(mu(z; theta), sigma_mu^2), theta = (Om, OL), radiation-less, H0 fixed.

Guide ("partial multivariate normal"): correlations among the two global parameters and between them and each
supernova's latent redshift, none between different supernovae.  The definition is in ref. [41], which is not in the
container; the reading used here (DESIGN.md R-pmvn) is the reparameterisation

    theta = m + L eps_g,                 eps_g ~ N(0, I_2),   L lower triangular with positive diagonal
    z_s   = a_s + c_s . eps_g + d_s e_s, e_s ~ N(0, 1),       d_s > 0

i.e. a multivariate normal whose Cholesky factor has an arrow pattern; entropy = sum log L_ii + sum log d_s + const.

Every evaluation of the model and of its gradients wrt (theta, z) is ONE call of `cosmo_snia_logjoint` (the fused CUDA
kernel); this file only draws the guide's samples, forms the reparameterised ELBO gradient from the kernel's outputs and
takes Adam steps -- torch tensor plumbing on the same device.  There is no autograd tape anywhere.
"""
import math


def mock_snia(n, *, Om=0.3, OL=0.7, H0=70.0, sigma_mu=0.14, sigma_z=0.04, beta=3.0, shape=3.0, seed=0, device="cuda"):
    """Mock data of the toy model (figure 4a): returns dict of device tensors z_true, z_obs, mu_obs, sigma_mu."""
    import torch
    from . import binding as cb
    g = torch.Generator(device=device).manual_seed(seed)
    # Gamma(shape, beta) for integer shape as a sum of exponentials (keeps the generator explicit and seeded)
    k = int(round(shape))
    if abs(shape - k) > 1e-12 or k < 1:
        raise ValueError("mock_snia draws integer gamma shapes only")
    u = torch.rand((k, n), dtype=torch.float64, device=device, generator=g)
    z = -torch.log1p(-u).sum(0) / beta
    one = lambda v: torch.tensor([v], dtype=torch.float64, device=device)
    mu, _ = cb.cosmo_eval(z, one(Om), one(OL), one(0.0), one(H0), cb.ELEMENTWISE, ("MU",))
    mu_obs = mu[0, 0] + sigma_mu * torch.randn(n, dtype=torch.float64, device=device, generator=g)
    z_obs = z + (1.0 + z) * sigma_z * torch.randn(n, dtype=torch.float64, device=device, generator=g)
    return {"z_true": z, "z_obs": z_obs, "mu_obs": mu_obs.contiguous(),
            "sigma_mu": torch.full((n,), sigma_mu, dtype=torch.float64, device=device)}


class _Adam:
    """Adam on a list of tensors with explicit gradients (ascent)."""

    def __init__(self, params, lrs, b1=0.9, b2=0.95, eps=1e-8):
        import torch
        self.p, self.lr, self.b1, self.b2, self.eps, self.t = params, lrs, b1, b2, eps, 0
        self.m = [torch.zeros_like(x) for x in params]
        self.v = [torch.zeros_like(x) for x in params]

    def step(self, grads, scale=1.0):
        self.t += 1
        c1, c2 = 1.0 - self.b1 ** self.t, 1.0 - self.b2 ** self.t
        for x, g, m, v, lr in zip(self.p, grads, self.m, self.v, self.lr):
            m.mul_(self.b1).add_(g, alpha=1.0 - self.b1)
            v.mul_(self.b2).addcmul_(g, g, value=1.0 - self.b2)
            x.add_((m / c1) / ((v / c2).sqrt() + self.eps), alpha=lr * scale)


def fit_snia_vi(z_obs, mu_obs, sigma_mu, *, sigma_z=0.04, beta=3.0, shape=3.0, H0=70.0, steps=400, n_samples=8, lr=0.02,
                init=(0.5, 0.5), seed=0, z_floor=1e-4, log_every=0):
    """Fit the PMVN guide by stochastic gradient ascent on the ELBO.  Returns a dict with the guide's parameters
    (`mean` [2], `chol` [2, 2], `cov` [2, 2], `z_mean` [N], `z_corr` [N, 2], `z_scale` [N]) and the ELBO trace."""
    import torch
    from . import binding as cb
    dev, f64 = z_obs.device, torch.float64
    N, S = z_obs.numel(), int(n_samples)
    g = torch.Generator(device=dev).manual_seed(seed)
    m = torch.tensor(init, dtype=f64, device=dev)
    Ld = torch.full((2,), math.log(0.05), dtype=f64, device=dev)          # log of the diagonal of L
    Lo = torch.zeros(1, dtype=f64, device=dev)                            # L[1, 0]
    a = z_obs.clamp_min(0.02).clone()
    c = torch.zeros((N, 2), dtype=f64, device=dev)
    ld = torch.log(0.5 * sigma_z * (1.0 + a))                             # log d_s
    # step sizes: the globals move on the scale of their posterior width, the per-supernova terms on that of sigma_z
    opt = _Adam([m, Ld, Lo, a, c, ld], [lr, 5.0 * lr, lr, 0.2 * lr, 0.2 * lr, 2.0 * lr])
    ws = torch.empty(cb.workspace_bytes(N, S, cb.OUTER, ("MU",), True), dtype=torch.uint8, device=dev)
    Or0 = torch.zeros(S, dtype=f64, device=dev)
    H0s = torch.full((S,), float(H0), dtype=f64, device=dev)
    trace = []
    for it in range(steps):
        eg = torch.randn((S, 2), dtype=f64, device=dev, generator=g)
        es = torch.randn((S, N), dtype=f64, device=dev, generator=g)
        Ldiag = Ld.exp()
        th0 = m[0] + Ldiag[0] * eg[:, 0]
        th1 = m[1] + Lo[0] * eg[:, 0] + Ldiag[1] * eg[:, 1]
        d = ld.exp()
        z = a[None, :] + eg @ c.T + d[None, :] * es
        inside = z > z_floor                                              # the support of the prior; clamped samples pass no gradient
        z = torch.where(inside, z, torch.full_like(z, z_floor)).contiguous()
        logp, gth, gz = cb.cosmo_snia_logjoint(z, z_obs, mu_obs, sigma_mu, sigma_z, beta, shape, th0.contiguous(), th1.contiguous(),
                                               Or0, H0s, workspace=ws)
        ok = torch.isfinite(logp)
        if not bool(ok.any()):
            raise RuntimeError("every guide sample left the model's domain; lower lr or change init")
        w = ok.to(f64) / ok.sum()
        gz = torch.where(inside & ok[:, None], gz, torch.zeros_like(gz))
        g0 = torch.where(ok, gth[0], torch.zeros_like(gth[0]))
        g1 = torch.where(ok, gth[1], torch.zeros_like(gth[1]))
        elbo = float((torch.where(ok, logp, torch.zeros_like(logp)) * w).sum() + Ld.sum() + ld.sum())
        trace.append(elbo)
        # reparameterised gradient of mean_s log p + entropy.  The terms that correlate a gradient with the noise that
        # produced it (scales and couplings) use the gradient minus its sample mean: E[eps] = 0, so this is the same
        # expectation (times (S-1)/S, undone below) without the large common part that vanishes only on average.
        gm = torch.stack([(g0 * w).sum(), (g1 * w).sum()])
        nok = float(ok.sum())
        ub = nok / max(nok - 1.0, 1.0)
        g0c = torch.where(ok, g0 - gm[0], torch.zeros_like(g0)) * ub
        g1c = torch.where(ok, g1 - gm[1], torch.zeros_like(g1)) * ub
        gLd = torch.stack([(g0c * eg[:, 0] * w).sum() * Ldiag[0] + 1.0, (g1c * eg[:, 1] * w).sum() * Ldiag[1] + 1.0])
        gLo = (g1c * eg[:, 0] * w).sum().reshape(1)
        gzw = gz * w[:, None]
        ga = gzw.sum(0)
        gzc = (gz - ga[None, :]) * (w * ub)[:, None]
        gc = gzc.T @ eg
        gld = (gzc * es).sum(0) * d + 1.0
        opt.step([gm, gLd, gLo, ga, gc, gld], scale=0.5 * (1.0 + math.cos(math.pi * it / steps)) * 0.95 + 0.05)
        if log_every and it % log_every == 0:
            print(f"step {it:5d}  ELBO {elbo:.4f}  mean {m.tolist()}  sd {Ld.exp().tolist()}", flush=True)
    Ldiag = Ld.exp()
    L = torch.zeros((2, 2), dtype=f64, device=dev)
    L[0, 0], L[1, 0], L[1, 1] = Ldiag[0], Lo[0], Ldiag[1]
    return {"mean": m, "chol": L, "cov": L @ L.T, "z_mean": a, "z_corr": c, "z_scale": ld.exp(), "elbo": trace}
