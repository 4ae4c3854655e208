"""cosmo_snia_loglike_static: the fused SN-Ia likelihood with its scratch in a static device array (no workspace, no allocation), for
callers that cannot call cudaMalloc.  Checked against the existing workspace path cosmo_snia_loglike on two calls in a row (the second
smaller than the first, so that stale scratch of the first call would show), plus the size limit.  Collected last on purpose
(pytest -x must not lose other tests to a failure here); passes alone in a fresh process and after the others."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cb():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    from paper_2212_01937_b200 import binding
    binding.lib()
    return binding


def _case(seed, N, S):
    rng = np.random.default_rng(seed)
    z = rng.uniform(0.01, 1.5, N)
    mu_obs = 5.0 * np.log10((1 + z) * z * 4282.7) + 25.0 + rng.normal(0.0, 0.1, N)      # any plausible data: only path equality is tested
    sigma = rng.uniform(0.05, 0.2, N)
    Om = rng.normal(0.3, 0.05, S); OL = rng.normal(0.7, 0.05, S); H0 = rng.normal(70.0, 2.0, S)
    Or = np.where(np.arange(S) % 2 == 0, 0.0, 9e-5)
    return z, mu_obs, sigma, Om, OL, Or, H0


def test_static_scratch_matches_workspace_path_twice(cb):
    import torch
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    assert cb.static_scratch_bytes() == 24 << 20
    for call, (seed, N, S) in enumerate(((1, 200_003, 70), (2, 30_011, 9))):          # ragged tails; second call smaller than the first
        a = [dev(x) for x in _case(seed, N, S)]
        ref_L, ref_g = cb.cosmo_snia_loglike(*a)
        logL = torch.full((S,), float("nan"), dtype=torch.float64, device="cuda")
        grad = torch.full((4, S), float("nan"), dtype=torch.float64, device="cuda")
        torch.cuda.synchronize()
        free0 = torch.cuda.mem_get_info()[0]
        cb.cosmo_snia_loglike_static(*a, logL=logL, grad=grad)
        torch.cuda.synchronize()
        if call == 1:                      # (the first use on a device may load the module: not an allocation of the call itself)
            assert torch.cuda.mem_get_info()[0] == free0, "the static-scratch call changed the amount of free device memory"
        L, g, rL, rg = logL.cpu().numpy(), grad.cpu().numpy(), ref_L.cpu().numpy(), ref_g.cpu().numpy()
        assert np.isfinite(L).all() and np.isfinite(g).all()
        # same kernels, same summation order: agreement to rounding; asserted at the tolerances the parity tests use (1e-10 on logL,
        # 1e-8 on gradients relative to the larger of the two)
        assert np.abs(L - rL).max() <= 1e-10 * np.abs(rL).max(), (call, np.abs(L - rL).max())
        assert (np.abs(g - rg) <= 1e-8 * np.maximum(np.abs(rg), np.abs(rg).max(axis=1, keepdims=True) * 1e-6)).all(), call
        assert np.array_equal(L, rL) and np.array_equal(g, rg), "same kernels and grid: expected bit-identical results"
    # want_grad = False, and the empty batch
    a = [dev(x) for x in _case(3, 4096, 3)]
    L1, g1 = cb.cosmo_snia_loglike_static(*a, want_grad=False)
    assert g1 is None and np.array_equal(L1.cpu().numpy(), cb.cosmo_snia_loglike(*a)[0].cpu().numpy())
    e = torch.empty(0, dtype=torch.float64, device="cuda")
    L0, g0 = cb.cosmo_snia_loglike_static(e, e, e, *a[3:])
    assert (L0 == 0).all() and (g0 == 0).all()


def test_static_scratch_rejects_sizes_beyond_its_maximum(cb):
    import torch
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda()
    # BASELINE.json config 4 (S = 256, N = 1e6) fits; twice the supernovae does not: 40 S ceil(N/512) bytes of partial sums
    S = 256
    z, mu_obs, sigma, Om, OL, Or, H0 = _case(4, 16, S)
    big = torch.zeros(2_100_000, dtype=torch.float64, device="cuda") + 0.5
    logL = torch.full((S,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(cb.CosmoError, match="static scratch"):
        cb.cosmo_snia_loglike_static(big, big, big, dev(Om), dev(OL), dev(Or), dev(H0), logL=logL)
    torch.cuda.synchronize()
    assert (logL == 7.0).all()             # nothing was launched
    ok = torch.zeros(1_000_000, dtype=torch.float64, device="cuda") + 0.5
    cb.cosmo_snia_loglike_static(ok, ok + 42.0, ok, dev(Om), dev(OL), dev(Or), dev(H0), logL=logL)
    torch.cuda.synchronize()
    assert torch.isfinite(logL).all()
