"""Times every C-ABI call on the BASELINE.json configs (seeded synthetic inputs, device-resident, CUDA events).  A measurement
script beside bench.py, not part of the package.

    python bench_calls.py [--steps 10] [--small] [--only config2,config5]

One JSON line per config: evals/s of the whole call and the mean duration of its dominant kernel (library hook).
bench.py stays the headline (config 3); this is the per-config table quoted in DESIGN.md / profiles/.
"""
import argparse
import json

import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main():
    import torch
    from paper_2212_01937_b200 import binding as cb, workloads as W

    ap = argparse.ArgumentParser()
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--small", action="store_true", help="1/10 of the sizes (smoke)")
    ap.add_argument("--only", default="")
    args = ap.parse_args()
    f = 10 if args.small else 1
    dev = lambda a, dt=None: (torch.from_numpy(np.ascontiguousarray(a)).cuda() if dt is None
                              else torch.from_numpy(np.ascontiguousarray(a)).cuda().to(dt))
    rng = np.random.default_rng(0)

    def timed(fn, evals, name, extra=None):
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        cb.profile(True)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        k_ms, k_n = cb.profile_mean_ms()
        cb.profile(False)
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        line = {"config": name, "evals_per_call": int(evals), "ms_per_call": ms, "evals_per_s": evals / (ms * 1e-3),
                "dominant_kernel_ms": k_ms}
        line.update(extra or {})
        print(json.dumps(line), flush=True)

    def want(name):
        return not args.only or name in args.only.split(",")

    if want("config1"):
        w = W.config1()
        a = [dev(x) for x in (w.z, w.Om, w.OL, w.Or, w.H0)]
        timed(lambda: cb.cosmo_eval(*a, cb.ELEMENTWISE, w.which), w.n_z, "config1 fwd D_C,mu N=1e4 one cosmology f64")
    if want("config2"):
        w = W.config2(n=1_000_000 // f)
        a = [dev(x) for x in (w.z, w.Om, w.OL, w.Or, w.H0)]
        out = torch.empty((4, 1, w.n_z), dtype=torch.float64, device="cuda")
        st = torch.empty((1, w.n_z), dtype=torch.uint8, device="cuda")
        timed(lambda: cb.cosmo_eval(*a, cb.ELEMENTWISE, w.which, out=out, status=st), w.n_z,
              "config2 fwd D_C,D_M,t_L,d_abs per-element cosmology f64")
        timed(lambda: cb.cosmo_eval(*a, cb.ELEMENTWISE, ("DC", "DM"), out=out[:2], status=st), w.n_z,
              "config2 fwd D_C,D_M only per-element cosmology f64")
    if want("config3"):
        w = W.config3(n=1_000_000 // f)
        a = [dev(x) for x in (w.z, w.Om, w.OL, w.Or, w.H0)]
        g = dev(w.grad_out)
        S, N = w.n_cosmo, w.n_z
        out = torch.empty((1, S, N), dtype=torch.float64, device="cuda")
        gz = torch.empty(N, dtype=torch.float64, device="cuda")
        gp = torch.empty((4, S), dtype=torch.float64, device="cuda")
        st = torch.empty((S, N), dtype=torch.uint8, device="cuda")
        ws = torch.empty(cb.workspace_bytes(N, S, cb.OUTER, w.which, True), dtype=torch.uint8, device="cuda")
        timed(lambda: cb.cosmo_vjp(*a, g, cb.OUTER, w.which, out=out, grad_z=gz, grad_params=gp, status=st, workspace=ws), S * N,
              "config3 fwd+VJP mu OUTER f64")
        timed(lambda: cb.cosmo_eval(*a, cb.OUTER, w.which, out=out, status=st, workspace=ws), S * N, "config3 fwd only mu OUTER f64")
        a32 = [dev(w.z, torch.float32)] + a[1:]
        g32, out32, gz32 = g.to(torch.float32), out.to(torch.float32), gz.to(torch.float32)
        timed(lambda: cb.cosmo_vjp(*a32, g32, cb.OUTER, w.which, out=out32, grad_z=gz32, grad_params=gp, status=st, workspace=ws), S * N,
              "config3 fwd+VJP mu OUTER f32")
    if want("outer6"):
        # every plane in OUTER mode (the SBI use, PAPER.md:287 fn.24): 10^6 redshifts x 16 cosmologies, all six outputs
        w = W.config3(n=1_000_000 // f, S=16, which=("DC", "DM", "DL", "MU", "TL", "DABS"))
        a = [dev(x) for x in (w.z, w.Om, w.OL, w.Or, w.H0)]
        g = dev(w.grad_out)
        S, N = w.n_cosmo, w.n_z
        out = torch.empty((6, S, N), dtype=torch.float64, device="cuda")
        gz = torch.empty(N, dtype=torch.float64, device="cuda")
        gp = torch.empty((4, S), dtype=torch.float64, device="cuda")
        st = torch.empty((S, N), dtype=torch.uint8, device="cuda")
        ws = torch.empty(cb.workspace_bytes(N, S, cb.OUTER, w.which, True), dtype=torch.uint8, device="cuda")
        timed(lambda: cb.cosmo_vjp(*a, g, cb.OUTER, w.which, out=out, grad_z=gz, grad_params=gp, status=st, workspace=ws), S * N,
              "OUTER all six outputs fwd+VJP, N=1e6 x S=16 f64")
        timed(lambda: cb.cosmo_eval(*a, cb.OUTER, w.which, out=out, status=st, workspace=ws), S * N, "OUTER all six outputs fwd only, N=1e6 x S=16 f64")
    if want("config4"):
        n = 1_000_000 // f
        z = rng.uniform(0.01, 1.5, n)
        one = lambda v: dev(np.array([v]))
        mu, _ = cb.cosmo_eval(dev(z), one(0.3), one(0.7), one(0.0), one(70.0), cb.ELEMENTWISE, ("MU",))   # timing only: any mu source does
        w = W.config4(lambda zz, *p: mu[0, 0].cpu().numpy(), n=n, S=256, seed=4)
        a = [dev(x) for x in (z, w.extra["mu_obs"], w.extra["sigma"], w.Om, w.OL, w.Or, w.H0)]
        logL = torch.empty(256, dtype=torch.float64, device="cuda")
        grad = torch.empty((4, 256), dtype=torch.float64, device="cuda")
        ws = torch.empty(cb.workspace_bytes(n, 256, cb.OUTER, ("MU",), True), dtype=torch.uint8, device="cuda")
        timed(lambda: cb.cosmo_snia_loglike(*a, logL=logL, grad=grad, workspace=ws), 256 * n, "config4 fused SN-Ia logL + grad S=256 f64")
    if want("logjoint"):
        n, S = 1_000_000 // f, 64
        zt = rng.gamma(3.0, 1 / 3.0, n) + 0.02
        one = lambda v: dev(np.array([v]))
        mu, _ = cb.cosmo_eval(dev(zt), one(0.3), one(0.7), one(0.0), one(70.0), cb.ELEMENTWISE, ("MU",))
        mu_obs = mu[0, 0] + 0.14 * torch.randn(n, dtype=torch.float64, device="cuda")
        z_obs = dev(zt + (1 + zt) * 0.04 * rng.standard_normal(n))
        z = (z_obs[None, :] + 0.03 * torch.randn((S, n), dtype=torch.float64, device="cuda")).abs() + 0.01
        sig = torch.full((n,), 0.14, dtype=torch.float64, device="cuda")
        P = [dev(rng.normal(0.3, 0.03, S)), dev(rng.normal(0.7, 0.03, S)), dev(np.zeros(S)), dev(rng.normal(70, 1, S))]
        ws = torch.empty(cb.workspace_bytes(n, S, cb.OUTER, ("MU",), True), dtype=torch.uint8, device="cuda")
        timed(lambda: cb.cosmo_snia_logjoint(z, z_obs, mu_obs.contiguous(), sig, 0.04, 3.0, 3.0, *P, workspace=ws), S * n,
              "section-4 log-joint with latent z (one VI step): N=1e6 SNe x S=64 samples, logp + grad_params + grad_z f64")
    if want("twolimit"):
        n = 1_000_000 // f
        z1 = dev(rng.uniform(0.0, 3.0, n)); z2 = z1 + dev(10.0 ** rng.uniform(-3.0, 0.8, n))
        P = [dev(rng.uniform(0.08, 0.6, n)), dev(rng.uniform(0.0, 1.2, n)), dev(rng.choice([0.0, 1e-5, 9e-5, 1e-3], n)), dev(rng.uniform(60, 80, n))]
        timed(lambda: cb.cosmo_eval2(z1, z2, *P, which=("DC", "DM", "TL", "DABS", "DA")), n,
              "two-limit forms (z1, z2), five outputs, per-element cosmology, forward f64")
        g = torch.randn((5, n), dtype=torch.float64, device="cuda")
        timed(lambda: cb.cosmo_eval2(z1, z2, *P, which=("DC", "DM", "TL", "DABS", "DA"), grad_out=g), n,
              "two-limit forms (z1, z2), five outputs, per-element cosmology, forward + VJP f64")
    if want("wmix"):
        w = W.wmix(n=1_000_000 // f)
        a = [dev(w[k]) for k in ("z", "Om", "OL", "Or", "Ow13", "Ow23", "H0")]
        timed(lambda: cb.cosmo_eval_w(*a, which=("DC", "DM", "DL", "MU")), len(w["z"]),
              "extra-w family (general quartic), D_C, D_M, D_L, mu + d/dz, per-element cosmology f64")
        gw = torch.randn((6, len(w["z"])), dtype=torch.float64, device="cuda")
        timed(lambda: cb.cosmo_eval_w(*a, which=("DC", "DM", "DL", "MU", "TL", "DABS"), grad_out=gw), len(w["z"]),
              "extra-w family (general quartic), all six outputs forward + VJP (6 parameter gradients), per-element cosmology f64")
        one = [dev(np.array([x])) for x in (0.27, 0.55, 8e-5, 0.06, 0.09, 70.0)]
        timed(lambda: cb.cosmo_eval_w(a[0], *one, which=("DC", "DM", "DL", "MU")), len(w["z"]),
              "extra-w family (general quartic), D_C, D_M, D_L, mu + d/dz, one shared cosmology f64")
    if want("config5"):
        w = W.config5(n=10_000_000 // f, n_struct=100_000 // f)
        a = [dev(x) for x in (w.z, w.Om, w.OL, w.Or, w.H0)]
        N = w.n_z
        g = torch.randn((6, 1, N), dtype=torch.float64, device="cuda")
        out = torch.empty((6, 1, N), dtype=torch.float64, device="cuda")
        gz = torch.empty(N, dtype=torch.float64, device="cuda")
        gp = torch.empty((4, N), dtype=torch.float64, device="cuda")
        st = torch.empty((1, N), dtype=torch.uint8, device="cuda")
        timed(lambda: cb.cosmo_vjp(*a, g, cb.ELEMENTWISE, w.which, out=out, grad_z=gz, grad_params=gp, status=st), N,
              "config5 fwd+VJP all six outputs per-element cosmology f64")
        timed(lambda: cb.cosmo_eval(*a, cb.ELEMENTWISE, w.which, out=out, status=st), N, "config5 fwd all six outputs f64")
        a32 = [dev(w.z, torch.float32)] + a[1:]
        g32, out32, gz32 = g.to(torch.float32), out.to(torch.float32), gz.to(torch.float32)
        timed(lambda: cb.cosmo_vjp(*a32, g32, cb.ELEMENTWISE, w.which, out=out32, grad_z=gz32, grad_params=gp, status=st), N,
              "config5 fwd+VJP all six outputs f32")


if __name__ == "__main__":
    main()
