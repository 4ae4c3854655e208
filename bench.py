#!/usr/bin/env python
"""bench.py -- headline measurement (contract: see DESIGN.md "Measurement").

Default workload: BASELINE.json configs[2] ("config3"): fused forward + analytic VJP of the distance modulus for a VI
minibatch, 10^6 sorted mock-SN redshifts x 64 cosmology samples = 6.4e7 evals per step, FP64, OUTER mode.  This is
the configuration BASELINE.json's metric ("distance+gradient evals/sec (FP64) ...") and its >=50 %-of-FP64-peak target
are quoted on.  One step = one pass of the whole hot path (prep kernel, fused forward+VJP kernel, reduction).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config {3,4,5}] [--dtype {f64,f32}]

--config 4: the fused SN-Ia likelihood (10^6 SNe x 256 samples); --config 5: the stress config (1.03e7 per-element cosmologies, all
six outputs, forward + VJP).  --dtype f32: the FP32 variant of configs 3 and 5 (clearly not the headline: "dtype": "f32").

N > 1 (torchrun): ONE array of N x 10^6 redshifts is cut into contiguous shards (sharding.shard_bounds), every rank evaluates its
shard against all cosmologies (weak scaling) and the parameter gradients [4][S] are summed with one NCCL all-reduce per step -- the
only exchange the path has.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "distance+gradient evals/sec (FP64)"
UNIT = "evals/s"
WORKLOADS = {
    3: "config3: fwd+VJP of mu, OUTER, N=1e6 sorted z x S=64 cosmologies (6.4e7 evals/step)",
    4: "config4: fused SN-Ia log-likelihood + parameter gradients, N=1e6 SNe x S=256 samples (2.56e8 evals/step)",
    5: "config5: stress, ELEMENTWISE fwd+VJP of all six outputs, 1.03e7 per-element cosmologies (1.03e7 evals/step)",
}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, choices=[3, 4, 5])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--n", type=int, default=None, help="redshifts per rank (default: the config's size)")
    ap.add_argument("--S", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


# ------------------------------------------------------------------------------------------ oracle legs
def oracle_rate(config, n_sample, S_sample, threads=None):
    """Times the oracle as it stands on a bounded sample of the same workload; returns (evals/s, cores, sample text)."""
    import oracle
    from paper_2212_01937_b200 import workloads as W
    cores = threads or oracle.max_threads()
    if config == 5:
        w = W.config5(n=n_sample, n_struct=max(8, n_sample // 100))
        t0 = time.perf_counter()
        oracle.observables_batch(w.z, w.Om, w.OL, w.Or, w.H0, with_grad=True, threads=cores)
        dt = time.perf_counter() - t0
        return w.n_z / dt, cores, f"{w.n_z} rows of config5 (all six outputs + all gradients)"
    w = W.config3(n=n_sample, S=S_sample, seed=3)
    Or = w.Or if config == 3 else np.zeros_like(w.Or)
    t0 = time.perf_counter()
    for s in range(S_sample):
        oracle.observables_batch(w.z, w.Om[s:s + 1], w.OL[s:s + 1], Or[s:s + 1], w.H0[s:s + 1], with_grad=True, threads=cores)
    dt = time.perf_counter() - t0
    return n_sample * S_sample / dt, cores, f"{n_sample} redshifts x {S_sample} cosmologies of config{config} (mu + all gradients)"


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n_s, S_s = (20_000, 4) if args.config != 5 else (60_000, 1)
    # torchrun exports OMP_NUM_THREADS=1 to every rank; here the other ranks have exited, so rank 0 uses the host's cores as at N=1
    threads = len(os.sched_getaffinity(0)) if int(os.environ.get("WORLD_SIZE", "1")) > 1 else None
    for _ in range(args.warmup):
        oracle_rate(args.config, 2000, 1, threads)
    rates = []
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r, cores, sample = oracle_rate(args.config, n_s, S_s, threads)
        rates.append(r)
    dt = time.perf_counter() - t0
    value = float(np.mean(rates))          # evals/s of the timed oracle calls (input generation excluded)
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f80 (x87 long double quadrature)", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "step": f"bounded sample: {sample}"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "cpu_model": cpu_model()},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler(threading.Thread):
    def __init__(self, index=0, period=0.005):
        super().__init__(daemon=True)
        self.period, self.samples, self.reasons, self.stop_flag = period, [], set(), False
        self.max_mhz = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {getattr(nv, k): k for k in dir(nv) if k.startswith("nvmlClocksThrottleReason") and isinstance(getattr(nv, k), int)}
        while not self.stop_flag:
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if bit and (r & bit) == bit and "None" not in name and "All" not in name:
                        self.reasons.add(name.replace("nvmlClocksThrottleReason", ""))
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self):
        s = sorted(self.samples)
        return {"sm_mhz": (s[len(s) // 2] if s else None), "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons),
                "samples": len(s)}


# ------------------------------------------------------------------------------------------ our arm
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_2212_01937_b200 import binding as cb, workloads as W, roofline as RL, sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    f32 = args.dtype == "f32"
    fdt = torch.float32 if f32 else torch.float64
    npdt = np.float32 if f32 else np.float64
    t = lambda a, dt=None: torch.from_numpy(np.ascontiguousarray(a)).to(dev) if dt is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev).to(dt)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    cfg = args.config
    # ---- the case: device-resident step(), host-buffer e2e step, bookkeeping for the roofline
    if cfg == 3:
        # ONE job of world x n redshifts, cut contiguously over the ranks; the same cosmology samples everywhere
        w = W.config3_shard(args.n or 1_000_000, world, rank, S=args.S or 64)
        N, S = w.n_z, w.n_cosmo
        evals, which = N * S, w.which
        z, Om, OL, Or, H0, gout = t(w.z, fdt), t(w.Om), t(w.OL), t(w.Or), t(w.H0), t(w.grad_out, fdt)
        out = torch.empty((len(which), S, N), dtype=fdt, device=dev)     # forward values are written too
        gz = torch.empty(N, dtype=fdt, device=dev)
        gp = torch.empty((4, S), dtype=torch.float64, device=dev)
        st = torch.empty((S, N), dtype=torch.uint8, device=dev)
        ws = torch.empty(max(256, cb.workspace_bytes(N, S, cb.OUTER, which, True)), dtype=torch.uint8, device=dev)
        reduced = [gp]

        def step():
            cb.cosmo_vjp(z, Om, OL, Or, H0, gout, cb.OUTER, which, out=out, grad_z=gz, grad_params=gp, status=st, workspace=ws)

        hz, hOm, hOL, hOr, hH0, hg = (pin(a) for a in (w.z, w.Om, w.OL, w.Or, w.H0, w.grad_out))
        hgz, hgp = pin(np.empty(N)), pin(np.empty((4, S)))

        def e2e_step():      # the step's result: grad_z[N] and grad_params[4][S] (pinned), read back every step
            if f32:
                return None
            cb.cosmo_eval_host(hz, hOm, hOL, hOr, hH0, cb.OUTER, which, grad_out=hg, want_out=False, want_status=False, grad_z=hgz, grad_params=hgp)
            return hz.nbytes + hg.nbytes + 4 * hOm.nbytes, hgz.nbytes + hgp.nbytes
        key = "config3_vjp_mu_" + args.dtype
        kernel = f"k_outer<{'float' if f32 else 'double'},false,false,VJP,MU>"
        alg_bytes = RL.BYTES_PER_EVAL_C3[args.dtype] * evals
        l2_note = f"inputs larger than L2 (grad_out {gout.numel() * gout.element_size() >> 20} MB per step), no flush"
        cfg_extra = {"n_z_per_gpu": N, "n_cosmo": S, "mode": "OUTER", "which": list(which)}
    elif cfg == 4:
        N, S = args.n or 1_000_000, args.S or 256
        rng = np.random.default_rng(4 + 1000 * rank)
        zz = rng.uniform(0.01, 1.5, N)
        one = lambda v: t(np.array([v]))
        mu0, _ = cb.cosmo_eval(t(zz), one(0.3), one(0.7), one(0.0), one(70.0), cb.ELEMENTWISE, ("MU",))     # timing only: any mu source does
        mu_true = mu0[0, 0].cpu().numpy()
        w = W.config4(lambda *_: mu_true, n=N, S=S, seed=4)
        w.z = zz
        evals, which = N * S, ("MU",)
        z, mu_obs, sigma = t(w.z, fdt), t(w.extra["mu_obs"], fdt), t(w.extra["sigma"], fdt)
        Om, OL, Or, H0 = t(w.Om), t(w.OL), t(w.Or), t(w.H0)
        logL = torch.empty(S, dtype=torch.float64, device=dev)
        grad = torch.empty((4, S), dtype=torch.float64, device=dev)
        ws = torch.empty(max(256, cb.workspace_bytes(N, S, cb.OUTER, which, True)), dtype=torch.uint8, device=dev)
        reduced = [logL, grad]

        def step():
            cb.cosmo_snia_loglike(z, mu_obs, sigma, Om, OL, Or, H0, logL=logL, grad=grad, workspace=ws)

        hin = [torch.from_numpy(np.ascontiguousarray(a.astype(npdt) if i < 3 else a)).pin_memory()
               for i, a in enumerate((w.z, w.extra["mu_obs"], w.extra["sigma"], w.Om, w.OL, w.Or, w.H0))]
        hout = [torch.empty(S, dtype=torch.float64).pin_memory(), torch.empty((4, S), dtype=torch.float64).pin_memory()]

        def e2e_step():     # this call has no host-buffer twin in the C ABI: pinned copies in, the device call, pinned copies out
            d = [h.to(dev, non_blocking=True) for h in hin]
            cb.cosmo_snia_loglike(*d, logL=logL, grad=grad, workspace=ws)
            hout[0].copy_(logL, non_blocking=True); hout[1].copy_(grad, non_blocking=True)
            torch.cuda.synchronize()
            return sum(h.numel() * h.element_size() for h in hin), sum(h.numel() * h.element_size() for h in hout)
        key = "config4_snia_" + args.dtype
        kernel = f"k_outer<{'float' if f32 else 'double'},false,false,SNIA,MU>"
        alg_bytes = float(3 * N * (4 if f32 else 8) * ((S + 15) // 16))       # z, mu_obs, sigma re-read once per chunk of 16 samples (L2-resident)
        l2_note = "24 MB of data re-read per 16-sample chunk (L2-resident by design); 2 MB L2-flush write between steps is not needed: compute-bound"
        cfg_extra = {"n_sne_per_gpu": N, "n_samples": S, "mode": "OUTER"}
    else:
        w = W.config5(n=args.n or 10_000_000, n_struct=(args.n or 10_000_000) // 100, seed=5 + 1000 * rank)
        N = w.n_z
        evals, which = N, w.which
        z, Om, OL, Or, H0, gout = t(w.z, fdt), t(w.Om), t(w.OL), t(w.Or), t(w.H0), t(w.grad_out, fdt)
        out = torch.empty((6, 1, N), dtype=fdt, device=dev)
        gz = torch.empty(N, dtype=fdt, device=dev)
        gp = torch.empty((4, N), dtype=torch.float64, device=dev)
        st = torch.empty((1, N), dtype=torch.uint8, device=dev)
        ws = torch.empty(max(256, cb.workspace_bytes(N, N, cb.ELEMENTWISE, which, True)), dtype=torch.uint8, device=dev)
        reduced = []

        def step():
            cb.cosmo_vjp(z, Om, OL, Or, H0, gout, cb.ELEMENTWISE, which, out=out, grad_z=gz, grad_params=gp, status=st, workspace=ws)

        hz, hOm, hOL, hOr, hH0, hg = (pin(a) for a in (w.z, w.Om, w.OL, w.Or, w.H0, w.grad_out))

        ho, hgz, hgp, hst = (pin(np.empty(sh, dtype=dt_)) for sh, dt_ in (((6, 1, N), np.float64), ((N,), np.float64), ((4, N), np.float64),
                                                                          ((1, N), np.uint8)))

        def e2e_step():
            if f32:
                return None
            cb.cosmo_eval_host(hz, hOm, hOL, hOr, hH0, cb.ELEMENTWISE, which, grad_out=hg, out=ho, grad_z=hgz, grad_params=hgp, status=hst)
            return hz.nbytes + hg.nbytes + 4 * hOm.nbytes, ho.nbytes + hgz.nbytes + hgp.nbytes + hst.nbytes
        key = "config5_vjp_all_" + args.dtype
        kernel = f"k_elem<{'float' if f32 else 'double'},true,true,true> + k_elem_redo"
        eb = 4 if f32 else 8
        alg_bytes = float(N * (eb + 32 + 6 * eb + 6 * eb + eb + 32 + 1))     # z, 4 params, grad_out, out, grad_z, grad_params, status
        l2_note = f"inputs larger than L2 ({int(alg_bytes) >> 20} MB per step), no flush"
        cfg_extra = {"n_per_gpu": N, "mode": "ELEMENTWISE", "which": list(which)}

    def full_step():
        step()
        if world > 1 and reduced:
            sharding.allreduce_sums(*reduced)     # the path's only exchange: per-sample sums over the z shards
    step_fn = full_step

    for _ in range(max(3, args.warmup)):
        step_fn()
    barrier()

    # ---- timed region: device-resident inputs (grad_out alone is 512 MB > 126 MB L2, so no L2 flush is needed)
    sampler = ClockSampler(local)
    sampler.start()
    cb.profile(True)
    l0 = cb.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        step_fn()
    e1.record()
    barrier()
    ms_total = e0.elapsed_time(e1)
    launches = cb.launch_count() - l0
    k_ms, k_n = cb.profile_mean_ms()
    cb.profile(False)
    if world > 1:
        tt = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms_total = float(tt.item())
    ms_step = ms_total / args.steps
    value = evals * world / (ms_step * 1e-3)

    # ---- unprofiled repeat (the profile hook serialises host and device): this is the number reported
    barrier()
    e0.record()
    for _ in range(args.steps):
        step_fn()
    e1.record()
    barrier()
    ms2 = e0.elapsed_time(e1)
    if world > 1:
        tt = torch.tensor([ms2], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        ms2 = float(tt.item())
    sampler.stop_flag = True
    sampler.join(timeout=1.0)
    launches_per_step = launches // max(1, args.steps)
    ms_step = ms2 / args.steps
    value = evals * world / (ms_step * 1e-3)

    # ---- end to end through the host-buffer path: pinned host inputs -> H2D -> kernels -> D2H, every step
    e2e = None
    e2e_steps = max(2, min(args.steps, 5))
    if e2e_step() is not None:           # warm (allocates staging); None: no host-buffer entry point for this dtype
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            h2d, d2h = e2e_step()
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / e2e_steps
        if world > 1:
            tt = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
            e2e_s = float(tt.item())
        e2e = {"value": evals * world / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": e2e_s * 1e3,
               "api": "cosmo_eval_host (pinned host buffers, chunked over three streams)" if cfg != 4 else
                      "pinned torch copies around cosmo_snia_loglike (the call has no host-buffer twin)"}

    # ---- ALU roofline: FMA peak of the arithmetic type measured live with the library's probe, kernel time from CUDA events on its stream
    peak_tflops = None
    if rank == 0:
        for _ in range(2):
            cb.probe_fma(args.dtype, 148 * 16, 2048)
        torch.cuda.synchronize()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        best = 0.0
        for _ in range(5):
            p0.record()
            flops, _ = cb.probe_fma(args.dtype, 148 * 16, 8192)
            p1.record()
            torch.cuda.synchronize()
            best = max(best, flops / (p0.elapsed_time(p1) * 1e-3) / 1e12)
        peak_tflops = best
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    fpe = RL.FLOPS_PER_EVAL.get(key)
    pipe = RL.PIPE_INST_PER_EVAL.get(key)
    achieved = fpe * evals / (k_ms * 1e-3) / 1e12 if (fpe and k_ms > 0) else None
    full_size = (cfg == 3 and (N, S) == (1_000_000, 64)) or (cfg == 4 and (N, S) == (1_000_000, 256)) or (cfg == 5 and N == 10_300_000)
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": (achieved / peak_tflops) if (achieved and peak_tflops) else None,
                "traffic": RL.DRAM_TRAFFIC_BYTES_PER_LAUNCH.get(key) if full_size else None,
                "traffic_unit": "bytes/launch (ncu dram read+write, profiles/)",
                "algorithmic_bytes": alg_bytes,
                "pipe_frac": (pipe * evals / (k_ms * 1e-3)) / (peak_tflops * 0.5e12) if (pipe and k_ms > 0 and peak_tflops) else None,
                "kernel": kernel, "kernel_ms": k_ms, "kernel_launches_timed": k_n,
                "flops_per_eval": fpe, "flops_source": RL.SOURCE.get(key), "flops_build_matches": RL.csrc_hash() == RL.CAPTURED_CSRC_HASH,
                "peak_source": f"measured live: cosmo_probe_fma_{args.dtype} (8 FMA chains/thread)",
                "nominal_tflops": RL.NOMINAL_FP64_TFLOPS if not f32 else RL.NOMINAL_FP32_TFLOPS,
                "hbm_gbs_achieved": alg_bytes / (k_ms * 1e-3) / 1e9 if k_ms > 0 else None}
    cpu_baseline = None
    if not args.no_cpu_baseline:
        n_s, S_s = (100_000, 4) if cfg != 5 else (300_000, 1)
        oracle_rate(cfg, 2000, 1)
        r, cores, sample = oracle_rate(cfg, n_s, S_s)
        r1, _, sample1 = oracle_rate(cfg, n_s // 10, 1 if cfg == 5 else 2, threads=1)     # the paper's setting: one thread
        cpu_baseline = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample, "cpu_model": cpu_model(),
                        "single_thread": {"value": r1, "unit": UNIT, "cores": 1, "sample": sample1}}
    line = {"metric": METRIC if not f32 else METRIC.replace("FP64", "FP32 variant"), "value": value, "unit": UNIT, "n_gpus": world,
            "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
            "data": "synthetic",
            "config": dict({"workload": WORKLOADS[cfg] + (", FP64" if not f32 else ", FP32 variant"), "l2": l2_note,
                            "parallelism": f"z-shard x{world}"}, **cfg_extra),
            "clocks": sampler.summary(),
            "e2e": e2e,
            "gpu_launches": int(launches), "gpu_launches_per_step": int(launches_per_step),
            "roofline": roofline, "cpu_baseline": cpu_baseline}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
