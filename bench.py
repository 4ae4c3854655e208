#!/usr/bin/env python
"""bench.py -- headline measurement (contract: see DESIGN.md "Measurement").

Workload: BASELINE.json configs[2] ("config3"): fused forward + analytic VJP of the distance modulus for a VI
minibatch, 10^6 sorted mock-SN redshifts x 64 cosmology samples = 6.4e7 evals per step, FP64, OUTER mode.  This is
the configuration BASELINE.json's metric ("distance+gradient evals/sec (FP64) ...") and its >=50 %-of-FP64-peak target
are quoted on.  One step = one pass of the whole hot path (prep kernel, fused forward+VJP kernel, reduction).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]

N > 1 (torchrun): every rank evaluates its own 10^6-redshift shard against all 64 cosmologies (weak scaling) and the
parameter gradients [4][64] are summed with one NCCL all-reduce per step -- the only exchange the path has.
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
WORKLOAD = "config3: fwd+VJP of mu, OUTER, N=1e6 sorted z x S=64 cosmologies (6.4e7 evals/step), FP64"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=1_000_000, help="redshifts per rank (default: the config's 10^6)")
    ap.add_argument("--S", type=int, default=64)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------ oracle legs
def oracle_rate(n_sample, S_sample, threads=None, seed=3):
    """Times the oracle as it stands on a bounded sample of the same workload; returns (evals/s, cores, sample text)."""
    import oracle
    rng = np.random.default_rng(seed)
    z = np.sort(rng.uniform(0.01, 1.5, n_sample))
    Om = rng.normal(0.3, 0.05, S_sample); OL = rng.normal(0.7, 0.05, S_sample); H0 = rng.normal(70.0, 2.0, S_sample)
    Or = np.full(S_sample, 9e-5)
    cores = threads or oracle.max_threads()
    t0 = time.perf_counter()
    for s in range(S_sample):
        oracle.observables_batch(z, Om[s:s + 1], OL[s:s + 1], Or[s:s + 1], H0[s:s + 1], with_grad=True, threads=cores)
    dt = time.perf_counter() - t0
    return n_sample * S_sample / dt, cores, f"{n_sample} redshifts x {S_sample} cosmologies of config3 (values + all gradients)"


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    n_s, S_s = 20_000, 4
    rates = []
    # torchrun exports OMP_NUM_THREADS=1 to every rank; here the other ranks have exited, so rank 0 uses the host's cores as at N=1
    threads = len(os.sched_getaffinity(0)) if int(os.environ.get("WORLD_SIZE", "1")) > 1 else None
    for _ in range(args.warmup):
        oracle_rate(2000, 1, threads)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r, cores, sample = oracle_rate(n_s, S_s, threads)
        rates.append(r)
    dt = time.perf_counter() - t0
    value = args.steps * n_s * S_s / dt
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f80 (x87 long double quadrature)", "data": "synthetic",
            "config": {"workload": WORKLOAD, "step": f"bounded sample: {sample}"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
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

    # seeded synthetic inputs of the config's shape; each rank draws its own redshift shard (same cosmology samples)
    w = W.config3(n=args.n, S=args.S, seed=3)
    if rank > 0:
        rng = np.random.default_rng(1000 + rank)
        w.z = np.sort(rng.uniform(0.01, 1.5, args.n))
        w.grad_out = rng.standard_normal(w.grad_out.shape)
    N, S = w.n_z, w.n_cosmo
    evals = N * S
    which = w.which
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    z, Om, OL, Or, H0, gout = t(w.z), t(w.Om), t(w.OL), t(w.Or), t(w.H0), t(w.grad_out)
    out = torch.empty((len(which), S, N), dtype=torch.float64, device=dev)     # forward values are written too
    gz = torch.empty(N, dtype=torch.float64, device=dev)
    gp = torch.empty((4, S), dtype=torch.float64, device=dev)
    st = torch.empty((S, N), dtype=torch.uint8, device=dev)
    ws = torch.empty(max(256, cb.workspace_bytes(N, S, cb.OUTER, which, True)), dtype=torch.uint8, device=dev)

    def step():
        cb.cosmo_vjp(z, Om, OL, Or, H0, gout, cb.OUTER, which, out=out, grad_z=gz, grad_params=gp, status=st, workspace=ws)
        if world > 1:
            sharding.allreduce_sums(gp)     # the path's only exchange: [4][S] parameter-gradient sums over the z shards

    for _ in range(max(3, args.warmup)):
        step()
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
        step()
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
        step()
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

    # ---- end to end through the host-buffer C-ABI call: pinned host inputs -> H2D -> kernels -> D2H, every step
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()
    hz, hOm, hOL, hOr, hH0, hg = (pin(a) for a in (w.z, w.Om, w.OL, w.Or, w.H0, w.grad_out))
    e2e_steps = max(2, min(args.steps, 5))
    cb.cosmo_eval_host(hz, hOm, hOL, hOr, hH0, cb.OUTER, which, grad_out=hg, want_out=False, want_status=False)   # warm (allocates scratch)
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        _, gz_h, gp_h, _ = cb.cosmo_eval_host(hz, hOm, hOL, hOr, hH0, cb.OUTER, which, grad_out=hg, want_out=False, want_status=False)
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    if world > 1:
        tt = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e_s = float(tt.item())
    h2d = hz.nbytes + hg.nbytes + 4 * hOm.nbytes
    d2h = gz_h.nbytes + gp_h.nbytes

    # ---- ALU roofline: DFMA peak measured live with the library's probe, kernel time from CUDA events on its stream
    peak_tflops = None
    if rank == 0:
        for _ in range(2):
            cb.probe_fma("f64", 148 * 16, 2048)
        torch.cuda.synchronize()
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        best = 0.0
        for _ in range(5):
            p0.record()
            flops, _ = cb.probe_fma("f64", 148 * 16, 8192)
            p1.record()
            torch.cuda.synchronize()
            best = max(best, flops / (p0.elapsed_time(p1) * 1e-3) / 1e12)
        peak_tflops = best
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return
    fpe = RL.FLOPS_PER_EVAL["config3_vjp_mu_f64"]
    achieved = fpe * evals / (k_ms * 1e-3) / 1e12 if k_ms > 0 else None
    roofline = {"bound": "alu", "achieved": achieved, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": (achieved / peak_tflops) if (achieved and peak_tflops) else None,
                "traffic": RL.DRAM_TRAFFIC_BYTES_PER_LAUNCH["config3_vjp_mu_f64"] if (N, S) == (1_000_000, 64) else None,
                "traffic_unit": "bytes/launch (ncu dram read+write, profiles/r01c_k_outer_vjp.md)",
                "algorithmic_bytes": RL.BYTES_PER_EVAL_C3 * evals,
                "fp64_pipe_frac": (RL.FP64_PIPE_INST_PER_EVAL["config3_vjp_mu_f64"] * evals / (k_ms * 1e-3)) / (peak_tflops * 0.5e12)
                if (k_ms > 0 and peak_tflops) else None,
                "kernel": "k_outer<double,false,false,VJP,MU>", "kernel_ms": k_ms, "kernel_launches_timed": k_n,
                "flops_per_eval": fpe, "peak_source": "measured live: cosmo_probe_fma_f64 (8 DFMA chains/thread)",
                "nominal_fp64_tflops": RL.NOMINAL_FP64_TFLOPS,
                "hbm_gbs_achieved": RL.BYTES_PER_EVAL_C3 * evals / (k_ms * 1e-3) / 1e9 if k_ms > 0 else None}
    cpu_baseline = None
    if not args.no_cpu_baseline:
        oracle_rate(2000, 1)
        r, cores, sample = oracle_rate(100_000, 4)
        cpu_baseline = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": WORKLOAD, "n_z_per_gpu": N, "n_cosmo": S, "mode": "OUTER", "which": list(which),
                       "l2": "inputs larger than L2 (grad_out 512 MB per step), no flush", "parallelism": f"z-shard x{world}"},
            "clocks": sampler.summary(),
            "e2e": {"value": evals * world / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "ms_per_step": e2e_s * 1e3, "api": "cosmo_eval_host (pinned host buffers)"},
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
