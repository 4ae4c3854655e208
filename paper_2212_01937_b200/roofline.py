"""Roofline bookkeeping for bench.py (no arithmetic of the method lives here).

The hot path is bound by the plain FP64 ALUs (nothing is a dense contraction; HBM traffic is <= 16 B per eval).
`achieved` = algorithmic FP64 flops per launch / kernel time, where the per-eval figure is the count of FP64
instructions the kernel executes per (z, cosmology) pair, measured ONCE with Nsight Compute SASS counters
(smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum, 2 flops per DFMA; profiles/ holds the capture and
DESIGN.md "Roofline" the derivation).  `peak` = the DFMA rate bench.py measures live with the library's FMA-chain
probe (cosmo_probe_fma_f64); the nominal figure beside it is 148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz.
"""

# FP64 work per eval of the config-3 fused forward+VJP kernel k_outer<double,false,false,VJP,MU> as committed, from the
# ncu captures profiles/r01b_k_outer_vjp.md and (re-captured for the committed build, same counts) profiles/r01c_k_outer_vjp.md
# (6.4e7 evals/launch):
#   DFMA 137.4, DMUL 98.7, DADD 24.5 thread-instructions per eval -> 2*137.4 + 98.7 + 24.5 = 397.9 flops
#   FP64-pipe instructions per eval (the above + 5.3 DSETP) = 265.9
# (earlier builds: profiles/r01_final_k_outer_vjp.md 430.6 flops / 300.1 pipe instructions; first working version,
#  profiles/r01_k_outer_vjp.md: 774.8 / 513.7.  Fewer flops for the same result is the point: compare evals/s across
#  builds, and the roofline fraction within one.)
FLOPS_PER_EVAL = {
    "config3_vjp_mu_f64": 397.9,
}
# instructions per eval on the arithmetic pipe of the dtype (FP64: DFMA + DMUL + DADD + DSETP)
PIPE_INST_PER_EVAL = {
    "config3_vjp_mu_f64": 265.9,
}
# dram__bytes_read.sum + dram__bytes_write.sum of that kernel, per launch (same capture)
DRAM_TRAFFIC_BYTES_PER_LAUNCH = {
    "config3_vjp_mu_f64": 544.13e6 + 635.70e6,
}
# where each entry comes from
SOURCE = {
    "config3_vjp_mu_f64": "profiles/r01c_k_outer_vjp.md",
}

# nominal B200 vector peaks (context only; the denominator is the measured probe): 148 SMs x lanes x 2 x 1.965 GHz
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12

# algorithmic HBM bytes per eval, config 3 as bench.py runs it (z, params and constants stay on chip): grad_out read, out + status
# written, z / grad_z amortised over S
BYTES_PER_EVAL_C3 = {"f64": 8.0 + 8.0 + 1.0 + (8.0 + 8.0) / 64.0, "f32": 4.0 + 4.0 + 1.0 + (4.0 + 4.0) / 64.0}
