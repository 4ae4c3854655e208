"""Roofline bookkeeping for bench.py (no arithmetic of the method lives here).

The hot path is bound by the plain FP64 ALUs (nothing is a dense contraction; HBM traffic is <= 16 B per eval).
`achieved` = algorithmic FP64 flops per launch / kernel time, where the per-eval figure is the count of FP64
instructions the kernel executes per (z, cosmology) pair, measured ONCE with Nsight Compute SASS counters
(smsp__sass_thread_inst_executed_op_{dfma,dmul,dadd}_pred_on.sum, 2 flops per DFMA; profiles/ holds the capture and
DESIGN.md "Roofline" the derivation).  `peak` = the DFMA rate bench.py measures live with the library's FMA-chain
probe (cosmo_probe_fma_f64); the nominal figure beside it is 148 SMs x 64 FP64 FMA lanes x 2 x 1.965 GHz.
"""

# Arithmetic work per eval of the dominant kernel of each bench.py arm, from Nsight Compute SASS counters of the committed build
# (profiles/r02_k_outer_vjp.md, profiles/r02_other_kernels.md + .csv).  flops = 2 x FMA + MUL + ADD of the arithmetic type; "pipe"
# = instructions that occupy that type's pipe.  Fewer flops for the same result is the point of most optimisations here: compare evals/s
# across builds, and the roofline fraction within one.  (Round 1: config 3 397.9 flops / 265.9 pipe instructions.)
#   config3_vjp_mu_f64  k_outer<double,0,0,VJP,MU>, 6.4e7 evals/launch: DFMA 135.05, DMUL 98.23, DADD 25.23 per eval
#   config3_vjp_mu_f32  k_outer<float,0,0,VJP,MU>:  FFMA 78.47, FMUL 80.14, FADD 13.70 per eval (204.7 FP32 instructions in all)
#   config4_snia_f64    k_outer<double,0,0,SNIA,MU>, 2.56e8 evals/launch: DFMA 150.60, DMUL 105.40, DADD 35.41 per eval
#   config5_vjp_all_f64 k_elem<double,1,1,1,0> (+ k_elem_redo on 2.5 % of the elements), 1.03e7 evals: DFMA 1036.6, DMUL 602.6, DADD 210.6 per eval
#                       (2135 FP64 instructions before the d_abs recurrences were solved directly and sinn() lost its libm tiers)
#   config5_vjp_all_f32 k_elem<float,1,1,1,0>: FFMA 506.9, FMUL 409.4, FADD 194.3 per eval (FP32 flops only are counted), plus 351 FP64
#                       instructions per eval (the per-element root solve, which stays FP64)
FLOPS_PER_EVAL = {
    "config3_vjp_mu_f64": 393.5,
    "config3_vjp_mu_f32": 250.8,
    "config4_snia_f64": 442.0,
    "config5_vjp_all_f64": 2886.3,
    "config5_vjp_all_f32": 1617.5,
}
# instructions per eval on the arithmetic pipe of the dtype
PIPE_INST_PER_EVAL = {
    "config3_vjp_mu_f64": 264.8,
    "config3_vjp_mu_f32": 204.7,
    "config4_snia_f64": 298.4,
    "config5_vjp_all_f64": 1928.2,
    "config5_vjp_all_f32": 1327.2,
}
# dram__bytes_read.sum + dram__bytes_write.sum of that kernel, per launch (same captures)
DRAM_TRAFFIC_BYTES_PER_LAUNCH = {
    "config3_vjp_mu_f64": 544.20e6 + 640.53e6,
    "config3_vjp_mu_f32": 272e6 + 305e6,
    "config4_snia_f64": 25e6,
    "config5_vjp_all_f64": 907e6 + 897e6,
    "config5_vjp_all_f32": 618e6 + 587e6,
}
# where each entry comes from
SOURCE = {
    "config3_vjp_mu_f64": "profiles/r02_k_outer_vjp.md",
    "config3_vjp_mu_f32": "profiles/r02_other_kernels.csv",
    "config4_snia_f64": "profiles/r02_other_kernels.csv",
    "config5_vjp_all_f64": "profiles/r02_other_kernels.csv",
    "config5_vjp_all_f32": "profiles/r02_other_kernels.csv",
}

# nominal B200 vector peaks (context only; the denominator is the measured probe): 148 SMs x lanes x 2 x 1.965 GHz
NOMINAL_FP64_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
NOMINAL_FP32_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12

# algorithmic HBM bytes per eval, config 3 as bench.py runs it (z, params and constants stay on chip): grad_out read, out + status
# written, z / grad_z amortised over S
BYTES_PER_EVAL_C3 = {"f64": 8.0 + 8.0 + 1.0 + (8.0 + 8.0) / 64.0, "f32": 4.0 + 4.0 + 1.0 + (4.0 + 4.0) / 64.0}


# The per-eval figures above belong to ONE build of the kernels.  csrc_hash() fingerprints the CUDA sources; CAPTURED_CSRC_HASH is the
# fingerprint at the time of the ncu captures.  bench.py reports whether the two agree ("flops_build_matches"), so that a later kernel
# change cannot silently carry a stale flop count into the roofline fraction.
CAPTURED_CSRC_HASH = "2d35a26358a87058"


def csrc_hash() -> str:
    import hashlib
    import os
    d = os.path.join(os.path.dirname(os.path.abspath(__file__)), "csrc")
    h = hashlib.sha256()
    for f in sorted(os.listdir(d)):
        if f.endswith((".cu", ".cuh")):
            h.update(f.encode())
            h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]
