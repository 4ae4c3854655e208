/* cosmo_b200_diag.h -- DIAGNOSTIC entry points of libcosmo_b200.so: measurement and test hooks, not part of the product surface
 * (include/cosmo_b200.h).  Used by bench.py (ALU peak probes, kernel timing, launch count) and by the tests (the device Carlson
 * functions on their own).  Same conventions as cosmo_b200.h: device pointers, asynchronous on `stream`, 0 or a negative COSMO_E_* code.
 */
#ifndef COSMO_B200_DIAG_H
#define COSMO_B200_DIAG_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* The device Carlson functions of the hot path on their own (eqs. (2.6), (2.7), (2.9); duplication
 * algorithm of ref. [10]), in the real-symmetric form the path uses: for each i
 *   rf[i] = R_F(x, m+h, m-h),  rd[i] = R_D(m+h, m-h, x),  rj[i] = R_J(x, m+h, m-h, p),   h^2 = s[i]
 * with x > 0, p > 0 and either s >= 0 with m - h > 0 (three positive reals) or s < 0 (a complex-conjugate pair m +- i|h|).
 * All arrays have length n (device pointers). */
int cosmo_carlson_pair(const double* x, const double* m, const double* s, const double* p, int64_t n, double* rf, double* rd,
                       double* rj, void* stream);

/* ALU roofline probes: each thread runs `iters` rounds of 8 independent dependent-FMA chains (FP64 / FP32) and
 * stores one value per thread in sink[blocks*256].  flops = blocks * 256 * iters * 8 * 2.  Used by bench.py to
 * measure the DFMA / FFMA peak that the roofline fraction is quoted against. */
int cosmo_probe_fma_f64(int blocks, int iters, double* sink, void* stream);
int cosmo_probe_fma_f32(int blocks, int iters, float* sink, void* stream);

/* Optional timing of the DOMINANT kernel of each call (the OUTER / ELEMENTWISE evaluation kernel, not prep/reduce) with
 * CUDA events recorded on the launching stream.  cosmo_profile(1) starts (and resets) the statistics, cosmo_profile(0)
 * stops; cosmo_profile_mean_ms synchronises on the last recorded launch and returns the mean duration in ms over the
 * launches since the reset (count in *n_launches, nullable).  When on, each call first waits for the previous call's
 * kernel to finish (host side), so leave it off outside measurements.  Not thread-safe. */
int cosmo_profile(int on);
double cosmo_profile_mean_ms(int64_t* n_launches);

/* number of kernels the library has launched in this process (all entry points) */
int64_t cosmo_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif /* COSMO_B200_DIAG_H */
