// cosmo_types.cuh -- shared definitions of the CUDA path (no arithmetic of the method lives here).
//
// Notation follows arXiv:2212.01937: x = 1+z, E^2(x) of eq. (2.2),
// the three fundamental integrals I0, T, A of eqs. (2.3)-(2.5) without their
// unit prefactors.  DESIGN.md "Real-quadratic form" explains how the root tuple r of eq. (3.2)
// is carried as two real quadratic factors.
#pragma once
#include <math.h>
#include <stdint.h>
#include <string.h>

#ifdef __CUDACC__
#define CB_HD __host__ __device__ __forceinline__
#define CB_HD_NOINLINE static __host__ __device__ __noinline__

#else
#define CB_HD inline
#define CB_HD_NOINLINE static inline
#endif

namespace cb {

// Fast FP64 reciprocal / square root for the per-element path on the device: MUFU seed (2^-20, measured) + one cubic step (error
// ~ 2^-58), no special-case handling -- the IEEE sequences cost 3-5 times the instructions and, inlined some 40 times per element,
// push the ELEMENTWISE kernels out of the instruction cache (profiles/).  Arguments: finite, normal, non-zero (cb_sqrt0 also takes 0).
// On the host (tests/hostcheck) they are the plain operations.
CB_HD double cb_rcp(double b) {
#ifdef __CUDA_ARCH__
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(b));
    const double e = fma(-b, r, 1.0);
    return fma(r, fma(e, e, e), r);
#else
    return 1.0 / b;
#endif
}
CB_HD double cb_div(double a, double b) {
#ifdef __CUDA_ARCH__
    const double r = cb_rcp(b), q = a * r;
    return fma(fma(-b, q, a), r, q);              // one correction step on the quotient
#else
    return a / b;
#endif
}
CB_HD double cb_sqrt0(double a) {                 // sqrt(a), a >= 0
#ifdef __CUDA_ARCH__
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(a));
    const double t = a * y;
    const double e = fma(-t, y, 1.0);
    const double r = fma(t * e, fma(0.375, e, 0.5), t);
    return a > 0.0 ? r : 0.0;
#else
    return sqrt(a);
#endif
}

// units: DESIGN.md reading R-units (the paper is silent)
constexpr double C_KM_S = 299792.458;             // km/s
constexpr double HUBBLE_GYR = 977.7922216807891;  // (1 km/s/Mpc)^-1 in Gyr
constexpr double FIVE_OVER_LN10 = 2.171472409516259138;

// Numeric constants of the per-element path.  On the device they live in the constant bank so that FP64 instructions
// take them as c[bank][offset] operands (a 64-bit literal otherwise costs two moves every time registers run short).
struct KTab {
    double third, two_thirds, sixteenth_inv;                      // 1/3, 2/3, 1/16
    double five_over_ln10, half_ln_2pi;
    double rf[7];      // R_F series: -1/10, 1/24, -5/208, 1/14, -3/44, 1/16, 3/104
    double rj[11];     // R_D/R_J series: -3/14, 9/88, -1/16, 1/6, -9/52, 45/272, 3/40, -9/68, -3/22, 3/20, 3/26
    double fo[11];     // 1/(2j+1)!
    double go[11];     // 1/(2j)!
    double dfo[11];    // j/(2j+1)!
    double rc[10];     // 1/3, 1/5, ..., 1/21
};
#define CB_KTAB_INIT {                                                                                                          \
    1.0 / 3, 2.0 / 3, 1.0 / 16, 2.171472409516259138, 0.91893853320467274178,                                                  \
    {-0.1, 1.0 / 24, -5.0 / 208, 1.0 / 14, -3.0 / 44, 1.0 / 16, 3.0 / 104},                                                    \
    {-3.0 / 14, 9.0 / 88, -1.0 / 16, 1.0 / 6, -9.0 / 52, 45.0 / 272, 3.0 / 40, -9.0 / 68, -3.0 / 22, 3.0 / 20, 3.0 / 26},      \
    {1.0, 1.0 / 6.0, 1.0 / 120.0, 1.0 / 5040.0, 1.0 / 362880.0, 1.0 / 39916800.0, 1.0 / 6227020800.0, 1.0 / 1307674368000.0,   \
     1.0 / 355687428096000.0, 1.0 / 121645100408832000.0, 1.0 / 51090942171709440000.0},                                       \
    {1.0, 0.5, 1.0 / 24.0, 1.0 / 720.0, 1.0 / 40320.0, 1.0 / 3628800.0, 1.0 / 479001600.0, 1.0 / 87178291200.0,                \
     1.0 / 20922789888000.0, 1.0 / 6402373705728000.0, 1.0 / 2432902008176640000.0},                                           \
    {0.0, 1.0 / 6.0, 2.0 / 120.0, 3.0 / 5040.0, 4.0 / 362880.0, 5.0 / 39916800.0, 6.0 / 6227020800.0, 7.0 / 1307674368000.0,   \
     8.0 / 355687428096000.0, 9.0 / 121645100408832000.0, 10.0 / 51090942171709440000.0},                                      \
    {1.0 / 3, 1.0 / 5, 1.0 / 7, 1.0 / 9, 1.0 / 11, 1.0 / 13, 1.0 / 15, 1.0 / 17, 1.0 / 19, 1.0 / 21}}
#ifdef __CUDACC__
static __constant__ KTab KT_dev = CB_KTAB_INIT;
#endif
static const KTab KT_host = CB_KTAB_INIT;
#ifdef __CUDA_ARCH__
#define CB_KT KT_dev
#else
#define CB_KT KT_host
#endif

// `which` bits, planes in ascending bit order (include/cosmo_b200.h)
enum : unsigned { W_DC = 1, W_DM = 2, W_DL = 4, W_MU = 8, W_TL = 16, W_DABS = 32, W_DA = 64, W_VC = 128, W_AGE = 256, W_ALL = 511 };
constexpr int N_PLANES = 9;                        // number of `which` bits
// status bits (include/cosmo_b200.h)
enum : unsigned { ST_ROOT_ON_PATH = 1, ST_UNSUPPORTED = 2, ST_DL_NONPOS = 4, ST_ITER_CAP = 8, ST_GRAD_ILLCOND = 16,
                  ST_INTERNAL_REDO = 128 };   // internal: never leaves the library
// cancellation factor of the gradient bases (cosmo_obs.cuh, grad_basis) above which an element's gradient integrals are taken from
// quadrature instead (grad_quad).  FP64: basis error ~ 2e-16 x cond (measured on config 5: <= 4e-10 below 1e6).
constexpr double GRAD_COND_LIMIT = 1.0e6;
constexpr double GRAD_COND_LIMIT_F32 = 30.0;

// depth of the perturbative d_abs recursions: rows k = 0 .. REC_KS of the moment recurrence for the value,
// k = 3 .. REC_KJ + 1 for the gradient's J'_5, J'_6, each solved directly (cosmo_eval.cuh, band_solve).  The truncation costs
// ~ ((Or/Om) x)^depth; where that exceeds the tolerance the direct forms take over (eq. (3.9), whose cancellation Om/(Or x) is then
// mild; the exact gradient basis, guarded by the cancellation check).
#ifndef CB_REC_KS
#define CB_REC_KS 8
#endif
#ifndef CB_REC_KJ
#define CB_REC_KJ 12
#endif
constexpr int REC_KS = CB_REC_KS, REC_KJ = CB_REC_KJ;

constexpr int NIT_CAP = 14;   // duplication steps never exceed this (status bit 8 when hit)

// Per-cosmology constant block ("S3" of the hot path).  E^2(x) = Q1(x) Q2(x),
//   Q1(x) = (Or x + m)(x - rn)        (the two negative real roots  -m/Or  and  rn;  Or = 0: linear)
//   Q2(x) = x^2 + b x + c             (the remaining pair: complex-conjugate or two reals)
template <typename T>
struct Cosmo {
    T Or, m, rn, b, c;
    T Om, Ok, OL, H0;
    T q11, q21;        // Q1(1), Q2(1)
    T sD, sDr;         // disc(Q1) disc(Q2) / 4  and sqrt|.|   (u13^2 - u14^2)^2 = 4 z^4 sD
    T theta;           // 2 f1 h2 + 2 h1 f2 - g1 g2 :  u12^2 - (u13^2+u14^2)/2 = z^2 theta / 2
    T W;               // Or^2 Q2(-m/Or) = m^2 - Or b m + Or^2 c
    T kf;              // (Or + m)/(1 - rn)
    T ck;              // sqrt(kf / Q2(1))
    T xlim;            // smallest real root of E^2 above 1 (+inf if none): x >= xlim -> status 1
    T dH, tH;          // c/H0 [Mpc], 1/H0 [Gyr]
    // lookback time, eq. (3.8) with i = big root, j = rn
    T p5c, Gp, qhc, OrM;
    // absorption distance, eq. (3.9) with (i,j,k,l) = (rn, pair, pair, big); (B.3) when Or = 0
    T Q2n, aF, WoOr, sig, mOrn, C1, F1, iOm;   // C1 = (1-rn) Q2(1), F1 = sqrt(C1/(Or+m)), iOm = 1/Om
    // gradient basis coefficients: dX/dtheta = -1/2 sum_j G[theta][j] basis_j
    T GI[3][5];        // X = I0 : basis (I0, K, b0, b1, b2)
    T GT[3][6];        // X = T  : basis (I0, K, b0, b1, b2, T)
    T GA[3][7];        // X = A  : basis (I0, K, b0, b1, b2, b3 (b4 when Or = 0), A)
    T Tinf, dTinf[3];  // int_1^inf dx/(x E) and its derivatives wrt (Om, OL, Or): age(z) = tH (Tinf - T(z))  (W_AGE only)
    T GJ[5][5];        // J'_p = int x^p dx / E^3, p = 0..4, over the basis (I0, K, b0, b1, b2)  (d_abs gradient)
    unsigned status;
    unsigned cubic;    // bit 0: Or == 0 (cubic case, appendix B.1);  bit 1: two complex pairs (cosmo_c4.cuh; m, rn hold g1, h1);
                       // bit 2: gradient bases unusable (a root pair's gap has closed, e.g. OL = 0): quadrature for every element;
                       // bit 3: bases large enough that some redshift may exceed GRAD_COND_LIMIT: the OUTER kernels take the
                       //        checked row for this cosmology (the ELEMENTWISE kernels check every element anyway)
};

constexpr int COSMO_NFIELDS = 115;   // floating-point members of Cosmo<T>, in declaration order
static_assert(sizeof(Cosmo<double>) == COSMO_NFIELDS * sizeof(double) + 2 * sizeof(unsigned), "Cosmo<T> layout");
static_assert(sizeof(Cosmo<float>) == COSMO_NFIELDS * sizeof(float) + 2 * sizeof(unsigned), "Cosmo<T> layout");

// FP64 block -> arithmetic type of the per-element path
template <typename T>
CB_HD void convert_cosmo(const Cosmo<double>& a, Cosmo<T>& b) {
    const double* pa = reinterpret_cast<const double*>(&a);
    T* pb = reinterpret_cast<T*>(&b);
    for (int i = 0; i < COSMO_NFIELDS; ++i) pb[i] = (T)pa[i];
    b.status = a.status;
    b.cubic = a.cubic;
}

}  // namespace cb
