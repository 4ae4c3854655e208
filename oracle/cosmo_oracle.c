/* cosmo_oracle.c -- ORACLE. TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, obviously-correct CPU implementation of what the hot path of
 * arXiv:2212.01937 ("Analytic auto-differentiable LCDM cosmography") computes,
 * written from the paper's DEFINITIONS, in x87 80-bit `long double`.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load it.  It shares no code with the CUDA path
 * (paper_2212_01937_b200/csrc) and neither includes the other.
 *
 * What is here, with the passage each part follows (PAPER.md = /root/reference/PAPER.md):
 *
 *  (1) oracle_integrals      : the three fundamental integrals, eqs. (2.3)-(2.5)
 *                               with E^2 of eq. (2.2) and
 *                              Omega_k = 1 - sum of the others, z1 = 0,
 *                              by adaptive 21-point Gauss-Kronrod quadrature -- the
 *                              method the paper itself validates against (PAPER.md:233,
 *                              :243 fn.18).  These integrals are the plain definition
 *                              of what eqs. (3.7)-(3.9) re-express exactly.
 *                              Parameter derivatives: Leibniz's integrand rule applied
 *                              to the same integrals (the route PAPER.md:285 fn.23
 *                              names), by the same quadrature.
 *  (2) oracle_observables    : D_C, D_M (sin/sinh curvature transform), D_L=(1+z)D_M,
 *                              mu = 5 log10(D_L / 10 pc) (PAPER.md:277 fn.22),
 *                              lookback time, absorption distance, and
 *                              their total derivatives wrt (z, Om, OL, Or, H0).
 *                              DESIGN.md readings R-units, R-sinn.
 *  (3) oracle_age            : int_z^inf of eq. (2.4) -- used only to pin
 *                              (1) through lookback + age(z) = age(0).
 *  (4) oracle_rf/rc/rd/rj    : independent scalar Carlson symmetric integrals, eqs.
 *                              (2.6)-(2.9), complex arguments, by the
 *                              duplication algorithm the paper cites (ref. [10],
 *                              PAPER.md:113, :420; the algorithm itself is not printed in
 *                              the paper: this follows its statement in DLMF 19.36(i),
 *                              ref. [12]).  Not used by (1)-(3); used by tests to check
 *                              that the paper's closed forms equal the quadrature.
 *  (5) oracle_snia_loglike   : the Gaussian mu-likelihood of PAPER.md:283 summed over
 *                              objects, with parameter gradients, by direct summation.
 *  (6)-(10)                  : further down, each with its own header: the section-4 log-joint, the two-limit forms, the
 *                              derived observables, the extra constant-w components (chi family; then all six observables
 *                              with every gradient).
 *
 * Pins (tests/test_oracle_*.py): closed forms (Einstein-de Sitter, de Sitter, Milne,
 * radiation-only, flat LCDM t_L/age/d_abs, Mattig), flat-LCDM 2F1 expression,
 * 40-digit mpmath quadrature goldens, central finite differences of every gradient,
 * lookback<->age consistency, Carlson special values / identities / SciPy elliprX.
 *
 * Build: python oracle/build.py  (gcc -O2 -fopenmp, no -ffast-math).
 */
#include <complex.h>
#include <float.h>
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <string.h>

#ifdef _OPENMP
#include <omp.h>
#endif

#include "gk21_nodes.h"

#if LDBL_MANT_DIG < 64
#error "oracle needs an extended-precision long double (x87 80-bit or wider)"
#endif

typedef long double ld;
typedef long double complex ldc;

/* ---- units (reading R-units; the paper is silent) ---- */
#define C_KM_S 299792.458L                   /* speed of light, km/s (exact, SI)         */
#define HUBBLE_GYR 977.7922216807891L        /* (1 km/s/Mpc)^-1 in Gyr (Julian years)    */

int oracle_ldbl_mant_dig(void) { return LDBL_MANT_DIG; }
int oracle_max_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
void oracle_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ======================================================================================
 * (1) quadrature of the defining integrals
 * ====================================================================================== */

/* integrand components, all as functions of u = ln(1+z'), x = e^u, dz' = x du:
 *   0 I0 = int dz'/E                 (2.3) without c/H0
 *   1 T  = int dz'/((1+z')E)         (2.4) without 1/H0
 *   2 A  = int (1+z')^2 dz'/E        (2.5) without c/H0
 *   3..5   dI0/d(Om,OL,Or)   6..8 dT/d(Om,OL,Or)   9..11 dA/d(Om,OL,Or)
 * with dE^2/dOm = x^3-x^2, dE^2/dOL = 1-x^2, dE^2/dOr = x^4-x^2 (Omega_k eliminated,
 * PAPER.md:73) and d(E^-1)/dtheta = -1/2 (dE^2/dtheta) E^-3 (Leibniz rule). */
#define NV 12

typedef struct { ld Om, OL, Or, Ok; int nv; } cosmo_t;

static inline ld E2_of_x(const cosmo_t *c, ld x) {
    /* eq. (2.2), written exactly as printed */
    return c->Or * x * x * x * x + c->Om * x * x * x + c->Ok * x * x + c->OL;
}

/* returns kappa >= 1, the rounding amplification of E^2 at x (sum of |terms| / |sum|), used only
 * by the acceptance test's rounding floor (near a loitering phase E^2 is a small difference of O(1) terms) */
static ld integrand_u(const cosmo_t *c, ld u, ld f[NV]) {
    ld x = expl(u);
    ld E2 = E2_of_x(c, x);
    ld kappa = (c->Or * x * x * x * x + c->Om * x * x * x + fabsl(c->Ok) * x * x + fabsl(c->OL)) / fabsl(E2);
    ld E = sqrtl(E2);
    f[0] = x / E;
    f[1] = 1.0L / E;
    f[2] = x * x * x / E;
    if (c->nv > 3) {
        ld E3 = E2 * E;
        ld x2 = x * x;
        ld zz = expm1l(u); /* x - 1 without cancellation at small z */
        ld dOm = x2 * zz, dOL = -zz * (x + 1.0L), dOr = x2 * zz * (x + 1.0L); /* x^3-x^2, 1-x^2, x^4-x^2 */
        ld w0 = -0.5L * x / E3, w1 = -0.5L / E3, w2 = -0.5L * x2 * x / E3;
        f[3] = w0 * dOm; f[4] = w0 * dOL; f[5] = w0 * dOr;
        f[6] = w1 * dOm; f[7] = w1 * dOL; f[8] = w1 * dOr;
        f[9] = w2 * dOm; f[10] = w2 * dOL; f[11] = w2 * dOr;
    }
    return kappa;
}

/* one 21-point Gauss-Kronrod panel on [a,b]; K = Kronrod estimate, G = embedded Gauss */
static void gk21_panel(const cosmo_t *c, ld a, ld b, ld K[NV], ld G[NV], ld Kabs[NV]) {
    ld h = 0.5L * (b - a), m = 0.5L * (a + b), f[NV];
    int nv = c->nv;
    for (int v = 0; v < nv; ++v) K[v] = G[v] = Kabs[v] = 0.0L;
    for (int i = 0; i < 21; ++i) {
        ld kappa = integrand_u(c, m + h * GK21_X[i], f);
        for (int v = 0; v < nv; ++v) {
            K[v] += GK21_WK[i] * f[v];
            G[v] += GK21_WG[i] * f[v];
            Kabs[v] += GK21_WK[i] * fabsl(f[v]) * kappa;
        }
    }
    for (int v = 0; v < nv; ++v) { K[v] *= h; G[v] *= h; Kabs[v] *= h; }
}

/* adaptive bisection: a panel is accepted when, for every component, |K-G| is below
 * tol * |scale| * (panel width / total width), or below the rounding floor of the panel sum
 * (GK_ROUND * LDBL_EPSILON * int |f| kappa, kappa = rounding amplification of E^2); the accepted value is K.  For these analytic integrands the
 * Kronrod value is far more accurate than |K-G| indicates. */
#define GK_TOL 1e-16L
#define GK_ROUND 64.0L
#define GK_MAXDEPTH 60
#define GK_MAXPANELS 20000 /* safety net; oracle_integrals returns -2 when hit */

static void gk21_adapt(const cosmo_t *c, ld a, ld b, ld frac, const ld scale[NV], int depth,
                       ld acc[NV], int *npanels) {
    ld K[NV], G[NV], Kabs[NV];
    gk21_panel(c, a, b, K, G, Kabs);
    int ok = 1;
    for (int v = 0; v < c->nv; ++v) {
        ld err = fabsl(K[v] - G[v]);
        if (err > GK_TOL * scale[v] * frac && err > GK_ROUND * LDBL_EPSILON * Kabs[v]) ok = 0;
        if (err != err) ok = 1; /* NaN integrand (E^2 < 0 between the validity samples): give up, NaN propagates */
    }
    if (ok || depth >= GK_MAXDEPTH || *npanels >= GK_MAXPANELS) {
        for (int v = 0; v < c->nv; ++v) acc[v] += K[v];
        ++*npanels;
        return;
    }
    ld m = 0.5L * (a + b);
    gk21_adapt(c, a, m, 0.5L * frac, scale, depth + 1, acc, npanels);
    gk21_adapt(c, m, b, 0.5L * frac, scale, depth + 1, acc, npanels);
}

/* out[0..2] = I0,T,A ; if with_grad out[3..11] = their d/d(Om,OL,Or).  Returns panels used,
 * or -1 if E^2 <= 0 somewhere on the path -- found by a scan of 65 points or by the quadrature itself (unphysical, no Big Bang). */
int oracle_integrals(ld z, ld Om, ld OL, ld Or, int with_grad, ld out[NV]) {
    cosmo_t c = { Om, OL, Or, 1.0L - Om - OL - Or, with_grad ? NV : 3 };
    for (int v = 0; v < NV; ++v) out[v] = 0.0L;
    if (!(z > -1.0L)) return -1;
    if (z == 0.0L) return 0;
    ld U = log1pl(z);
    /* validity: E^2 must stay positive on the path */
    for (int i = 0; i <= 64; ++i) {
        ld x = expl(U * i / 64.0L);
        if (!(E2_of_x(&c, x) > 0.0L)) return -1;
    }
    /* first pass on fixed panels gives the scale used by the acceptance test */
    ld scale[NV], K[NV], G[NV], Kabs[NV];
    gk21_panel(&c, 0.0L, U, K, G, Kabs);
    for (int v = 0; v < c.nv; ++v) scale[v] = fabsl(K[v]);
    int npanels = 0;
    /* integrate on panels of width <= 1 in u (a decade of 1+z is ~2.3 panels) */
    int nseg = (int)ceill(fabsl(U));
    if (nseg < 1) nseg = 1;
    for (int s = 0; s < nseg; ++s) {
        ld a = U * s / nseg, b = U * (s + 1) / nseg;
        gk21_adapt(&c, a, b, 1.0L / nseg, scale, 0, out, &npanels);
    }
    if (npanels >= GK_MAXPANELS) return -2;
    /* a stretch with E^2 <= 0 that is narrower than the scan's step (two real roots close to each other on the path) is met by the
     * quadrature instead: sqrt of a negative number.  Same verdict as the scan's. */
    if (out[0] != out[0] || out[1] != out[1] || out[2] != out[2]) return -1;
    return npanels;
}

/* ======================================================================================
 * (3) age: int_z^inf dz'/((1+z')E) = int_0^{a} a' da'/sqrt(P(a')),  P = Or + Om a + Ok a^2 + OL a^4,
 *     with a' = s^2 so that the Or = 0 endpoint behaviour sqrt(a') becomes polynomial.
 * ====================================================================================== */
static ld age_integrand_s(const cosmo_t *c, ld s) {
    ld a = s * s;
    ld P = c->Or + c->Om * a + c->Ok * a * a + c->OL * a * a * a * a;
    /* a da = s^2 * 2 s ds ; if Or == 0 factor s out of sqrt(P) analytically */
    if (c->Or == 0.0L) {
        ld P1 = c->Om + c->Ok * a + c->OL * a * a * a; /* P / a */
        return 2.0L * s * s / sqrtl(P1);
    }
    return 2.0L * s * s * s / sqrtl(P);
}
static ld age_panel(const cosmo_t *c, ld a, ld b, ld *G) {
    ld h = 0.5L * (b - a), m = 0.5L * (a + b), K = 0.0L;
    *G = 0.0L;
    for (int i = 0; i < 21; ++i) {
        ld f = age_integrand_s(c, m + h * GK21_X[i]);
        K += GK21_WK[i] * f;
        *G += GK21_WG[i] * f;
    }
    *G *= h;
    return K * h;
}
static ld age_adapt(const cosmo_t *c, ld a, ld b, ld tolabs, int depth) {
    ld G, K = age_panel(c, a, b, &G);
    if (fabsl(K - G) <= tolabs || depth >= GK_MAXDEPTH) return K;
    ld m = 0.5L * (a + b);
    return age_adapt(c, a, m, 0.5L * tolabs, depth + 1) + age_adapt(c, m, b, 0.5L * tolabs, depth + 1);
}
/* H0 * age at redshift z (dimensionless) */
ld oracle_age_dimless(ld z, ld Om, ld OL, ld Or) {
    cosmo_t c = { Om, OL, Or, 1.0L - Om - OL - Or, 3 };
    ld smax = sqrtl(1.0L / (1.0L + z));
    ld G, K0 = age_panel(&c, 0.0L, smax, &G);
    return age_adapt(&c, 0.0L, smax, GK_TOL * fabsl(K0), 0);
}

/* ======================================================================================
 * (2) observables and their total derivatives
 * ====================================================================================== */
enum { OBS_DC = 0, OBS_DM, OBS_DL, OBS_MU, OBS_TL, OBS_DABS, N_OBS };
enum { WRT_Z = 0, WRT_OM, WRT_OL, WRT_OR, WRT_H0, N_WRT };

/* sinn(k, chi) = sinh(sqrt(k) chi)/sqrt(k) (k>0), sin(sqrt(-k) chi)/sqrt(-k) (k<0), chi (k=0);
 * also d/dchi and d/dk at fixed chi.  Series in w = k chi^2 for small |w| (the closed forms cancel). */
static void sinn_transform(ld k, ld chi, ld *F, ld *dF_dI, ld *dF_dk) {
    ld w = k * chi * chi;
    if (fabsl(w) < 1e-2L) {
        /* F = chi sum w^n/(2n+1)!, dF/dI = sum w^n/(2n)!, dF/dk = chi^3 sum n w^(n-1)/(2n+1)! */
        ld S = 0, C = 0, D = 0, term_s = 1.0L, term_c = 1.0L; /* w^n/(2n+1)!, w^n/(2n)! */
        ld wpow_prev_over = 0.0L;                              /* w^(n-1)/(2n+1)!       */
        for (int n = 0; n < 12; ++n) {
            S += term_s; C += term_c;
            if (n >= 1) D += n * wpow_prev_over;
            /* advance to n+1 */
            wpow_prev_over = term_s / ((2.0L * n + 2) * (2.0L * n + 3)); /* w^n/(2n+3)! */
            term_s = term_s * w / ((2.0L * n + 2) * (2.0L * n + 3));
            term_c = term_c * w / ((2.0L * n + 1) * (2.0L * n + 2));
        }
        *F = chi * S; *dF_dI = C; *dF_dk = chi * chi * chi * D;
        return;
    }
    if (k > 0) {
        ld s = sqrtl(k);
        ld sh = sinhl(s * chi), ch = coshl(s * chi);
        *F = sh / s; *dF_dI = ch; *dF_dk = (chi * ch - sh / s) / (2.0L * k);
    } else {
        ld s = sqrtl(-k);
        ld sn = sinl(s * chi), cs = cosl(s * chi);
        *F = sn / s; *dF_dI = cs; *dF_dk = (chi * cs - sn / s) / (2.0L * k);
    }
}

/* val[N_OBS], grad[N_OBS][N_WRT] (grad may be NULL).  Units: H0 in km/s/Mpc, distances in Mpc,
 * t_L in Gyr, mu in mag.  Returns 0, or -1 invalid path (values NaN), or 1 if D_L <= 0 (mu = NaN). */
int oracle_observables(ld z, ld Om, ld OL, ld Or, ld H0, ld val[N_OBS], ld *grad /* [N_OBS*N_WRT] or NULL */) {
    ld q[NV];
    int rc = oracle_integrals(z, Om, OL, Or, grad != NULL, q);
    if (rc < 0) {
        for (int i = 0; i < N_OBS; ++i) val[i] = NAN;
        if (grad) for (int i = 0; i < N_OBS * N_WRT; ++i) grad[i] = NAN;
        return -1;
    }
    ld Ok = 1.0L - Om - OL - Or;
    ld x = 1.0L + z;
    ld E = sqrtl(Or * x * x * x * x + Om * x * x * x + Ok * x * x + OL);
    ld dH = C_KM_S / H0, tH = HUBBLE_GYR / H0;
    ld I0 = q[0], T = q[1], A = q[2];
    ld F, Fi, Fk;
    sinn_transform(Ok, I0, &F, &Fi, &Fk);
    val[OBS_DC] = dH * I0;
    val[OBS_DM] = dH * F;
    val[OBS_DL] = x * dH * F;
    int status = 0;
    if (val[OBS_DL] > 0) val[OBS_MU] = 5.0L * log10l(val[OBS_DL]) + 25.0L; /* D_L in Mpc; 10 pc = 1e-5 Mpc */
    else { val[OBS_MU] = NAN; status = 1; }
    val[OBS_TL] = tH * T;
    val[OBS_DABS] = dH * A;
    if (!grad) return status;
    ld (*g)[N_WRT] = (ld (*)[N_WRT])grad;
    /* d/dz = integrand at the upper limit */
    ld dI_dz = 1.0L / E, dT_dz = 1.0L / (x * E), dA_dz = x * x / E;
    g[OBS_DC][WRT_Z] = dH * dI_dz;
    g[OBS_DM][WRT_Z] = dH * Fi * dI_dz;
    g[OBS_DL][WRT_Z] = dH * F + x * g[OBS_DM][WRT_Z];
    g[OBS_TL][WRT_Z] = tH * dT_dz;
    g[OBS_DABS][WRT_Z] = dH * dA_dz;
    for (int p = 0; p < 3; ++p) { /* Om, OL, Or ; dOk/dtheta = -1 for each */
        ld dI = q[3 + p], dT = q[6 + p], dA = q[9 + p];
        g[OBS_DC][WRT_OM + p] = dH * dI;
        g[OBS_DM][WRT_OM + p] = dH * (Fi * dI - Fk);
        g[OBS_DL][WRT_OM + p] = x * g[OBS_DM][WRT_OM + p];
        g[OBS_TL][WRT_OM + p] = tH * dT;
        g[OBS_DABS][WRT_OM + p] = dH * dA;
    }
    g[OBS_DC][WRT_H0] = -val[OBS_DC] / H0;
    g[OBS_DM][WRT_H0] = -val[OBS_DM] / H0;
    g[OBS_DL][WRT_H0] = -val[OBS_DL] / H0;
    g[OBS_TL][WRT_H0] = -val[OBS_TL] / H0;
    g[OBS_DABS][WRT_H0] = -val[OBS_DABS] / H0;
    for (int w = 0; w < N_WRT; ++w)
        g[OBS_MU][w] = (status == 0) ? 5.0L / logl(10.0L) * g[OBS_DL][w] / val[OBS_DL] : NAN;
    return status;
}

/* Batch over n elements (OpenMP over elements).  Parameter arrays have length n_cosmo in {1, n}
 * (n_cosmo == 1 broadcasts).  val: [n][N_OBS]; grad: [n][N_OBS][N_WRT] or NULL; status: [n] or NULL.
 * Inputs are doubles (the very values the GPU path is given); outputs long double. */
void oracle_observables_batch(int64_t n, const double *z, const double *Om, const double *OL, const double *Or,
                              const double *H0, int64_t n_cosmo, ld *val, ld *grad, int32_t *status) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t j = (n_cosmo == 1) ? 0 : i;
        int rc = oracle_observables((ld)z[i], (ld)Om[j], (ld)OL[j], (ld)Or[j], (ld)H0[j], val + i * N_OBS,
                                    grad ? grad + i * N_OBS * N_WRT : NULL);
        if (status) status[i] = rc;
    }
}

/* ======================================================================================
 * (2b) further derived observables of PAPER.md:95: angular-diameter distance
 *      D_A = D_M/(1+z), comoving volume out to z over the whole sky V_C = 4 pi int_0^chi D_M^2 dchi'
 *      (ref. [59] eq. (13.60)), and the age at z, int_z^inf of eq. (2.4), with their total derivatives
 *      wrt (z, Om, OL, Or, H0).  val[3] = {DA [Mpc], VC [Mpc^3], AGE [Gyr]}, grad[3][5].
 *      The age gradient integrals are Leibniz integrals of the same integrand, in a = 1/(1+z'), a = s^2:
 *        d(H0 age)/dtheta = -1/2 int_0^{a_z} q_theta(a) P(a)^{-3/2} da,  q = a^2-a^3 (Om), a^5-a^3 (OL), a-a^3 (Or).
 * ====================================================================================== */
static void age_grad_integrand_s(const cosmo_t *c, ld s, ld f[4]) {
    ld a = s * s;
    if (c->Or == 0.0L) {
        /* P = a P1, P^{3/2} = a^{3/2} P1^{3/2}; da = 2 s ds = 2 a^{1/2} ds */
        ld P1 = c->Om + c->Ok * a + c->OL * a * a * a, r = P1 * sqrtl(P1);
        f[0] = 2.0L * a / sqrtl(P1);                      /* a da / sqrt(P) = 2 s^2 ds / sqrt(P1) */
        f[1] = 2.0L * (a - a * a) / r;                    /* (a^2 - a^3) a^{-3/2} 2 a^{1/2} */
        f[2] = 2.0L * (a * a * a * a - a * a) / r;
        f[3] = 2.0L * (1.0L - a * a) / r;
        return;
    }
    ld P = c->Or + c->Om * a + c->Ok * a * a + c->OL * a * a * a * a, r = P * sqrtl(P);
    f[0] = 2.0L * s * a / sqrtl(P);
    f[1] = 2.0L * s * (a * a - a * a * a) / r;
    f[2] = 2.0L * s * (a * a * a * a * a - a * a * a) / r;
    f[3] = 2.0L * s * (a - a * a * a) / r;
}
static void age_grad_panel(const cosmo_t *c, ld a, ld b, ld K[4], ld G[4]) {
    ld h = 0.5L * (b - a), m = 0.5L * (a + b), f[4];
    for (int v = 0; v < 4; ++v) K[v] = G[v] = 0.0L;
    for (int i = 0; i < 21; ++i) {
        age_grad_integrand_s(c, m + h * GK21_X[i], f);
        for (int v = 0; v < 4; ++v) { K[v] += GK21_WK[i] * f[v]; G[v] += GK21_WG[i] * f[v]; }
    }
    for (int v = 0; v < 4; ++v) { K[v] *= h; G[v] *= h; }
}
static void age_grad_adapt(const cosmo_t *c, ld a, ld b, const ld tolabs[4], int depth, ld acc[4], int *npanels) {
    ld K[4], G[4];
    age_grad_panel(c, a, b, K, G);
    int ok = 1;
    for (int v = 0; v < 4; ++v) {
        ld err = fabsl(K[v] - G[v]);
        if (err > tolabs[v]) ok = 0;
        if (err != err) ok = 1;   /* NaN/inf integrand (e.g. a divergent gradient integral when Om = 0): give up, it propagates */
    }
    if (ok || depth >= GK_MAXDEPTH || *npanels >= GK_MAXPANELS) { for (int v = 0; v < 4; ++v) acc[v] += K[v]; ++*npanels; return; }
    ld m = 0.5L * (a + b), t2[4];
    for (int v = 0; v < 4; ++v) t2[v] = 0.5L * tolabs[v];
    age_grad_adapt(c, a, m, t2, depth + 1, acc, npanels);
    age_grad_adapt(c, m, b, t2, depth + 1, acc, npanels);
}

/* V_C / (4 pi d_H^3) = v(k, chi) = int_0^chi F(k, chi')^2 dchi' and its partial wrt k; F = sinn transform (dv/dchi = F^2) */
static void volume_transform(ld k, ld chi, ld *v, ld *dv_dk) {
    ld w = k * chi * chi;
    if (fabsl(w) < 1e-2L) {
        /* v = chi^3 sum_{j>=1} 4^j w^(j-1) / (2 (2j+1)!),  dv/dk = chi^5 sum_{j>=2} (j-1) 4^j w^(j-2) / (2 (2j+1)!) */
        ld S = 0, D = 0, coef = 1.0L; /* 4^j/(2j+1)! */
        ld wp1 = 1.0L, wp2 = 1.0L;
        for (int j = 1; j < 14; ++j) {
            coef = coef * 4.0L / ((2.0L * j) * (2.0L * j + 1.0L));
            S += 0.5L * coef * wp1;
            if (j >= 2) { D += 0.5L * (j - 1) * coef * wp2; wp2 *= w; }
            wp1 *= w;
        }
        *v = chi * chi * chi * S; *dv_dk = chi * chi * chi * chi * chi * D;
        return;
    }
    if (k > 0) {
        /* v = (sinh(2 s chi)/(2 s) - chi)/(2k), s = sqrt(k);  d/dk of the numerator = chi cosh/(2k) - sinh/(4 k s) */
        ld s = sqrtl(k), sh2 = sinhl(2.0L * s * chi), ch2 = coshl(2.0L * s * chi);
        *v = (sh2 / (2.0L * s) - chi) / (2.0L * k);
        ld dnum = chi * ch2 / (2.0L * k) - sh2 / (4.0L * k * s);
        *dv_dk = dnum / (2.0L * k) - (*v) / k;
    } else {
        /* with kk = -k: v = (chi - sin(2 s chi)/(2 s))/(2 kk), s = sqrt(kk) */
        ld kk = -k, s = sqrtl(kk), sn2 = sinl(2.0L * s * chi), cs2 = cosl(2.0L * s * chi);
        *v = (chi - sn2 / (2.0L * s)) / (2.0L * kk);
        ld dnum = -(chi * cs2 / (2.0L * kk) - sn2 / (4.0L * kk * s));
        ld dv_dkk = dnum / (2.0L * kk) - (*v) / kk;
        *dv_dk = -dv_dkk;
    }
}

int oracle_derived(ld z, ld Om, ld OL, ld Or, ld H0, ld val[3], ld *grad /* [3*N_WRT] or NULL */) {
    ld base[N_OBS], bgrad[N_OBS * N_WRT];
    int rc = oracle_observables(z, Om, OL, Or, H0, base, bgrad);
    if (rc < 0) {
        for (int i = 0; i < 3; ++i) val[i] = NAN;
        if (grad) for (int i = 0; i < 3 * N_WRT; ++i) grad[i] = NAN;
        return -1;
    }
    ld (*bg)[N_WRT] = (ld (*)[N_WRT])bgrad;
    ld x = 1.0L + z, Ok = 1.0L - Om - OL - Or, dH = C_KM_S / H0, tH = HUBBLE_GYR / H0;
    ld I0 = base[OBS_DC] / dH;
    /* D_A */
    val[0] = base[OBS_DM] / x;
    /* V_C */
    ld v, dv_dk, F, Fi, Fk;
    volume_transform(Ok, I0, &v, &dv_dk);
    sinn_transform(Ok, I0, &F, &Fi, &Fk);
    const ld FOURPI = 12.566370614359172953850573533118L;
    val[1] = FOURPI * dH * dH * dH * v;
    /* age */
    cosmo_t c = { Om, OL, Or, Ok, 3 };
    ld smax = sqrtl(1.0L / x), K0[4], G0[4], tol[4], acc[4] = {0, 0, 0, 0};
    age_grad_panel(&c, 0.0L, smax, K0, G0);
    for (int i = 0; i < 4; ++i) tol[i] = GK_TOL * fabsl(K0[i]) + 1e-30L;
    int npanels = 0;
    age_grad_adapt(&c, 0.0L, smax, tol, 0, acc, &npanels);
    val[2] = tH * acc[0];
    if (!grad) return rc;
    ld (*g)[N_WRT] = (ld (*)[N_WRT])grad;
    for (int w = 0; w < N_WRT; ++w) g[0][w] = bg[OBS_DM][w] / x;
    g[0][WRT_Z] -= base[OBS_DM] / (x * x);
    /* dv = F^2 dI0 + dv_dk dk ; dI0/dtheta = grad(DC)/dH (params), dI0/dz = 1/E */
    ld E = sqrtl(Or * x * x * x * x + Om * x * x * x + Ok * x * x + OL);
    g[1][WRT_Z] = FOURPI * dH * dH * dH * F * F / E;
    for (int p = 0; p < 3; ++p) {
        ld dI = bg[OBS_DC][WRT_OM + p] / dH;
        g[1][WRT_OM + p] = FOURPI * dH * dH * dH * (F * F * dI - dv_dk);
    }
    g[1][WRT_H0] = -3.0L * val[1] / H0;
    g[2][WRT_Z] = -tH / (x * E);
    for (int p = 0; p < 3; ++p) g[2][WRT_OM + p] = tH * (-0.5L) * acc[1 + p];
    g[2][WRT_H0] = -val[2] / H0;
    return rc;
}

void oracle_derived_batch(int64_t n, const double *z, const double *Om, const double *OL, const double *Or,
                          const double *H0, int64_t n_cosmo, ld *val, ld *grad, int32_t *status) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t j = (n_cosmo == 1) ? 0 : i;
        int rc = oracle_derived((ld)z[i], (ld)Om[j], (ld)OL[j], (ld)Or[j], (ld)H0[j], val + i * 3, grad ? grad + i * 3 * N_WRT : NULL);
        if (status) status[i] = rc;
    }
}

/* ======================================================================================
 * (5) SN Ia Gaussian mu-likelihood: mu_obs_n | mu_n ~ N(mu_n, sigma_n^2)
 *     logL = sum_n [ -1/2 ((mu_obs_n - mu_n)/sigma_n)^2 - ln sigma_n - 1/2 ln 2 pi ]
 *     dlogL/dtheta = sum_n ((mu_obs_n - mu_n)/sigma_n^2) dmu_n/dtheta,  theta in (Om, OL, Or, H0)
 *     one cosmology; out = {logL, d/dOm, d/dOL, d/dOr, d/dH0}.  Long-double accumulation in index order.
 * ====================================================================================== */
int oracle_snia_loglike(int64_t n, const double *z, const double *mu_obs, const double *sigma, double Om, double OL,
                        double Or, double H0, int with_grad, ld out[5]) {
    ld acc[5] = { 0, 0, 0, 0, 0 };
    int bad = 0;
    const ld half_ln_2pi = 0.5L * logl(2.0L * acosl(-1.0L));
#pragma omp parallel
    {
        ld loc[5] = { 0, 0, 0, 0, 0 };
        int locbad = 0;
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            ld val[N_OBS], grad[N_OBS * N_WRT];
            int rc = oracle_observables((ld)z[i], (ld)Om, (ld)OL, (ld)Or, (ld)H0, val, with_grad ? grad : NULL);
            if (rc != 0) { locbad = 1; continue; }
            ld s = (ld)sigma[i];
            ld r = ((ld)mu_obs[i] - val[OBS_MU]) / s;
            loc[0] += -0.5L * r * r - logl(s) - half_ln_2pi;
            if (with_grad)
                for (int p = 0; p < 4; ++p) loc[1 + p] += (r / s) * grad[OBS_MU * N_WRT + WRT_OM + p];
        }
#pragma omp critical
        {
            for (int k = 0; k < 5; ++k) acc[k] += loc[k];
            bad |= locbad;
        }
    }
    for (int k = 0; k < 5; ++k) out[k] = acc[k];
    return bad ? -1 : 0;
}

/* ======================================================================================
 * (4) independent scalar Carlson integrals, complex arguments, duplication (DLMF 19.36(i))
 *     r = requested relative accuracy.  csqrtl is the principal root (Re >= 0) throughout.
 * ====================================================================================== */
#define CARLSON_R 1e-18L
#define CARLSON_MAXIT 200

static ld max3(ld a, ld b, ld c) { return fmaxl(a, fmaxl(b, c)); }

ldc oracle_rf_c(ldc x, ldc y, ldc z) {
    ldc A0 = (x + y + z) / 3.0L, A = A0;
    ld Q = powl(3.0L * CARLSON_R, -1.0L / 6.0L) * max3(cabsl(A0 - x), cabsl(A0 - y), cabsl(A0 - z));
    ld f = 1.0L; /* 4^n */
    for (int n = 0; n < CARLSON_MAXIT && !(Q / f < cabsl(A)); ++n) {
        ldc sx = csqrtl(x), sy = csqrtl(y), sz = csqrtl(z);
        ldc lam = sx * sy + sx * sz + sy * sz;
        A = (A + lam) / 4.0L; x = (x + lam) / 4.0L; y = (y + lam) / 4.0L; z = (z + lam) / 4.0L;
        f *= 4.0L;
    }
    ldc X = 1.0L - x / A, Y = 1.0L - y / A, Z = -X - Y; /* = (A0-x0)/(4^n A_n) etc. */
    ldc E2 = X * Y - Z * Z, E3 = X * Y * Z;
    return (1.0L - E2 / 10.0L + E3 / 14.0L + E2 * E2 / 24.0L - 3.0L * E2 * E3 / 44.0L - 5.0L * E2 * E2 * E2 / 208.0L +
            3.0L * E3 * E3 / 104.0L + E2 * E2 * E3 / 16.0L) / csqrtl(A);
}

/* R_C(x,y) = R_F(x,y,y); real y < 0 (with real x >= 0): Cauchy principal value */
ldc oracle_rc_c(ldc x, ldc y) {
    if (cimagl(y) == 0.0L && creall(y) < 0.0L && cimagl(x) == 0.0L && creall(x) >= 0.0L) {
        ld xr = creall(x), yr = creall(y);
        return sqrtl(xr / (xr - yr)) * oracle_rc_c(xr - yr, -yr);
    }
    ldc A0 = (x + 2.0L * y) / 3.0L, A = A0, y0 = y;
    ld Q = powl(3.0L * CARLSON_R, -1.0L / 8.0L) * cabsl(A0 - x);
    ld f = 1.0L;
    for (int n = 0; n < CARLSON_MAXIT && !(Q / f < cabsl(A)); ++n) {
        ldc lam = 2.0L * csqrtl(x) * csqrtl(y) + y;
        A = (A + lam) / 4.0L; x = (x + lam) / 4.0L; y = (y + lam) / 4.0L;
        f *= 4.0L;
    }
    ldc s = (y0 - A0) / (f * A);
    ldc s2 = s * s;
    return (1.0L + s2 * (3.0L / 10.0L + s * (1.0L / 7.0L + s * (3.0L / 8.0L + s * (9.0L / 22.0L + s * (159.0L / 208.0L + s * (9.0L / 8.0L))))))) /
           csqrtl(A);
}

static ldc carlson_series_dj(ldc E2, ldc E3, ldc E4, ldc E5) {
    return 1.0L - 3.0L * E2 / 14.0L + E3 / 6.0L + 9.0L * E2 * E2 / 88.0L - 3.0L * E4 / 22.0L - 9.0L * E2 * E3 / 52.0L +
           3.0L * E5 / 26.0L - E2 * E2 * E2 / 16.0L + 3.0L * E3 * E3 / 40.0L + 3.0L * E2 * E4 / 20.0L +
           45.0L * E2 * E2 * E3 / 272.0L - 9.0L * (E3 * E4 + E2 * E5) / 68.0L;
}

ldc oracle_rd_c(ldc x, ldc y, ldc z) {
    ldc A0 = (x + y + 3.0L * z) / 5.0L, A = A0, x0 = x, y0 = y, sum = 0.0L;
    ld Q = powl(CARLSON_R / 4.0L, -1.0L / 6.0L) * max3(cabsl(A0 - x), cabsl(A0 - y), cabsl(A0 - z));
    ld f = 1.0L;
    for (int n = 0; n < CARLSON_MAXIT && !(Q / f < cabsl(A)); ++n) {
        ldc sx = csqrtl(x), sy = csqrtl(y), sz = csqrtl(z);
        ldc lam = sx * sy + sx * sz + sy * sz;
        sum += 1.0L / (f * sz * (z + lam));
        A = (A + lam) / 4.0L; x = (x + lam) / 4.0L; y = (y + lam) / 4.0L; z = (z + lam) / 4.0L;
        f *= 4.0L;
    }
    ldc X = (A0 - x0) / (f * A), Y = (A0 - y0) / (f * A), Z = -(X + Y) / 3.0L;
    ldc E2 = X * Y - 6.0L * Z * Z, E3 = (3.0L * X * Y - 8.0L * Z * Z) * Z, E4 = 3.0L * (X * Y - Z * Z) * Z * Z,
        E5 = X * Y * Z * Z * Z;
    return carlson_series_dj(E2, E3, E4, E5) / (f * A * csqrtl(A)) + 3.0L * sum;
}

/* R_J(x,y,z,p); real p < 0 with real non-negative x,y,z: Cauchy principal value via DLMF 19.20.14 */
ldc oracle_rj_c(ldc x, ldc y, ldc z, ldc p) {
    if (cimagl(p) == 0.0L && creall(p) < 0.0L && cimagl(x) == 0.0L && cimagl(y) == 0.0L && cimagl(z) == 0.0L) {
        ld a = creall(x), b = creall(y), c = creall(z), t;
        /* order a <= b <= c */
        if (a > b) { t = a; a = b; b = t; }
        if (b > c) { t = b; b = c; c = t; }
        if (a > b) { t = a; a = b; b = t; }
        ld q = -creall(p);
        /* DLMF 19.20.14: (q + y) R_J(x,y,z,-q) = (p - y) R_J(x,y,z,p) - 3 R_F(x,y,z) + 3 sqrt(xyz/(xz+pq)) R_C(xz+pq, pq),
         * p = y + (z-y)(y-x)/(y+q), valid for y between x and z; here y := b (the middle one), x := a, z := c. */
        ld pp = b + (c - b) * (b - a) / (b + q);
        ldc rj = oracle_rj_c(a, b, c, pp);
        ldc rf = oracle_rf_c(a, b, c);
        ld xzpq = a * c + pp * q;
        ldc rc = oracle_rc_c(xzpq, pp * q);
        return ((pp - b) * rj - 3.0L * rf + 3.0L * sqrtl(a * b * c / xzpq) * rc) / (q + b);
    }
    ldc A0 = (x + y + z + 2.0L * p) / 5.0L, A = A0, x0 = x, y0 = y, z0 = z, sum = 0.0L;
    ldc delta = (p - x) * (p - y) * (p - z);
    ld Q = powl(CARLSON_R / 4.0L, -1.0L / 6.0L) *
           fmaxl(max3(cabsl(A0 - x), cabsl(A0 - y), cabsl(A0 - z)), cabsl(A0 - p));
    ld f = 1.0L;
    for (int n = 0; n < CARLSON_MAXIT && !(Q / f < cabsl(A)); ++n) {
        ldc sx = csqrtl(x), sy = csqrtl(y), sz = csqrtl(z), sp = csqrtl(p);
        ldc lam = sx * sy + sx * sz + sy * sz;
        ldc d = (sp + sx) * (sp + sy) * (sp + sz);
        ldc e = delta / (f * f * f * d * d);
        sum += oracle_rc_c(1.0L, 1.0L + e) / (f * d);
        A = (A + lam) / 4.0L; x = (x + lam) / 4.0L; y = (y + lam) / 4.0L; z = (z + lam) / 4.0L; p = (p + lam) / 4.0L;
        f *= 4.0L;
    }
    ldc X = (A0 - x0) / (f * A), Y = (A0 - y0) / (f * A), Z = (A0 - z0) / (f * A), P = (-X - Y - Z) / 2.0L;
    ldc E2 = X * Y + X * Z + Y * Z - 3.0L * P * P, E3 = X * Y * Z + 2.0L * E2 * P + 4.0L * P * P * P,
        E4 = (2.0L * X * Y * Z + E2 * P + 3.0L * P * P * P) * P, E5 = X * Y * Z * P * P;
    return carlson_series_dj(E2, E3, E4, E5) / (f * A * csqrtl(A)) + 6.0L * sum;
}

/* ctypes-friendly wrappers: double in, long double (re, im) out */
void oracle_rf(double xr, double xi, double yr, double yi, double zr, double zi, ld out[2]) {
    ldc r = oracle_rf_c(xr + I * (ld)xi, yr + I * (ld)yi, zr + I * (ld)zi);
    out[0] = creall(r); out[1] = cimagl(r);
}
void oracle_rc(double xr, double xi, double yr, double yi, ld out[2]) {
    ldc r = oracle_rc_c(xr + I * (ld)xi, yr + I * (ld)yi);
    out[0] = creall(r); out[1] = cimagl(r);
}
void oracle_rd(double xr, double xi, double yr, double yi, double zr, double zi, ld out[2]) {
    ldc r = oracle_rd_c(xr + I * (ld)xi, yr + I * (ld)yi, zr + I * (ld)zi);
    out[0] = creall(r); out[1] = cimagl(r);
}
void oracle_rj(double xr, double xi, double yr, double yi, double zr, double zi, double pr, double pi_, ld out[2]) {
    ldc r = oracle_rj_c(xr + I * (ld)xi, yr + I * (ld)yi, zr + I * (ld)zi, pr + I * (ld)pi_);
    out[0] = creall(r); out[1] = cimagl(r);
}

/* GK21 rule exposed for the quadrature-rule pin (exactness degree, weights) */
void oracle_gk21_rule(ld x[21], ld wk[21], ld wg[21]) {
    memcpy(x, GK21_X, sizeof(GK21_X)); memcpy(wk, GK21_WK, sizeof(GK21_WK)); memcpy(wg, GK21_WG, sizeof(GK21_WG));
}

/* ======================================================================================
 * (6) the log-joint of the paper's section-4 toy model with LATENT redshifts:
 *       mu_obs_n | z_n, theta ~ N(mu(z_n; theta), sigma_mu_n^2)
 *       z_obs_n  | z_n        ~ N(z_n, (1+z_n)^2 sigma_z^2)                      (photometric-redshift toy model)
 *       z_n                  ~ Gamma(shape, rate beta):  p(z) = beta^shape z^(shape-1) e^(-beta z) / Gamma(shape)
 *     (the paper fixes beta = 3, sigma_mu = 0.14, sigma_z = 0.04 and does not print the shape: DESIGN.md reading R-prior.)
 *     out = {log p, d/dOm, d/dOL, d/dOr, d/dH0};  gz[n] = d log p / d z_n  (nullable).  One cosmology, direct summation.
 * ====================================================================================== */
int oracle_snia_logjoint(int64_t n, const double *z, const double *z_obs, const double *mu_obs, const double *sigma_mu,
                         double sigma_z, double beta, double shape, double Om, double OL, double Or, double H0,
                         int with_grad, ld out[5], ld *gz) {
    ld acc[5] = { 0, 0, 0, 0, 0 };
    int bad = 0;
    const ld half_ln_2pi = 0.5L * logl(2.0L * acosl(-1.0L));
    const ld prior_norm = (ld)shape * logl((ld)beta) - lgammal((ld)shape);
#pragma omp parallel
    {
        ld loc[5] = { 0, 0, 0, 0, 0 };
        int locbad = 0;
#pragma omp for schedule(static)
        for (int64_t i = 0; i < n; ++i) {
            ld val[N_OBS], grad[N_OBS * N_WRT];
            int rc = oracle_observables((ld)z[i], (ld)Om, (ld)OL, (ld)Or, (ld)H0, val, with_grad ? grad : NULL);
            if (rc != 0) { locbad = 1; if (gz) gz[i] = NAN; continue; }
            ld zi = (ld)z[i], x = 1.0L + zi;
            ld s = (ld)sigma_mu[i], r = ((ld)mu_obs[i] - val[OBS_MU]) / s;
            ld sz = x * (ld)sigma_z, rz = ((ld)z_obs[i] - zi) / sz;
            loc[0] += (-0.5L * r * r - logl(s) - half_ln_2pi) + (-0.5L * rz * rz - logl(sz) - half_ln_2pi)
                      + (prior_norm + ((ld)shape - 1.0L) * logl(zi) - (ld)beta * zi);
            if (with_grad) {
                for (int p = 0; p < 4; ++p) loc[1 + p] += (r / s) * grad[OBS_MU * N_WRT + WRT_OM + p];
                if (gz) gz[i] = (r / s) * grad[OBS_MU * N_WRT + WRT_Z]
                                + (rz / sz + rz * rz / x - 1.0L / x)                 /* d/dz of the photo-z term */
                                + (((ld)shape - 1.0L) / zi - (ld)beta);              /* d/dz of the prior         */
            }
        }
#pragma omp critical
        {
            for (int k = 0; k < 5; ++k) acc[k] += loc[k];
            bad |= locbad;
        }
    }
    for (int k = 0; k < 5; ++k) out[k] = acc[k];
    return bad ? -1 : 0;
}

/* ======================================================================================
 * (7) the TWO-LIMIT forms of eqs. (2.3)-(2.5) (PAPER.md:88-93 define chi(z1,z2), t(z1,z2), d_abs(z1,z2)):
 *     same quadrature on [ln(1+z1), ln(1+z2)].  out[12] as oracle_integrals.
 *     oracle_observables2: val[5] = {D_C12, D_M12 (sinn of the comoving distance between z1 and z2), t12, d_abs12,
 *     D_A12 = D_M12/(1+z2)} and grad[5][6] wrt (z1, z2, Om, OL, Or, H0).
 * ====================================================================================== */
int oracle_integrals2(ld z1, ld z2, ld Om, ld OL, ld Or, int with_grad, ld out[NV]) {
    cosmo_t c = { Om, OL, Or, 1.0L - Om - OL - Or, with_grad ? NV : 3 };
    for (int v = 0; v < NV; ++v) out[v] = 0.0L;
    if (!(z1 > -1.0L) || !(z2 > -1.0L)) return -1;
    if (z1 == z2) return 0;
    ld U1 = log1pl(z1), U2 = log1pl(z2);
    for (int i = 0; i <= 64; ++i) {
        ld x = expl(U1 + (U2 - U1) * i / 64.0L);
        if (!(E2_of_x(&c, x) > 0.0L)) return -1;
    }
    ld scale[NV], K[NV], G[NV], Kabs[NV];
    gk21_panel(&c, U1, U2, K, G, Kabs);
    for (int v = 0; v < c.nv; ++v) scale[v] = fabsl(K[v]);
    int npanels = 0;
    int nseg = (int)ceill(fabsl(U2 - U1));
    if (nseg < 1) nseg = 1;
    for (int s = 0; s < nseg; ++s) {
        ld a = U1 + (U2 - U1) * s / nseg, b = U1 + (U2 - U1) * (s + 1) / nseg;
        gk21_adapt(&c, a, b, 1.0L / nseg, scale, 0, out, &npanels);
    }
    if (npanels >= GK_MAXPANELS) return -2;
    return npanels;
}

int oracle_observables2(ld z1, ld z2, ld Om, ld OL, ld Or, ld H0, ld val[5], ld *grad /* [5*6] or NULL */) {
    ld q[NV];
    int rc = oracle_integrals2(z1, z2, Om, OL, Or, grad != NULL, q);
    if (rc < 0) {
        for (int i = 0; i < 5; ++i) val[i] = NAN;
        if (grad) for (int i = 0; i < 30; ++i) grad[i] = NAN;
        return -1;
    }
    ld Ok = 1.0L - Om - OL - Or, x1 = 1.0L + z1, x2 = 1.0L + z2;
    cosmo_t c = { Om, OL, Or, Ok, 3 };
    ld E1 = sqrtl(E2_of_x(&c, x1)), E2 = sqrtl(E2_of_x(&c, x2));
    ld dH = C_KM_S / H0, tH = HUBBLE_GYR / H0;
    ld F, Fi, Fk;
    sinn_transform(Ok, q[0], &F, &Fi, &Fk);
    val[0] = dH * q[0]; val[1] = dH * F; val[2] = tH * q[1]; val[3] = dH * q[2]; val[4] = dH * F / x2;
    if (!grad) return 0;
    ld (*g)[6] = (ld (*)[6])grad;
    /* d/dz1 = -integrand(z1), d/dz2 = +integrand(z2) */
    g[0][0] = -dH / E1;            g[0][1] = dH / E2;
    g[1][0] = -dH * Fi / E1;       g[1][1] = dH * Fi / E2;
    g[2][0] = -tH / (x1 * E1);     g[2][1] = tH / (x2 * E2);
    g[3][0] = -dH * x1 * x1 / E1;  g[3][1] = dH * x2 * x2 / E2;
    g[4][0] = g[1][0] / x2;        g[4][1] = g[1][1] / x2 - val[1] / (x2 * x2);
    for (int p = 0; p < 3; ++p) {
        g[0][2 + p] = dH * q[3 + p];
        g[1][2 + p] = dH * (Fi * q[3 + p] - Fk);
        g[2][2 + p] = tH * q[6 + p];
        g[3][2 + p] = dH * q[9 + p];
        g[4][2 + p] = g[1][2 + p] / x2;
    }
    for (int o = 0; o < 5; ++o) g[o][5] = -val[o] / H0;
    return 0;
}

void oracle_observables2_batch(int64_t n, const double *z1, const double *z2, const double *Om, const double *OL, const double *Or,
                               const double *H0, int64_t n_cosmo, ld *val, ld *grad, int32_t *status) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t j = (n_cosmo == 1) ? 0 : i;
        int rc = oracle_observables2((ld)z1[i], (ld)z2[i], (ld)Om[j], (ld)OL[j], (ld)Or[j], (ld)H0[j], val + i * 5, grad ? grad + i * 30 : NULL);
        if (status) status[i] = rc;
    }
}

/* ======================================================================================
 * (9) extra components with constant equation of state w in {-2/3, -1/3} (PAPER.md:82 fn.4):
 *       E^2(x) = Or x^4 + Om x^3 + (Ok + Ow13) x^2 + Ow23 x + OL,   Ok = 1 - Om - OL - Or - Ow13 - Ow23,
 *     each component evolving as x^(3(1+w)) (fn.4 with constant w); the curvature of the transverse distance is Ok
 *     alone.  chi family only: I0 = int_1^x dx'/E (eq. (2.3)), then D_C, D_M, D_L, mu as in (2), and
 *     their d/dz (the integrand at the upper limit, chained).  Same adaptive GK21 in u = ln x as (1), written out
 *     again for this polynomial so that (1) stays exactly as pinned. */
typedef struct { ld a4, a3, a2, a1, a0; } poly4_t;

static inline ld w_E2(const poly4_t *p, ld x) { return (((p->a4 * x + p->a3) * x + p->a2) * x + p->a1) * x + p->a0; }

static void w_panel(const poly4_t *p, ld a, ld b, ld *K, ld *G, ld *Kabs) {
    ld h = 0.5L * (b - a), m = 0.5L * (a + b);
    *K = *G = *Kabs = 0.0L;
    for (int i = 0; i < 21; ++i) {
        ld x = expl(m + h * GK21_X[i]);
        ld E2 = w_E2(p, x);
        ld kappa = ((((fabsl(p->a4) * x + fabsl(p->a3)) * x + fabsl(p->a2)) * x + fabsl(p->a1)) * x + fabsl(p->a0)) / fabsl(E2);
        ld f = x / sqrtl(E2);                       /* dx/E = x du/E */
        *K += GK21_WK[i] * f; *G += GK21_WG[i] * f; *Kabs += GK21_WK[i] * fabsl(f) * kappa;
    }
    *K *= h; *G *= h; *Kabs *= h;
}

static void w_adapt(const poly4_t *p, ld a, ld b, ld frac, ld scale, int depth, ld *acc, int *npanels) {
    ld K, G, Kabs;
    w_panel(p, a, b, &K, &G, &Kabs);
    ld err = fabsl(K - G);
    int ok = !(err > GK_TOL * scale * frac && err > GK_ROUND * LDBL_EPSILON * Kabs);
    if (err != err) ok = 1;
    if (ok || depth >= GK_MAXDEPTH || *npanels >= GK_MAXPANELS) { *acc += K; ++*npanels; return; }
    ld m = 0.5L * (a + b);
    w_adapt(p, a, m, 0.5L * frac, scale, depth + 1, acc, npanels);
    w_adapt(p, m, b, 0.5L * frac, scale, depth + 1, acc, npanels);
}

/* val[4] = D_C, D_M, D_L [Mpc], mu [mag]; dz[4] = their d/dz.  Returns 0, -1 (E^2 <= 0 on the path or z <= -1:
 * NaN) or 1 (D_L <= 0: mu NaN). */
int oracle_w_chi(ld z, ld Om, ld OL, ld Or, ld Ow13, ld Ow23, ld H0, ld val[4], ld dz[4]) {
    ld Ok = 1.0L - Om - OL - Or - Ow13 - Ow23;
    poly4_t p = { Or, Om, Ok + Ow13, Ow23, OL };
    for (int i = 0; i < 4; ++i) val[i] = dz[i] = NAN;
    if (!(z > -1.0L)) return -1;
    ld U = log1pl(z), I0 = 0.0L;
    for (int i = 0; i <= 64; ++i)
        if (!(w_E2(&p, expl(U * i / 64.0L)) > 0.0L)) return -1;
    if (z != 0.0L) {
        ld K, G, Kabs;
        w_panel(&p, 0.0L, U, &K, &G, &Kabs);
        int npanels = 0, nseg = (int)ceill(fabsl(U));
        if (nseg < 1) nseg = 1;
        for (int s = 0; s < nseg; ++s) w_adapt(&p, U * s / nseg, U * (s + 1) / nseg, 1.0L / nseg, fabsl(K), 0, &I0, &npanels);
    }
    ld x = 1.0L + z, E = sqrtl(w_E2(&p, x)), dH = C_KM_S / H0;
    ld F, Fi, Fk;
    sinn_transform(Ok, I0, &F, &Fi, &Fk);
    val[0] = dH * I0; val[1] = dH * F; val[2] = x * dH * F;
    dz[0] = dH / E; dz[1] = dH * Fi / E; dz[2] = dH * F + x * dz[1];
    if (!(val[2] > 0)) return 1;
    val[3] = 5.0L * log10l(val[2]) + 25.0L;
    dz[3] = 5.0L / logl(10.0L) * dz[2] / val[2];
    return 0;
}

/* batch; parameter arrays of length n_cosmo in {1, n}; val, dz: [n][4] */
void oracle_w_chi_batch(int64_t n, const double *z, const double *Om, const double *OL, const double *Or, const double *Ow13,
                        const double *Ow23, const double *H0, int64_t n_cosmo, ld *val, ld *dz, int32_t *status) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t j = (n_cosmo == 1) ? 0 : i;
        int rc = oracle_w_chi((ld)z[i], (ld)Om[j], (ld)OL[j], (ld)Or[j], (ld)Ow13[j], (ld)Ow23[j], (ld)H0[j], val + i * 4, dz + i * 4);
        if (status) status[i] = rc;
    }
}

/* ======================================================================================
 * (10) the w family in full (rest): all three integrals of eqs. (2.3)-(2.5) for the polynomial of (9), the six
 *      observables of (2) and their total derivatives with respect to (z, Om, OL, Or, Ow13, Ow23, H0), Ok = 1 - (sum of the five
 *      densities) eliminated: by Leibniz' rule
 *        dE^2/dOm = x^3 - x^2, dE^2/dOL = 1 - x^2, dE^2/dOr = x^4 - x^2, dE^2/dOw13 = x^2 - x^2 = 0, dE^2/dOw23 = x - x^2,
 *      and dOk/dtheta = -1 for each of the five in the curvature transform.  Same adaptive GK21 in u = ln x, written out for this
 *      integrand set so that (1) and (9) stay exactly as pinned.
 *      q[15] = I0, T, A, then d I0 / d(Om, OL, Or, Ow23), d T / d(..), d A / d(..)   (Ow13: identically zero, not stored).
 * ====================================================================================== */
#define NVW 15
static ld w_integrand_full(const poly4_t *p, int nv, ld u, ld f[NVW]) {
    ld x = expl(u);
    ld E2 = w_E2(p, x);
    ld kappa = ((((fabsl(p->a4) * x + fabsl(p->a3)) * x + fabsl(p->a2)) * x + fabsl(p->a1)) * x + fabsl(p->a0)) / fabsl(E2);
    ld E = sqrtl(E2);
    f[0] = x / E; f[1] = 1.0L / E; f[2] = x * x * x / E;
    if (nv > 3) {
        ld E3 = E2 * E, x2 = x * x, zz = expm1l(u);
        ld d[4] = { x2 * zz, -zz * (x + 1.0L), x2 * zz * (x + 1.0L), -x * zz };      /* x^3-x^2, 1-x^2, x^4-x^2, x-x^2 */
        ld w[3] = { -0.5L * x / E3, -0.5L / E3, -0.5L * x2 * x / E3 };
        for (int k = 0; k < 3; ++k)
            for (int t = 0; t < 4; ++t) f[3 + 4 * k + t] = w[k] * d[t];
    }
    return kappa;
}
static void w_panel_full(const poly4_t *p, int nv, ld a, ld b, ld K[NVW], ld G[NVW], ld Kabs[NVW]) {
    ld h = 0.5L * (b - a), m = 0.5L * (a + b), f[NVW];
    for (int v = 0; v < nv; ++v) K[v] = G[v] = Kabs[v] = 0.0L;
    for (int i = 0; i < 21; ++i) {
        ld kappa = w_integrand_full(p, nv, m + h * GK21_X[i], f);
        for (int v = 0; v < nv; ++v) { K[v] += GK21_WK[i] * f[v]; G[v] += GK21_WG[i] * f[v]; Kabs[v] += GK21_WK[i] * fabsl(f[v]) * kappa; }
    }
    for (int v = 0; v < nv; ++v) { K[v] *= h; G[v] *= h; Kabs[v] *= h; }
}
static void w_adapt_full(const poly4_t *p, int nv, ld a, ld b, ld frac, const ld scale[NVW], int depth, ld acc[NVW], int *npanels) {
    ld K[NVW], G[NVW], Kabs[NVW];
    w_panel_full(p, nv, a, b, K, G, Kabs);
    int ok = 1;
    for (int v = 0; v < nv; ++v) {
        ld err = fabsl(K[v] - G[v]);
        if (err > GK_TOL * scale[v] * frac && err > GK_ROUND * LDBL_EPSILON * Kabs[v]) ok = 0;
        if (err != err) ok = 1;
    }
    if (ok || depth >= GK_MAXDEPTH || *npanels >= GK_MAXPANELS) { for (int v = 0; v < nv; ++v) acc[v] += K[v]; ++*npanels; return; }
    ld m = 0.5L * (a + b);
    w_adapt_full(p, nv, a, m, 0.5L * frac, scale, depth + 1, acc, npanels);
    w_adapt_full(p, nv, m, b, 0.5L * frac, scale, depth + 1, acc, npanels);
}

enum { WWRT_Z = 0, WWRT_OM, WWRT_OL, WWRT_OR, WWRT_OW13, WWRT_OW23, WWRT_H0, N_WWRT };

/* val[N_OBS] (order of (2): DC, DM, DL, MU, TL, DABS), grad[N_OBS][N_WWRT] (nullable).  Returns 0, -1 (invalid path: NaN) or 1 (D_L <= 0). */
int oracle_w_observables(ld z, ld Om, ld OL, ld Or, ld Ow13, ld Ow23, ld H0, ld val[N_OBS], ld *grad) {
    ld Ok = 1.0L - Om - OL - Or - Ow13 - Ow23;
    poly4_t p = { Or, Om, Ok + Ow13, Ow23, OL };
    for (int i = 0; i < N_OBS; ++i) val[i] = NAN;
    if (grad) for (int i = 0; i < N_OBS * N_WWRT; ++i) grad[i] = NAN;
    if (!(z > -1.0L)) return -1;
    ld U = log1pl(z), q[NVW];
    int nv = grad ? NVW : 3;
    for (int v = 0; v < NVW; ++v) q[v] = 0.0L;
    for (int i = 0; i <= 64; ++i)
        if (!(w_E2(&p, expl(U * i / 64.0L)) > 0.0L)) return -1;
    if (z != 0.0L) {
        ld scale[NVW], K[NVW], G[NVW], Kabs[NVW];
        w_panel_full(&p, nv, 0.0L, U, K, G, Kabs);
        for (int v = 0; v < nv; ++v) scale[v] = fabsl(K[v]);
        int npanels = 0, nseg = (int)ceill(fabsl(U));
        if (nseg < 1) nseg = 1;
        for (int s = 0; s < nseg; ++s) w_adapt_full(&p, nv, U * s / nseg, U * (s + 1) / nseg, 1.0L / nseg, scale, 0, q, &npanels);
    }
    ld x = 1.0L + z, E = sqrtl(w_E2(&p, x)), dH = C_KM_S / H0, tH = HUBBLE_GYR / H0;
    ld I0 = q[0], T = q[1], A = q[2], F, Fi, Fk;
    sinn_transform(Ok, I0, &F, &Fi, &Fk);
    val[OBS_DC] = dH * I0; val[OBS_DM] = dH * F; val[OBS_DL] = x * dH * F;
    int status = 0;
    if (val[OBS_DL] > 0) val[OBS_MU] = 5.0L * log10l(val[OBS_DL]) + 25.0L;
    else { val[OBS_MU] = NAN; status = 1; }
    val[OBS_TL] = tH * T; val[OBS_DABS] = dH * A;
    if (!grad) return status;
    ld (*g)[N_WWRT] = (ld (*)[N_WWRT])grad;
    g[OBS_DC][WWRT_Z] = dH / E;
    g[OBS_DM][WWRT_Z] = dH * Fi / E;
    g[OBS_DL][WWRT_Z] = dH * F + x * g[OBS_DM][WWRT_Z];
    g[OBS_TL][WWRT_Z] = tH / (x * E);
    g[OBS_DABS][WWRT_Z] = dH * x * x / E;
    const int col[5] = { 0, 1, 2, -1, 3 };             /* Om, OL, Or, Ow13 (no E^2 dependence), Ow23 -> column of q */
    for (int t = 0; t < 5; ++t) {
        ld dI = col[t] >= 0 ? q[3 + col[t]] : 0.0L, dT = col[t] >= 0 ? q[7 + col[t]] : 0.0L, dA = col[t] >= 0 ? q[11 + col[t]] : 0.0L;
        g[OBS_DC][WWRT_OM + t] = dH * dI;
        g[OBS_DM][WWRT_OM + t] = dH * (Fi * dI - Fk);           /* dOk/dtheta = -1 */
        g[OBS_DL][WWRT_OM + t] = x * g[OBS_DM][WWRT_OM + t];
        g[OBS_TL][WWRT_OM + t] = tH * dT;
        g[OBS_DABS][WWRT_OM + t] = dH * dA;
    }
    for (int o = 0; o < N_OBS; ++o) if (o != OBS_MU) g[o][WWRT_H0] = -val[o] / H0;
    for (int w = 0; w < N_WWRT; ++w)
        g[OBS_MU][w] = (status == 0) ? 5.0L / logl(10.0L) * g[OBS_DL][w] / val[OBS_DL] : NAN;
    return status;
}

void oracle_w_observables_batch(int64_t n, const double *z, const double *Om, const double *OL, const double *Or, const double *Ow13,
                                const double *Ow23, const double *H0, int64_t n_cosmo, ld *val, ld *grad, int32_t *status) {
#pragma omp parallel for schedule(dynamic, 64)
    for (int64_t i = 0; i < n; ++i) {
        int64_t j = (n_cosmo == 1) ? 0 : i;
        int rc = oracle_w_observables((ld)z[i], (ld)Om[j], (ld)OL[j], (ld)Or[j], (ld)Ow13[j], (ld)Ow23[j], (ld)H0[j], val + i * N_OBS,
                                      grad ? grad + i * N_OBS * N_WWRT : NULL);
        if (status) status[i] = rc;
    }
}
