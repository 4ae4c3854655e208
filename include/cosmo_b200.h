/* cosmo_b200.h -- C ABI of the B200-native LCDM+radiation cosmography library (libcosmo_b200.so).
 *
 * What the calls compute (PAPER.md = arXiv:2212.01937 text; DESIGN.md lists every reading of it):
 *   E^2(z) = Or (1+z)^4 + Om (1+z)^3 + Ok (1+z)^2 + OL,  Ok = 1 - Om - OL - Or      eq. (2.2)
 *   chi   = (c/H0) int_0^z dz'/E                                                       eq. (2.3)
 *   t     = (1/H0) int_0^z dz'/((1+z')E)          (lookback time)                      eq. (2.4)
 *   d_abs = (c/H0) int_0^z (1+z')^2 dz'/E                                              eq. (2.5)
 * evaluated in closed form by Carlson's symmetric integrals R_F, R_J, R_D, R_C, eqs. (3.7)-(3.9)
 * and (B.1)-(B.3) when Or = 0, plus the derived observables of PAPER.md:95 and :277 fn.22:
 *   D_C = chi;  D_M = (c/H0) sinn(sqrt|Ok| I0)/sqrt|Ok|  (sin for Ok<0, sinh for Ok>0);  D_L = (1+z) D_M;
 *   mu = 5 log10(D_L / 10 pc);  t_L = t;  d_abs;
 *   and D_A = D_M/(1+z) [Mpc], the comoving volume of the whole sky out to z,
 *   V_C = 4 pi int_0^chi D_M^2 dchi' [Mpc^3], and the age at z, int_z^inf of eq. (2.4) [Gyr].
 *   (The age plane is formed as t(0 -> inf) - t(0 -> z), once per cosmology and once per redshift: its relative error is that of
 *   t_L times t(inf)/age(z) -- 1e-13 below z = 10, 1e-10 at z = 1000.  The early-universe age to full precision is the t plane of
 *   cosmo_eval2 between z and z2 = 1e10 plus the remainder of the leading term beyond it, 2/(3 sqrt(Om)) z2^(-3/2) / H0 (matter) or
 *   1/(2 sqrt(Or)) z2^(-2) / H0 (radiation): 1e-14 at every z, tests/test_gpu_parity.py::test_age_high_z.)
 * and their analytic gradients with respect to z and (Om, OL, Or, H0), Ok eliminated.
 *
 * Units: H0 in km/s/Mpc; distances in Mpc (c = 299792.458 km/s); t_L in Gyr (1/H0 = 977.7922216807891/H0 Gyr); mu in mag.
 *
 * Conventions for every call:
 *   - every pointer is a DEVICE pointer owned by the caller unless marked "host"; the device-pointer calls allocate nothing
 *     (scratch comes in through `workspace`); only cosmo_eval_host, which takes host pointers, keeps device staging buffers of
 *     its own (released by cosmo_host_release);
 *   - the call only enqueues kernels on `stream` (a cudaStream_t passed as void*; NULL = legacy default stream),
 *     it never synchronises; results are valid after the stream reaches the end of the enqueued work;
 *   - return value 0 = enqueued; negative = COSMO_E_* below, nothing was launched (argument errors) or the CUDA
 *     launch failed (COSMO_E_CUDA; cosmo_last_cuda_error() gives the cudaError_t);
 *   - per-element domain problems never abort: the element's outputs are NaN and its status byte carries
 *       1  a root of E^2 lies on (0, z] (no-Big-Bang region)
 *       2  unsupported input: Om <= 0, Or < 0, OL < 0, H0 <= 0, z <= -1, non-finite, or a root structure that could not be
 *          factorised (the method needs E^2 of degree 3 or 4)
 *       4  D_L <= 0 (closed universe at/after the antipode): mu is NaN, the other outputs are valid
 *       8  the duplication loop hit its iteration cap before Carlson's stopping rule was met; from cosmo_eval_w also: t_L or d_abs
 *          came out not-a-number on a valid path (an isolated coincidence inside the complex Carlson functions: reported, not silent)
 *      16  a parameter gradient of this element is not served to the documented accuracy (set by the VJP calls; values valid).
 *          Where roots of E^2 (nearly) coincide the closed-form gradient bases cancel -- the 1/prod(r_j - r_k) of PAPER.md:320-345 --
 *          and the element's gradient integrals are taken from Gauss-Legendre quadrature of their definition instead (also at
 *          OL = 0: Einstein-de Sitter, open and closed matter models), so this bit is left for: a near-repeated pair whose centre
 *          lies ON the path while the bases cancel, and the gradient of the age plane when the bases are singular (OL = 0).
 */
#ifndef COSMO_B200_H
#define COSMO_B200_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ELEMENTWISE: n_cosmo == n_z (one cosmology per redshift) or n_cosmo == 1; rows = 1.
 * OUTER      : every redshift with every cosmology (PAPER.md:287 fn.24); rows = n_cosmo, element (s, n) at [s*n_z + n]. */
typedef enum { COSMO_ELEMENTWISE = 0, COSMO_OUTER = 1 } cosmo_mode;

/* `which` bitmask; the selected planes are stored in ascending bit order: out[plane][row][n]. */
enum { COSMO_DC = 1, COSMO_DM = 2, COSMO_DL = 4, COSMO_MU = 8, COSMO_TL = 16, COSMO_DABS = 32,
       COSMO_DA = 64, COSMO_VC = 128, COSMO_AGE = 256 };

enum {
    COSMO_OK = 0,
    COSMO_E_NULL = -1,      /* a required pointer is NULL                        */
    COSMO_E_SIZE = -2,      /* negative size, or n_cosmo incompatible with mode  */
    COSMO_E_WHICH = -3,     /* which == 0 or has unknown bits                    */
    COSMO_E_MODE = -4,      /* unknown mode                                      */
    COSMO_E_WORKSPACE = -5, /* ws_bytes < cosmo_workspace_bytes(...)             */
    COSMO_E_CUDA = -6,      /* kernel launch failed                              */
    COSMO_E_STATIC_LIMIT = -7 /* problem too large for the fixed static scratch of cosmo_snia_loglike_static */
};

/* SoA cosmological parameters, each of length n_cosmo.  Always FP64, also for the _f32 entry points
 * (reading R-fp32). */
typedef struct { const double *Om, *OL, *Or, *H0; } cosmo_params;

/* Bytes of scratch the calls below need (device memory, 256-byte aligned, contents undefined on entry and exit).  ELEMENTWISE calls
 * with one cosmology per redshift need none for the forward and a work list of n_z 32-bit indices for the VJP (n_z < 2^32). */
size_t cosmo_workspace_bytes(int64_t n_z, int64_t n_cosmo, int mode, uint32_t which, int with_grad);

/* Forward.  z[n_z]; out[n_which][rows][n_z]; status: nullable, [rows][n_z] bytes. */
int cosmo_eval(const double* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which,
               double* out, uint8_t* status, void* workspace, size_t ws_bytes, void* stream);

/* Fused forward + vector-Jacobian product (no tape).  grad_out has the layout of out.  out: nullable.
 * grad_z[n_z]            = sum over rows and planes of grad_out * d out / d z        (overwritten)
 * grad_params[4][n_cosmo] = sum over the redshifts that use cosmology s, order (Om, OL, Or, H0), total derivatives
 *                           with Ok = 1 - Om - OL - Or eliminated                     (overwritten)
 * Invalid elements (status 1, 2) contribute NaN. */
int cosmo_vjp(const double* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which,
              const double* grad_out, double* out, double* grad_z, double* grad_params, uint8_t* status,
              void* workspace, size_t ws_bytes, void* stream);

/* Fused distance-modulus -> Gaussian log-likelihood for S cosmology samples over N supernovae:
 *   logL[s] = sum_n [ -1/2 ((mu_obs[n] - mu(z[n]; theta_s)) / sigma[n])^2 - ln sigma[n] - 1/2 ln 2 pi ]
 *   grad[4][S] = d logL[s] / d (Om, OL, Or, H0)   (nullable)
 * Elements with status != 0 contribute NaN. */
int cosmo_snia_loglike(const double* z, const double* mu_obs, const double* sigma, int64_t N, cosmo_params p, int64_t S,
                       double* logL, double* grad, void* workspace, size_t ws_bytes, void* stream);

/* The same likelihood WITHOUT a workspace and without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it): the scratch is a static device array of COSMO_STATIC_SCRATCH_BYTES (24 MiB)
 * that every GPU loading the library holds until the process exits.  Same kernels and results as cosmo_snia_loglike (FP64).
 *   Limit: align256(928 S) + align256(40 S ceil(N / 512)) <= COSMO_STATIC_SCRATCH_BYTES, e.g. S = 256 samples x N <= 1.04e6 supernovae
 *   (BASELINE.json config 4 fits) or S = 64 x N <= 4.2e6; beyond it the call returns COSMO_E_STATIC_LIMIT and launches nothing.
 *   The call runs no cudaMalloc / cudaFree / allocating routine; its first use on a device asks the runtime for the array's address
 *   (cudaGetSymbolAddress, with the CURRENT device: `stream` must belong to it).
 *   All calls on a GPU share the array and it keeps the last call's contents (every call overwrites what it reads, nothing has to be
 *   cleared): calls that may overlap on the device -- different streams without ordering between them, different host threads -- race.
 *   Serialise them, or use cosmo_snia_loglike with one workspace per stream. */
#define COSMO_STATIC_SCRATCH_BYTES (24u << 20)
int cosmo_snia_loglike_static(const double* z, const double* mu_obs, const double* sigma, int64_t N, cosmo_params p, int64_t S,
                              double* logL, double* grad, void* stream);
size_t cosmo_static_scratch_bytes(void);

/* Log-joint of the paper's section-4 toy model with LATENT redshifts (one step of its variational fit evaluates this
 * and its gradient for S posterior samples): for sample s with redshifts z[s][0..N) and cosmology theta_s
 *   log p[s] = sum_n [ ln N(mu_obs[n] | mu(z[s][n]; theta_s), sigma_mu[n]^2) + ln N(z_obs[n] | z[s][n], (1+z[s][n])^2 sigma_z^2)
 *                      + ln Gamma(z[s][n]; shape, rate beta) ]
 *   grad[4][S]    = d log p[s] / d (Om, OL, Or, H0)      (nullable)
 *   grad_z[S][N]  = d log p[s] / d z[s][n]               (nullable)
 * (the paper fixes beta = 3, sigma_mu = 0.14, sigma_z = 0.04; it does not print the gamma shape: DESIGN.md reading R-prior.)
 * Workspace: cosmo_workspace_bytes(N, S, COSMO_OUTER, COSMO_MU, 1). */
int cosmo_snia_logjoint(const double* z, const double* z_obs, const double* mu_obs, const double* sigma_mu, double sigma_z,
                        double beta, double shape, int64_t N, cosmo_params p, int64_t S, double* logp, double* grad, double* grad_z,
                        void* workspace, size_t ws_bytes, void* stream);

/* FP32 variants: z, out, grad_out, grad_z, mu_obs, sigma are float and the per-element arithmetic is FP32;
 * parameters, the per-cosmology constants (root solve) and the reduced outputs grad_params / logL / grad stay FP64. */
int cosmo_eval_f32(const float* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which,
                   float* out, uint8_t* status, void* workspace, size_t ws_bytes, void* stream);
int cosmo_vjp_f32(const float* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which,
                  const float* grad_out, float* out, float* grad_z, double* grad_params, uint8_t* status,
                  void* workspace, size_t ws_bytes, void* stream);
int cosmo_snia_loglike_f32(const float* z, const float* mu_obs, const float* sigma, int64_t N, cosmo_params p, int64_t S,
                           double* logL, double* grad, void* workspace, size_t ws_bytes, void* stream);

/* Host-buffer convenience (every pointer is a HOST pointer; allocates device scratch, copies in, runs cosmo_vjp or
 * cosmo_eval (grad_out == NULL), copies out, synchronises).  This is the end-to-end call bench.py times as `e2e`. */
int cosmo_eval_host(const double* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which,
                    const double* grad_out, double* out, double* grad_z, double* grad_params, uint8_t* status);

/* TWO-LIMIT forms (PAPER.md:88-93 define chi(z1,z2), t(z1,z2), d_abs(z1,z2); eqs. (3.7)-(3.9) are two-limit as printed), one
 * (z1[i], z2[i], cosmology) per element; n_cosmo in {1, n}.  `which` may hold COSMO_DC (comoving distance between z1 and z2),
 * COSMO_DM (transverse distance between them, d_H sinn(...)), COSMO_TL (t(z1,z2)), COSMO_DABS, COSMO_DA (= D_M12/(1+z2));
 * planes out[n_which][n] in ascending bit order.  grad_out == NULL: forward (out required).  Otherwise also the VJP:
 * grad_z1[n], grad_z2[n], grad_params[4][n] (per element, order Om, OL, Or, H0; out nullable).  status as above.
 * workspace: cosmo_eval2_workspace_bytes(n, grad_out != NULL) bytes of device scratch. */
int cosmo_eval2(const double* z1, const double* z2, int64_t n, cosmo_params p, int64_t n_cosmo, uint32_t which, const double* grad_out,
                double* out, double* grad_z1, double* grad_z2, double* grad_params, uint8_t* status, void* workspace, size_t ws_bytes,
                void* stream);
/* scratch of cosmo_eval2: 0 for the forward call (workspace may be NULL), a work list of up to n indices with the VJP (n < 2^32) */
size_t cosmo_eval2_workspace_bytes(int64_t n, int with_grad);

/* EXTRA CONSTANT-w COMPONENTS (PAPER.md:82 fn.4: E^2 must be a polynomial of degree <= 4, which admits w in
 * {-1, -2/3, -1/3, 0, 1/3}):  E^2(x) = Or x^4 + Om x^3 + (Ok + Ow13) x^2 + Ow23 x + OL with Ok = 1 - Om - OL - Or - Ow13 - Ow23
 * (the curvature of the transverse distance is Ok alone).  `which` from COSMO_DC, COSMO_DM, COSMO_DL, COSMO_MU (eq. (3.7)/(B.1) on a
 * general real factorisation of the quartic), COSMO_TL, COSMO_DABS (eqs. (3.8)/(3.9), (B.2)/(B.3) with the polynomial's complex roots
 * and complex Carlson functions, as the paper formulates them).  One (z[i], cosmology) per element, parameter
 * arrays of length n_cosmo in {1, n} (device pointers).
 *   out[n_which][n] in ascending bit order (nullable with grad_out); dout_dz (nullable), same shape: d plane / dz.
 *   grad_out (nullable, [n_which][n]): also the VJP, per element: grad_z[n] and grad_params[6][n] in the order
 *   (Om, OL, Or, Ow13, Ow23, H0), total derivatives with Ok eliminated.  Their density part is the quadrature of the Leibniz integrals
 *   (a general quartic offers no fixed root structure for the closed-form gradient bases); status 16 where a root of E^2 sits too close
 *   to the path for that rule.
 *   status (nullable): 1 root of E^2 on the path / E^2 <= 0; 2 unsupported input or factorisation failure -- also set, with NaN in the
 *   t_L / d_abs planes only, where E^2 has degree <= 2 with distinct roots (the method needs degree 3 or 4; monomials
 *   E^2 = a x^n are served in closed form); 4 D_L <= 0; 8 iteration cap; 16 as above.
 *   workspace: cosmo_eval_w_workspace_bytes(n_cosmo) bytes: a shared cosmology is factored once per call into it; with per-element
 *   cosmologies it holds the work list of the second pass (elements that need the general root solve), n < 2^32. */
int cosmo_eval_w(const double* z, int64_t n, const double* Om, const double* OL, const double* Or, const double* Ow13,
                 const double* Ow23, const double* H0, int64_t n_cosmo, uint32_t which, const double* grad_out, double* out,
                 double* dout_dz, double* grad_z, double* grad_params, uint8_t* status, void* workspace, size_t ws_bytes, void* stream);
size_t cosmo_eval_w_workspace_bytes(int64_t n_cosmo);

/* frees the device staging buffers cosmo_eval_host keeps between calls (no-op if there are none) */
void cosmo_host_release(void);

int cosmo_last_cuda_error(void);
const char* cosmo_strerror(int code);
const char* cosmo_version(void);

#ifdef __cplusplus
}
#endif
#endif /* COSMO_B200_H */
