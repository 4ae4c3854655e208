"""Per-row tolerances of the parity tests (test helper; no arithmetic of the method's evaluation: only the DEFINITIONS of E^2,
eq. (2.2), and of the curvature transform are used to state how well-conditioned each row is).

BASELINE.json asks for relative error <= 1e-11 (FP64 values), <= 1e-8 (FP64 gradients), <= 2e-5 (FP32).  Those hold as MAXIMA on
every row whose result is well-conditioned.  Two families of rows are not, for ANY evaluation method in that precision, and get
the tolerance their conditioning allows instead of being left out:

  loitering   E^2 has a near-double root next to the path (config 5 block a: OL = OL_crit - delta): the integrand ~ 1/sqrt(E^2_min),
              and a rounding error eps in the inputs moves E^2_min by ~ eps, i.e. the integrals by ~ eps / E^2_min relative.
              Row tolerance: tol x max(1, LOITER_C x eps / (tol x E^2_min)).
  antipode    closed models with sqrt|Ok| I0 near a multiple of pi: D_M = d_H sin(a)/sqrt|Ok| -> 0, so a relative error tau of I0
              becomes tau x |a cot a| of D_M (and of D_L; mu = 5 log10 D_L gets the ABSOLUTE error 5/ln10 x that).
              Row tolerance of D_M, D_L: tol_I0 x max(1, |a cot a|).
"""
import numpy as np

from paper_2212_01937_b200 import workloads as W

EPS = np.finfo(np.float64).eps
LOITER_C = 8.0          # measured: error x E^2_min / eps <= 1 on config 5 block a; 8 is the margin
FIVE_OVER_LN10 = 5.0 / np.log(10.0)


def row_conditioning(z, Om, OL, Or, H0, I0_ref, tol):
    """returns (tau_int, amp_dm): per-row relative tolerance of the three integrals and the amplification I0 -> D_M"""
    z, Om, OL, Or = (np.asarray(a, dtype=np.float64) for a in (z, Om, OL, Or))
    e2min = np.maximum(W.e2_min_on_path(z, Om, OL, Or), 1e-300)
    tau = tol * np.maximum(1.0, LOITER_C * EPS / (tol * e2min))
    Ok = 1.0 - Om - OL - Or
    a = np.sqrt(np.abs(Ok)) * np.abs(np.asarray(I0_ref, dtype=np.float64))
    with np.errstate(divide="ignore", invalid="ignore"):
        amp = np.where(Ok < 0, np.abs(a / np.tan(a)), np.where(Ok > 0, np.abs(a / np.tanh(np.maximum(a, 1e-300))), 1.0))
    amp = np.maximum(1.0, np.nan_to_num(amp, nan=1.0, posinf=1e300))
    return tau, amp


def value_tolerance(name, tau, amp, mu_ref=None):
    """relative tolerance per row of plane `name` given the integrals' tolerance tau and the D_M amplification amp"""
    if name in ("DC", "TL", "DABS", "AGE"):
        return tau
    if name in ("DM", "DL", "DA"):
        return tau * amp + 4 * EPS
    if name == "MU":
        return tau + FIVE_OVER_LN10 * (tau * amp + 4 * EPS) / np.maximum(np.abs(mu_ref), 1e-300)
    if name == "VC":
        return 3 * tau * amp
    raise KeyError(name)


def grad_tolerance(name, tau, amp, tol_val, tol_grad, val_ref=None, mu_ref=None):
    """relative tolerance per row of the gradients of plane `name` (denominator max(|ref|, 1e-3 |value|), reading R-tol):
    the stated gradient tolerance, inflated on ill-conditioned rows by the same factors as the value; the gradients of mu carry
    1/D_L, hence D_L's own relative error on top."""
    infl = tau / tol_val
    if name in ("DC", "TL", "DABS", "AGE"):
        return tol_grad * infl
    if name in ("DM", "DL", "DA", "VC"):
        return tol_grad * infl * amp
    if name == "MU":
        return tol_grad * infl * amp + (tau * amp + 4 * EPS)
    raise KeyError(name)
