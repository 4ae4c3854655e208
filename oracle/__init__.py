"""ORACLE -- test infrastructure, not the product.

ctypes binding of oracle/liboracle.so (plain C, long double; see cosmo_oracle.c for what each
function computes and the passage of PAPER.md it follows).  Only tests/, __graft_entry__.smoke()
and bench.py's cpu_baseline / --impl reference legs may import this package.  It imports nothing
from paper_2212_01937_b200 and shares no code with the CUDA path.
"""
import ctypes as C
import numpy as np

from .build import build as _build

OBS = ("DC", "DM", "DL", "MU", "TL", "DABS")        # order of the observable axis
WRT = ("z", "Om", "OL", "Or", "H0")                 # order of the derivative axis
N_OBS, N_WRT, NV = 6, 5, 12

_lib = None
_LD = C.c_longdouble
_LDP = C.POINTER(C.c_longdouble)
_DP = C.POINTER(C.c_double)


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_integrals.argtypes = [_LD, _LD, _LD, _LD, C.c_int, _LDP]
        _lib.oracle_integrals.restype = C.c_int
        _lib.oracle_age_dimless.argtypes = [_LD, _LD, _LD, _LD]
        _lib.oracle_age_dimless.restype = _LD
        _lib.oracle_observables.argtypes = [_LD] * 5 + [_LDP, _LDP]
        _lib.oracle_observables.restype = C.c_int
        _lib.oracle_observables_batch.argtypes = [C.c_int64, _DP, _DP, _DP, _DP, _DP, C.c_int64, _LDP, _LDP,
                                                  C.POINTER(C.c_int32)]
        _lib.oracle_observables_batch.restype = None
        _lib.oracle_derived_batch.argtypes = [C.c_int64, _DP, _DP, _DP, _DP, _DP, C.c_int64, _LDP, _LDP, C.POINTER(C.c_int32)]
        _lib.oracle_derived_batch.restype = None
        _lib.oracle_snia_loglike.argtypes = [C.c_int64, _DP, _DP, _DP] + [C.c_double] * 4 + [C.c_int, _LDP]
        _lib.oracle_snia_loglike.restype = C.c_int
        _lib.oracle_observables2_batch.argtypes = [C.c_int64, _DP, _DP, _DP, _DP, _DP, _DP, C.c_int64, _LDP, _LDP, C.POINTER(C.c_int32)]
        _lib.oracle_observables2_batch.restype = None
        _lib.oracle_w_chi_batch.argtypes = [C.c_int64] + [_DP] * 7 + [C.c_int64, _LDP, _LDP, C.POINTER(C.c_int32)]
        _lib.oracle_w_chi_batch.restype = None
        _lib.oracle_w_observables_batch.argtypes = [C.c_int64] + [_DP] * 7 + [C.c_int64, _LDP, _LDP, C.POINTER(C.c_int32)]
        _lib.oracle_w_observables_batch.restype = None
        _lib.oracle_snia_logjoint.argtypes = [C.c_int64, _DP, _DP, _DP, _DP] + [C.c_double] * 7 + [C.c_int, _LDP, _LDP]
        _lib.oracle_snia_logjoint.restype = C.c_int
        for name, nin in (("oracle_rf", 6), ("oracle_rc", 4), ("oracle_rd", 6), ("oracle_rj", 8)):
            f = getattr(_lib, name)
            f.argtypes = [C.c_double] * nin + [_LDP]
            f.restype = None
        _lib.oracle_gk21_rule.argtypes = [_LDP, _LDP, _LDP]
        _lib.oracle_max_threads.restype = C.c_int
        _lib.oracle_set_threads.argtypes = [C.c_int]
        _lib.oracle_ldbl_mant_dig.restype = C.c_int
        assert _lib.oracle_ldbl_mant_dig() >= 64
    return _lib


def _ldp(a):
    return a.ctypes.data_as(_LDP)


def _dp(a):
    return a.ctypes.data_as(_DP)


def integrals(z, Om, OL, Or, with_grad=True):
    """(I0, T, A[, dI0/d(Om,OL,Or), dT/d(..), dA/d(..)]) as np.longdouble[12]; eqs (2.3)-(2.5) without units."""
    out = np.zeros(NV, dtype=np.longdouble)
    rc = lib().oracle_integrals(_LD(z), _LD(Om), _LD(OL), _LD(Or), int(with_grad), _ldp(out))
    if rc < 0:
        out[:] = np.nan
    return out


def age_dimless(z, Om, OL, Or):
    """H0 * int_z^inf dt."""
    return np.longdouble(lib().oracle_age_dimless(_LD(z), _LD(Om), _LD(OL), _LD(Or)))


def observables(z, Om, OL, Or, H0, with_grad=True):
    """Scalar call with long-double inputs: val[6], grad[6,5] (np.longdouble), status."""
    val = np.zeros(N_OBS, dtype=np.longdouble)
    grad = np.zeros((N_OBS, N_WRT), dtype=np.longdouble)
    rc = lib().oracle_observables(_LD(z), _LD(Om), _LD(OL), _LD(Or), _LD(H0), _ldp(val),
                                  _ldp(grad) if with_grad else None)
    return val, (grad if with_grad else None), rc


def observables_batch(z, Om, OL, Or, H0, with_grad=True, threads=None):
    """z[n] float64; Om, OL, Or, H0 each scalar or float64[n].  Returns val[n,6], grad[n,6,5] or None,
    status[n] (0 ok, -1 invalid path, 1 D_L<=0), all values np.longdouble."""
    z = np.ascontiguousarray(z, dtype=np.float64)
    n = z.shape[0]
    ps = [np.ascontiguousarray(np.atleast_1d(p), dtype=np.float64) for p in (Om, OL, Or, H0)]
    n_cosmo = ps[0].shape[0]
    assert all(p.shape[0] == n_cosmo for p in ps) and n_cosmo in (1, n)
    val = np.zeros((n, N_OBS), dtype=np.longdouble)
    grad = np.zeros((n, N_OBS, N_WRT), dtype=np.longdouble) if with_grad else None
    status = np.zeros(n, dtype=np.int32)
    L = lib()
    if threads:
        L.oracle_set_threads(int(threads))
    L.oracle_observables_batch(n, _dp(z), *[_dp(p) for p in ps], n_cosmo, _ldp(val),
                               _ldp(grad) if with_grad else None, status.ctypes.data_as(C.POINTER(C.c_int32)))
    return val, grad, status


DERIVED = ("DA", "VC", "AGE")                       # order of oracle_derived's observable axis


def derived_batch(z, Om, OL, Or, H0, with_grad=True, threads=None):
    """Further derived observables: D_A [Mpc], V_C [Mpc^3, whole sky], age at z [Gyr].
    Returns val[n,3], grad[n,3,5] or None, status[n]; np.longdouble."""
    z = np.ascontiguousarray(z, dtype=np.float64)
    n = z.shape[0]
    ps = [np.ascontiguousarray(np.atleast_1d(p), dtype=np.float64) for p in (Om, OL, Or, H0)]
    n_cosmo = ps[0].shape[0]
    assert all(p.shape[0] == n_cosmo for p in ps) and n_cosmo in (1, n)
    val = np.zeros((n, 3), dtype=np.longdouble)
    grad = np.zeros((n, 3, N_WRT), dtype=np.longdouble) if with_grad else None
    status = np.zeros(n, dtype=np.int32)
    L = lib()
    if threads:
        L.oracle_set_threads(int(threads))
    L.oracle_derived_batch(n, _dp(z), *[_dp(p) for p in ps], n_cosmo, _ldp(val), _ldp(grad) if with_grad else None,
                           status.ctypes.data_as(C.POINTER(C.c_int32)))
    return val, grad, status


def snia_loglike(z, mu_obs, sigma, Om, OL, Or, H0, with_grad=True):
    """One cosmology: np.longdouble[5] = logL, dlogL/d(Om, OL, Or, H0)."""
    z, mu_obs, sigma = (np.ascontiguousarray(a, dtype=np.float64) for a in (z, mu_obs, sigma))
    out = np.zeros(5, dtype=np.longdouble)
    rc = lib().oracle_snia_loglike(z.shape[0], _dp(z), _dp(mu_obs), _dp(sigma), float(Om), float(OL), float(Or),
                                   float(H0), int(with_grad), _ldp(out))
    if rc != 0:
        out[:] = np.nan
    return out


OBS2 = ("DC", "DM", "TL", "DABS", "DA")              # two-limit observables
WRT2 = ("z1", "z2", "Om", "OL", "Or", "H0")


def observables2_batch(z1, z2, Om, OL, Or, H0, with_grad=True, threads=None):
    """Two-limit forms of eqs. (2.3)-(2.5): val[n,5] (OBS2), grad[n,5,6] (WRT2) or None, status[n]."""
    z1 = np.ascontiguousarray(z1, dtype=np.float64); z2 = np.ascontiguousarray(z2, dtype=np.float64)
    n = z1.shape[0]
    ps = [np.ascontiguousarray(np.atleast_1d(p), dtype=np.float64) for p in (Om, OL, Or, H0)]
    n_cosmo = ps[0].shape[0]
    assert z2.shape[0] == n and all(p.shape[0] == n_cosmo for p in ps) and n_cosmo in (1, n)
    val = np.zeros((n, 5), dtype=np.longdouble)
    grad = np.zeros((n, 5, 6), dtype=np.longdouble) if with_grad else None
    status = np.zeros(n, dtype=np.int32)
    L = lib()
    if threads:
        L.oracle_set_threads(int(threads))
    L.oracle_observables2_batch(n, _dp(z1), _dp(z2), *[_dp(p) for p in ps], n_cosmo, _ldp(val), _ldp(grad) if with_grad else None,
                                status.ctypes.data_as(C.POINTER(C.c_int32)))
    return val, grad, status


OBSW = ("DC", "DM", "DL", "MU")


def w_chi_batch(z, Om, OL, Or, Ow13, Ow23, H0, threads=None):
    """chi family with extra constant-w components, w = -1/3 and -2/3 (PAPER.md:82 fn.4):
    val[n,4] (OBSW), dz[n,4] = d val / dz, status[n] (0 ok, -1 invalid path, 1 D_L <= 0)."""
    z = np.ascontiguousarray(z, dtype=np.float64)
    n = z.shape[0]
    ps = [np.ascontiguousarray(np.atleast_1d(p), dtype=np.float64) for p in (Om, OL, Or, Ow13, Ow23, H0)]
    n_cosmo = ps[0].shape[0]
    assert all(p.shape[0] == n_cosmo for p in ps) and n_cosmo in (1, n)
    val = np.zeros((n, 4), dtype=np.longdouble)
    dz = np.zeros((n, 4), dtype=np.longdouble)
    status = np.zeros(n, dtype=np.int32)
    L = lib()
    if threads:
        L.oracle_set_threads(int(threads))
    L.oracle_w_chi_batch(n, _dp(z), *[_dp(p) for p in ps], n_cosmo, _ldp(val), _ldp(dz), status.ctypes.data_as(C.POINTER(C.c_int32)))
    return val, dz, status


WRTW = ("z", "Om", "OL", "Or", "Ow13", "Ow23", "H0")


def w_observables_batch(z, Om, OL, Or, Ow13, Ow23, H0, with_grad=True, threads=None):
    """All six observables (OBS order) with extra constant-w components and their total derivatives (WRTW order):
    val[n,6], grad[n,6,7] or None, status[n] (0 ok, -1 invalid path, 1 D_L <= 0).  PAPER.md:82 fn.4; SURVEY NEXT-3."""
    z = np.ascontiguousarray(z, dtype=np.float64)
    n = z.shape[0]
    ps = [np.ascontiguousarray(np.atleast_1d(p), dtype=np.float64) for p in (Om, OL, Or, Ow13, Ow23, H0)]
    n_cosmo = ps[0].shape[0]
    assert all(p.shape[0] == n_cosmo for p in ps) and n_cosmo in (1, n)
    val = np.zeros((n, N_OBS), dtype=np.longdouble)
    grad = np.zeros((n, N_OBS, 7), dtype=np.longdouble) if with_grad else None
    status = np.zeros(n, dtype=np.int32)
    L = lib()
    if threads:
        L.oracle_set_threads(int(threads))
    L.oracle_w_observables_batch(n, _dp(z), *[_dp(p) for p in ps], n_cosmo, _ldp(val), _ldp(grad) if with_grad else None,
                                 status.ctypes.data_as(C.POINTER(C.c_int32)))
    return val, grad, status


def snia_logjoint(z, z_obs, mu_obs, sigma_mu, sigma_z, beta, shape, Om, OL, Or, H0, with_grad=True):
    """Log-joint of the section-4 toy model with latent redshifts, one cosmology:
    (np.longdouble[5] = log p, d/d(Om, OL, Or, H0);  grad_z[n] np.longdouble or None)."""
    z, z_obs, mu_obs, sigma_mu = (np.ascontiguousarray(a, dtype=np.float64) for a in (z, z_obs, mu_obs, sigma_mu))
    out = np.zeros(5, dtype=np.longdouble)
    gz = np.zeros(z.shape[0], dtype=np.longdouble) if with_grad else None
    rc = lib().oracle_snia_logjoint(z.shape[0], _dp(z), _dp(z_obs), _dp(mu_obs), _dp(sigma_mu), float(sigma_z), float(beta),
                                    float(shape), float(Om), float(OL), float(Or), float(H0), int(with_grad), _ldp(out),
                                    _ldp(gz) if with_grad else None)
    if rc != 0:
        out[:] = np.nan
    return out, gz


def _carlson(name, *args):
    out = np.zeros(2, dtype=np.longdouble)
    flat = []
    for a in args:
        a = complex(a)
        flat += [a.real, a.imag]
    getattr(lib(), name)(*flat, _ldp(out))
    return out[0] if out[1] == 0 else complex(out[0], out[1])


def rf(x, y, z): return _carlson("oracle_rf", x, y, z)       # eq. (2.6)
def rc(x, y): return _carlson("oracle_rc", x, y)             # eq. (2.8)
def rd(x, y, z): return _carlson("oracle_rd", x, y, z)       # eq. (2.9)
def rj(x, y, z, p): return _carlson("oracle_rj", x, y, z, p)  # eq. (2.7)


def gk21_rule():
    x, wk, wg = (np.zeros(21, dtype=np.longdouble) for _ in range(3))
    lib().oracle_gk21_rule(_ldp(x), _ldp(wk), _ldp(wg))
    return x, wk, wg


def max_threads():
    return int(lib().oracle_max_threads())
