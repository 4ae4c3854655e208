"""Thin Python binding of the C ABI in include/cosmo_b200.h: argument marshalling only.

Every step of the hot path runs inside libcosmo_b200.so's CUDA kernels.  PyTorch supplies device memory and the
current stream.  There is no CPU path: loading fails loudly if the library is missing, and every call requires
CUDA tensors.
"""
from __future__ import annotations

import ctypes as C
import os

HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(HERE, "libcosmo_b200.so")

ELEMENTWISE, OUTER = 0, 1
DC, DM, DL, MU, TL, DABS, DA, VC, AGE = 1, 2, 4, 8, 16, 32, 64, 128, 256
WHICH_BITS = {"DC": DC, "DM": DM, "DL": DL, "MU": MU, "TL": TL, "DABS": DABS, "DA": DA, "VC": VC, "AGE": AGE}
WHICH_ORDER = ("DC", "DM", "DL", "MU", "TL", "DABS", "DA", "VC", "AGE")

# every symbol include/cosmo_b200.h and include/cosmo_b200_diag.h declare
SYMBOLS = ("cosmo_host_release", "cosmo_snia_loglike_static", "cosmo_static_scratch_bytes", "cosmo_eval2_workspace_bytes", "cosmo_eval_w_workspace_bytes", "cosmo_workspace_bytes", "cosmo_eval", "cosmo_vjp", "cosmo_snia_loglike", "cosmo_eval_f32", "cosmo_vjp_f32",
           "cosmo_snia_loglike_f32", "cosmo_snia_logjoint", "cosmo_eval2", "cosmo_eval_w", "cosmo_eval_host", "cosmo_carlson_pair", "cosmo_probe_fma_f64", "cosmo_probe_fma_f32",
           "cosmo_profile", "cosmo_profile_mean_ms",
           "cosmo_launch_count", "cosmo_last_cuda_error", "cosmo_strerror", "cosmo_version")


class CosmoParams(C.Structure):
    _fields_ = [("Om", C.c_void_p), ("OL", C.c_void_p), ("Or", C.c_void_p), ("H0", C.c_void_p)]


class CosmoError(RuntimeError):
    pass


_lib = None


def lib():
    """dlopen the CUDA library (no GPU needed to load it); raises if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise CosmoError(f"{LIB_PATH} is missing: build it with `python -m paper_2212_01937_b200.build` "
                         "(there is no CPU fallback)")
    L = C.CDLL(LIB_PATH)
    vp, i64, u32, sz, ci = C.c_void_p, C.c_int64, C.c_uint32, C.c_size_t, C.c_int
    L.cosmo_workspace_bytes.argtypes = [i64, i64, ci, u32, ci]
    L.cosmo_workspace_bytes.restype = sz
    for name in ("cosmo_eval", "cosmo_eval_f32"):
        f = getattr(L, name)
        f.argtypes = [vp, i64, CosmoParams, i64, ci, u32, vp, vp, vp, sz, vp]
        f.restype = ci
    for name in ("cosmo_vjp", "cosmo_vjp_f32"):
        f = getattr(L, name)
        f.argtypes = [vp, i64, CosmoParams, i64, ci, u32, vp, vp, vp, vp, vp, vp, sz, vp]
        f.restype = ci
    for name in ("cosmo_snia_loglike", "cosmo_snia_loglike_f32"):
        f = getattr(L, name)
        f.argtypes = [vp, vp, vp, i64, CosmoParams, i64, vp, vp, vp, sz, vp]
        f.restype = ci
    L.cosmo_snia_loglike_static.argtypes = [vp, vp, vp, i64, CosmoParams, i64, vp, vp, vp]
    L.cosmo_snia_loglike_static.restype = ci
    L.cosmo_static_scratch_bytes.restype = sz
    L.cosmo_eval_host.argtypes = [vp, i64, CosmoParams, i64, ci, u32, vp, vp, vp, vp, vp]
    L.cosmo_eval_host.restype = ci
    for name in ("cosmo_probe_fma_f64", "cosmo_probe_fma_f32"):
        f = getattr(L, name)
        f.argtypes = [ci, ci, vp, vp]
        f.restype = ci
    L.cosmo_snia_logjoint.argtypes = [vp, vp, vp, vp, C.c_double, C.c_double, C.c_double, i64, CosmoParams, i64, vp, vp, vp, vp, sz, vp]
    L.cosmo_snia_logjoint.restype = ci
    L.cosmo_eval2.argtypes = [vp, vp, i64, CosmoParams, i64, u32, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    L.cosmo_eval2_workspace_bytes.argtypes = [i64, ci]
    L.cosmo_eval2_workspace_bytes.restype = sz
    L.cosmo_eval2.restype = ci
    L.cosmo_eval_w.argtypes = [vp, i64, vp, vp, vp, vp, vp, vp, i64, u32, vp, vp, vp, vp, vp, vp, vp, sz, vp]
    L.cosmo_eval_w_workspace_bytes.argtypes = [i64]
    L.cosmo_eval_w_workspace_bytes.restype = sz
    L.cosmo_eval_w.restype = ci
    L.cosmo_carlson_pair.argtypes = [vp, vp, vp, vp, i64, vp, vp, vp, vp]
    L.cosmo_carlson_pair.restype = ci
    L.cosmo_launch_count.restype = i64
    L.cosmo_profile.argtypes = [ci]
    L.cosmo_profile.restype = ci
    L.cosmo_profile_mean_ms.argtypes = [C.POINTER(i64)]
    L.cosmo_profile_mean_ms.restype = C.c_double
    L.cosmo_last_cuda_error.restype = ci
    L.cosmo_strerror.argtypes = [ci]
    L.cosmo_strerror.restype = C.c_char_p
    L.cosmo_version.restype = C.c_char_p
    _lib = L
    return L


def which_mask(which) -> int:
    if isinstance(which, int):
        return which
    m = 0
    for w in which:
        m |= WHICH_BITS[w]
    return m


def which_names(mask: int):
    return tuple(n for n in WHICH_ORDER if mask & WHICH_BITS[n])


def _check(rc: int):
    if rc != 0:
        L = lib()
        msg = L.cosmo_strerror(rc).decode()
        if rc == -6:
            msg += f" [cudaError {L.cosmo_last_cuda_error()}]"
        raise CosmoError(f"cosmo_b200 error {rc}: {msg}")


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise CosmoError("CUDA device required: the hot path runs only in CUDA kernels (no CPU fallback)")
    return torch


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


def _dev(t, dtype, torch, name):
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise CosmoError(f"{name}: expected a contiguous CUDA tensor of dtype {dtype}")
    return t


def _params(Om, OL, Or, H0, torch):
    ps = [_dev(p, torch.float64, torch, "params") for p in (Om, OL, Or, H0)]
    n = ps[0].numel()
    if any(p.numel() != n for p in ps):
        raise CosmoError("Om, OL, Or, H0 must have the same length")
    return CosmoParams(*[p.data_ptr() for p in ps]), n, ps


def _stream(torch):
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def workspace_bytes(n_z, n_cosmo, mode, which, with_grad) -> int:
    return int(lib().cosmo_workspace_bytes(n_z, n_cosmo, mode, which_mask(which), int(with_grad)))


def _given(t, shape, dtype, torch, name, device):
    """a caller-supplied output buffer: contiguous CUDA tensor of the expected dtype, element count and device"""
    if t is None:
        return None
    n = 1
    for d in shape:
        n *= d
    if not (t.is_cuda and t.dtype == dtype and t.is_contiguous() and t.numel() == n and t.device == device):
        raise CosmoError(f"{name}: expected a contiguous {dtype} CUDA tensor with {n} elements {tuple(shape)} on {device}")
    return t


def _workspace(torch, nbytes, device, workspace):
    if workspace is not None:
        if not (workspace.is_cuda and workspace.is_contiguous() and workspace.device == device):
            raise CosmoError(f"workspace: expected a contiguous CUDA tensor on {device}")
        if workspace.numel() * workspace.element_size() < nbytes:
            raise CosmoError("workspace tensor too small")
        return workspace
    return torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)


def cosmo_eval(z, Om, OL, Or, H0, mode=ELEMENTWISE, which=("DC",), out=None, status=None, workspace=None):
    """Forward.  Returns (out[n_which, rows, n_z], status[rows, n_z] uint8)."""
    torch = _torch()
    mask = which_mask(which)
    f32 = z.dtype == torch.float32
    dt = torch.float32 if f32 else torch.float64
    _dev(z, dt, torch, "z")
    P, n_cosmo, keep = _params(Om, OL, Or, H0, torch)
    n_z = z.numel()
    rows = n_cosmo if mode == OUTER else 1
    nw = bin(mask).count("1")
    _given(out, (nw, rows, n_z), dt, torch, "out", z.device)
    _given(status, (rows, n_z), torch.uint8, torch, "status", z.device)
    if out is None:
        out = torch.empty((nw, rows, n_z), dtype=dt, device=z.device)
    if status is None:
        status = torch.empty((rows, n_z), dtype=torch.uint8, device=z.device)
    ws_b = workspace_bytes(n_z, n_cosmo, mode, mask, False)
    ws = _workspace(torch, ws_b, z.device, workspace)
    fn = lib().cosmo_eval_f32 if f32 else lib().cosmo_eval
    with torch.cuda.device(z.device):          # kernels and stream of the tensors' device, whatever the current one is
        _check(fn(_ptr(z), n_z, P, n_cosmo, mode, mask, _ptr(out), _ptr(status), _ptr(ws), ws.numel() * ws.element_size(), _stream(torch)))
    return out, status


def cosmo_vjp(z, Om, OL, Or, H0, grad_out, mode=ELEMENTWISE, which=("DC",), want_out=False, out=None, grad_z=None,
              grad_params=None, status=None, workspace=None):
    """Fused forward + VJP.  Returns (grad_z[n_z], grad_params[4, n_cosmo] float64, out or None, status)."""
    torch = _torch()
    mask = which_mask(which)
    f32 = z.dtype == torch.float32
    dt = torch.float32 if f32 else torch.float64
    _dev(z, dt, torch, "z")
    _dev(grad_out, dt, torch, "grad_out")
    P, n_cosmo, keep = _params(Om, OL, Or, H0, torch)
    n_z = z.numel()
    rows = n_cosmo if mode == OUTER else 1
    nw = bin(mask).count("1")
    if grad_out.numel() != nw * rows * n_z:
        raise CosmoError("grad_out must have shape [n_which, rows, n_z]")
    _given(out, (nw, rows, n_z), dt, torch, "out", z.device)
    _given(grad_z, (n_z,), dt, torch, "grad_z", z.device)
    _given(grad_params, (4, n_cosmo), torch.float64, torch, "grad_params", z.device)
    _given(status, (rows, n_z), torch.uint8, torch, "status", z.device)
    if want_out and out is None:
        out = torch.empty((nw, rows, n_z), dtype=dt, device=z.device)
    if grad_z is None:
        grad_z = torch.empty(n_z, dtype=dt, device=z.device)
    if grad_params is None:
        grad_params = torch.empty((4, n_cosmo), dtype=torch.float64, device=z.device)
    if status is None:
        status = torch.empty((rows, n_z), dtype=torch.uint8, device=z.device)
    ws_b = workspace_bytes(n_z, n_cosmo, mode, mask, True)
    ws = _workspace(torch, ws_b, z.device, workspace)
    fn = lib().cosmo_vjp_f32 if f32 else lib().cosmo_vjp
    with torch.cuda.device(z.device):
        _check(fn(_ptr(z), n_z, P, n_cosmo, mode, mask, _ptr(grad_out), _ptr(out), _ptr(grad_z), _ptr(grad_params), _ptr(status),
                  _ptr(ws), ws.numel() * ws.element_size(), _stream(torch)))
    return grad_z, grad_params, out, status


def cosmo_snia_loglike(z, mu_obs, sigma, Om, OL, Or, H0, want_grad=True, logL=None, grad=None, workspace=None):
    """Fused SN-Ia Gaussian log-likelihood.  Returns (logL[S], grad[4, S] or None), float64."""
    torch = _torch()
    f32 = z.dtype == torch.float32
    dt = torch.float32 if f32 else torch.float64
    for t, nm in ((z, "z"), (mu_obs, "mu_obs"), (sigma, "sigma")):
        _dev(t, dt, torch, nm)
    P, S, keep = _params(Om, OL, Or, H0, torch)
    N = z.numel()
    _given(logL, (S,), torch.float64, torch, "logL", z.device)
    _given(grad, (4, S), torch.float64, torch, "grad", z.device)
    if mu_obs.numel() != N or sigma.numel() != N:
        raise CosmoError("z, mu_obs and sigma must have the same length")
    if logL is None:
        logL = torch.empty(S, dtype=torch.float64, device=z.device)
    if want_grad and grad is None:
        grad = torch.empty((4, S), dtype=torch.float64, device=z.device)
    ws_b = workspace_bytes(N, S, OUTER, MU, True)
    ws = _workspace(torch, ws_b, z.device, workspace)
    fn = lib().cosmo_snia_loglike_f32 if f32 else lib().cosmo_snia_loglike
    with torch.cuda.device(z.device):
        _check(fn(_ptr(z), _ptr(mu_obs), _ptr(sigma), N, P, S, _ptr(logL), _ptr(grad), _ptr(ws), ws.numel() * ws.element_size(), _stream(torch)))
    return logL, grad


def cosmo_snia_loglike_static(z, mu_obs, sigma, Om, OL, Or, H0, want_grad=True, logL=None, grad=None):
    """cosmo_snia_loglike without workspace or allocation inside the library (static device scratch of 24 MiB, shared by all calls on the
    GPU: do not overlap calls).  FP64.  Pass logL / grad to keep this wrapper from allocating the outputs.  Raises CosmoError (-7) when
    (N, S) exceeds the static scratch.  Returns (logL[S], grad[4, S] or None)."""
    torch = _torch()
    for t, nm in ((z, "z"), (mu_obs, "mu_obs"), (sigma, "sigma")):
        _dev(t, torch.float64, torch, nm)
    P, S, keep = _params(Om, OL, Or, H0, torch)
    N = z.numel()
    if logL is None:
        logL = torch.empty(S, dtype=torch.float64, device=z.device)
    if want_grad and grad is None:
        grad = torch.empty((4, S), dtype=torch.float64, device=z.device)
    with torch.cuda.device(z.device):          # the static array's address is taken for the CURRENT device
        _check(lib().cosmo_snia_loglike_static(_ptr(z), _ptr(mu_obs), _ptr(sigma), N, P, S, _ptr(logL), _ptr(grad), _stream(torch)))
    return logL, grad


def static_scratch_bytes() -> int:
    return int(lib().cosmo_static_scratch_bytes())


def cosmo_snia_logjoint(z, z_obs, mu_obs, sigma_mu, sigma_z, beta, shape, Om, OL, Or, H0, want_grad=True, workspace=None):
    """Log-joint with latent redshifts z[S, N].  Returns (logp[S], grad[4, S] or None, grad_z[S, N] or None)."""
    torch = _torch()
    for t, nm in ((z, "z"), (z_obs, "z_obs"), (mu_obs, "mu_obs"), (sigma_mu, "sigma_mu")):
        _dev(t, torch.float64, torch, nm)
    P, S, keep = _params(Om, OL, Or, H0, torch)
    N = z_obs.numel()
    if z.numel() != S * N:
        raise CosmoError("z must have shape [S, N]")
    logp = torch.empty(S, dtype=torch.float64, device=z.device)
    grad = torch.empty((4, S), dtype=torch.float64, device=z.device) if want_grad else None
    gz = torch.empty((S, N), dtype=torch.float64, device=z.device) if want_grad else None
    ws = _workspace(torch, workspace_bytes(N, S, OUTER, MU, True), z.device, workspace)
    _check(lib().cosmo_snia_logjoint(_ptr(z), _ptr(z_obs), _ptr(mu_obs), _ptr(sigma_mu), float(sigma_z), float(beta), float(shape), N, P, S,
                                     _ptr(logp), _ptr(grad), _ptr(gz), _ptr(ws), ws.numel(), _stream(torch)))
    return logp, grad, gz


def cosmo_eval2(z1, z2, Om, OL, Or, H0, which=("DC",), grad_out=None, want_out=True, workspace=None):
    """Two-limit forms between z1 and z2 (elementwise).  Returns (out[n_which, n] or None, grad_z1, grad_z2, grad_params[4, n], status);
    the gradients are None without grad_out.  which from DC, DM, TL, DABS, DA."""
    torch = _torch()
    mask = which_mask(which)
    _dev(z1, torch.float64, torch, "z1"); _dev(z2, torch.float64, torch, "z2")
    P, n_cosmo, keep = _params(Om, OL, Or, H0, torch)
    n = z1.numel()
    nw = bin(mask).count("1")
    out = torch.empty((nw, n), dtype=torch.float64, device=z1.device) if (want_out or grad_out is None) else None
    status = torch.empty(n, dtype=torch.uint8, device=z1.device)
    g1 = g2 = gp = None
    if grad_out is not None:
        _dev(grad_out, torch.float64, torch, "grad_out")
        g1 = torch.empty(n, dtype=torch.float64, device=z1.device)
        g2 = torch.empty(n, dtype=torch.float64, device=z1.device)
        gp = torch.empty((4, n), dtype=torch.float64, device=z1.device)
    ws_b = int(lib().cosmo_eval2_workspace_bytes(n, int(grad_out is not None)))
    ws = _workspace(torch, ws_b, z1.device, workspace) if ws_b else None
    _check(lib().cosmo_eval2(_ptr(z1), _ptr(z2), n, P, n_cosmo, mask, _ptr(grad_out), _ptr(out), _ptr(g1), _ptr(g2), _ptr(gp), _ptr(status),
                             _ptr(ws), ws_b, _stream(torch)))
    return out, g1, g2, gp, status


def cosmo_eval_w(z, Om, OL, Or, Ow13, Ow23, H0, which=("DC",), want_dz=True, grad_out=None, workspace=None):
    """Extra constant-w components w = -1/3 (Ow13) and w = -2/3 (Ow23), PAPER.md:82 fn.4 (elementwise; parameters of length 1 or n).
    which from DC, DM, DL, MU, TL, DABS.  Returns (out[n_which, n], dout_dz[n_which, n] or None, status[n]); with grad_out also
    (grad_z[n], grad_params[6, n]) appended, the parameters in the order (Om, OL, Or, Ow13, Ow23, H0)."""
    torch = _torch()
    mask = which_mask(which)
    _dev(z, torch.float64, torch, "z")
    n = z.numel()
    ps = []
    for t, nm in ((Om, "Om"), (OL, "OL"), (Or, "Or"), (Ow13, "Ow13"), (Ow23, "Ow23"), (H0, "H0")):
        _dev(t, torch.float64, torch, nm)
        ps.append(t)
    n_cosmo = ps[0].numel()
    if any(t.numel() != n_cosmo for t in ps):
        raise CosmoError("parameter arrays must have equal lengths")
    nw = bin(mask).count("1")
    out = torch.empty((nw, n), dtype=torch.float64, device=z.device)
    dz = torch.empty((nw, n), dtype=torch.float64, device=z.device) if want_dz else None
    status = torch.empty(n, dtype=torch.uint8, device=z.device)
    gz = gp = None
    if grad_out is not None:
        _dev(grad_out, torch.float64, torch, "grad_out")
        if grad_out.numel() != nw * n:
            raise CosmoError("grad_out must have shape [n_which, n]")
        gz = torch.empty(n, dtype=torch.float64, device=z.device)
        gp = torch.empty((6, n), dtype=torch.float64, device=z.device)
    ws_b = int(lib().cosmo_eval_w_workspace_bytes(n_cosmo))
    ws = _workspace(torch, ws_b, z.device, workspace)
    _check(lib().cosmo_eval_w(_ptr(z), n, *[_ptr(t) for t in ps], n_cosmo, mask, _ptr(grad_out), _ptr(out), _ptr(dz), _ptr(gz), _ptr(gp),
                              _ptr(status), _ptr(ws), ws_b, _stream(torch)))
    if grad_out is None:
        return out, dz, status
    return out, dz, status, gz, gp


def cosmo_eval_host(z, Om, OL, Or, H0, mode=ELEMENTWISE, which=("DC",), grad_out=None, want_out=True, want_status=True, out=None,
                    grad_z=None, grad_params=None, status=None):
    """Host-buffer call (numpy float64 arrays in, numpy out): H2D + kernels + D2H inside the library, synchronous.  Pass pinned arrays
    (inputs and, through out / grad_z / grad_params / status, outputs) for full PCIe speed; outputs not passed are allocated here."""
    import numpy as np
    _torch()
    mask = which_mask(which)
    arrs = [np.ascontiguousarray(a, dtype=np.float64) for a in (z, Om, OL, Or, H0)]
    n_z, n_cosmo = arrs[0].shape[0], arrs[1].shape[0]
    rows = n_cosmo if mode == OUTER else 1
    nw = bin(mask).count("1")
    vp = lambda a: C.c_void_p(a.ctypes.data) if a is not None else C.c_void_p(0)
    P = CosmoParams(*[a.ctypes.data for a in arrs[1:]])

    def buf(given, shape, dtype, want):
        if given is not None:
            if given.shape != shape or given.dtype != dtype or not given.flags.c_contiguous:
                raise CosmoError(f"output buffer: expected a C-contiguous {dtype} array of shape {shape}")
            return given
        return np.empty(shape, dtype=dtype) if want else None
    out = buf(out, (nw, rows, n_z), np.float64, want_out or grad_out is None)
    status = buf(status, (rows, n_z), np.uint8, want_status)
    gz = gp = None
    if grad_out is not None:
        grad_out = np.ascontiguousarray(grad_out, dtype=np.float64)
        if grad_out.size != nw * rows * n_z:
            raise CosmoError("grad_out must have shape [n_which, rows, n_z]")
        gz = buf(grad_z, (n_z,), np.float64, True)
        gp = buf(grad_params, (4, n_cosmo), np.float64, True)
    _check(lib().cosmo_eval_host(vp(arrs[0]), n_z, P, n_cosmo, mode, mask, vp(grad_out), vp(out), vp(gz), vp(gp), vp(status)))
    return out, gz, gp, status


def carlson_pair(x, m, s, p):
    """R_F(x, m+h, m-h), R_D(m+h, m-h, x), R_J(x, m+h, m-h, p) with h^2 = s, by the hot path's device functions"""
    torch = _torch()
    for t in (x, m, s, p):
        _dev(t, torch.float64, torch, "carlson_pair argument")
    n = x.numel()
    rf, rd, rj = (torch.empty(n, dtype=torch.float64, device=x.device) for _ in range(3))
    _check(lib().cosmo_carlson_pair(_ptr(x), _ptr(m), _ptr(s), _ptr(p), n, _ptr(rf), _ptr(rd), _ptr(rj), _stream(torch)))
    return rf, rd, rj


def cosmo_host_release():
    """frees the device staging buffers cosmo_eval_host keeps between calls"""
    f = lib().cosmo_host_release
    f.restype = None
    f()


def probe_fma(dtype="f64", blocks=148 * 8, iters=4096):
    """Launch the FMA-chain roofline probe on the current stream; returns flops of the launch."""
    torch = _torch()
    dt = torch.float64 if dtype == "f64" else torch.float32
    sink = torch.empty(blocks * 256, dtype=dt, device="cuda")
    fn = lib().cosmo_probe_fma_f64 if dtype == "f64" else lib().cosmo_probe_fma_f32
    _check(fn(blocks, iters, _ptr(sink), _stream(torch)))
    return blocks * 256 * iters * 8 * 2, sink


def profile(on: bool):
    """start/stop CUDA-event timing of the dominant kernel of each call (see include/cosmo_b200.h)"""
    _check(lib().cosmo_profile(int(on)))


def profile_mean_ms():
    n = C.c_int64(0)
    ms = lib().cosmo_profile_mean_ms(C.byref(n))
    return float(ms), int(n.value)


def launch_count() -> int:
    return int(lib().cosmo_launch_count())


def version() -> str:
    return lib().cosmo_version().decode()
