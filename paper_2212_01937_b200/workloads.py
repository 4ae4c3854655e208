"""Seeded synthetic inputs for the five BASELINE.json configs (recipe: DESIGN.md "Input recipe").

This module serves BOTH the oracle-side tests and the CUDA-side tests/bench.  It holds none of the
method's arithmetic: only random draws and, for the structured stress rows of config 5, linear
solves on the DEFINITION of E^2 (eq. (2.2)) that place roots where the config asks.
It imports neither `oracle` nor the CUDA binding.

The paper's own workloads are mock/synthetic (redshift grids of PAPER.md:233,:247; mock SNe Ia of
PAPER.md:283,:297), so these inputs do not stand in for any public dataset.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

__all__ = ["Workload", "config1", "config2", "config3", "config3_shard", "config4", "config5", "invalid_rows", "e2_min_on_path"]


@dataclass
class Workload:
    name: str
    mode: str                      # "elementwise" | "outer"
    z: np.ndarray                  # float64 [N]
    Om: np.ndarray                 # float64 [S] (S == 1, N (elementwise) or #cosmologies (outer))
    OL: np.ndarray
    Or: np.ndarray
    H0: np.ndarray
    which: tuple                   # names of the outputs, ascending bit order
    grad_out: np.ndarray | None = None   # [n_which][rows][N]
    extra: dict = field(default_factory=dict)

    @property
    def n_z(self):
        return self.z.shape[0]

    @property
    def n_cosmo(self):
        return self.Om.shape[0]

    @property
    def n_evals(self):
        return self.n_z * (self.n_cosmo if self.mode == "outer" else 1)


def e2_min_on_path(z, Om, OL, Or):
    """min of E^2(x) (eq. 2.2) over x in [1, 1+z], from its stationary points (dE^2/dx = x(4 Or x^2 + 3 Om x + 2 Ok))."""
    z, Om, OL, Or = np.broadcast_arrays(*(np.asarray(a, dtype=np.float64) for a in (z, Om, OL, Or)))
    Ok = 1.0 - Om - OL - Or
    xmax = 1.0 + z

    def e2(x):
        return Or * x ** 4 + Om * x ** 3 + Ok * x ** 2 + OL

    m = np.minimum(e2(np.ones_like(xmax)), e2(xmax))
    disc = 9.0 * Om ** 2 - 32.0 * Or * Ok
    with np.errstate(invalid="ignore", divide="ignore"):
        sq = np.sqrt(np.where(disc >= 0, disc, np.nan))
        cands = [np.where(Or > 0, (-3.0 * Om + s * sq) / (8.0 * np.where(Or > 0, Or, 1.0)), np.nan) for s in (1.0, -1.0)]
        cands.append(np.where(Or == 0, -2.0 * Ok / (3.0 * Om), np.nan))
    for xs in cands:
        ok = np.isfinite(xs) & (xs > 1.0) & (xs < xmax)
        m = np.where(ok, np.minimum(m, e2(np.where(ok, xs, 1.0))), m)
    return m


def config1(n: int = 10_000, seed: int = 1) -> Workload:
    """Flat LCDM, one cosmology (0.3, 0.7, 0, 70), z ~ U(0.01, 2); outputs D_C and mu, forward only."""
    rng = np.random.default_rng(seed)
    z = 0.01 + 1.99 * rng.random(n)
    one = lambda v: np.array([v], dtype=np.float64)
    return Workload("config1", "elementwise", z, one(0.3), one(0.7), one(0.0), one(70.0), ("DC", "MU"))


def config2(n: int = 1_000_000, seed: int = 2) -> Workload:
    """General LCDM + radiation + curvature, one cosmology per element; D_C, D_M, t_L, d_abs forward."""
    rng = np.random.default_rng(seed)

    def draw(m):
        z = rng.uniform(0.001, 5.0, m)
        Om = rng.uniform(0.05, 0.6, m)
        OL = rng.uniform(0.0, 1.2, m)
        Or = 10.0 ** rng.uniform(-5.0, -3.0, m)
        H0 = rng.uniform(60.0, 80.0, m)
        return z, Om, OL, Or, H0

    cols = list(draw(n))
    for _ in range(100):   # redraw rows in the no-Big-Bang region so that n valid rows remain
        bad = ~(e2_min_on_path(cols[0], cols[1], cols[2], cols[3]) > 1e-3)
        if not bad.any():
            break
        new = draw(int(bad.sum()))
        for c, v in zip(cols, new):
            c[bad] = v
    z, Om, OL, Or, H0 = cols
    return Workload("config2", "elementwise", z, Om, OL, Or, H0, ("DC", "DM", "TL", "DABS"))


def _vi_samples(rng, S, Or_value):
    Om = rng.normal(0.3, 0.05, S)
    OL = rng.normal(0.7, 0.05, S)
    Or = np.full(S, Or_value)
    H0 = rng.normal(70.0, 2.0, S)
    return Om, OL, Or, H0


def config3(n: int = 1_000_000, S: int = 64, seed: int = 3, which=("MU",)) -> Workload:
    """VI minibatch: n sorted mock-SN redshifts x S cosmology samples, forward + VJP; grad_out ~ N(0,1) [1][S][n]."""
    rng = np.random.default_rng(seed)
    z = np.sort(rng.uniform(0.01, 1.5, n))
    Om, OL, Or, H0 = _vi_samples(rng, S, 9e-5)
    g = rng.standard_normal((len(which), S, n))
    return Workload("config3", "outer", z, Om, OL, Or, H0, tuple(which), grad_out=g)


def config3_shard(n_per_rank: int, world: int, rank: int, S: int = 64, seed: int = 3, which=("MU",)) -> Workload:
    """Rank `rank`'s part of ONE config-3 job of world x n_per_rank sorted redshifts (multi-GPU runs): the global
    redshift array is drawn and sorted once and cut contiguously (sharding.shard_bounds); the upstream gradient of a shard is drawn
    from (seed, shard index), so the job on `world` ranks and the same job on one rank (its shards concatenated) see identical inputs."""
    from .sharding import shard_bounds
    rng = np.random.default_rng(seed)
    z = np.sort(rng.uniform(0.01, 1.5, n_per_rank * world))
    Om, OL, Or, H0 = _vi_samples(rng, S, 9e-5)
    lo, hi = shard_bounds(n_per_rank * world, world, rank)
    g = np.random.default_rng([seed, rank]).standard_normal((len(which), S, hi - lo))
    return Workload("config3", "outer", z[lo:hi], Om, OL, Or, H0, tuple(which), grad_out=g)


def config4(mu_fn, n: int = 1_000_000, S: int = 256, seed: int = 4) -> Workload:
    """Fused SN-Ia likelihood.  mu_fn(z, Om, OL, Or, H0) -> mu[n] supplies the noiseless distance moduli of the
    fiducial cosmology (0.3, 0.7, 0, 70): tests pass the ORACLE's mu; for timing-only runs any mu source does.
    sigma = 0.1 per object; S samples drawn as config 3 but radiation-less (reading R-c4)."""
    rng = np.random.default_rng(seed)
    z = rng.uniform(0.01, 1.5, n)
    noise = rng.normal(0.0, 0.1, n)
    sigma = np.full(n, 0.1)
    Om, OL, Or, H0 = _vi_samples(rng, S, 0.0)
    mu_true = np.asarray(mu_fn(z, 0.3, 0.7, 0.0, 70.0), dtype=np.float64)
    return Workload("config4", "outer", z, Om, OL, Or, H0, ("MU",),
                    extra={"mu_obs": mu_true + noise, "sigma": sigma})


def _solve_Om_OL(Or, rows, rhs):
    """Solve the 2x2 real systems  rows[...,2,2] @ (Om, OL) = rhs[...,2]  (E^2 is linear in Om, OL at fixed Or)."""
    a, b, c, d = rows[..., 0, 0], rows[..., 0, 1], rows[..., 1, 0], rows[..., 1, 1]
    det = a * d - b * c
    Om = (rhs[..., 0] * d - b * rhs[..., 1]) / det
    OL = (a * rhs[..., 1] - c * rhs[..., 0]) / det
    return Om, OL


def _e2_linear_rows(x):
    """E^2(x) = Or (x^4 - x^2) + Om (x^3 - x^2) + OL (1 - x^2) + x^2  (Ok eliminated): coefficient of (Om, OL)."""
    return np.stack([x ** 3 - x ** 2, 1.0 - x ** 2], axis=-1)


def _block_a(rng, m, Or):
    """Just inside the no-Big-Bang boundary: (Om, OL_crit) put a DOUBLE root of E^2 at x_d > 1; OL = OL_crit - delta."""
    xd = rng.uniform(2.5, 6.0, m)
    row0 = _e2_linear_rows(xd)
    row1 = np.stack([3 * xd ** 2 - 2 * xd, -2 * xd], axis=-1)        # d/dx of the coefficients
    rhs = np.stack([-(Or * (xd ** 4 - xd ** 2) + xd ** 2), -(Or * (4 * xd ** 3 - 2 * xd) + 2 * xd)], axis=-1)
    Om, OLc = _solve_Om_OL(Or, np.stack([row0, row1], axis=-2), rhs)
    delta = 10.0 ** rng.uniform(-6.0, -1.0, m)
    z = (xd - 1.0) * rng.uniform(1.05, 3.0, m)                        # past the loitering redshift
    return z, Om, OLc - delta, {"delta": delta, "x_d": xd}


def _block_b(rng, m, Or):
    """Near-degenerate REAL pair: two real roots of E^2 in x in (0,1) separated by gap (recollapsing closed models)."""
    xc = rng.uniform(0.03, 0.35, m)
    gap = np.minimum(10.0 ** rng.uniform(-6.0, -1.0, m), xc)
    x1, x2 = xc - 0.5 * gap, xc + 0.5 * gap
    rows = np.stack([_e2_linear_rows(x1), _e2_linear_rows(x2)], axis=-2)
    rhs = np.stack([-(Or * (x1 ** 4 - x1 ** 2) + x1 ** 2), -(Or * (x2 ** 4 - x2 ** 2) + x2 ** 2)], axis=-1)
    Om, OL = _solve_Om_OL(Or, rows, rhs)
    z = 10.0 ** rng.uniform(-2.0, 1.0, m)
    return z, Om, OL, {"gap": gap, "x_c": xc}


def _block_c(rng, m, Or):
    """Complex-conjugate pair with Re x > 1 (yellow region of Fig. 1): roots at xr +- i y."""
    xr = rng.uniform(1.05, 6.0, m)
    y = rng.uniform(0.05, 3.0, m)
    rho = xr + 1j * y
    cm = rho ** 3 - rho ** 2
    cl = 1.0 - rho ** 2
    r = -(Or * (rho ** 4 - rho ** 2) + rho ** 2)
    rows = np.stack([np.stack([cm.real, cl.real], axis=-1), np.stack([cm.imag, cl.imag], axis=-1)], axis=-2)
    Om, OL = _solve_Om_OL(Or, rows, np.stack([r.real, r.imag], axis=-1))
    z = (xr - 1.0) * rng.uniform(0.5, 4.0, m)
    return z, Om, OL, {"x_re": xr, "x_im": y}


def _structured(rng, maker, m):
    """Draw until m rows satisfy Om in (0.02, 3), OL in [0, 3), |Ok| <= 0.5, E^2 > 0 on the path."""
    out = None
    need = m
    for _ in range(400):
        k = max(4 * need, 256)
        Or = rng.choice(np.array([0.0, 9e-5, 1e-3]), k)
        z, Om, OL, info = maker(rng, k, Or)
        with np.errstate(all="ignore"):
            ok = ((Om > 0.02) & (Om < 3.0) & (OL >= 0.0) & (OL < 3.0) & (np.abs(1.0 - Om - OL - Or) <= 0.5)
                  & (e2_min_on_path(z, Om, OL, Or) > 0.0))
        cols = [z[ok], Om[ok], OL[ok], Or[ok]] + [v[ok] for v in info.values()]
        out = cols if out is None else [np.concatenate([a, b]) for a, b in zip(out, cols)]
        need = m - out[0].shape[0]
        if need <= 0:
            break
    assert out is not None and out[0].shape[0] >= m, "structured block generator starved"
    out = [a[:m] for a in out]
    return out[0], out[1], out[2], out[3], dict(zip(info.keys(), out[4:]))


def config5(n: int = 10_000_000, n_struct: int = 100_000, seed: int = 5) -> Workload:
    """Stress: n random rows (z log-uniform in [1e-4, 1100], Ok ~ U(-.5,.5), Om ~ U(.05,1.5), Or in {0, 9e-5, 1e-3})
    followed by three structured blocks of n_struct rows each (a: near no-Big-Bang boundary, b: near-degenerate
    real pair, c: c.c. pair with Re x > 1).  Elementwise; all six outputs; forward + VJP with grad_out ~ N(0,1)."""
    rng = np.random.default_rng(seed)

    def draw(m):
        z = 10.0 ** rng.uniform(-4.0, np.log10(1100.0), m)
        Or = rng.choice(np.array([0.0, 9e-5, 1e-3]), m)
        Ok = rng.uniform(-0.5, 0.5, m)
        Om = rng.uniform(0.05, 1.5, m)
        OL = 1.0 - Om - Or - Ok
        return z, Om, OL, Or

    cols = list(draw(n))
    for _ in range(200):
        bad = (cols[2] < 0.0) | ~(e2_min_on_path(cols[0], cols[1], cols[2], cols[3]) > 1e-3)
        if not bad.any():
            break
        new = draw(int(bad.sum()))
        for c, v in zip(cols, new):
            c[bad] = v
    blocks = {"random": (0, n)}
    infos = {}
    start = n
    for name, maker in (("a_boundary", _block_a), ("b_real_pair", _block_b), ("c_cc_pair_re_gt_1", _block_c)):
        z, Om, OL, Or, info = _structured(rng, maker, n_struct)
        cols = [np.concatenate([c, v]) for c, v in zip(cols, (z, Om, OL, Or))]
        blocks[name] = (start, start + n_struct)
        infos[name] = info
        start += n_struct
    z, Om, OL, Or = cols
    H0 = rng.uniform(60.0, 80.0, z.shape[0])
    which = ("DC", "DM", "DL", "MU", "TL", "DABS")
    g = rng.standard_normal((len(which), 1, z.shape[0]))
    return Workload("config5", "elementwise", z, Om, OL, Or, H0, which, grad_out=g,
                    extra={"blocks": blocks, "info": infos})


def invalid_rows():
    """Hand-built rows for the status path: (z, Om, OL, Or, H0, expected status bit).
    1: E^2 has a root on (0, z] (no-Big-Bang region); 2: unsupported (degree < 3 / negative density /
    z <= -1); 4: D_L <= 0 (closed universe past the antipode)."""
    rows = [
        (8.0, 0.05, 1.5, 0.0, 70.0, 1),
        (8.0, 0.05, 1.5, 9e-5, 70.0, 1),
        (3.0, 0.01, 1.2, 1e-5, 70.0, 1),
        (1.0, 0.0, 1.0, 0.0, 70.0, 2),
        (1.0, -0.1, 0.7, 9e-5, 70.0, 2),
        (1.0, 0.3, -0.2, 9e-5, 70.0, 2),
        (1.0, 0.3, 0.7, -1e-5, 70.0, 2),
        (-1.5, 0.3, 0.7, 9e-5, 70.0, 2),
    ]
    return rows


def wmix(n: int = 20_000, seed: int = 7):
    """Inputs for the extra-w family (PAPER.md:82 fn.4): per-element cosmologies with components of w = -1/3 and
    w = -2/3 beside matter, Lambda, radiation and curvature; log-uniform z in [1e-3, 10].  The first rows are the structural
    cases: single-component universes and polynomials of every degree 0..4.  Returns dict of float64 arrays
    z, Om, OL, Or, Ow13, Ow23, H0."""
    rng = np.random.default_rng(seed)
    z = 10.0 ** rng.uniform(-3.0, 1.0, n)
    Om = rng.uniform(0.05, 0.5, n)
    OL = rng.uniform(0.0, 0.9, n)
    Or = rng.choice([0.0, 1e-5, 9e-5, 1e-3], n)
    Ow13 = np.where(rng.random(n) < 0.9, rng.uniform(0.0, 0.3, n), rng.uniform(-0.05, 0.0, n))
    Ow23 = np.where(rng.random(n) < 0.9, rng.uniform(0.0, 0.3, n), rng.uniform(-0.05, 0.0, n))
    H0 = rng.uniform(60.0, 80.0, n)
    special = [  # (Om, OL, Or, Ow13, Ow23)
        (0.0, 0.0, 0.0, 0.0, 1.0),      # E^2 = x
        (0.0, 0.0, 0.0, 1.0, 0.0),      # E^2 = x^2, flat
        (0.0, 0.0, 0.0, 0.0, 0.0),      # Milne
        (0.0, 1.0, 0.0, 0.0, 0.0),      # de Sitter: degree 0
        (1.0, 0.0, 0.0, 0.0, 0.0),      # Einstein-de Sitter
        (0.0, 0.0, 1.0, 0.0, 0.0),      # radiation only
        (0.0, 0.65, 0.0, 0.0, 0.35),    # degree 1
        (0.0, 0.65, 0.0, 0.35, 0.0),    # degree 2, flat
        (0.35, 0.0, 0.0, 0.0, 0.65),    # degree 3 without constant term
        (0.3, 0.7, 0.0, 0.0, 0.0), (0.3, 0.7, 9e-5, 0.0, 0.0), (0.27, 0.55, 8e-5, 0.06, 0.09),
    ]
    k = min(len(special), n)
    for i in range(k):
        Om[i], OL[i], Or[i], Ow13[i], Ow23[i] = special[i]
    return {"z": z, "Om": Om, "OL": OL, "Or": Or, "Ow13": Ow13, "Ow23": Ow23, "H0": H0}
