// cosmo_eval.cuh -- hot-path steps S4-S8 for ONE (z, cosmology) pair, templated on the arithmetic type.
//
// S4 radicands u_ij, S5 fused Carlson duplication (ref. [10]; eqs. (2.6)-(2.9)
// PAPER.md:115-131), S6 reductions eqs. (3.7)-(3.9) / (B.1)-(B.3),
// S7 observables (PAPER.md:95, :277 fn.22), S8 analytic gradients (eq. (2.10); appendix A).
//
// Real-quadratic form: with E^2 = Q1 Q2, the three arguments of R_F in eq. (3.7) are
//   xa = u12^2            = ( sqrt(Q1(x) Q2(1)) + sqrt(Q1(1) Q2(x)) )^2              (real, positive)
//   u13^2, u14^2 = mp +- h,  mp = xa - z^2 theta / 2,  h^2 = s = z^4 sD              (complex-conjugate pair when s < 0)
// and one duplication step (lambda = sum of pairwise products of the square roots) acts on (xa, mp, s) with
// real arithmetic only:  sqrt(y) sqrt(ybar) = sqrt(mp^2 - s),  sqrt(y) + sqrt(ybar) = sqrt(2 (mp + sqrt(mp^2 - s))).
#pragma once
#include "cosmo_types.cuh"

namespace cb {

template <typename T> struct Num;
template <> struct Num<double> {
    static CB_HD double sqrt_(double a) { return sqrt(a); }
    static CB_HD double log_(double a) { return log(a); }
    static CB_HD double exp_(double a) { return exp(a); }
    static CB_HD double atan_(double a) { return atan(a); }
    static CB_HD void sincos_(double a, double* s, double* c) { *s = sin(a); *c = cos(a); }
    static CB_HD double fma_(double a, double b, double c) { return fma(a, b, c); }
    static CB_HD double abs_(double a) { return fabs(a); }
    static CB_HD double max_(double a, double b) { return fmax(a, b); }
    static constexpr double QF = 400.0;    // (3 r)^(-1/6), r = 1e-16 (R_F stopping rule, ref. [10])
    static constexpr double QJ = 600.0;    // (r/4)^(-1/6)            (R_D, R_J)
    static constexpr double RC_SMALL = 0.03;
};
template <> struct Num<float> {
    static CB_HD float sqrt_(float a) { return sqrtf(a); }
    static CB_HD float log_(float a) { return logf(a); }
    static CB_HD float exp_(float a) { return expf(a); }
    static CB_HD float atan_(float a) { return atanf(a); }
    static CB_HD void sincos_(float a, float* s, float* c) { *s = sinf(a); *c = cosf(a); }
    static CB_HD float fma_(float a, float b, float c) { return fmaf(a, b, c); }
    static CB_HD float abs_(float a) { return fabsf(a); }
    static CB_HD float max_(float a, float b) { return fmaxf(a, b); }
    static constexpr float QF = 12.0f;     // r = 1e-7
    static constexpr float QJ = 19.0f;
    static constexpr float RC_SMALL = 0.25f;
};

// vote policy: the duplication loop runs until EVERY lane of the warp has converged (branch-light, no divergence)
struct VoteNone { CB_HD bool any(bool p) const { return p; } };
#ifdef __CUDACC__
struct VoteWarp { __device__ __forceinline__ bool any(bool p) const { return __any_sync(0xffffffffu, p); } };
#endif

// R_C(1, 1+e), e > -1 (eq. (2.8)): atan(sqrt e)/sqrt e or atanh(sqrt -e)/sqrt -e.
template <typename T>
CB_HD T rc1(T e) {
    using N = Num<T>;
    if (N::abs_(e) < N::RC_SMALL) {
        T s = T(1.0 / 21);
        s = N::fma_(s, -e, T(1.0 / 19)); s = N::fma_(s, -e, T(1.0 / 17)); s = N::fma_(s, -e, T(1.0 / 15));
        s = N::fma_(s, -e, T(1.0 / 13)); s = N::fma_(s, -e, T(1.0 / 11)); s = N::fma_(s, -e, T(1.0 / 9));
        s = N::fma_(s, -e, T(1.0 / 7)); s = N::fma_(s, -e, T(1.0 / 5)); s = N::fma_(s, -e, T(1.0 / 3));
        return N::fma_(s, -e, T(1));
    }
    if (e > T(0)) { T r = N::sqrt_(e); return N::atan_(r) / r; }
    T r = N::sqrt_(-e);
    return T(0.5) * N::log_((T(1) + r) / (T(1) - r)) / r;
}
// R_C(x, y) for x >= 0, y > 0
template <typename T>
CB_HD T rc(T x, T y) { return rc1<T>(y / x - T(1)) / Num<T>::sqrt_(x); }

// Carlson's degree-7 series in the elementary symmetric functions (R_D / R_J form, ref. [10] as in DLMF 19.36.2)
template <typename T>
CB_HD T series_J(T E2, T E3, T E4, T E5) {
    return T(1) - T(3.0 / 14) * E2 + T(1.0 / 6) * E3 + T(9.0 / 88) * E2 * E2 - T(3.0 / 22) * E4 - T(9.0 / 52) * E2 * E3
           + T(3.0 / 26) * E5 - T(1.0 / 16) * E2 * E2 * E2 + T(3.0 / 40) * E3 * E3 + T(3.0 / 20) * E2 * E4
           + T(45.0 / 272) * E2 * E2 * E3 - T(9.0 / 68) * (E3 * E4 + E2 * E5);
}

// what one element needs from the fused Carlson pass
template <typename T>
struct Core {
    T I0, TT, AA;      // eqs. (2.3)-(2.5) without unit prefactors
    T K;               // int (Or x + m)/(x - rn) dx/E  (second kind; basis function of the gradients)
    T E;               // E(z)
    T Em1;             // E(z) - 1, cancellation-free
    unsigned status;
};

// S4-S6.  kT: lookback integral, kA: absorption integral, kK: the second-kind integral K (needs R_D).
template <typename T, bool kT, bool kA, bool kK, typename Vote>
CB_HD void eval_core(const Cosmo<T>& C, T z, const Vote& vote, Core<T>& R) {
    using N = Num<T>;
    constexpr bool kD = kK || kA;          // R_D tail needed
    const T x = T(1) + z;
    const T z2 = z * z;
    unsigned st = C.status;
    if (!(x > T(0))) st |= ST_UNSUPPORTED;
    if (x >= C.xlim) st |= ST_ROOT_ON_PATH;
    // ---- S4 radicands
    const T lin = N::fma_(C.Or, x, C.m);                 // Or x + m
    const T xmr = x - C.rn;
    const T q1x = lin * xmr;
    const T q2x = N::fma_(x + C.b, x, C.c);
    const T ra = N::sqrt_(q1x * C.q21), rb = N::sqrt_(C.q11 * q2x);
    const T U12 = ra + rb;
    T xa = U12 * U12;
    T mp = N::fma_(T(-0.5) * z2, C.theta, xa);
    T s = z2 * z2 * C.sD;
    const T xa0 = xa, m0 = mp, s0 = s;
    const T hs = z2 * C.sDr;                             // |h|
    // E(z) and E(z) - 1 (for d/dz and the boundary terms of the gradients)
    const T E2 = q1x * q2x;
    const T Ev = N::sqrt_(E2);
    {
        T t = N::fma_(C.Or, N::fma_(N::fma_(x + T(1), x, T(1)), x, T(1)), N::fma_(C.Om, N::fma_(x + T(1), x, T(1)), C.Ok * (x + T(1))));
        R.Em1 = z * t / (Ev + T(1));
    }
    R.E = Ev;
    // ---- R_J parameters
    T p5 = T(0), p0 = T(0), dl5 = T(0), dl0 = T(0), p5_0 = T(0), p0_0 = T(0);
    if (kT) {
        p5 = N::fma_(z2, C.p5c, xa);
        p5_0 = p5;
        T pm = p5 - mp;
        dl5 = (p5 - xa) * N::fma_(pm, pm, -s);
    }
    const bool quartA = kA && !C.cubic;
    if (kA) {
        p0 = quartA ? N::fma_(-C.Or * z2, C.Q2n, xa) : xa;
        p0_0 = p0;
        T pm = p0 - mp;
        dl0 = (p0 - xa) * N::fma_(pm, pm, -s);
    }
    // ---- stopping rule (ref. [10]): 4^-n Q < |A_n| for every series that is summed
    const T dxm = N::abs_(xa - mp);
    const T QFv = N::QF * (T(2.0 / 3) * dxm + hs);
    const T QDv = kD ? N::QJ * (T(3.0 / 5) * dxm + hs) : T(0);
    T Q5v = T(0), Q0v = T(0);
    if (kT) {
        T A0 = (xa + T(2) * mp + T(2) * p5) * T(0.2);
        Q5v = N::QJ * N::max_(N::max_(N::abs_(A0 - xa), N::abs_(A0 - mp) + hs), N::abs_(A0 - p5));
    }
    if (kA) {
        T A0 = (xa + T(2) * mp + T(2) * p0) * T(0.2);
        Q0v = N::QJ * N::max_(N::max_(N::abs_(A0 - xa), N::abs_(A0 - mp) + hs), N::abs_(A0 - p0));
    }
    // ---- S5 fused duplication
    T f = T(1), tailD = T(0), sum5 = T(0), sum0 = T(0);
    int nit = 0;
    for (;;) {
        bool more = f * QFv >= N::abs_(xa + T(2) * mp) * T(1.0 / 3);
        if (kD) more = more || (f * QDv >= N::abs_(T(3) * xa + T(2) * mp) * T(0.2));
        if (kT) more = more || (f * Q5v >= N::abs_(xa + T(2) * mp + T(2) * p5) * T(0.2));
        if (kA) more = more || (f * Q0v >= N::abs_(xa + T(2) * mp + T(2) * p0) * T(0.2));
        more = more && (st == 0);
        if (nit >= NIT_CAP) { if (more) st |= ST_ITER_CAP; more = false; }
        if (!vote.any(more)) break;
        const T sx = N::sqrt_(xa);
        const T spd = N::sqrt_(N::fma_(mp, mp, -s));
        const T sa = N::sqrt_(T(2) * (mp + spd));
        const T lam = N::fma_(sx, sa, spd);
        if (kD) tailD += f / (sx * (xa + lam));
        if (kT) {
            const T rp = N::sqrt_(p5);
            const T d = (rp + sx) * (p5 + N::fma_(rp, sa, spd));
            const T e = f * f * f * dl5 / (d * d);
            sum5 += f / d * rc1<T>(e);
            p5 = T(0.25) * (p5 + lam);
        }
        if (kA) {
            const T rp = N::sqrt_(p0);
            const T d = (rp + sx) * (p0 + N::fma_(rp, sa, spd));
            const T e = f * f * f * dl0 / (d * d);
            sum0 += f / d * rc1<T>(e);
            p0 = T(0.25) * (p0 + lam);
        }
        xa = T(0.25) * (xa + lam);
        mp = T(0.25) * (mp + lam);
        s *= T(1.0 / 16);
        f *= T(0.25);
        ++nit;
    }
    // ---- series: R_F
    T RF;
    {
        const T An = (xa + T(2) * mp) * T(1.0 / 3);
        const T g = f / An;
        const T dl = (xa0 - m0) * T(1.0 / 3) * g;
        const T vs = s0 * g * g;
        const T e2 = T(-3) * dl * dl - vs;
        const T e3 = T(-2) * dl * (dl * dl - vs);
        const T S = T(1) - T(0.1) * e2 + T(1.0 / 14) * e3 + T(1.0 / 24) * e2 * e2 - T(3.0 / 44) * e2 * e3
                    - T(5.0 / 208) * e2 * e2 * e2 + T(3.0 / 104) * e3 * e3 + T(1.0 / 16) * e2 * e2 * e3;
        RF = S / N::sqrt_(An);
    }
    R.I0 = T(2) * z * RF;                                 // eq. (3.7) / (B.1)
    // ---- series: R_D(u13^2, u14^2, u12^2)
    T RD = T(0);
    if (kD) {
        const T AD = (T(3) * xa + T(2) * mp) * T(0.2);
        const T g = f / AD;
        const T dd = (xa0 - m0) * T(0.2) * g;
        const T XY = T(9) * dd * dd - s0 * g * g;
        const T Z = T(-2) * dd, Z2 = Z * Z;
        const T e2 = XY - T(6) * Z2;
        const T e3 = (T(3) * XY - T(8) * Z2) * Z;
        const T e4 = T(3) * (XY - Z2) * Z2;
        const T e5 = XY * Z2 * Z;
        RD = f * series_J<T>(e2, e3, e4, e5) / (AD * N::sqrt_(AD)) + T(3) * tailD;
    }
    const T rU = T(1) / U12;
    if (kK) {
        // K = 2 z [ z^2/3 W R_D + sqrt((Or x + m) kf / (x - rn)) / u12 ]   (Carlson's [p_n = -3] integral)
        R.K = T(2) * z * N::fma_(z2 * T(1.0 / 3) * C.W, RD, N::sqrt_(lin * C.kf / xmr) * rU);
    }
    auto rj_series = [&](T p_n, T p_init, T sum) -> T {
        const T An = (xa + T(2) * mp + T(2) * p_n) * T(0.2);
        const T A0 = (xa0 + T(2) * m0 + T(2) * p_init) * T(0.2);
        const T g = f / An;
        const T X = (A0 - xa0) * g;
        const T am = A0 - m0;
        const T YpZ = T(2) * am * g;
        const T YZ = N::fma_(am, am, -s0) * g * g;
        const T P = T(-0.5) * (X + YpZ);
        const T XYZ = X * YZ;
        const T P2 = P * P;
        const T e2 = N::fma_(X, YpZ, YZ) - T(3) * P2;
        const T e3 = XYZ + T(2) * e2 * P + T(4) * P2 * P;
        const T e4 = (T(2) * XYZ + e2 * P + T(3) * P2 * P) * P;
        const T e5 = XYZ * P2;
        return f * series_J<T>(e2, e3, e4, e5) / (An * N::sqrt_(An)) + T(6) * sum;
    };
    if (kT) {
        // eq. (3.8) with i = big root, j = rn, scaled so that Or -> 0 reproduces (B.2)
        const T RJ5 = rj_series(p5, p5_0, sum5);
        const T qh = x * p5_0 * C.qhc / lin;
        const T sh = N::fma_(z2, C.OL, qh);
        R.TT = T(2) * z * (z2 * T(1.0 / 3) * C.Gp * RJ5 + rc<T>(sh, qh) - C.OrM * RF);
    }
    if (kA) {
        const T bnd = N::sqrt_(xmr * (T(1) - C.rn)) * rU;
        if (quartA) {
            // eq. (3.9) with (i,j,k,l) = (rn, pair, pair, big)
            const T RJ0 = rj_series(p0, p0_0, sum0);
            const T q0 = p0_0 / ((T(1) - C.rn) * xmr);
            const T s0q = N::fma_(C.Or, z2, q0);
            const T t1 = N::sqrt_(xmr * q2x / lin) - N::sqrt_((T(1) - C.rn) * C.q21 / (C.Or + C.m));
            const T t2 = z * C.aF * RF;
            const T t3 = z * C.WoOr * N::fma_(z2 * T(1.0 / 3) * C.Q2n, RD, bnd / N::sqrt_(lin * (C.Or + C.m)));
            const T t4 = z * C.sig * N::fma_(z2 * T(1.0 / 3) * C.Q2n * C.mOrn, RJ0, rc<T>(s0q, q0));
            R.AA = (t1 + t2) + (t3 + t4);
        } else {
            // eq. (B.3) with i = rn
            R.AA = T(2.0 / 3) * z * (R.Em1 / (C.m * z) + C.aF * RF
                                     + T(2) * C.sig * N::fma_(z2 * T(1.0 / 3) * C.Q2n * C.m, RD, bnd));
            if (z == T(0)) R.AA = T(0);
        }
    }
    R.status = st;
}

// unified curvature transform in w = Ok I0^2 (reading R-sinn):
//   F = I0 f(w), dF/dI0 = g(w), dF/dOk = I0^3 f'(w);  f = sum w^j/(2j+1)!, g = sum w^j/(2j)!
template <typename T>
CB_HD void sinn(T k, T I0, T& F, T& Fi, T& Fk) {
    using N = Num<T>;
    const T w = k * I0 * I0;
    if (N::abs_(w) <= T(1)) {
        T sf = T(1.0 / 51090942171709440000.0), sg = T(1.0 / 2432902008176640000.0), sd = T(10.0 / 51090942171709440000.0);
        const double FO[10] = {1.0 / 121645100408832000.0, 1.0 / 355687428096000.0, 1.0 / 1307674368000.0, 1.0 / 6227020800.0,
                               1.0 / 39916800.0, 1.0 / 362880.0, 1.0 / 5040.0, 1.0 / 120.0, 1.0 / 6.0, 1.0};
        const double GO[10] = {1.0 / 6402373705728000.0, 1.0 / 20922789888000.0, 1.0 / 87178291200.0, 1.0 / 479001600.0,
                               1.0 / 3628800.0, 1.0 / 40320.0, 1.0 / 720.0, 1.0 / 24.0, 0.5, 1.0};
#pragma unroll
        for (int j = 0; j < 10; ++j) {
            sf = N::fma_(sf, w, T(FO[j]));
            sg = N::fma_(sg, w, T(GO[j]));
            if (j < 9) sd = N::fma_(sd, w, T((9 - j) * FO[j]));
        }
        F = I0 * sf; Fi = sg; Fk = I0 * I0 * I0 * sd;
        return;
    }
    if (k > T(0)) {
        const T sq = N::sqrt_(k), y = sq * I0, ey = N::exp_(y), iey = T(1) / ey;
        const T sh = T(0.5) * (ey - iey), ch = T(0.5) * (ey + iey);
        F = sh / sq; Fi = ch; Fk = (I0 * ch - F) / (T(2) * k);
    } else {
        const T sq = N::sqrt_(-k);
        T sn, cs;
        N::sincos_(sq * I0, &sn, &cs);
        F = sn / sq; Fi = cs; Fk = (I0 * cs - F) / (T(2) * k);
    }
}

}  // namespace cb
