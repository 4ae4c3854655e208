// cosmo_c4.cuh -- slow path for the one root structure the real-quadratic labelling of DESIGN.md section 2 cannot
// serve: E^2 with NO real negative root (two complex-conjugate pairs; needs Om^2 < ~4 Or Ok, about 1 row in 10^4 of
// config 2).  There eqs. (3.8)/(3.9) single out a COMPLEX root r_i, so the R_J parameter
// u_i5^2 / u_i0^2 is complex while x = u12^2, y = u13^2, z = u14^2 stay real (each u is invariant under the conjugation
// that swaps the members of both pairs).  This file evaluates the paper's formulae as printed, in complex arithmetic
// only where it is needed (the p-track of R_J, R_C, and the algebraic coefficients).  FP64 always.  For the gradients it
// also returns K = int_1^x N_K / E^3 with N_K = Or^2 Re (x - r1)^2 Q2(x): the real part of Carlson's [+1, -1, -1, -3] integral
// int sqrt(t - r1) / ((t - r2)^(3/2) sqrt((t - r3)(t - r4))) dt = (2/3) d13 d14 dz^3 R_D(u13^2, u14^2, u12^2) + 2 dz X1 Y1 / (X2 Y2 u12)
// (the same R_D term eq. (3.9) carries), which for r2 = conj(r1) equals Or^(3/2) int (t - r1)^2 Q2 / E^3 dt.  It plays the part
// the [p_n = -3] integral of the real root plays in the gradient bases of cosmo_prep.cuh.
#pragma once
#include "cosmo_eval.cuh"

namespace cb {

struct cx { double re, im; };
CB_HD cx cx_(double r, double i = 0.0) { cx c; c.re = r; c.im = i; return c; }
CB_HD cx operator+(cx a, cx b) { return cx_(a.re + b.re, a.im + b.im); }
CB_HD cx operator-(cx a, cx b) { return cx_(a.re - b.re, a.im - b.im); }
CB_HD cx operator-(cx a) { return cx_(-a.re, -a.im); }
CB_HD cx operator*(cx a, cx b) { return cx_(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
CB_HD cx operator*(double s, cx a) { return cx_(s * a.re, s * a.im); }
// Division, modulus and square root: IEEE operations by default -- the rare two-complex-pairs rows of the hot path carry eq. (3.9)'s
// Om/Or cancellation and need every bit.  A translation unit that defines CB_CX_FAST before including this header (tu_w.cu: the extra-w
// family, where complex arithmetic is the main path and the stated d_abs tolerance is 1e-10) gets the MUFU-seeded forms of cosmo_types.cuh.
#if defined(CB_CX_FAST) && defined(__CUDA_ARCH__)
CB_HD double cx_rcp_(double a) { return cb_rcp(a); }
CB_HD double cx_sqrt_(double a) { return cb_sqrt0(a); }
CB_HD double cx_abs(cx a) { return cb_sqrt0(a.re * a.re + a.im * a.im); }
#else
CB_HD double cx_rcp_(double a) { return 1.0 / a; }
CB_HD double cx_sqrt_(double a) { return sqrt(a); }
CB_HD double cx_abs(cx a) { return hypot(a.re, a.im); }
#endif
CB_HD cx operator/(cx a, cx b) {
    const double d = cx_rcp_(b.re * b.re + b.im * b.im);
    return cx_((a.re * b.re + a.im * b.im) * d, (a.im * b.re - a.re * b.im) * d);
}
CB_HD cx cx_conj(cx a) { return cx_(a.re, -a.im); }
CB_HD cx cx_sqrt(cx a) {      // principal square root (Re >= 0)
    const double r = cx_abs(a);
    if (r == 0.0) return cx_(0.0);
    if (a.re >= 0.0) { const double t = cx_sqrt_(0.5 * (r + a.re)); return cx_(t, 0.5 * a.im * cx_rcp_(t)); }
    const double t = cx_sqrt_(0.5 * (r - a.re));
    return cx_(0.5 * fabs(a.im) * cx_rcp_(t), a.im >= 0.0 ? t : -t);
}
CB_HD cx cx_log(cx a) { return cx_(log(cx_abs(a)), atan2(a.im, a.re)); }

// R_C(1, 1+e) for complex e (eq. (2.8)): series near 0, else ln((1+s)/(1-s))/(2s) with s = sqrt(-e)
CB_HD cx cx_rc1(cx e) {
    if (cx_abs(e) < 0.03) {
        cx s = cx_(CB_KT.rc[9]);
        for (int j = 8; j >= 0; --j) s = cx_(CB_KT.rc[j]) - s * e;
        return cx_(1.0) - s * e;
    }
    const cx s = cx_sqrt(-e);
    return cx_log((cx_(1.0) + s) / (cx_(1.0) - s)) / (2.0 * s);
}
// R_C(x, y), complex, y != 0
CB_HD cx cx_rc(cx x, cx y) { return cx_rc1(y / x - cx_(1.0)) / cx_sqrt(x); }

// R_F(x,y,z), R_D(x,y,z) (last argument z) and R_J(x,y,z,p) for real positive x, y, z and complex p, ref. [10] duplication
struct C4Carlson { double RF, RDz; cx RJ; };
CB_HD void c4_carlson(double x, double y, double z, cx p, bool want_j, C4Carlson& out) {
    const double x0 = x, y0 = y, z0 = z;
    const cx delta = (p - cx_(x)) * (p - cx_(y)) * (p - cx_(z));
    const double AF0 = (x + y + z) / 3.0, AD0 = (x + y + 3.0 * z) / 5.0;
    const cx AJ0 = 0.2 * (cx_(x + y + z) + 2.0 * p);
    const double dev = fmax(fmax(fabs(AF0 - x), fabs(AF0 - y)), fabs(AF0 - z)) + fmax(fabs(AD0 - x), fmax(fabs(AD0 - y), fabs(AD0 - z)));
    const double devJ = want_j ? fmax(fmax(cx_abs(AJ0 - cx_(x)), cx_abs(AJ0 - cx_(y))), fmax(cx_abs(AJ0 - cx_(z)), cx_abs(AJ0 - p))) : 0.0;
    double f = 1.0, tailD = 0.0;
    cx sumJ = cx_(0.0);
    for (int it = 0; it < 2 * NIT_CAP; ++it) {
        const double AF = (x + y + z) / 3.0, AD = (x + y + 3.0 * z) / 5.0;
        const cx AJ = 0.2 * (cx_(x + y + z) + 2.0 * p);
        if (f * 600.0 * dev < fmin(AF, AD) && (!want_j || f * 600.0 * devJ < cx_abs(AJ))) break;
        const double sx = sqrt(x), sy = sqrt(y), sz = sqrt(z);
        const double lam = sx * sy + sx * sz + sy * sz;
        tailD += f / (sz * (z + lam));
        if (want_j) {
            const cx sp = cx_sqrt(p);
            const cx d = (sp + cx_(sx)) * (sp + cx_(sy)) * (sp + cx_(sz));
            const cx e = (f * f * f) * delta / (d * d);
            sumJ = sumJ + (f * cx_rc1(e)) / d;
            p = 0.25 * (p + cx_(lam));
        }
        x = 0.25 * (x + lam); y = 0.25 * (y + lam); z = 0.25 * (z + lam);
        f *= 0.25;
    }
    {
        const double A = (x + y + z) / 3.0, g = f / A;
        const double X = (AF0 - x0) * g, Y = (AF0 - y0) * g, Z = -X - Y;
        const double e2 = X * Y - Z * Z, e3 = X * Y * Z;
        out.RF = (1.0 - e2 / 10.0 + e3 / 14.0 + e2 * e2 / 24.0 - 3.0 * e2 * e3 / 44.0 - 5.0 * e2 * e2 * e2 / 208.0 + 3.0 * e3 * e3 / 104.0
                  + e2 * e2 * e3 / 16.0) / sqrt(A);
    }
    {
        const double A = (x + y + 3.0 * z) / 5.0, g = f / A;
        const double X = (AD0 - x0) * g, Y = (AD0 - y0) * g, Z = -(X + Y) / 3.0;
        const double e2 = X * Y - 6.0 * Z * Z, e3 = (3.0 * X * Y - 8.0 * Z * Z) * Z, e4 = 3.0 * (X * Y - Z * Z) * Z * Z, e5 = X * Y * Z * Z * Z;
        out.RDz = f * series_J<double>(e2, e3, e4, e5) / (A * sqrt(A)) + 3.0 * tailD;
    }
    out.RJ = cx_(0.0);
    if (want_j) {
        const cx A = 0.2 * (cx_(x + y + z) + 2.0 * p);
        const cx g = cx_(f) / A;
        const cx X = (AJ0 - cx_(x0)) * g, Y = (AJ0 - cx_(y0)) * g, Z = (AJ0 - cx_(z0)) * g;
        const cx P = -0.5 * (X + Y + Z);
        const cx XYZ = X * Y * Z, P2 = P * P;
        const cx e2 = X * Y + X * Z + Y * Z - 3.0 * P2;
        const cx e3 = XYZ + 2.0 * (e2 * P) + 4.0 * (P2 * P);
        const cx e4 = (2.0 * XYZ + e2 * P + 3.0 * (P2 * P)) * P;
        const cx e5 = XYZ * P2;
        const double* c = CB_KT.rj;
        const cx S = cx_(1.0) + c[0] * e2 + c[3] * e3 + c[1] * (e2 * e2) + c[8] * e4 + c[4] * (e2 * e3) + c[10] * e5 + c[2] * (e2 * e2 * e2)
                     + c[6] * (e3 * e3) + c[9] * (e2 * e4) + c[5] * (e2 * e2 * e3) + c[7] * (e3 * e4 + e2 * e5);
        out.RJ = (f * S) / (A * cx_sqrt(A)) + 6.0 * sumJ;
    }
}

// I0, T, A of eqs. (3.7)-(3.9) with the roots r_1 = conj(r_2) of Q1 = Or x^2 + g1 x + h1 and r_3 = conj(r_4) of
// Q2 = x^2 + b x + c, permutation (i, j, k, l) = (1, 2, 3, 4); everything in x = 1 + z (d_i5 = -rho_i), between the limits
// x1 = 1 + z1 and x = 1 + z2 (the hot path calls it with x1 = 1).  dz = z2 - z1 comes in from the caller: formed as x - x1 it
// would carry the rounding of 1 + z, eps/z of every result at small z (3.7e-11 at z = 1e-6 before this was an argument).
// (never inlined: a rare path must not cost the hot kernels registers)
CB_HD_NOINLINE void eval_c4(double Or, double g1, double h1, double b, double c, double x1, double x, double dz, bool want_T, bool want_A,
                   double& I0, double& TT, double& AA, double& KK) {
    const double D1 = 4.0 * Or * h1 - g1 * g1, D2 = 4.0 * c - b * b;       // both > 0 here
    const cx r1 = cx_(-g1 / (2.0 * Or), sqrt(D1) / (2.0 * Or)), r2 = cx_conj(r1);
    const cx r3 = cx_(-0.5 * b, 0.5 * sqrt(D2)), r4 = cx_conj(r3);
    const cx X1 = cx_sqrt(cx_(x) - r1), Y1 = cx_sqrt(cx_(x1) - r1), X3 = cx_sqrt(cx_(x) - r3), Y3 = cx_sqrt(cx_(x1) - r3);
    const cx X2 = cx_conj(X1), Y2 = cx_conj(Y1), X4 = cx_conj(X3), Y4 = cx_conj(Y3);
    const cx u12 = X1 * X2 * Y3 * Y4 + Y1 * Y2 * X3 * X4;
    const cx u13 = X1 * X3 * Y2 * Y4 + Y1 * Y3 * X2 * X4;
    const cx u14 = X1 * X4 * Y2 * Y3 + Y1 * Y4 * X2 * X3;
    const double xa = u12.re * u12.re, ya = u13.re * u13.re, za = u14.re * u14.re;    // imaginary parts vanish identically
    const cx d12 = r2 - r1, d13 = r3 - r1, d14 = r4 - r1, d23 = r3 - r2, d24 = r4 - r2;
    const double ia = 1.0 / sqrt(Or);
    C4Carlson K;
    // (3.8): i = 1, j = 2:  u_i5^2 = u12^2 - dz^2 d13 d14 d25/d15, d_n5 = -rho_n
    const cx p5 = cx_(xa) - (dz * dz) * (d13 * d14 * (r2 / r1));
    c4_carlson(ya, za, xa, p5, want_T, K);
    I0 = ia * 2.0 * dz * K.RF;
    KK = sqrt(Or) * (((2.0 / 3.0) * dz * dz * dz * K.RDz) * (d13 * d14) + (2.0 * dz) * ((X1 * Y1) / (X2 * Y2 * u12))).re;
    TT = 0.0; AA = 0.0;
    if (want_T) {
        const cx q5 = (cx_(x * x1) / ((cx_(x1) - r1) * (cx_(x) - r1))) * p5;
        const cx s5 = q5 + (dz * dz) * (r3 * r4 * (r2 / r1));
        const cx br = cx_(K.RF) - ((dz * dz / 3.0) * (d12 * d13 * d14 / (-r1)) * K.RJ + cx_rc(s5, q5));
        TT = ia * ((2.0 * dz) * (br / r1)).re;
    }
    if (want_A) {
        // (3.9): (i, j, k, l) = (1, 3, 4, 2): R_D(u13^2, u14^2, u12^2) is real, u_i0^2 = u12^2 - dz^2 d13 d14
        const cx p0 = cx_(xa) - (dz * dz) * (d13 * d14);
        C4Carlson K0;
        c4_carlson(ya, za, xa, p0, true, K0);
        const cx q0 = p0 / ((cx_(x1) - r1) * (cx_(x) - r1));
        const cx s0 = q0 + cx_(dz * dz);
        // boundary term [F] between the limits, F = X1 X3 X4 / X2, F^2 = N(x)/(x - r2), N = (x - r1) Q2.  Close limits: the difference
        // through F^2, with the factor dz taken out of N(x)(x1 - r2) - N(x1)(x - r2) = dz ([N; x, x1] (x1 - r2) - N(x1)) analytically
        // (subtracted directly it loses eps/dz: 2e-10 of d_abs at z = 1e-4)
        const cx Fx = X1 * X3 * X4 / X2, F1 = Y1 * Y3 * Y4 / Y2;
        cx bnd = Fx - F1;
        if (fabs(dz) <= 0.05 * fmin(x, x1)) {
            const cx br1 = cx_(b) - r1, cr1 = cx_(c) - b * r1;                              // N = x^3 + br1 x^2 + cr1 x - c r1
            const cx dd = cx_(x * x + x * x1 + x1 * x1) + (x + x1) * br1 + cr1;             // divided difference [N; x, x1]
            const cx N1 = (x1 * x1 + b * x1 + c) * (cx_(x1) - r1);
            bnd = dz * ((dd * (cx_(x1) - r2) - N1) / ((cx_(x) - r2) * (cx_(x1) - r2) * (Fx + F1)));
        }
        const cx sig = r1 + r2 + r3 + r4;
        const cx t2 = dz * ((2.0 * (r1 * r1) - d13 * d14) * cx_(K0.RF));
        const cx t3 = dz * ((d23 * d24) * (((dz * dz / 3.0) * (d13 * d14)) * cx_(K0.RDz) + (X1 * Y1) / (X2 * Y2 * u12)));
        const cx t4 = dz * (sig * (cx_rc(s0, q0) - ((dz * dz / 3.0) * (d13 * d14 * d12)) * K0.RJ));
        AA = ia * (bnd + t2 + t3 + t4).re;
    }
}

}  // namespace cb
