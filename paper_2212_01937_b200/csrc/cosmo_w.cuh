// cosmo_w.cuh -- chi family (D_C, D_M, D_L, mu and their d/dz) when E^2 carries extra components with constant equation of
// state w = -1/3 and w = -2/3 (PAPER.md:82 fn.4: the method needs E^2 to be a polynomial of degree <= 4, i.e.
// w in {-1, -2/3, -1/3, 0, 1/3}):
//     E^2(x) = Or x^4 + Om x^3 + (Ok + Ow13) x^2 + Ow23 x + OL,      Ok = 1 - Om - OL - Or - Ow13 - Ow23.
// The x^1 term removes the structure the hot path's factorisation relies on (cosmo_prep.cuh), so this is a GENERAL real
// quartic: roots by Aberth's simultaneous iteration in complex arithmetic, grouped into two REAL quadratics
// Q1 = f1 x^2 + g1 x + h1, Q2 = f2 x^2 + g2 x + h2 (conjugates together, real roots with their neighbours; leading
// coefficients may vanish: a root at infinity is a constant factor).  Eq. (3.7)/(B.1) then needs no root singled
// out: I0 = 2 z R_F(u12^2, u13^2, u14^2) with the real-symmetric arguments of cosmo_eval.cuh,
//     u12 = sqrt(Q1(x) Q2(1)) + sqrt(Q1(1) Q2(x)),  u13^2, u14^2 = u12^2 - z^2 Theta / 2 +- z^2 sqrt(disc1 disc2) / 2,
// and the same duplication code.  ELEMENTWISE, FP64, forward values and d/dz (= integrand at z, chained); parameter
// gradients, t_L and d_abs of this family are not built (eqs. (3.8)/(3.9) single out a root).
#pragma once
#include "cosmo_obs.cuh"

namespace cb {

struct WCosmo {
    double f1, g1, h1, f2, g2, h2;     // E^2 = Q1 Q2
    double q11, q21, theta, sD, sDr;   // Q1(1), Q2(1), apolar invariant, disc1 disc2 / 4 and sqrt|.|
    double rr[4];                      // real roots (path check)
    int nreal;
    double Ok, dH;
    unsigned status;
};

CB_HD cx w_poly(const double* a, int n, cx x, cx& dp) {       // Horner: value and derivative
    cx p = cx_(a[n]);
    dp = cx_(0.0);
    for (int i = n - 1; i >= 0; --i) { dp = dp * x + p; p = p * x + cx_(a[i]); }
    return p;
}

CB_HD void w_prep(double Om, double OL, double Or, double Ow13, double Ow23, double H0, WCosmo& W) {
    const double Ok = 1.0 - Om - OL - Or - Ow13 - Ow23;
    const double a[5] = {OL, Ow23, Ok + Ow13, Om, Or};
    W.Ok = Ok; W.dH = C_KM_S / H0;
    W.status = 0; W.nreal = 0;
    for (int i = 0; i < 4; ++i) W.rr[i] = 0.0;
    bool fin = H0 > 0.0;
    for (int i = 0; i < 5; ++i) fin = fin && (fabs(a[i]) < 1e300);       // also false for NaN
    int n = 4;
    while (n > 0 && a[n] == 0.0) --n;
    W.f1 = W.g1 = 0.0; W.h1 = a[n]; W.f2 = W.g2 = 0.0; W.h2 = 1.0;       // n == 0: E^2 = const
    if (!fin) { W.status = ST_UNSUPPORTED; n = 0; }
    cx r[4];
    if (n >= 1) {
        // roots at x = 0 (absent low-order components, e.g. x^3 for Einstein-de Sitter) are exact and multiple: take them out first
        int m0 = 0;
        while (m0 < n && a[m0] == 0.0) ++m0;
        const int nd = n - m0;                                             // degree of the deflated polynomial
        double c[5], R = 0.0;
        for (int i = 0; i <= nd; ++i) c[i] = a[i + m0] / a[n];
        for (int i = 0; i < nd; ++i) R = fmax(R, fabs(c[i]));
        R += 1.0;                                                          // Cauchy bound
        for (int k = 0; k < nd; ++k) {
            const double ang = 6.283185307179586 * k / nd + 0.4;
            r[k] = cx_(R * cos(ang), R * sin(ang));
        }
        for (int k = nd; k < n; ++k) r[k] = cx_(0.0);
        for (int it = 0; it < 200 && nd > 0; ++it) {
            double big = 0.0;
            for (int k = 0; k < nd; ++k) {
                cx dp;
                const cx p = w_poly(c, nd, r[k], dp);
                if (cx_abs(p) == 0.0) continue;
                const cx w = p / dp;
                cx sum = cx_(0.0);
                for (int j = 0; j < nd; ++j)
                    if (j != k) sum = sum + cx_(1.0) / (r[k] - r[j]);
                const cx d = w / (cx_(1.0) - w * sum);
                r[k] = r[k] - d;
                big = fmax(big, cx_abs(d) / fmax(cx_abs(r[k]), 1e-300));
            }
            if (big < 4e-16) break;
        }
        // group into real quadratics: a root with a significant imaginary part goes with its conjugate, real ones are
        // sorted and paired with their neighbours
        bool used[4] = {false, false, false, false};
        double qb[2] = {0.0, 0.0}, qc[2] = {0.0, 0.0};                     // monic quadratics x^2 + qb x + qc
        int nq = 0;
        for (int k = 0; k < n; ++k) {
            if (used[k] || !(fabs(r[k].im) > 1e-9 * cx_abs(r[k]))) continue;
            int best = -1; double bd = 1e308;
            for (int j = 0; j < n; ++j) {
                if (j == k || used[j]) continue;
                const double dd = cx_abs(r[j] - cx_conj(r[k]));
                if (dd < bd) { bd = dd; best = j; }
            }
            if (best < 0) { W.status |= ST_UNSUPPORTED; break; }
            used[k] = used[best] = true;
            const double re = 0.5 * (r[k].re + r[best].re);
            const cx pr = r[k] * r[best];
            if (nq < 2) { qb[nq] = -2.0 * re; qc[nq] = pr.re; ++nq; }
        }
        double rl[4]; int nr = 0;
        for (int k = 0; k < n; ++k)
            if (!used[k]) rl[nr++] = r[k].re;
        for (int i = 1; i < nr; ++i) {                                     // insertion sort
            const double v = rl[i]; int j = i - 1;
            while (j >= 0 && rl[j] > v) { rl[j + 1] = rl[j]; --j; }
            rl[j + 1] = v;
        }
        W.nreal = nr;
        for (int i = 0; i < nr; ++i) W.rr[i] = rl[i];
        // quadratics from real neighbours; with an odd number of real roots the smallest stays a linear factor
        int ir = 0;
        double lin = 0.0; bool has_lin = false;
        if ((nr & 1) != 0) { lin = rl[0]; has_lin = true; ir = 1; }
        for (; ir + 1 < nr && nq < 2; ir += 2) { qb[nq] = -(rl[ir] + rl[ir + 1]); qc[nq] = rl[ir] * rl[ir + 1]; ++nq; }
        // assemble Q1 (carries the leading coefficient) and Q2
        const double lead = a[n];
        if (n == 4) { W.f1 = lead; W.g1 = lead * qb[0]; W.h1 = lead * qc[0]; W.f2 = 1.0; W.g2 = qb[1]; W.h2 = qc[1]; }
        else if (n == 3) { W.f1 = 0.0; W.g1 = lead; W.h1 = -lead * lin; W.f2 = 1.0; W.g2 = qb[0]; W.h2 = qc[0]; }
        else if (n == 2) { W.f1 = 0.0; W.g1 = 0.0; W.h1 = lead; W.f2 = 1.0; W.g2 = qb[0]; W.h2 = qc[0]; }
        else { W.f1 = 0.0; W.g1 = 0.0; W.h1 = lead; W.f2 = 0.0; W.g2 = 1.0; W.h2 = -lin; }
        if ((n == 4 && (nq != 2 || has_lin)) || (n == 3 && (nq != 1 || !has_lin)) || (n == 2 && nq != 1) || (n == 1 && !has_lin))
            W.status |= ST_UNSUPPORTED;
        // the product must reproduce the coefficients
        const double e4 = W.f1 * W.f2, e3 = W.f1 * W.g2 + W.g1 * W.f2, e2 = W.f1 * W.h2 + W.g1 * W.g2 + W.h1 * W.f2,
                     e1 = W.g1 * W.h2 + W.h1 * W.g2, e0 = W.h1 * W.h2;
        const double sc = fabs(a[0]) + fabs(a[1]) + fabs(a[2]) + fabs(a[3]) + fabs(a[4]);
        const double res = fabs(e4 - a[4]) + fabs(e3 - a[3]) + fabs(e2 - a[2]) + fabs(e1 - a[1]) + fabs(e0 - a[0]);
        if (!(res <= 1e-11 * sc)) W.status |= ST_UNSUPPORTED;
    }
    W.q11 = W.f1 + W.g1 + W.h1;
    W.q21 = W.f2 + W.g2 + W.h2;
    W.theta = 2.0 * W.f1 * W.h2 + 2.0 * W.h1 * W.f2 - W.g1 * W.g2;
    W.sD = 0.25 * (W.g1 * W.g1 - 4.0 * W.f1 * W.h1) * (W.g2 * W.g2 - 4.0 * W.f2 * W.h2);
    W.sDr = sqrt(fabs(W.sD));
}

// values v[4] = D_C, D_M, D_L, mu and dz[4] = their d/dz
template <typename Vote>
CB_HD unsigned w_eval(const WCosmo& W, double z, const Vote& vote, double v[4], double dz[4]) {
    const double x = 1.0 + z, z2 = z * z;
    unsigned st[1] = {W.status};
    if (!(x > 0.0)) st[0] |= ST_UNSUPPORTED;
    for (int i = 0; i < W.nreal; ++i)
        if ((W.rr[i] >= fmin(1.0, x)) && (W.rr[i] <= fmax(1.0, x))) st[0] |= ST_ROOT_ON_PATH;
    const double q1x = fma(fma(W.f1, x, W.g1), x, W.h1), q2x = fma(fma(W.f2, x, W.g2), x, W.h2);
    const double a1 = q1x * W.q21, a2 = W.q11 * q2x;
    if (!(a1 > 0.0) || !(a2 > 0.0)) st[0] |= ST_ROOT_ON_PATH;          // E^2 <= 0 on the way (or NaN input)
    const double ra = sqrt(a1), rb = sqrt(a2), U12 = ra + rb;
    double xa[1] = {U12 * U12}, mp[1], s[1], p5[1] = {0.0}, p0[1] = {0.0};
    const double hd = 0.5 * z2 * W.theta, hs = z2 * W.sDr;
    mp[0] = xa[0] - hd;
    s[0] = z2 * z2 * W.sD;
    const double dl5[1] = {0.0}, dl0[1] = {0.0}, Qc[1] = {carlson_Qc<double>(hd, hs, false)}, Q5v[1] = {0.0}, Q0v[1] = {0.0};
    double g2, tailD[1], sum5[1], sum0[1];
    carlson_dup<double, false, false, false, 1, Vote>(xa, mp, s, p5, p0, dl5, dl0, Qc, Q5v, Q0v, st, vote, g2, tailD, sum5, sum0);
    const double RF = carlson_rf_series<double>(xa[0], mp[0], g2, hd, s[0]);
    const double I0 = 2.0 * z * RF;                                        // eq. (3.7) / (B.1)
    const double iE = 1.0 / (ra * rb);                                     // E(1) = 1: a1 a2 = E^2(x)
    double F, Fi, Fk;
    sinn<double>(W.Ok, I0, F, Fi, Fk);
    v[0] = W.dH * I0; v[1] = W.dH * F; v[2] = x * v[1];
    dz[0] = W.dH * iE; dz[1] = W.dH * Fi * iE; dz[2] = fma(x, dz[1], v[1]);
    if (v[2] > 0.0) {
        v[3] = fma(CB_KT.five_over_ln10, log(v[2]), 25.0);
        dz[3] = CB_KT.five_over_ln10 * dz[2] / v[2];
    } else {
        v[3] = dz[3] = NAN;
        if (!(st[0] & (ST_ROOT_ON_PATH | ST_UNSUPPORTED))) st[0] |= ST_DL_NONPOS;
    }
    if (st[0] & (ST_ROOT_ON_PATH | ST_UNSUPPORTED))
        for (int i = 0; i < 4; ++i) v[i] = dz[i] = NAN;
    return st[0];
}

}  // namespace cb
