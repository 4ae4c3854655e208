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
    double Ok, dH, tH;
    double a[5];                       // E^2 = a[0] + a[1] x + .. + a[4] x^4
    cx rt[4];                          // its roots in x, sorted by decreasing modulus (t_L, d_abs: eqs. (3.8)/(3.9) single roots out)
    int deg;                           // degree of E^2
    int iA;                            // index in rt of r_i of eq. (3.9): the smallest real root other than rt[0], else rt[3]
    unsigned status;
};

CB_HD cx w_poly(const double* a, int n, cx x, cx& dp) {       // Horner: value and derivative
    cx p = cx_(a[n]);
    dp = cx_(0.0);
    for (int i = n - 1; i >= 0; --i) { dp = dp * x + p; p = p * x + cx_(a[i]); }
    return p;
}

// every structure (degrees 0-4, roots at 0, four real roots, ...): never inlined, the kernels reach it through w_prep's fall-back
CB_HD_NOINLINE void w_prep_general(double Om, double OL, double Or, double Ow13, double Ow23, double H0, WCosmo& W) {
    const double Ok = 1.0 - Om - OL - Or - Ow13 - Ow23;
    const double a[5] = {OL, Ow23, Ok + Ow13, Om, Or};
    W.Ok = Ok; W.dH = C_KM_S / H0; W.tH = HUBBLE_GYR / H0;
    for (int i = 0; i < 5; ++i) W.a[i] = a[i];
    for (int i = 0; i < 4; ++i) W.rt[i] = cx_(0.0);
    W.deg = 0; W.iA = 3;
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
        // Fast path for the usual structure (degree 3 or 4, no root at 0, matter present): Bairstow's iteration for a real quadratic
        // factor x^2 + b x + c from the pair of a0 + a3 x^3 ~ 0 (x = rho e^{+-i pi/3}, rho = cbrt(a0/a3)), then the two quadratic
        // formulas.  ~10 x cheaper than the simultaneous iteration below, which remains the fall-back (and serves every other case).
        bool fast = false;
        if (m0 == 0 && nd >= 3 && a[3] > 0.0 && a[0] > 0.0) {
            const double rho = cbrt(a[0] / a[3]);
            double bb = -rho, cc = rho * rho, q2 = a[4], q1 = 0.0, q0 = 0.0;
            const double sc = fabs(a[0]) + fabs(a[1]) + fabs(a[2]) + fabs(a[3]) + fabs(a[4]);
            for (int it = 0; it < 16; ++it) {
                q1 = a[3] - bb * q2; q0 = a[2] - bb * q1 - cc * q2;
                const double r1 = a[1] - bb * q0 - cc * q1, r0 = a[0] - cc * q0;
                if (fabs(r1) + fabs(r0) <= 1e-15 * sc) { fast = true; break; }
                const double s1 = q1 - bb * q2, s0 = q0 - cc * q2;
                const double u1 = s0 - bb * s1, u0 = -cc * s1;
                const double det = u1 * s0 - u0 * s1;
                if (det == 0.0 || !(fabs(det) < 1e300)) break;
                bb += (r1 * s0 - r0 * s1) / det;
                cc += (u1 * r0 - u0 * r1) / det;
            }
            if (fast) {
                q1 = a[3] - bb * q2; q0 = a[2] - bb * q1 - cc * q2;
                auto quad_roots = [](double A, double B, double Cc, cx& ra, cx& rb) {       // A x^2 + B x + Cc, A != 0
                    const double disc = B * B - 4.0 * A * Cc;
                    if (disc < 0.0) { const double sq = sqrt(-disc); ra = cx_(-B / (2.0 * A), sq / (2.0 * A)); rb = cx_conj(ra); }
                    else { const double t = -0.5 * (B + copysign(sqrt(disc), B)); ra = cx_(t / A); rb = cx_(t != 0.0 ? Cc / t : 0.0); }
                };
                quad_roots(1.0, bb, cc, r[0], r[1]);
                if (nd == 4) quad_roots(q2, q1, q0, r[2], r[3]);
                else r[2] = cx_(-q0 / q1);
            }
        }
        double prev_big = 1e300;
        for (int it = 0; it < 200 && nd > 0 && !fast; ++it) {
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
            // at rounding level the steps stop shrinking (a root with a close neighbour settles to ~sqrt(eps) steps): stop instead of
            // spending the remaining sweeps on noise; the coefficient-residual check below still guards the result
            if (big < 1e-7 && big > 0.25 * prev_big) break;
            prev_big = big;
        }
        W.deg = n;
        for (int k = 0; k < n; ++k) W.rt[k] = r[k];
        for (int i = 1; i < n; ++i) {                                       // insertion sort by decreasing modulus
            const cx v = W.rt[i]; int j = i - 1;
            while (j >= 0 && cx_abs(W.rt[j]) < cx_abs(v)) { W.rt[j + 1] = W.rt[j]; --j; }
            W.rt[j + 1] = v;
        }
        W.iA = 3;
        for (int k = 1; k < n; ++k)
            if (fabs(W.rt[k].im) <= 1e-9 * cx_abs(W.rt[k])) W.iA = k;
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

// S1-S3 of the w family.  Fast front end for the usual structure -- degree 3 or 4 with matter and a constant term, and at least one
// complex-conjugate pair: Bairstow's iteration for a real quadratic factor x^2 + b x + c of E^2 from the pair of a0 + a3 x^3 ~ 0
// (x = rho e^{+-i pi/3}, rho = cbrt(a0/a3)) splits E^2 into the two real quadratics directly; roots by the quadratic formula; no
// indexed arrays, fast reciprocals.  Anything else (and any doubt: no convergence, both factors with real roots, where the pairing
// of the four real roots matters) goes to w_prep_general.
// kDefer (main pass of k_w): anything but the fast structure is only marked ST_INTERNAL_REDO (W then holds E^2 = 1, harmless to
// evaluate); the kernel lists such elements and its second pass runs them through the general solve.
template <bool kDefer = false>
CB_HD void w_prep(double Om, double OL, double Or, double Ow13, double Ow23, double H0, WCosmo& W) {
    const double Ok = 1.0 - Om - OL - Or - Ow13 - Ow23;
    const double a0 = OL, a1 = Ow23, a2 = Ok + Ow13, a3 = Om, a4 = Or;
    const double sc = fabs(a0) + fabs(a1) + fabs(a2) + fabs(a3) + fabs(a4);
    bool ok = (H0 > 0.0) && (a0 > 0.0) && (a3 > 0.0) && (a4 >= 0.0) && (sc < 1e300);
    double bb = 0.0, cc = 0.0, q2 = a4, q1 = 0.0, q0 = 0.0;
    if (ok) {
        const double rho = cbrt(a0 * cb_rcp(a3));
        bb = -rho; cc = rho * rho;
        bool conv = false;
        for (int it = 0; it < 16; ++it) {
            q1 = a3 - bb * q2; q0 = a2 - bb * q1 - cc * q2;
            const double r1 = a1 - bb * q0 - cc * q1, r0 = a0 - cc * q0;
            if (fabs(r1) + fabs(r0) <= 1e-15 * sc) { conv = true; break; }
            const double s1 = q1 - bb * q2, s0 = q0 - cc * q2;
            const double u1 = s0 - bb * s1, u0 = -cc * s1;
            const double det = u1 * s0 - u0 * s1;
            if (det == 0.0 || !(fabs(det) < 1e300)) break;
            const double idet = cb_rcp(det);
            bb += (r1 * s0 - r0 * s1) * idet;
            cc += (u1 * r0 - u0 * r1) * idet;
        }
        ok = conv;
    }
    const bool quart = a4 > 0.0;
    const double d2 = bb * bb - 4.0 * cc;                         // disc of x^2 + b x + c
    const double d1 = q1 * q1 - 4.0 * q2 * q0;                    // disc of q2 x^2 + q1 x + q0 (quartic case)
    // the pairing is forced only if a conjugate pair exists; three or four real roots: general path (pairs real roots with neighbours)
    ok = ok && ((d2 < 0.0) || (quart && d1 < 0.0)) && (quart || q1 != 0.0);
    if (!ok) {
        if (!kDefer) { w_prep_general(Om, OL, Or, Ow13, Ow23, H0, W); return; }
        W.f1 = W.g1 = 0.0; W.h1 = 1.0; W.f2 = W.g2 = 0.0; W.h2 = 1.0;
        W.q11 = W.q21 = 1.0; W.theta = W.sD = W.sDr = 0.0;
        W.rr[0] = W.rr[1] = W.rr[2] = W.rr[3] = 0.0; W.nreal = 0;
        W.Ok = 0.0; W.dH = W.tH = 1.0;
        W.a[0] = 1.0; W.a[1] = W.a[2] = W.a[3] = W.a[4] = 0.0;
        W.rt[0] = W.rt[1] = W.rt[2] = W.rt[3] = cx_(0.0);
        W.deg = 0; W.iA = 3;
        W.status = ST_INTERNAL_REDO;
        return;
    }
    W.Ok = Ok;
    { const double iH = cb_rcp(H0); W.dH = C_KM_S * iH; W.tH = HUBBLE_GYR * iH; }
    W.a[0] = a0; W.a[1] = a1; W.a[2] = a2; W.a[3] = a3; W.a[4] = a4;
    W.status = 0;
    W.deg = quart ? 4 : 3;
    W.f1 = quart ? q2 : 0.0; W.g1 = q1; W.h1 = q0; W.f2 = 1.0; W.g2 = bb; W.h2 = cc;
    // roots of the two factors
    cx ra, rb, rc_, rd;                                           // (ra, rb) of Q2, (rc_, rd) of Q1 (rd unused for the cubic)
    int nr = 0;
    double real0 = 0.0, real1 = 0.0, real2 = 0.0;                 // real roots, ascending where two come from one quadratic
    if (d2 < 0.0) { const double sq = cb_sqrt0(-d2); ra = cx_(-0.5 * bb, 0.5 * sq); rb = cx_conj(ra); }
    else {
        const double t = -0.5 * (bb + copysign(cb_sqrt0(d2), bb));
        const double x1 = t, x2 = (t != 0.0) ? cc * cb_rcp(t) : 0.0;
        ra = cx_(x1); rb = cx_(x2);
        real0 = fmin(x1, x2); real1 = fmax(x1, x2); nr = 2;
    }
    if (quart) {
        const double i2 = cb_rcp(2.0 * q2);
        if (d1 < 0.0) { rc_ = cx_(-q1 * i2, cb_sqrt0(-d1) * i2); rd = cx_conj(rc_); }
        else {
            const double t = -0.5 * (q1 + copysign(cb_sqrt0(d1), q1));
            const double x1 = t * cb_rcp(q2), x2 = (t != 0.0) ? q0 * cb_rcp(t) : 0.0;
            rc_ = cx_(x1); rd = cx_(x2);
            real0 = fmin(x1, x2); real1 = fmax(x1, x2); nr = 2;   // (d2 < 0 here: the only real roots)
        }
    } else {
        const double xl = -q0 * cb_rcp(q1);
        rc_ = cx_(xl); rd = cx_(0.0);
        if (nr == 0) { real0 = xl; nr = 1; }
        else { real2 = fmax(real1, xl); const double lo = fmin(real0, xl), mid = fmax(real0, fmin(real1, xl)); real0 = lo; real1 = mid; nr = 3; }
    }
    W.nreal = nr; W.rr[0] = real0; W.rr[1] = real1; W.rr[2] = real2; W.rr[3] = 0.0;
    // roots by decreasing modulus (sorting network on four scalars; the cubic's fourth slot has modulus -1 and stays last)
    double ma = ra.re * ra.re + ra.im * ra.im, mb = rb.re * rb.re + rb.im * rb.im, mc = rc_.re * rc_.re + rc_.im * rc_.im,
           md = quart ? rd.re * rd.re + rd.im * rd.im : -1.0;
    auto cswap = [](cx& u, double& mu, cx& v, double& mv) { if (mu < mv) { const cx t = u; u = v; v = t; const double m = mu; mu = mv; mv = m; } };
    cswap(ra, ma, rb, mb); cswap(rc_, mc, rd, md); cswap(ra, ma, rc_, mc); cswap(rb, mb, rd, md); cswap(rb, mb, rc_, mc);
    W.rt[0] = ra; W.rt[1] = rb; W.rt[2] = rc_; W.rt[3] = rd;
    W.iA = 3;
    if (fabs(rb.im) <= 1e-9 * sqrt(mb)) W.iA = 1;
    if (fabs(rc_.im) <= 1e-9 * sqrt(mc)) W.iA = 2;
    if (quart && fabs(rd.im) <= 1e-9 * sqrt(md)) W.iA = 3;
    // the product must reproduce the coefficients
    const double e4 = W.f1, e3 = W.f1 * W.g2 + W.g1, e2 = W.f1 * W.h2 + W.g1 * W.g2 + W.h1, e1 = W.g1 * W.h2 + W.h1 * W.g2, e0 = W.h1 * W.h2;
    const double res = fabs(e4 - a4) + fabs(e3 - a3) + fabs(e2 - a2) + fabs(e1 - a1) + fabs(e0 - a0);
    if (!(res <= 1e-11 * sc)) W.status |= ST_UNSUPPORTED;
    W.q11 = W.f1 + W.g1 + W.h1;
    W.q21 = W.f2 + W.g2 + W.h2;
    W.theta = 2.0 * W.f1 * W.h2 + 2.0 * W.h1 * W.f2 - W.g1 * W.g2;
    W.sD = 0.25 * (W.g1 * W.g1 - 4.0 * W.f1 * W.h1) * d2;
    W.sDr = cb_sqrt0(fabs(W.sD));
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
    const double ra = cb_sqrt0(a1), rb = cb_sqrt0(a2), U12 = ra + rb;
    double xa[1] = {U12 * U12}, mp[1], s[1], p5[1] = {0.0}, p0[1] = {0.0};
    const double hd = 0.5 * z2 * W.theta, hs = z2 * W.sDr;
    mp[0] = xa[0] - hd;
    s[0] = z2 * z2 * W.sD;
    const double dl5[1] = {0.0}, dl0[1] = {0.0}, Qc[1] = {carlson_Qc<double>(hd, hs, false)}, Q5v[1] = {0.0}, Q0v[1] = {0.0};
    double g2, tailD[1], sum5[1], sum0[1];
    carlson_dup<double, false, false, false, 1, Vote>(xa, mp, s, p5, p0, dl5, dl0, Qc, Q5v, Q0v, st, vote, g2, tailD, sum5, sum0);
    const double RF = carlson_rf_series<double>(xa[0], mp[0], g2, hd, s[0]);
    const double I0 = 2.0 * z * RF;                                        // eq. (3.7) / (B.1)
    const double iE = cb_rcp(ra * rb);                                     // E(1) = 1: a1 a2 = E^2(x)
    double F, Fi, Fk;
    sinn<double>(W.Ok, I0, F, Fi, Fk);
    v[0] = W.dH * I0; v[1] = W.dH * F; v[2] = x * v[1];
    dz[0] = W.dH * iE; dz[1] = W.dH * Fi * iE; dz[2] = fma(x, dz[1], v[1]);
    if (v[2] > 0.0) {
        v[3] = fma(CB_KT.five_over_ln10, Num<double>::log_(v[2]), 25.0);
        dz[3] = CB_KT.five_over_ln10 * dz[2] * cb_rcp(v[2]);
    } else {
        v[3] = dz[3] = NAN;
        if (!(st[0] & (ST_ROOT_ON_PATH | ST_UNSUPPORTED))) st[0] |= ST_DL_NONPOS;
    }
    if (st[0] & (ST_ROOT_ON_PATH | ST_UNSUPPORTED))
        for (int i = 0; i < 4; ++i) v[i] = dz[i] = NAN;
    return st[0];
}

// ---- t_L and d_abs on the general quartic (rest).  Eqs. (3.8)/(3.9) single out a root r_i, which may be complex here,
// so this is the paper's own formulation: complex roots, complex X_n, Y_n, u_ij and complex Carlson functions,
// principal square roots throughout.  Labelling ("r_i, r_j the biggest roots"), by modulus of
// the x-roots: t_L: r_i = the biggest; d_abs: r_l = the biggest, r_i = the smallest real root (the smallest root if none is real) --
// tried over all 24 labellings against the oracle on the seeded mix: the only one without failures (d_abs <= 5e-11: the Om/Or
// cancellation of eq. (3.9)).

// R_F(x,y,z), R_D(x,y,z) (last argument z) and R_J(x,y,z,p), all arguments complex: duplication, ref. [10] (DLMF 19.36(i))
struct CxCarlson { cx RF, RD, RJ; };
CB_HD void cx_carlson(cx x, cx y, cx z, cx p, bool want_j, CxCarlson& out) {
    const cx x0 = x, y0 = y, z0 = z;
    const cx delta = (p - x) * (p - y) * (p - z);
    const cx AF0 = (1.0 / 3.0) * (x + y + z), AD0 = 0.2 * (x + y + 3.0 * z), AJ0 = 0.2 * (x + y + z + 2.0 * p);
    const double dev = fmax(fmax(cx_abs(AF0 - x), cx_abs(AF0 - y)), cx_abs(AF0 - z)) + fmax(cx_abs(AD0 - x), fmax(cx_abs(AD0 - y), cx_abs(AD0 - z)));
    const double devJ = want_j ? fmax(fmax(cx_abs(AJ0 - x), cx_abs(AJ0 - y)), fmax(cx_abs(AJ0 - z), cx_abs(AJ0 - p))) : 0.0;
    double f = 1.0;
    cx tailD = cx_(0.0), sumJ = cx_(0.0);
    for (int it = 0; it < 2 * NIT_CAP; ++it) {
        const cx AF = (1.0 / 3.0) * (x + y + z), AD = 0.2 * (x + y + 3.0 * z), AJ = 0.2 * (x + y + z + 2.0 * p);
        if (f * 600.0 * dev < fmin(cx_abs(AF), cx_abs(AD)) && (!want_j || f * 600.0 * devJ < cx_abs(AJ))) break;
        const cx sx = cx_sqrt(x), sy = cx_sqrt(y), sz = cx_sqrt(z);
        const cx lam = sx * sy + sx * sz + sy * sz;
        tailD = tailD + cx_(f) / (sz * (z + lam));
        if (want_j) {
            const cx sp = cx_sqrt(p);
            const cx d = (sp + sx) * (sp + sy) * (sp + sz);
            const cx e = (f * f * f) * delta / (d * d);
            sumJ = sumJ + (f * cx_rc1(e)) / d;
            p = 0.25 * (p + lam);
        }
        x = 0.25 * (x + lam); y = 0.25 * (y + lam); z = 0.25 * (z + lam);
        f *= 0.25;
    }
    const double* c = CB_KT.rj;
    {
        const cx A = (1.0 / 3.0) * (x + y + z), g = cx_(f) / A;
        const cx X = (AF0 - x0) * g, Y = (AF0 - y0) * g, Z = -(X + Y);
        const cx e2 = X * Y - Z * Z, e3 = X * Y * Z;
        const cx S = cx_(1.0) - 0.1 * e2 + (1.0 / 14.0) * e3 + (1.0 / 24.0) * (e2 * e2) - (3.0 / 44.0) * (e2 * e3) - (5.0 / 208.0) * (e2 * e2 * e2)
                     + (3.0 / 104.0) * (e3 * e3) + (1.0 / 16.0) * (e2 * e2 * e3);
        out.RF = S / cx_sqrt(A);
    }
    {
        const cx A = 0.2 * (x + y + 3.0 * z), g = cx_(f) / A;
        const cx X = (AD0 - x0) * g, Y = (AD0 - y0) * g, Z = (-1.0 / 3.0) * (X + Y);
        const cx XY = X * Y, Z2 = Z * Z;
        const cx e2 = XY - 6.0 * Z2, e3 = (3.0 * XY - 8.0 * Z2) * Z, e4 = 3.0 * ((XY - Z2) * Z2), e5 = XY * Z2 * Z;
        const cx S = cx_(1.0) + c[0] * e2 + c[3] * e3 + c[1] * (e2 * e2) + c[8] * e4 + c[4] * (e2 * e3) + c[10] * e5 + c[2] * (e2 * e2 * e2)
                     + c[6] * (e3 * e3) + c[9] * (e2 * e4) + c[5] * (e2 * e2 * e3) + c[7] * (e3 * e4 + e2 * e5);
        out.RD = (f * S) / (A * cx_sqrt(A)) + 3.0 * tailD;
    }
    out.RJ = cx_(0.0);
    if (want_j) {
        const cx A = 0.2 * (x + y + z + 2.0 * p), g = cx_(f) / A;
        const cx X = (AJ0 - x0) * g, Y = (AJ0 - y0) * g, Z = (AJ0 - z0) * g;
        const cx P = -0.5 * (X + Y + Z);
        const cx XYZ = X * Y * Z, P2 = P * P;
        const cx e2 = X * Y + X * Z + Y * Z - 3.0 * P2;
        const cx e3 = XYZ + 2.0 * (e2 * P) + 4.0 * (P2 * P);
        const cx e4 = (2.0 * XYZ + e2 * P + 3.0 * (P2 * P)) * P;
        const cx e5 = XYZ * P2;
        const cx S = cx_(1.0) + c[0] * e2 + c[3] * e3 + c[1] * (e2 * e2) + c[8] * e4 + c[4] * (e2 * e3) + c[10] * e5 + c[2] * (e2 * e2 * e2)
                     + c[6] * (e3 * e3) + c[9] * (e2 * e4) + c[5] * (e2 * e2 * e3) + c[7] * (e3 * e4 + e2 * e5);
        out.RJ = (f * S) / (A * cx_sqrt(A)) + 6.0 * sumJ;
    }
}

// T = int_1^x dx/(x E), A = int_1^x x^2 dx/E for E^2 of degree 4 or 3 with the roots W.rt (x-roots, so d_i5 = -rho_i), and for
// E^2 = a x^n (every root at 0: elementary).  Returns false where the method does not apply (degree <= 2 with distinct roots).
// dz = x - 1 comes in as z (formed here it would carry the rounding of 1 + z: eps/z of both integrals).
// Branches: the formulae hold with sqrt(x - r) continued from a conjugate pair, i.e. with X_j X_k = +sqrt((x - r_j)(x - r_k)) for the
// two members of a pair.  Principal square roots do that for complex pairs; for two REAL roots to the right of the path (loitering-type
// models) they give (i a)(i a') = -a a' instead, which flips the sign of the odd terms (the boundary terms): every second such root
// takes the conjugate branch.  Real roots are taken as exactly real (the sign of a rounding-level imaginary part would pick the branch).
CB_HD void w_roots_sqrt(const cx* r, int n, double x, cx* X, cx* Y, bool* isreal) {
    const double hi = fmax(1.0, x);
    int nright = 0;
    for (int k = 0; k < n; ++k) {
        isreal[k] = fabs(r[k].im) <= 1e-9 * cx_abs(r[k]);
        const cx rk = isreal[k] ? cx_(r[k].re) : r[k];
        X[k] = cx_sqrt(cx_(x) - rk); Y[k] = cx_sqrt(cx_(1.0) - rk);
        if (isreal[k] && rk.re > hi) {
            if (nright & 1) { X[k] = cx_conj(X[k]); Y[k] = cx_conj(Y[k]); }
            ++nright;
        }
    }
}
CB_HD_NOINLINE bool w_TA(const WCosmo& W, double x, double dz, bool want_T, bool want_A, double& TT, double& AA) {
    TT = AA = NAN;
    const double lead = W.a[W.deg];
    bool mono = true;
    for (int k = 0; k < W.deg; ++k) mono = mono && cx_abs(W.rt[k]) == 0.0;
    if (mono) {                                          // E = sqrt(lead) x^(deg/2)
        const double h = 0.5 * W.deg, il = 1.0 / sqrt(lead), lx = log1p(dz);
        TT = (h == 0.0) ? il * lx : il * -expm1(-h * lx) / h;
        AA = (h == 3.0) ? il * lx : il * expm1((3.0 - h) * lx) / (3.0 - h);
        return true;
    }
    if (W.deg < 3) return false;
    const double ia = 1.0 / sqrt(lead);
    if (W.deg == 4) {
        const cx* r = W.rt;
        cx X[4], Y[4];
        bool isreal[4];
        w_roots_sqrt(r, 4, x, X, Y, isreal);
        auto usq = [&](int a, int b, int c, int e) { const cx u = X[a] * X[b] * Y[c] * Y[e] + Y[a] * Y[b] * X[c] * X[e]; return u * u; };
        auto pair = [&](int a, int b) { int c = -1, e = -1; for (int m = 0; m < 4; ++m) if (m != a && m != b) { if (c < 0) c = m; else e = m; } return usq(a, b, c, e); };
        auto d = [&](int a, int b) { return r[b] - r[a]; };
        const double lo = fmin(1.0, x);
        CxCarlson K;
        // the conjugate partner of root a (the other root closest to conj(r_a))
        auto partner = [&](int a) { int best = -1; double db = 1e300; for (int m = 0; m < 4; ++m) if (m != a) { const double dd = cx_abs(r[m] - cx_conj(r[a])); if (dd < db) { db = dd; best = m; } } return best; };
        if (want_T) {                    // eq. (3.8): r_i = the biggest non-zero REAL root left of the path where there is one (any j, k, l
                                         // then); else a complex root with ITS CONJUGATE as r_j (the labelling of cosmo_c4.cuh: the
                                         // products X_i X_j, Y_i Y_j are then real and the principal branches consistent)
            int i = -1, j, k, l;
            for (int m = 3; m >= 0; --m)
                if (isreal[m] && r[m].re < lo && r[m].re != 0.0) i = m;    // the roots are sorted by decreasing modulus
            if (i >= 0) {
                int o[3], c = 0;
                for (int m = 0; m < 4; ++m) if (m != i) o[c++] = m;
                j = o[0]; k = o[1]; l = o[2];
            } else {
                i = 0;                                                     // the pair further to the left, as cosmo_factor picks Q1
                double best = 1e300;
                for (int m = 0; m < 4; ++m) if (!isreal[m] && r[m].re < best) { best = r[m].re; i = m; }
                j = partner(i);
                k = -1; l = -1;
                for (int m = 0; m < 4; ++m) if (m != i && m != j) { if (k < 0) k = m; else l = m; }
            }
            const cx Pij = pair(i, j), Pik = pair(i, k), Pil = pair(i, l);
            const cx p5 = Pij - (dz * dz) * (d(i, k) * d(i, l) * (r[j] / r[i]));
            cx_carlson(Pij, Pik, Pil, p5, true, K);
            const cx q5 = (cx_(x) / ((cx_(1.0) - r[i]) * (cx_(x) - r[i]))) * p5;
            const cx s5 = q5 + (dz * dz) * (r[k] * r[l] * (r[j] / r[i]));
            const cx br = K.RF - ((dz * dz / 3.0) * (d(i, j) * d(i, k) * d(i, l) / (-r[i])) * K.RJ + cx_rc(s5, q5));
            TT = ia * ((2.0 * dz) * (br / r[i])).re;
        }
        if (want_A) {                    // eq. (3.9), (i, j, k, l) = (rn, pair, pair, big) of the hot path: r_i = the smallest REAL root left
                                         // of the path, r_l = the biggest root (the biggest real one left of the path if that one lies to
                                         // the right); without real roots left of the path, the complex pair further to the left (r_i and
                                         // its conjugate r_l, the labelling of cosmo_c4.cuh); r_j, r_k the other two
            int i = -1, l = -1;
            for (int m = 0; m < 4; ++m)
                if (isreal[m] && r[m].re < lo) { if (l < 0) l = m; i = m; }   // sorted by decreasing modulus: first = biggest, last = smallest
            // (a much bigger complex pair -- Om = 0 with little radiation: +- i sqrt(a2/Or) -- serves as r_l like the big real root does)
            if (i > 0 && !(isreal[0] && !(r[0].re < lo))) l = 0;
            if (l < 0 || i == l) {
                // the biggest pair whose real part lies left of the path (as r_j, r_k a much bigger pair would multiply the cancellation
                // of eq. (3.9) by its modulus squared), else the left-most one
                double best = 1e300;
                i = -1;
                for (int m = 3; m >= 0; --m) if (!isreal[m] && r[m].re < lo) i = m;
                if (i < 0) { i = 0; for (int m = 0; m < 4; ++m) if (!isreal[m] && r[m].re < best) { best = r[m].re; i = m; } }
                l = partner(i);
            }
            int j = -1, k = -1;
            for (int m = 0; m < 4; ++m)
                if (m != i && m != l) { if (j < 0) j = m; else k = m; }
            const cx Uij = pair(i, j), Uik = pair(i, k), Uil = pair(i, l);
            const cx p0 = Uij - (dz * dz) * (d(i, k) * d(i, l));
            cx_carlson(Uij, Uik, Uil, p0, true, K);                      // R_D's last argument is u_il^2
            const cx q0 = p0 / ((cx_(1.0) - r[i]) * (cx_(x) - r[i]));
            const cx s0 = q0 + cx_(dz * dz);
            // boundary term [F], F^2 = N(x)/(x - r_l), N = (x - r_i)(x - r_j)(x - r_k); close limits: through F^2 with dz taken out of
            // N(x)(1 - r_l) - N(1)(x - r_l) analytically (cosmo_c4.cuh does the same; subtracted directly it loses eps/dz)
            const cx Fx = X[i] * X[j] * X[k] / X[l], F1 = Y[i] * Y[j] * Y[k] / Y[l];
            cx bnd = Fx - F1;
            if (fabs(dz) <= 0.05 * lo) {
                const cx e1 = r[i] + r[j] + r[k], e2 = r[i] * r[j] + r[i] * r[k] + r[j] * r[k];
                const cx dd = cx_(x * x + x + 1.0) - (x + 1.0) * e1 + e2;                       // [N; x, 1]
                const cx N1 = (cx_(1.0) - r[i]) * (cx_(1.0) - r[j]) * (cx_(1.0) - r[k]);
                bnd = dz * ((dd * (cx_(1.0) - r[l]) - N1) / ((cx_(x) - r[l]) * (cx_(1.0) - r[l]) * (Fx + F1)));
            }
            const cx uil = X[i] * X[l] * Y[j] * Y[k] + Y[i] * Y[l] * X[j] * X[k];
            const cx sig = r[0] + r[1] + r[2] + r[3];
            const cx t2 = dz * ((2.0 * (r[i] * r[i]) - d(i, j) * d(i, k)) * K.RF);
            const cx t3 = dz * ((d(j, l) * d(k, l)) * (((dz * dz / 3.0) * (d(i, j) * d(i, k))) * K.RD + (X[i] * Y[i]) / (X[l] * Y[l] * uil)));
            const cx B0 = cx_rc(s0, q0) - ((dz * dz / 3.0) * (d(i, j) * d(i, k) * d(i, l))) * K.RJ;     // = int (x - r_i) dx / (2 dz sqrt(lead) E)
            const cx t4 = dz * (sig * B0);
            AA = ia * (bnd + t2 + t3 + t4).re;
            // The groups of eq. (3.9) cancel by ~ a3/(a4 x).  Where radiation is a perturbation of a model with matter the
            // same Carlson values are assembled through the moment recurrence of the hot path (cosmo_eval.cuh, band_solve; DESIGN.md
            // "d_abs") with the x^1 term of this family: u_0 = I0, u_1 = 2 dz B0 / sqrt(lead) + r_i I0, d_abs integral = u_2.
            if (W.a[3] > 0.0) {
                constexpr int KS = REC_KS;
                double bk[KS + 1], u2[KS + 1], trunc, e2m1 = 0.0;
                {
                    double dk = 0.0;                               // x^j - 1 = x (x^(j-1) - 1) + dz
                    for (int m = 0; m <= 4; ++m) { e2m1 = fma(W.a[m], dk, e2m1); dk = fma(x, dk, dz); }       // E^2 - 1 (the coefficients sum to 1)
                }
                const double Ex = sqrt(1.0 + e2m1), Em1 = e2m1 / (Ex + 1.0);
                {
                    double dk = 0.0;
                    for (int m = 0; m <= KS; ++m) { bk[m] = fma(dk, Ex, Em1); dk = fma(x, dk, dz); }          // x^m E(x) - E(1)
                }
                const double I0 = ia * 2.0 * dz * K.RF.re;
                const double u1 = (ia * (2.0 * dz) * B0 + I0 * r[i]).re;
                band_solve<double, KS + 1, 2, 1, 0, 0, true>(W.a[3], W.a[0], W.a[4], W.a[2], bk, u1, I0, 0.0, x, u2, trunc, W.a[1]);
                if (trunc <= 1e-15 * fabs(u2[0])) AA = u2[0];
            }
        }
        return true;
    }
    // degree 3: eqs. (B.2), (B.3) with r_i = the biggest root (any labelling does; tested over all six)
    const cx* r = W.rt;
    cx X[3], Y[3];
    bool isreal[3];
    w_roots_sqrt(r, 3, x, X, Y, isreal);
    const cx u0 = X[0] * Y[1] * Y[2] + Y[0] * X[1] * X[2], u1 = X[1] * Y[0] * Y[2] + Y[1] * X[0] * X[2], u2 = X[2] * Y[0] * Y[1] + Y[2] * X[0] * X[1];
    CxCarlson K;
    if (want_T) {
        const cx p5 = u0 * u0 + (dz * dz) * r[0];
        cx_carlson(u0 * u0, u1 * u1, u2 * u2, p5, true, K);
        const cx s5 = Y[0] * Y[1] * Y[2] * cx_(x) + X[0] * X[1] * X[2];
        TT = ia * ((2.0 * dz) * ((dz * dz / 3.0) * K.RJ + cx_rc(s5 * s5, cx_(x) * p5))).re;
    }
    if (want_A) {
        cx_carlson(u1 * u1, u2 * u2, u0 * u0, cx_(1.0), false, K);       // R_D(u_j^2, u_k^2, u_i^2)
        const cx d01 = r[1] - r[0], d02 = r[2] - r[0], sig = r[0] + r[1] + r[2];
        const cx Gx = X[0] * X[1] * X[2], G1 = Y[0] * Y[1] * Y[2];                              // G^2 = N(x) = (x - r_0)(x - r_1)(x - r_2)
        cx dG = Gx - G1;
        if (fabs(dz) <= 0.05 * fmin(1.0, x)) {
            const cx e2 = r[0] * r[1] + r[0] * r[2] + r[1] * r[2];
            dG = dz * ((cx_(x * x + x + 1.0) - (x + 1.0) * sig + e2) / (Gx + G1));              // dz [N; x, 1] / (G(x) + G(1))
        }
        const cx b3 = dG + dz * ((3.0 * (r[0] * r[0]) - d01 * d02) * K.RF)
                      + (2.0 * dz) * (sig * (((dz * dz / 3.0) * (d01 * d02)) * K.RD + (X[0] * Y[0]) / u0));
        AA = ia * ((2.0 / 3.0) * b3).re;
    }
    return true;
}

// Gradient integrals of the w family: int D_theta p_X / E^3 dx over [1, x], theta = (Om, OL, Or, Ow23), D_theta = x^3 - x^2, 1 - x^2,
// x^4 - x^2, x - x^2 (Ow13 enters E^2 like curvature: no dependence at fixed sum), p_X = 1, 1/x, x^2 (X = I0, T, A): out[12] = [X][theta].
// By the 12-point Gauss-Legendre rule on panels of ratio <= 2 in x - c, as grad_quad() of the hot path (cosmo_obs.cuh), with c placed so
// that the panel widths follow the distance to the nearest root left of the path.  A general quartic has no fixed root structure to
// build the hot path's gradient bases on, so this family takes the quadrature for every element; where a root sits too close to the path
// for the rule to converge (Bernstein parameter < 3.5 for some root) the element is flagged ST_GRAD_ILLCOND instead.
CB_HD_NOINLINE unsigned w_grad_quad(const WCosmo& W, double z, double out[12]) {
    const double X12[12] = {0.00921968287664037465, 0.0479413718147625717, 0.115048662902847656, 0.206341022856691276, 0.316084250500909903,
                            0.437383295744265542, 0.562616704255734458, 0.683915749499090097, 0.793658977143308724, 0.884951337097152344,
                            0.952058628185237428, 0.990780317123359625};
    const double W12[12] = {0.0235876681932559136, 0.0534696629976592155, 0.0800391642716731132, 0.101583713361532961, 0.116746268269177404,
                            0.124573522906701393, 0.124573522906701393, 0.116746268269177404, 0.101583713361532961, 0.0800391642716731132,
                            0.0534696629976592155, 0.0235876681932559136};
    for (int i = 0; i < 12; ++i) out[i] = 0.0;
    const double X2 = 1.0 + z;
    const double lo = fmin(1.0, X2), hi = fmax(1.0, X2);
    if (!(lo > 0.0) || z == 0.0) return 0u;
    double dmin = 1e300;                                   // distance of the nearest root left of the path from its start
    for (int k = 0; k < W.deg; ++k)
        if (W.rt[k].re < lo) dmin = fmin(dmin, hypot(lo - W.rt[k].re, W.rt[k].im));
    const double c = lo - fmin(dmin, 1e6 * lo);
    const double q = (X2 - c) / (1.0 - c), qa = q >= 1.0 ? q : 1.0 / q;
    int np = 1;
    double r = q;
    if (qa > 2.0) {
        const double lr = log(q);
        np = (int)ceil(fabs(lr) * 1.4426950408889634);
        if (np > 64) np = 64;
        r = exp(lr / np);
    }
    unsigned st = 0u;
    const double rr = r >= 1.0 ? r : 1.0 / r;
    for (int k = 0; k < W.deg; ++k) {                      // Bernstein parameter of every root against the panel next to it
        const double a0 = W.rt[k].re, y0 = fabs(W.rt[k].im);
        double wre, h;
        if (a0 < lo) { h = 0.5 * (lo - c) * (rr - 1.0); wre = (lo - a0) / h + 1.0; }
        else if (a0 > hi) { h = 0.5 * (hi - c) * (1.0 - 1.0 / rr); wre = (a0 - hi) / h + 1.0; }
        else { h = 0.5 * (a0 - c) * (rr - 1.0); wre = 0.0; }
        const double wim = y0 / h;
        const double a = 0.5 * (hypot(wre + 1.0, wim) + hypot(wre - 1.0, wim));
        if (!(a + sqrt(fmax(a * a - 1.0, 0.0)) >= 3.5)) st = (unsigned)ST_GRAD_ILLCOND;
    }
    double wd = (np == 1) ? z : z * (r - 1.0) / (q - 1.0), tlo = 0.0;
    for (int k = 0; k < np; ++k) {
#pragma unroll
        for (int i = 0; i < 12; ++i) {
            const double t = fma(wd, X12[i], tlo), x = 1.0 + t;
            const double e2 = fma(fma(fma(fma(W.a[4], x, W.a[3]), x, W.a[2]), x, W.a[1]), x, W.a[0]);
            const double ie = Num<double>::rsqrt_(e2), f = (W12[i] * wd) * (ie * ie) * (ie * t);
            const double x2 = x * x, xp1 = x + 1.0, ix = cb_rcp(x);
            const double d[4] = {f * x2, -f * xp1, f * x2 * xp1, -f * x};
#pragma unroll
            for (int th = 0; th < 4; ++th) { out[th] += d[th]; out[4 + th] = fma(d[th], ix, out[4 + th]); out[8 + th] = fma(d[th], x2, out[8 + th]); }
        }
        tlo += wd;
        wd *= r;
    }
    return st;
}

// One element of the w family: values v[6] = D_C, D_M, D_L, mu, t_L, d_abs; dz[6] = d v / dz; with want_grad also
// gp[6][6] = d v[o] / d (Om, OL, Or, Ow13, Ow23, H0).  Status as w_eval, plus 2 (unsupported) with NaN in the t_L / d_abs planes
// where E^2 has degree <= 2 with distinct roots (eqs. (3.8)/(3.9), (B.2)/(B.3) need degree 3 or 4), plus 16.
template <typename Vote>
CB_HD unsigned w_eval_full(const WCosmo& W, double z, const Vote& vote, bool want_T, bool want_A, bool want_grad, double v[6], double dz[6],
                           double gp[6][6]) {
    double v4[4], d4[4];
    unsigned st = w_eval<Vote>(W, z, vote, v4, d4);
    for (int o = 0; o < 4; ++o) { v[o] = v4[o]; dz[o] = d4[o]; }
    v[4] = v[5] = dz[4] = dz[5] = NAN;
    const bool bad = (st & (ST_ROOT_ON_PATH | ST_UNSUPPORTED)) != 0;
    const double x = 1.0 + z;
    if ((want_T || want_A) && !bad) {
        double TT, AA;
        if (w_TA(W, x, z, want_T, want_A, TT, AA)) {
            const double E = W.dH / d4[0];                 // d D_C / dz = d_H / E
            if (want_T) { v[4] = W.tH * TT; dz[4] = W.tH / (x * E); }
            if (want_A) { v[5] = W.dH * AA; dz[5] = W.dH * x * x / E; }
            // a closed form that came out not-a-number on a valid path (an isolated coincidence inside the complex Carlson functions:
            // one row in 3e4 of the wide-prior comparison, on the device only) is reported, not passed on silently
            if ((want_T && !isfinite(TT)) || (want_A && !isfinite(AA))) st |= ST_ITER_CAP;
        } else {
            st |= ST_UNSUPPORTED;
        }
    }
    if (!want_grad) return st;
    for (int o = 0; o < 6; ++o)
        for (int t = 0; t < 6; ++t) gp[o][t] = NAN;
    if (bad) return st;
    double q[12];
    st |= w_grad_quad(W, z, q);
    const double I0 = v[0] / W.dH;
    double F, Fi, Fk;
    sinn<double>(W.Ok, I0, F, Fi, Fk);
    const int col[5] = {0, 1, 2, -1, 3};                   // Om, OL, Or, Ow13 (no E^2 dependence), Ow23 -> column of q
    const double k5 = CB_KT.five_over_ln10;
    for (int t = 0; t < 5; ++t) {
        const double dI = col[t] >= 0 ? -0.5 * q[col[t]] : 0.0, dT = col[t] >= 0 ? -0.5 * q[4 + col[t]] : 0.0, dA = col[t] >= 0 ? -0.5 * q[8 + col[t]] : 0.0;
        gp[0][t] = W.dH * dI;
        gp[1][t] = W.dH * (Fi * dI - Fk);                  // d Ok / d theta = -1 for each of the five densities
        gp[2][t] = x * gp[1][t];
        gp[3][t] = (v[2] > 0.0) ? k5 * gp[2][t] / v[2] : NAN;
        gp[4][t] = W.tH * dT;
        gp[5][t] = W.dH * dA;
    }
    const double iH0 = W.dH * (1.0 / C_KM_S);
    for (int o = 0; o < 6; ++o) gp[o][5] = -v[o] * iH0;
    gp[3][5] = -k5 * iH0;
    return st;
}

}  // namespace cb
