// cosmo_prep.cuh -- hot-path steps S1-S3: coefficients, validity, root solve, per-cosmology constants.
//
// Always FP64 (reading R-fp32: the per-cosmology block stays FP64 in every variant).
//
// Root solve (eq. (3.2); :249 "numerical root-finding worked better than the
// algebraic formulae").  The polynomial in x = 1+z is  P(x) = Or x^4 + Om x^3 + Ok x^2 + OL
// (eq. (2.2)).  Its roots are never formed one by one: P is split into two REAL quadratic
// factors  P = (Or x + m)(x - rn) * (x^2 + b x + c), which stay finite for Or -> 0 (cubic case of
// appendix B.1) and for OL -> 0, and which carry a complex-conjugate pair and a real
// pair (near-degenerate or not) by the same two real numbers (b, c).
#pragma once
#include "cosmo_types.cuh"

namespace cb {

// Solve the n x n system M a = rhs_k (k < nrhs) in place by Gaussian elimination with partial pivoting.
// M is row-major [n][n+nrhs] augmented.  Singular systems leave inf/nan (degenerate roots).
template <int N, int NR>
CB_HD void solve_aug(double (&M)[N][N + NR]) {
    for (int col = 0; col < N; ++col) {
        int piv = col;
        double best = fabs(M[col][col]);
        for (int r = col + 1; r < N; ++r) {
            double v = fabs(M[r][col]);
            if (v > best) { best = v; piv = r; }
        }
        if (piv != col) {
            for (int k = col; k < N + NR; ++k) { double t = M[col][k]; M[col][k] = M[piv][k]; M[piv][k] = t; }
        }
        double inv = 1.0 / M[col][col];
        for (int r = col + 1; r < N; ++r) {
            double f = M[r][col] * inv;
            for (int k = col + 1; k < N + NR; ++k) M[r][k] = fma(-f, M[col][k], M[r][k]);
        }
    }
    for (int col = N - 1; col >= 0; --col) {
        double inv = 1.0 / M[col][col];
        for (int k = N; k < N + NR; ++k) {
            double s = M[col][k];
            for (int j = col + 1; j < N; ++j) s = fma(-M[col][j], M[j][k], s);
            M[col][k] = s * inv;
        }
    }
}

// N_k(x) = k x^(k-1) E^2 - x^k (E^2)'/2 : d(x^k / E)/dx = N_k / E^3.  Adds coef * N_k to column `dst` (rows = powers).
template <int ROWS, int COLS>
CB_HD void add_Nk(double (&M)[ROWS][COLS], int dst, int k, const double e[5]) {
    for (int p = 0; p < 5; ++p) {
        if (k > 0 && p + k - 1 < ROWS) M[p + k - 1][dst] += k * e[p];
        if (p > 0 && p - 1 + k < ROWS) M[p - 1 + k][dst] -= 0.5 * p * e[p];
    }
}

// S1-S3.  want_grad: 0 none, 1 chi-family (GI), 2 all (GI, GT, GA).
CB_HD void cosmo_prep(double Om, double OL, double Or, double H0, int want_grad, Cosmo<double>& C) {
    const double Ok = 1.0 - Om - OL - Or;
    C.Om = Om; C.OL = OL; C.Or = Or; C.Ok = Ok; C.H0 = H0;
    C.dH = C_KM_S / H0; C.tH = HUBBLE_GYR / H0;
    C.cubic = (Or == 0.0);
    unsigned st = 0;
    // the method needs degree 3 or 4 and non-negative densities (include/cosmo_b200.h)
    if (!(Or >= 0.0) || !(Om > 0.0) || !(OL >= 0.0) || !(H0 > 0.0) || !isfinite(Ok) || !isfinite(H0)) st |= ST_UNSUPPORTED;

    // --- big root as m = -Or * rho_big: m^4 - Om m^3 + Ok Or m^2 + OL Or^3 = 0, m ~ Om (Newton; m = Om when Or = 0)
    double disc = Om * Om - 4.0 * Or * Ok;
    double m = 0.5 * (Om + sqrt(fmax(disc, 0.0)));
    const double Or3OL = OL * Or * Or * Or, OkOr = Ok * Or;
    for (int it = 0; it < 4; ++it) {
        double f = fma(fma(m - Om, m, OkOr), m * m, Or3OL);
        double fp = fma(fma(4.0, m, -3.0 * Om), m, 2.0 * OkOr) * m;
        m -= f / fp;
    }
    // --- deflate: P = (Or x + m)(x^3 + c2 x^2 + c1 x + c0), finite as Or -> 0
    const double c0 = OL / m;
    const double c1 = -Or * c0 / m;
    const double c2 = (Ok - Or * c1) / m;
    // --- the non-positive real root rn of the cubic: closed form, then Newton on the cubic
    double rn;
    {
        const double p = c1 - c2 * c2 * (1.0 / 3.0);
        const double q = c2 * c2 * c2 * (2.0 / 27.0) - c2 * c1 * (1.0 / 3.0) + c0;
        const double D = 0.25 * q * q + p * p * p * (1.0 / 27.0);
        double t;
        if (D > 0.0) {
            double A = -copysign(cbrt(0.5 * fabs(q) + sqrt(D)), q);
            t = (A != 0.0) ? A - p / (3.0 * A) : 0.0;
        } else {
            double r = 2.0 * sqrt(fmax(-p * (1.0 / 3.0), 0.0));
            double arg = (r > 0.0) ? 3.0 * q / (p * r) : 1.0;
            arg = fmin(1.0, fmax(-1.0, arg));
            double phi = acos(arg) * (1.0 / 3.0);
            const double TWO_PI_3 = 2.0943951023931954923;
            double t0 = r * cos(phi), t1 = r * cos(phi - TWO_PI_3), t2 = r * cos(phi - 2.0 * TWO_PI_3);
            t = fmin(t0, fmin(t1, t2));
        }
        rn = t - c2 * (1.0 / 3.0);
        for (int it = 0; it < 3; ++it) {
            double Cv = fma(fma(rn + c2, rn, c1), rn, c0);
            double Cp = fma(fma(3.0, rn, 2.0 * c2), rn, c1);
            if (Cp != 0.0) rn -= Cv / Cp;
        }
    }
    double b = c2 + rn;
    double c = fma(rn, b, c1);
    // --- Bairstow polish of (b, c) on the ORIGINAL polynomial (coefficients span orders of magnitude)
    for (int it = 0; it < 2; ++it) {
        double q2 = Or, q1 = Om - b * q2, q0 = Ok - b * q1 - c * q2;
        double r1 = -b * q0 - c * q1, r0 = OL - c * q0;
        double s1 = q1 - b * q2, s0 = q0 - c * q2;
        double u1 = s0 - b * s1, u0 = -c * s1;
        double det = u1 * s0 - u0 * s1;
        if (det != 0.0 && isfinite(det)) {
            b += (r1 * s0 - r0 * s1) / det;
            c += (u1 * r0 - u0 * r1) / det;
        }
    }
    // re-derive (m, rn) from the polished pair: quotient P / (x^2 + b x + c) = Or x^2 + g1 x + h1
    {
        double g1 = Om - b * Or, h1 = Ok - b * g1 - c * Or;
        // (Or x + m)(x - rn): g1 = m - Or rn, h1 = -m rn.  One Newton step on (m, rn) keeps them consistent.
        double F1 = (m - Or * rn) - g1, F2 = (-m * rn) - h1;
        // J = [[1, -Or], [-rn, -m]]
        double det = -m - Or * rn;
        if (det != 0.0) {
            double dm = (F1 * (-m) - (-Or) * F2) / det;
            double dr = (1.0 * F2 - (-rn) * F1) / det;
            m -= dm; rn -= dr;
        }
    }
    // factorisation check: coefficients of the product against (Or, Om, Ok, 0, OL)
    {
        double g1 = m - Or * rn, h1 = -m * rn;
        double e3 = Or * b + g1, e2 = Or * c + g1 * b + h1, e1 = g1 * c + h1 * b, e0 = h1 * c;
        double scale = fabs(Om) + fabs(Ok) + fabs(OL) + fabs(Or);
        double res = fabs(e3 - Om) + fabs(e2 - Ok) + fabs(e1) + fabs(e0 - OL);
        if (!(res <= 1e-9 * scale) || !(m > 0.0) || !(rn <= 1e-12)) st |= ST_UNSUPPORTED;   // also catches NaN
    }
    // --- no real negative root (two complex pairs): factor P = (Or x^2 + g1 x + h1)(x^2 + b x + c) by Bairstow from the
    // small pair x^2 ~ -OL/Ok; such rows are evaluated by the complex slow path of cosmo_c4.cuh (C.m, C.rn carry g1, h1)
    if ((st & ST_UNSUPPORTED) && Or > 0.0 && Om > 0.0 && OL >= 0.0 && H0 > 0.0 && Ok > 0.0 && isfinite(Ok)) {
        double bb = 0.0, cc = OL / Ok;
        for (int it = 0; it < 12; ++it) {
            double q2 = Or, q1 = Om - bb * q2, q0 = Ok - bb * q1 - cc * q2;
            double r1 = -bb * q0 - cc * q1, r0 = OL - cc * q0;
            double s1 = q1 - bb * q2, s0 = q0 - cc * q2;
            double u1 = s0 - bb * s1, u0 = -cc * s1;
            double det = u1 * s0 - u0 * s1;
            if (det == 0.0 || !isfinite(det)) break;
            bb += (r1 * s0 - r0 * s1) / det;
            cc += (u1 * r0 - u0 * r1) / det;
        }
        const double g1 = Om - bb * Or, h1 = Ok - bb * g1 - cc * Or;
        const double e1 = g1 * cc + h1 * bb, e0 = h1 * cc;
        const double scale = fabs(Om) + fabs(Ok) + fabs(OL) + fabs(Or);
        if (fabs(e1) + fabs(e0 - OL) <= 1e-9 * scale && 4.0 * Or * h1 - g1 * g1 > 0.0 && 4.0 * cc - bb * bb > 0.0) {
            st &= ~ST_UNSUPPORTED;
            C.cubic |= 2u;
            m = g1; rn = h1; b = bb; c = cc;
        }
    }
    C.m = m; C.rn = rn; C.b = b; C.c = c;
    // --- per-cosmology constants (S3)
    const double f1 = Or, g1 = m - Or * rn, h1 = -m * rn;
    C.q11 = (Or + m) * (1.0 - rn);
    C.q21 = 1.0 + b + c;
    const double D1r = m + Or * rn;              // sqrt(disc Q1)
    const double D2 = b * b - 4.0 * c;           // disc Q2: < 0 complex-conjugate pair, > 0 real pair
    C.sD = 0.25 * D1r * D1r * D2;
    C.sDr = sqrt(fabs(C.sD));
    C.theta = 2.0 * f1 * c + 2.0 * h1 - g1 * b;
    C.W = fma(Or, fma(Or, c, -b * m), m * m);
    C.kf = (Or + m) / (1.0 - rn);
    C.ck = sqrt(C.kf / C.q21);
    // validity: a real root of E^2 in (1, 1+z] -- only the pair can sit there
    C.xlim = INFINITY;
    if (D2 >= 0.0 && -0.5 * b > 1.0) {
        double sq = sqrt(D2);
        C.xlim = (b < 0.0) ? c / (0.5 * (-b + sq)) : 0.5 * (-b - sq);   // smaller root, cancellation-free
    }
    if (!(C.q21 > 0.0)) st |= ST_UNSUPPORTED;
    // lookback time constants
    C.p5c = rn * C.W / m;
    C.Gp = D1r * C.W / (m * m);
    C.qhc = m * m / (Or + m);
    C.OrM = Or / m;
    // absorption distance constants
    C.Q2n = fma(rn + b, rn, c);
    C.mOrn = D1r;
    C.C1 = (1.0 - rn) * C.q21;
    C.F1 = sqrt(C.C1 / (Or + m));
    C.iOm = 1.0 / Om;
    if (C.cubic & 1u) {
        C.aF = 3.0 * rn * rn - C.Q2n;
        C.sig = -Ok / Om;                 // sum of the three roots
        C.WoOr = 0.0;
    } else {
        C.aF = 2.0 * rn * rn - C.Q2n;
        C.sig = -Om / Or;                 // sum of the four roots (Vieta)
        C.WoOr = C.W / Or;
    }
    C.status = st;
    if (!want_grad) return;

    // --- gradient basis coefficients: polynomial identities in x, solved per cosmology
    const double e[5] = {OL, 0.0, Ok, Om, Or};
    const double NK[5] = {m * m * c, m * m * b + 2.0 * Or * m * c, m * m + 2.0 * Or * m * b + Or * Or * c,
                          2.0 * Or * m + Or * Or * b, Or * Or};
    {   // I0 and T share the 5x5 matrix: columns E^2, N_K, N_0, N_1, N_2 ; rhs: 3 for I0 then 3 for T
        double M[5][5 + 6];
        for (int r = 0; r < 5; ++r) for (int k = 0; k < 11; ++k) M[r][k] = 0.0;
        for (int p = 0; p < 5; ++p) { M[p][0] = e[p]; M[p][1] = NK[p]; }
        add_Nk(M, 2, 0, e); add_Nk(M, 3, 1, e); add_Nk(M, 4, 2, e);
        // D_theta = dE^2/dtheta with Ok eliminated: x^3 - x^2, 1 - x^2, x^4 - x^2
        M[3][5] = 1.0; M[2][5] = -1.0;
        M[0][6] = 1.0; M[2][6] = -1.0;
        M[4][7] = 1.0; M[2][7] = -1.0;
        // T: D_theta / x - aT E^2 / x with aT = D_theta(0)/OL (the 1/x pole goes to the forward T)
        const double aT[3] = {0.0, 1.0 / OL, 0.0};
        M[2][8] = 1.0; M[1][8] = -1.0;                       // x^2 - x
        M[1][9] = -1.0;                                      // (1 - x^2)/x = 1/x - x
        M[3][10] = 1.0; M[1][10] = -1.0;                     // x^3 - x
        for (int p = 1; p < 5; ++p) M[p - 1][9] -= aT[1] * e[p];
        solve_aug<5, 6>(M);
        for (int t = 0; t < 3; ++t) {
            for (int j = 0; j < 5; ++j) { C.GI[t][j] = M[j][5 + t]; C.GT[t][j] = M[j][8 + t]; }
            C.GT[t][5] = aT[t];
        }
    }
    if (want_grad < 2) return;
    {   // A: x^2 D_theta over columns E^2, N_K, N_0, N_1, N_2, N_3 (N_4 when Or = 0), x^2 E^2
        double M[7][7 + 3];
        for (int r = 0; r < 7; ++r) for (int k = 0; k < 10; ++k) M[r][k] = 0.0;
        for (int p = 0; p < 5; ++p) { M[p][0] = e[p]; M[p][1] = NK[p]; M[p + 2][6] = e[p]; }
        add_Nk(M, 2, 0, e); add_Nk(M, 3, 1, e); add_Nk(M, 4, 2, e); add_Nk(M, 5, (C.cubic & 1u) ? 4 : 3, e);
        M[5][7] = 1.0; M[4][7] = -1.0;
        M[2][8] = 1.0; M[4][8] = -1.0;
        M[6][9] = 1.0; M[4][9] = -1.0;
        solve_aug<7, 3>(M);
        for (int t = 0; t < 3; ++t) for (int j = 0; j < 7; ++j) C.GA[t][j] = M[j][7 + t];
    }
}

}  // namespace cb
