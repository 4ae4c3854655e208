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

// S1-S2: coefficients, validity, root solve.  Fills Om, OL, Or, Ok, H0, dH, tH, the factorisation (m, rn, b, c), status and the
// structure bits 0, 1 of C.cubic; cosmo_constants() derives everything else from these.
CB_HD void cosmo_factor(double Om, double OL, double Or, double H0, Cosmo<double>& C) {
    const double Ok = 1.0 - Om - OL - Or;
    C.Om = Om; C.OL = OL; C.Or = Or; C.Ok = Ok; C.H0 = H0;
    { const double iH = cb_rcp(H0); C.dH = C_KM_S * iH; C.tH = HUBBLE_GYR * iH; }
    C.cubic = (Or == 0.0);
    unsigned st = 0;
    // the method needs degree 3 or 4 and non-negative densities (include/cosmo_b200.h)
    if (!(Or >= 0.0) || !(Om > 0.0) || !(OL >= 0.0) || !(H0 > 0.0) || !isfinite(Ok) || !isfinite(H0)) st |= ST_UNSUPPORTED;

    // --- big root as m = -Or * rho_big: m^4 - Om m^3 + Ok Or m^2 + OL Or^3 = 0, m ~ Om (Newton; m = Om when Or = 0)
    double disc = Om * Om - 4.0 * Or * Ok;
    double m = 0.5 * (Om + cb_sqrt0(fmax(disc, 0.0)));
    const double Or3OL = OL * Or * Or * Or, OkOr = Ok * Or;
    for (int it = 0; it < 4; ++it) {
        double f = fma(fma(m - Om, m, OkOr), m * m, Or3OL);
        double fp = fma(fma(4.0, m, -3.0 * Om), m, 2.0 * OkOr) * m;
        m -= cb_div(f, fp);
    }
    // --- deflate: P = (Or x + m)(x^3 + c2 x^2 + c1 x + c0), finite as Or -> 0
    const double im = cb_rcp(m);
    const double c0 = OL * im;
    const double c1 = -Or * c0 * im;
    const double c2 = (Ok - Or * c1) * im;
    // --- the non-positive real root rn of the cubic: closed form, then Newton on the cubic
    double rn;
    {
        const double p = c1 - c2 * c2 * (1.0 / 3.0);
        const double q = c2 * c2 * c2 * (2.0 / 27.0) - c2 * c1 * (1.0 / 3.0) + c0;
        const double D = 0.25 * q * q + p * p * p * (1.0 / 27.0);
        double t;
        if (D > 0.0) {
            double A = -copysign(cbrt(0.5 * fabs(q) + cb_sqrt0(D)), q);
            t = (A != 0.0) ? A - cb_div(p, 3.0 * A) : 0.0;
        } else {
            double r = 2.0 * cb_sqrt0(fmax(-p * (1.0 / 3.0), 0.0));
            double arg = (r > 0.0) ? cb_div(3.0 * q, p * r) : 1.0;
            arg = fmin(1.0, fmax(-1.0, arg));
            double phi = acos(arg) * (1.0 / 3.0);
            const double TWO_PI_3 = 2.0943951023931954923;
            t = r * cos(phi - 2.0 * TWO_PI_3);       // the smallest of the three real roots: phi in [0, pi/3]
        }
        rn = t - c2 * (1.0 / 3.0);
        // OL = 0 exactly: x = 0 is a root (double when Or = 0) and the closed form, at its discriminant's zero, may return the
        // simple positive root of a closed matter model instead
        if (c0 == 0.0) rn = 0.0;
        for (int it = 0; it < 3; ++it) {
            double Cv = fma(fma(rn + c2, rn, c1), rn, c0);
            double Cp = fma(fma(3.0, rn, 2.0 * c2), rn, c1);
            if (Cp != 0.0) rn -= cb_div(Cv, Cp);
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
            const double idt = cb_rcp(det);
            b += (r1 * s0 - r0 * s1) * idt;
            c += (u1 * r0 - u0 * r1) * idt;
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
            const double idt = cb_rcp(det);
            double dm = (F1 * (-m) - (-Or) * F2) * idt;
            double dr = (1.0 * F2 - (-rn) * F1) * idt;
            m -= dm; rn -= dr;
        }
    }
    // factorisation check: coefficients of the product against (Or, Om, Ok, 0, OL)
    {
        double g1 = m - Or * rn, h1 = -m * rn;
        double e3 = Or * b + g1, e2 = Or * c + g1 * b + h1, e1 = g1 * c + h1 * b, e0 = h1 * c;
        double scale = fabs(Om) + fabs(Ok) + fabs(OL) + fabs(Or);
        double res = fabs(e3 - Om) + fabs(e2 - Ok) + fabs(e1) + fabs(e0 - OL);
        if (!(res <= 1e-13 * scale) || !(m > 0.0) || !(rn <= 1e-12)) st |= ST_UNSUPPORTED;   // also catches NaN
    }
    // --- the labelled solve failed (the two negative roots nearly coincide, or there is no real negative root at all): factor
    // P = (Or x^2 + g1 x + h1)(x^2 + b x + c) by Bairstow.  Starts: the small pair x^2 ~ -OL/Ok (Ok > 0), the quadratic the failed solve
    // ended with, and the pair of Or x^4 + OL = 0 with positive real part (large Or); the first that reproduces the coefficients is
    // classified: two negative real roots in one factor -> the real labelling (m, rn from that factor); two complex pairs -> the
    // complex slow path of cosmo_c4.cuh (C.m, C.rn carry g1, h1).
    if ((st & ST_UNSUPPORTED) && Or > 0.0 && Om > 0.0 && OL >= 0.0 && H0 > 0.0 && isfinite(Ok) && isfinite(H0)) {
        const double rho2 = sqrt(OL / Or);
        const double sb[3] = {0.0, b, -sqrt(2.0 * rho2)}, sc[3] = {OL / Ok, c, rho2};
        for (int start = (Ok > 0.0 ? 0 : 1); start < 3 && (st & ST_UNSUPPORTED); ++start) {
            double bb = sb[start], cc = sc[start];
            if (!isfinite(bb) || !isfinite(cc)) continue;
            for (int it = 0; it < 24; ++it) {
                double q2 = Or, q1 = Om - bb * q2, q0 = Ok - bb * q1 - cc * q2;
                double r1 = -bb * q0 - cc * q1, r0 = OL - cc * q0;
                double s1 = q1 - bb * q2, s0 = q0 - cc * q2;
                double u1 = s0 - bb * s1, u0 = -cc * s1;
                double det = u1 * s0 - u0 * s1;
                if (det == 0.0 || !isfinite(det)) break;
                bb += (r1 * s0 - r0 * s1) / det;
                cc += (u1 * r0 - u0 * r1) / det;
            }
            double g1 = Om - bb * Or, h1 = Ok - bb * g1 - cc * Or;
            const double e1 = g1 * cc + h1 * bb, e0 = h1 * cc;
            const double scale = fabs(Om) + fabs(Ok) + fabs(OL) + fabs(Or);
            if (!(fabs(e1) + fabs(e0 - OL) <= 1e-13 * scale)) continue;
            double d1 = g1 * g1 - 4.0 * Or * h1, d2 = bb * bb - 4.0 * cc;
            // OL = 0 with a complex pair: E^2 = x^2 (Or x^2 + Om x + Ok).  The real labelling would need Q1 = Or x x, i.e. m = 0 (its
            // formulae divide by m); the complex slow path takes the double root at 0 as its second "pair" (r3 = r4 = 0) as it stands:
            // it is the limit OL -> 0+ of the two-complex-pairs structure, where the small pair is +- i sqrt(OL/Ok)
            if (bb == 0.0 && cc == 0.0 && d1 < 0.0) {
                st &= ~ST_UNSUPPORTED;
                C.cubic |= 2u;
                m = g1; rn = h1; b = 0.0; c = 0.0;
                break;
            }
            // a factor with two non-positive real roots becomes Q1 = (Or x + m)(x - rn)
            if (d2 >= 0.0 && bb >= 0.0 && cc >= 0.0 && !(d1 >= 0.0 && g1 >= 0.0 && h1 >= 0.0)) {
                const double tb = g1 / Or, tc = h1 / Or;
                g1 = Or * bb; h1 = Or * cc; bb = tb; cc = tc;
                d1 = g1 * g1 - 4.0 * Or * h1; d2 = bb * bb - 4.0 * cc;
            }
            if (d1 >= 0.0 && g1 >= 0.0 && h1 >= 0.0) {
                const double sq = sqrt(d1);
                m = 0.5 * (g1 + sq);
                rn = -h1 / m;
                b = bb; c = cc;
                st &= ~ST_UNSUPPORTED;
            } else if (d1 < 0.0 && d2 < 0.0) {
                // Q1 takes the pair further to the left (the counterpart of {big, neg} on the real path: r_i of eqs. (3.8)/(3.9),
                // PAPER.md:225 "biggest roots"), Q2 the other one
                if (bb * Or > g1) { const double tb = g1 / Or, tc = h1 / Or; g1 = Or * bb; h1 = Or * cc; bb = tb; cc = tc; }
                st &= ~ST_UNSUPPORTED;
                C.cubic |= 2u;
                m = g1; rn = h1; b = bb; c = cc;
            }
        }
    }
    C.m = m; C.rn = rn; C.b = b; C.c = c;
    C.status = st;
}

// S3: the per-cosmology constants of eqs. (3.7)-(3.9) from the factorisation (cheap: a few divisions and square roots, so the
// ELEMENTWISE kernels can afford to form them again after the duplication loop instead of keeping them in registers across it)
CB_HD void cosmo_constants(Cosmo<double>& C) {
    const double Om = C.Om, OL = C.OL, Or = C.Or, Ok = C.Ok, m = C.m, rn = C.rn, b = C.b, c = C.c;
    unsigned st = C.status;
    const double f1 = Or, g1 = m - Or * rn, h1 = -m * rn;
    C.q11 = (Or + m) * (1.0 - rn);
    C.q21 = 1.0 + b + c;
    const double D1r = m + Or * rn;              // sqrt(disc Q1)
    const double D2 = b * b - 4.0 * c;           // disc Q2: < 0 complex-conjugate pair, > 0 real pair
    C.sD = 0.25 * D1r * D1r * D2;
    C.sDr = cb_sqrt0(fabs(C.sD));
    C.theta = 2.0 * f1 * c + 2.0 * h1 - g1 * b;
    C.W = fma(Or, fma(Or, c, -b * m), m * m);
    C.kf = cb_div(Or + m, 1.0 - rn);
    C.ck = cb_sqrt0(cb_div(C.kf, C.q21));
    // validity: a real root of E^2 in (1, 1+z] -- only the pair can sit there
    C.xlim = INFINITY;
    if (D2 >= 0.0 && -0.5 * b > 1.0) {
        double sq = sqrt(D2);
        C.xlim = (b < 0.0) ? c / (0.5 * (-b + sq)) : 0.5 * (-b - sq);   // smaller root, cancellation-free
    }
    if (!(C.q21 > 0.0)) st |= ST_UNSUPPORTED;
    // lookback time constants
    const double im = cb_rcp(m), iOrm = cb_rcp(Or + m);
    C.p5c = rn * C.W * im;
    C.Gp = D1r * C.W * (im * im);
    C.qhc = m * m * iOrm;
    C.OrM = Or * im;
    // absorption distance constants
    C.Q2n = fma(rn + b, rn, c);
    C.mOrn = D1r;
    C.C1 = (1.0 - rn) * C.q21;
    C.F1 = cb_sqrt0(C.C1 * iOrm);
    C.iOm = cb_rcp(Om);
    if (C.cubic & 1u) {
        C.aF = 3.0 * rn * rn - C.Q2n;
        C.sig = -Ok * C.iOm;              // sum of the three roots
        C.WoOr = 0.0;
    } else {
        C.aF = 2.0 * rn * rn - C.Q2n;
        const double iOr = cb_rcp(Or);
        C.sig = -Om * iOr;                // sum of the four roots (Vieta)
        C.WoOr = C.W * iOr;
    }
    C.status = st;
}

// The per-cosmology block again, from its few defining numbers (ELEMENTWISE kernels, after the duplication loop): the values pass
// through an empty asm statement, so the compiler has to form the derived constants anew here instead of carrying ~30 of them in
// registers (or local memory) across the loop.
CB_HD double cb_launder(double v) {
#ifdef __CUDA_ARCH__
    asm volatile("" : "+d"(v));
#endif
    return v;
}
template <typename T>
CB_HD void cosmo_reconstitute(const Cosmo<T>& C, Cosmo<double>& D) {
    D.Om = cb_launder((double)C.Om); D.OL = cb_launder((double)C.OL); D.Or = cb_launder((double)C.Or);
    D.Ok = 1.0 - D.Om - D.OL - D.Or;
    D.H0 = 0.0;                                   // not used after the loop: dH, tH are
    D.dH = cb_launder((double)C.dH); D.tH = cb_launder((double)C.tH);
    D.m = cb_launder((double)C.m); D.rn = cb_launder((double)C.rn); D.b = cb_launder((double)C.b); D.c = cb_launder((double)C.c);
    D.status = C.status; D.cubic = C.cubic;
    cosmo_constants(D);
    D.Tinf = (double)C.Tinf; D.dTinf[0] = (double)C.dTinf[0]; D.dTinf[1] = (double)C.dTinf[1]; D.dTinf[2] = (double)C.dTinf[2];
}

// Gradient bases: polynomial identities in x, solved per cosmology.  For a polynomial D(x) of degree <= 4,
//   int D / E^3 dx = a I0 + bK K + c0 b_0 + c1 b_1 + c2 b_2,     b_k = [x^k / E] between the limits,
// where (a, bK, c0, c1, c2) multiply the columns E^2, N_K, N_0, N_1, N_2 (N_k = k x^(k-1) E^2 - x^k (E^2)'/2) and solve the 5x5
// system whose rows are the powers x^0..x^4.  With e = (OL, 0, Ok, Om, Or):
//   x^0: e0 a + NK0 bK            + e0 c1             = D0
//   x^1:        NK1 bK - e2 c0             + 2 e0 c2  = D1
//   x^2: e2 a + NK2 bK - 1.5 e3 c0                    = D2     <- pivot on Om (> 0): c0
//   x^3: e3 a + NK3 bK - 2 e4 c0 - 0.5 e3 c1 + e2 c2  = D3
//   x^4: e4 a + NK4 bK           - e4 c1   + 0.5 e3 c2 = D4    <- pivot on Om: c2
// Eliminating c0 and c2 leaves a 3x3 system in (a, bK, c1), solved by its adjugate: no pivot search, no indexed storage, so the
// solver (16 numbers) and every row it produces stay in registers.  k_prep stores the rows the OUTER kernels need in Cosmo<T>; the
// ELEMENTWISE kernels, with one cosmology per element, produce each row right where it is consumed (cosmo_obs.cuh, grad_basis).
struct GradSolve {
    double e0, e2, e3, e4, k0, k2, al0, be0, al2, be2, de2;
    double i00, i01, i02, i10, i11, i12, i20, i21, i22;
    bool cubic, singular;

    CB_HD void init(const Cosmo<double>& C) {
        const double Or = C.Or, m = C.m, rn = C.rn, b = C.b, c = C.c;
        e0 = C.OL; e2 = C.Ok; e3 = C.Om; e4 = Or;
        cubic = (C.cubic & 1u) != 0;
        // N_K = P_K(x) (x^2 + b x + c).  Real labelling: P_K = (Or x + m)^2 (the [p_n = -3] integral of the root rn).  Two complex
        // pairs (C.m, C.rn carry g1, h1 of Q1 = Or x^2 + g1 x + h1 with roots r1 = conj(r2)): P_K = Or^2 Re (x - r1)^2
        // = Or^2 x^2 + Or g1 x + g1^2/2 - Or h1, the real part of Carlson's [+1, -3] integral of the pair (cosmo_c4.cuh).
        const bool c4 = (C.cubic & 2u) != 0;
        const double pk2 = Or * Or, pk1 = c4 ? Or * m : 2.0 * Or * m, pk0 = c4 ? 0.5 * m * m - Or * rn : m * m;
        const double NK0 = pk0 * c, NK1 = pk0 * b + pk1 * c, NK2 = pk0 + pk1 * b + pk2 * c, NK3 = pk1 + pk2 * b, NK4 = pk2;
        k2 = 2.0 * cb_rcp(e3); k0 = k2 * (1.0 / 3.0);
        al0 = e2 * k0; be0 = NK2 * k0;                              // c0 = al0 a + be0 bK - k0 D2
        al2 = -e4 * k2; be2 = -NK4 * k2; de2 = e4 * k2;             // c2 = al2 a + be2 bK + de2 c1 + k2 D4
        // 3x3 rows: (x^0), (x^1), (x^3)
        const double m00 = e0, m01 = NK0, m02 = e0;
        const double m10 = -e2 * al0 + 2.0 * e0 * al2, m11 = NK1 - e2 * be0 + 2.0 * e0 * be2, m12 = 2.0 * e0 * de2;
        const double m20 = e3 - 2.0 * e4 * al0 + e2 * al2, m21 = NK3 - 2.0 * e4 * be0 + e2 * be2, m22 = -0.5 * e3 + e2 * de2;
        const double c00 = m11 * m22 - m12 * m21, c01 = m12 * m20 - m10 * m22, c02 = m10 * m21 - m11 * m20;
        const double det = m00 * c00 + m01 * c01 + m02 * c02;
        const double idet = (det != 0.0) ? cb_rcp(det) : INFINITY;
        i00 = c00 * idet; i01 = (m02 * m21 - m01 * m22) * idet; i02 = (m01 * m12 - m02 * m11) * idet;
        i10 = c01 * idet; i11 = (m00 * m22 - m02 * m20) * idet; i12 = (m02 * m10 - m00 * m12) * idet;
        i20 = c02 * idet; i21 = (m01 * m20 - m00 * m21) * idet; i22 = (m00 * m11 - m01 * m10) * idet;
        // The bases become linearly dependent as the gap g of the pair x^2 + b x + c closes (the 1/prod(r_j - r_k) of appendix A,
        // PAPER.md:320-345; OL -> 0 is the commonest way there: the pair tends to +-sqrt(-OL/Ok) and at OL = 0 the system is singular).
        // The per-element cancellation factor (grad_basis) decides where they are still accurate; a singular system is marked here.
        singular = !isfinite(idet);
    }
    // coefficients (a, bK, c0, c1, c2) of the polynomial D0 + D1 x + .. + D4 x^4
    CB_HD void solve5(double D0, double D1, double D2, double D3, double D4, double* out5) const {
        const double g0 = -k0 * D2, g2 = k2 * D4;
        const double r0 = D0, r1 = D1 + e2 * g0 - 2.0 * e0 * g2, r2 = D3 + 2.0 * e4 * g0 - e2 * g2;
        const double av = i00 * r0 + i01 * r1 + i02 * r2;
        const double bv = i10 * r0 + i11 * r1 + i12 * r2;
        const double c1v = i20 * r0 + i21 * r1 + i22 * r2;
        out5[0] = av; out5[1] = bv;
        out5[2] = al0 * av + be0 * bv + g0;
        out5[3] = c1v;
        out5[4] = al2 * av + be2 * bv + de2 * c1v + g2;
    }
    // X = I0: D_theta = dE^2/dtheta with Ok eliminated: x^3 - x^2, 1 - x^2, x^4 - x^2 (theta = Om, OL, Or); basis (I0, K, b0, b1, b2)
    CB_HD void rowI(int t, double* g5) const { solve5(t == 1 ? 1.0 : 0.0, 0.0, -1.0, t == 0 ? 1.0 : 0.0, t == 2 ? 1.0 : 0.0, g5); }
    // X = T: D_theta / x - aT E^2 / x with aT = D_theta(0)/OL (the 1/x pole goes to the forward T): x^2 - x, 1/x - x, x^3 - x;
    // basis (I0, K, b0, b1, b2, T)
    CB_HD void rowT(int t, double* g6) const {
        const double aT = (t == 1) ? 1.0 / e0 : 0.0;
        if (t == 1) solve5(0.0, -1.0 - aT * e2, -aT * e3, -aT * e4, 0.0, g6);
        else solve5(0.0, -1.0, t == 0 ? 1.0 : 0.0, t == 2 ? 1.0 : 0.0, 0.0, g6);
        g6[5] = aT;
    }
    // the monomials themselves: J'_p = int x^p dx / E^3 (p = 0..4), used by the perturbative d_abs gradient
    CB_HD void rowJ(int p, double* g5) const { solve5(p == 0, p == 1, p == 2, p == 3, p == 4, g5); }
    // X = A: x^2 D_theta (x^5 - x^4, x^2 - x^4, x^6 - x^4) over the five columns above plus N_3 (N_4 when Or = 0) and x^2 E^2.
    // The rows x^5, x^6 involve only those two extra unknowns (c3, aA); their columns then move to the right-hand side
    // of the same 5x5 system.  Basis (I0, K, b0, b1, b2, b3 (b4 when Or = 0), A).
    CB_HD void rowA(int t, double* g7) const {
        const double D5 = (t == 0) ? 1.0 : 0.0, D6 = (t == 2) ? 1.0 : 0.0;
        double c3, aA, n2, n3, n4;
        if (cubic) {                // N_4 = (0,0,0,4 e0,0 | 3 e2, 2.5 e3);  x^2 E^2 = (0,0,e0,0,e2 | e3, 0)
            const double ie3 = 0.5 * k2;
            c3 = D6 * (0.4 * ie3);
            aA = (D5 - 3.0 * e2 * c3) * ie3;
            n2 = 0.0; n3 = 4.0 * e0; n4 = 0.0;
        } else {                    // N_3 = (0,0,3 e0,0,2 e2 | 1.5 e3, e4);  x^2 E^2 = (0,0,e0,0,e2 | e3, e4)
            const double id = cb_rcp(0.5 * e3 * e4);
            c3 = (D5 * e4 - e3 * D6) * id;
            aA = (1.5 * e3 * D6 - e4 * D5) * id;
            n2 = 3.0 * e0; n3 = 0.0; n4 = 2.0 * e2;
        }
        const double D2 = ((t == 1) ? 1.0 : 0.0) - c3 * n2 - aA * e0;
        const double D3 = -c3 * n3;
        const double D4 = -1.0 - c3 * n4 - aA * e2;
        solve5(0.0, 0.0, D2, D3, D4, g7);
        g7[5] = c3;
        g7[6] = aA;
    }
};

// S1-S3 with the stored gradient bases of the OUTER kernels.  want_grad: 0 none, 1 chi-family (GI, GT), 2 all (+ GJ, GA).
CB_HD void cosmo_prep(double Om, double OL, double Or, double H0, int want_grad, Cosmo<double>& C) {
    cosmo_factor(Om, OL, Or, H0, C);
    cosmo_constants(C);
    if (!want_grad) return;
    GradSolve G;
    G.init(C);
    if (G.singular) C.cubic |= 4u;      // bit 2: quadrature for every element (not in C.status: that would stop the duplication loop)
    for (int t = 0; t < 3; ++t) G.rowI(t, C.GI[t]);
    {   // screening for the OUTER kernels, which run the chi-family bases unchecked: at small z the basis values are ~ (1, kf, E'(1),
        // 1 - E'(1), 2 - E'(1)) x I0 and the result is compared with >= 1e-3 I0, so 1e3 sum_j |G_j| w_j bounds the cancellation factor
        // there (it falls with z).  Above the limit the cosmology takes the checked row (bit 3).
        double gmax = 0.0;
        for (int t = 0; t < 3; ++t) {
            const double g = fabs(C.GI[t][0]) + fabs(C.GI[t][1]) * fabs(C.kf) + 2.0 * (fabs(C.GI[t][2]) + fabs(C.GI[t][3]) + fabs(C.GI[t][4]));
            gmax = (g > gmax || !(g == g)) ? g : gmax;
        }
        if (!(1.0e3 * gmax <= GRAD_COND_LIMIT)) C.cubic |= 8u | (isfinite(gmax) ? 0u : 4u);
    }
    for (int t = 0; t < 3; ++t) G.rowT(t, C.GT[t]);
    if (want_grad < 2) return;
    for (int p = 0; p < 5; ++p) G.rowJ(p, C.GJ[p]);
    for (int t = 0; t < 3; ++t) G.rowA(t, C.GA[t]);
}

}  // namespace cb
