// cosmo_obs.cuh -- hot-path steps S7 (observables) and S8 (fused backward, no tape) for one element.
//
// S7: D_C = d_H I0, D_M = d_H sinn, D_L = (1+z) D_M, mu = 5 log10(D_L / 10 pc), t_L = T / H0, d_abs = d_H A
//     (PAPER.md:88-95, :277 fn.22; readings R-units, R-sinn).
// S8: d/dz = integrand at z; d/dH0 analytic; d/d(Om, OL, Or) with Ok eliminated from the SAME
//     forward intermediates (I0, K, T, A and boundary terms), DESIGN.md "Gradients" (replaces the tape of
//     eqs. (2.10)-(2.12) + appendix A, by their closed combination).
#pragma once
#include "cosmo_eval.cuh"
#include "cosmo_c4.cuh"

namespace cb {

template <typename T>
struct Obs {
    T v[N_PLANES];     // DC, DM, DL, MU, TL, DABS, DA, VC, AGE
    T F, Fi, Fk;       // curvature transform and its partials
    T Vk;              // d(V_C / (4 pi dH^3)) / dOk at fixed I0 (W_VC only)
    unsigned status;
};

// Rows whose E^2 has no real negative root (Cosmo::cubic bit 1): replace the fused real path's result by the complex
// slow path (cosmo_c4.cuh), including K, E, 1/E and E - 1 in the meaning the gradient bases of such rows expect.
template <typename T, bool kT, bool kA, bool kGrad>
CB_HD void apply_c4(const Cosmo<T>& C, T z, Core<T>& R) {
    if (!(C.cubic & 2u)) return;
    double I0, TT, AA, KK;
    eval_c4((double)C.Or, (double)C.m, (double)C.rn, (double)C.b, (double)C.c, 1.0, 1.0 + (double)z, (double)z, kT, kA, I0, TT, AA, KK);
    R.I0 = (T)I0; R.TT = (T)TT; R.AA = (T)AA; R.K = (T)KK;
    {
        const double x = 1.0 + (double)z, xp1 = x + 1.0, c2 = fma(xp1, x, 1.0);
        const double Ev = sqrt(fma(fma((double)C.Or, x, (double)C.m), x, (double)C.rn) * fma(x + (double)C.b, x, (double)C.c));
        const double t = fma((double)C.Or, fma(c2, x, 1.0), fma((double)C.Om, c2, (double)C.Ok * xp1));     // (E^2 - 1)/z
        R.E = (T)Ev; R.iE = (T)(1.0 / Ev); R.Em1 = (T)((double)z * t / (Ev + 1.0));
    }
    R.status = C.status | ((T(1) + z > T(0)) ? 0u : (unsigned)ST_UNSUPPORTED);
}

// Comoving volume over the whole sky, V_C = 4 pi dH^3 v, v(k, I0) = int_0^{I0} F(k, I)^2 dI (ref. [59] eq. (13.60)):
//   v = I0^3 h(w), dv/dk = I0^5 h'(w), w = Ok I0^2, h = sum_{j>=1} 4^j w^(j-1) / (2 (2j+1)!)  (|w| <= 1), closed forms beyond;
//   dv/dI0 = F^2.
template <typename T>
CB_HD void volume_libm(T k, T I0, T& v, T& vk) {
    using N = Num<T>;
    if (k > T(0)) {
        const T sq = N::sqrt_(k), y2 = T(2) * sq * I0, ey = N::exp_(y2), iey = T(1) / ey;
        const T sh2 = T(0.5) * (ey - iey), ch2 = T(0.5) * (ey + iey);
        v = (sh2 / (T(2) * sq) - I0) / (T(2) * k);
        vk = (I0 * ch2 / (T(2) * k) - sh2 / (T(4) * k * sq)) / (T(2) * k) - v / k;
    } else {
        const T kk = -k, sq = N::sqrt_(kk);
        T sn2, cs2;
        N::sincos_(T(2) * sq * I0, &sn2, &cs2);
        v = (I0 - sn2 / (T(2) * sq)) / (T(2) * kk);
        vk = -((-(I0 * cs2 / (T(2) * kk) - sn2 / (T(4) * kk * sq))) / (T(2) * kk) - v / kk);
    }
}
template <typename T>
CB_HD void volume(T k, T I0, T& v, T& vk) {
    using N = Num<T>;
    const T w = k * I0 * I0;
    const T I3 = I0 * I0 * I0;
    if (N::abs_(w) <= T(1)) {
        // coefficients 4^j / (2 (2j+1)!), j = 1..12
        const double H[12] = {1.0 / 3.0, 1.0 / 15.0, 2.0 / 315.0, 1.0 / 2835.0, 2.0 / 155925.0, 2.0 / 6081075.0, 4.0 / 638512875.0,
                              1.0 / 10854718875.0, 2.0 / 1856156927625.0, 2.0 / 194896477400625.0, 4.0 / 49308808782358125.0,
                              2.0 / 3698160658676859375.0};
        T sh = T(H[11]), sd = T(11.0 * H[11]);
#pragma unroll
        for (int j = 10; j >= 0; --j) {
            sh = N::fma_(sh, w, T(H[j]));
            if (j >= 1) sd = N::fma_(sd, w, T(j * H[j]));
        }
        v = I3 * sh;
        vk = I3 * I0 * I0 * sd;
        return;
    }
    volume_libm<T>(k, I0, v, vk);
}

// K elements of the same cosmology at once.  The common case (|Ok I0^2| <= 1/2, D_L > 0) is straight-line code for all K
// elements -- one basic block, so that the K dependency chains (three Horner polynomials and the ln series each) interleave
// in the FP64 pipe; everything else goes through the generic per-element forms.
template <typename T, bool kT, bool kA, int K>
CB_HD void observables_k(const Cosmo<T>& C, const T (&z)[K], const Core<T> (&R)[K], unsigned which, Obs<T> (&O)[K]) {
    using N = Num<T>;
    // elements whose path crosses a root or leaves the domain: every plane is NaN.  One select on the integral poisons
    // everything derived from it (the other integrals are selected below), instead of one select per plane.
    T I0[K];
    bool bad[K];
    T wmax = T(0);
#pragma unroll
    for (int k = 0; k < K; ++k) {
        bad[k] = (R[k].status & (ST_ROOT_ON_PATH | ST_UNSUPPORTED)) != 0;
        I0[k] = bad[k] ? T(NAN) : R[k].I0;
        wmax = N::max_(wmax, N::abs_(C.Ok * I0[k] * I0[k]));
    }
    if (wmax <= T(0.5)) {
#pragma unroll
        for (int k = 0; k < K; ++k) {
            T sf, sg, sd;
            sinn_poly<T, 7>(C.Ok * I0[k] * I0[k], sf, sg, sd);
            O[k].F = I0[k] * sf; O[k].Fi = sg; O[k].Fk = I0[k] * I0[k] * I0[k] * sd;
        }
    } else if (wmax <= T(1)) {                 // same straight-line form at degree 10 (next term 1/23! ~ 4e-23)
#pragma unroll
        for (int k = 0; k < K; ++k) {
            T sf, sg, sd;
            sinn_poly<T, 10>(C.Ok * I0[k] * I0[k], sf, sg, sd);
            O[k].F = I0[k] * sf; O[k].Fi = sg; O[k].Fk = I0[k] * I0[k] * I0[k] * sd;
        }
    } else {
        for (int k = 0; k < K; ++k) sinn<T>(C.Ok, I0[k], O[k].F, O[k].Fi, O[k].Fk);
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const T x = T(1) + z[k];
        unsigned st = R[k].status;
        O[k].v[0] = C.dH * I0[k];
        O[k].v[1] = C.dH * O[k].F;
        O[k].v[2] = x * O[k].v[1];
        O[k].v[3] = T(0);
        if (which & W_MU) {
            const bool pos = O[k].v[2] > T(0);              // branch-free: ln of a harmless stand-in, then select
            const T mu = N::fma_(T(CB_KT.five_over_ln10), N::log_(pos ? O[k].v[2] : T(1)), T(25));
            O[k].v[3] = pos ? mu : T(NAN);
            st |= (pos || bad[k]) ? 0u : (unsigned)ST_DL_NONPOS;
        }
        const T TT = kT ? (bad[k] ? T(NAN) : R[k].TT) : T(0);
        O[k].v[4] = C.tH * TT;
        O[k].v[5] = kA ? C.dH * (bad[k] ? T(NAN) : R[k].AA) : T(0);
        O[k].v[6] = O[k].v[7] = O[k].v[8] = T(0);
        O[k].Vk = T(0);
        if (which & W_DA) O[k].v[6] = O[k].v[1] / x;
        if (which & W_VC) {
            T v;
            volume<T>(C.Ok, I0[k], v, O[k].Vk);
            O[k].v[7] = T(12.566370614359172954) * C.dH * C.dH * C.dH * v;
        }
        if (kT && (which & W_AGE)) {
            O[k].v[8] = C.tH * (C.Tinf - TT);
            // the age's parameter gradient needs the T-basis at x -> infinity (prep_age): not available where that basis is singular
            if (!(C.dTinf[0] == C.dTinf[0]) && !bad[k]) st |= ST_GRAD_ILLCOND;
        }
        O[k].status = st;
    }
}

template <typename T, bool kT, bool kA>
CB_HD void observables(const Cosmo<T>& C, T z, const Core<T>& R, unsigned which, Obs<T>& O) {
    const T zz[1] = {z};
    const Core<T> RR[1] = {R};
    Obs<T> OO[1];
    observables_k<T, kT, kA, 1>(C, zz, RR, which, OO);
    O = OO[0];
}

// Age (int_z^inf of eq. (2.4)): age(z) = tH (Tinf - T(z)).  Tinf = int_1^inf dx/(x E) is one more evaluation of
// eq. (3.8) per cosmology at x = 1e10 (the formula is scale-free) plus the analytic remainder of the integrand's leading
// term beyond it (< 2e-15); its parameter derivatives use the same T-basis at that point.  FP64; called after cosmo_prep.
CB_HD void prep_age(Cosmo<double>& C, bool with_grad) {
    C.Tinf = NAN; C.dTinf[0] = C.dTinf[1] = C.dTinf[2] = NAN;
    if (C.status) return;
    const double X = 1.0e10, z = X - 1.0;
    Core<double> R;
    if (C.cubic & 2u) {
        R.I0 = R.TT = R.AA = R.K = R.E = R.iE = R.Em1 = 0.0;
        R.status = C.status;
        apply_c4<double, true, false, true>(C, z, R);
    } else {
        eval_core<double, true, false, true, VoteNone>(C, z, VoteNone(), R);
    }
    if (R.status) return;
    const double tail = (C.Or * X > C.Om) ? 0.5 / (sqrt(C.Or) * X * X) : (2.0 / 3.0) / (sqrt(C.Om) * X * sqrt(X));
    C.Tinf = R.TT + tail;
    if (!with_grad) { C.dTinf[0] = C.dTinf[1] = C.dTinf[2] = 0.0; return; }      // (NaN there means "basis singular" to observables_k)
    const double iE = R.iE;
    const double bt0 = -R.Em1 * iE, bt1 = (z - R.Em1) * iE, bt2 = (z * (X + 1.0) - R.Em1) * iE;
    GradSolve S;
    S.init(C);
    for (int t = 0; t < 3; ++t) {
        double g[6];
        S.rowT(t, g);
        C.dTinf[t] = -0.5 * (g[0] * R.I0 + g[1] * R.K + g[2] * bt0 + g[3] * bt1 + g[4] * bt2 + g[5] * R.TT);
    }
    // remainder beyond X of the Or-derivative, -1/2 int_X^inf (x^3 - x)/E^3 dx with E^2 ~ x^3 (Or x + Om): it decays only like
    // X^(-1/2) while matter dominates at X (2e-5/Om^1.5 at Or = 0); the Om and OL remainders are O(X^-3/2) and dropped.
    double rem;
    if (C.Or * X > 1.0e3 * C.Om) rem = 0.5 / (C.Or * sqrt(C.Or) * X * X);
    else rem = 2.0 * (2.0 * C.Or * X + C.Om) / (C.Om * C.Om * sqrt(X) * sqrt(C.Or * X + C.Om)) - 4.0 * sqrt(C.Or) / (C.Om * C.Om);
    C.dTinf[2] -= 0.5 * rem;
}

// ---- S8, first half: the parameter derivatives of the three integrals.
// Raw gradient integrals of one element over [1, 1+z] (Leibniz' rule: d X / d theta = -1/2 of these), theta = (Om, OL, Or),
// D_theta = dE^2/dtheta with Ok eliminated = x^3 - x^2, 1 - x^2, x^4 - x^2:
//   dI[t] = int D_theta / E^3 dx,   dT[t] = int D_theta / (x E^3) dx,   dA[t] = int x^2 D_theta / E^3 dx
template <typename T>
struct GradInt { T dI[3], dT[3], dA[3]; };

// From the gradient bases of cosmo_prep.cuh on the forward intermediates (the closed combination of
// eqs. (2.10)-(2.12) + appendix A).
// kCond: also return in *cond the cancellation factor of the evaluation, max over the requested families and theta of
// (sum_j |G_j basis_j|) / max(|result|, 1e-3 |forward integral|): the relative error of the result is ~ 2e-16 x cond in FP64.  It
// grows like 1 / prod(r_j - r_k) where roots of E^2 approach each other away from the path ("limits have to be
// explicitly implemented when arguments are repeated"); callers switch to grad_quad() above GRAD_COND_LIMIT.
// where the basis rows come from: stored per cosmology by k_prep (OUTER kernels) ...
template <typename T>
struct RowsStored {
    const Cosmo<T>& C;
    CB_HD void rowI(int t, T (&g)[5]) const { for (int j = 0; j < 5; ++j) g[j] = C.GI[t][j]; }
    CB_HD void rowT(int t, T (&g)[6]) const { for (int j = 0; j < 6; ++j) g[j] = C.GT[t][j]; }
    CB_HD void rowJ(int p, T (&g)[5]) const { for (int j = 0; j < 5; ++j) g[j] = C.GJ[p][j]; }
    CB_HD void rowA(int t, T (&g)[7]) const { for (int j = 0; j < 7; ++j) g[j] = C.GA[t][j]; }
};
// ... or produced right where they are consumed (ELEMENTWISE kernels: nothing to keep across the duplication loop)
template <typename T>
struct RowsSolved {
    const GradSolve& S;
    CB_HD void rowI(int t, T (&g)[5]) const { double d[5]; S.rowI(t, d); for (int j = 0; j < 5; ++j) g[j] = (T)d[j]; }
    CB_HD void rowT(int t, T (&g)[6]) const { double d[6]; S.rowT(t, d); for (int j = 0; j < 6; ++j) g[j] = (T)d[j]; }
    CB_HD void rowJ(int p, T (&g)[5]) const { double d[5]; S.rowJ(p, d); for (int j = 0; j < 5; ++j) g[j] = (T)d[j]; }
    CB_HD void rowA(int t, T (&g)[7]) const { double d[7]; S.rowA(t, d); for (int j = 0; j < 7; ++j) g[j] = (T)d[j]; }
};

// accumulator of the cancellation factor: kCond = 2 keeps its value (one division per result), kCond = 1 only whether it exceeds
// `limit` (a comparison per result: the form the kernels use)
template <typename T, int kCond>
struct CondAcc {
    T limit, cmax;
    bool over;
    CB_HD void add(T sa, T val, T fwd) {
        using N = Num<T>;
        const T den = N::max_(N::abs_(val), T(1e-3) * N::abs_(fwd));
        if (kCond == 2) { const T c = sa / den; cmax = (c > cmax || !(c == c)) ? c : cmax; }
        if (kCond == 1) over = over | !(sa <= limit * den);           // a NaN counts as exceeded
    }
};

template <typename T, bool kT, bool kA, int kCond, typename Rows>
CB_HD void grad_basis(const Cosmo<T>& C, const Rows& rows, T z, const Core<T>& R, GradInt<T>& D, T* cond = nullptr, T limit = T(0)) {
    using N = Num<T>;
    const T x = T(1) + z;
    const T iE = R.iE;
    // boundary terms b_k = x^k / E - 1 (cancellation-free)
    const T xp1 = x + T(1);
    const T n1 = z, n2 = z * xp1, n3 = z * N::fma_(xp1, x, T(1)), n4 = n2 * N::fma_(x, x, T(1));
    const T bt0 = -R.Em1 * iE, bt1 = (n1 - R.Em1) * iE, bt2 = (n2 - R.Em1) * iE;
    // |basis values|: sum_j |g_j b_j| = sum_j |g_j| |b_j| costs one FMA per term (the |.| of an operand is free)
    const T aI0 = N::abs_(R.I0), aK = N::abs_(R.K), a0 = N::abs_(bt0), a1 = N::abs_(bt1), a2 = N::abs_(bt2), aTT = N::abs_(R.TT);
    CondAcc<T, kCond> acc{limit, T(0), false};
    auto asum5 = [&](const T* g) {
        return N::fma_(N::abs_(g[0]), aI0, N::fma_(N::abs_(g[1]), aK, N::fma_(N::abs_(g[2]), a0, N::fma_(N::abs_(g[3]), a1, N::abs_(g[4]) * a2))));
    };
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        {
            T gi[5];
            rows.rowI(t, gi);
            D.dI[t] = gi[0] * R.I0 + gi[1] * R.K + gi[2] * bt0 + gi[3] * bt1 + gi[4] * bt2;
            if (kCond) acc.add(asum5(gi), D.dI[t], R.I0);
        }
        D.dT[t] = T(0); D.dA[t] = T(0);
        if (kT) {
            T g[6];
            rows.rowT(t, g);
            D.dT[t] = g[0] * R.I0 + g[1] * R.K + g[2] * bt0 + g[3] * bt1 + g[4] * bt2 + g[5] * R.TT;
            if (kCond) acc.add(N::fma_(N::abs_(g[5]), aTT, asum5(g)), D.dT[t], R.TT);
        }
    }
    if (kA) {
        const T btA = (((C.cubic & 1u) ? n4 : n3) - R.Em1) * iE;
        // d_abs gradient where radiation is a perturbation: the exact basis below multiplies the forward A by ~3/Or
        // (the x^5, x^6 rows), which loses Om/Or digits.  Instead J'_p = int x^p dx/E^3, p = 2, 3, 4, come from the basis and
        // J'_5.. follow from d(x^k / E) = N_k / E^3:  Om (k - 3/2) J'_{k+2} = [x^k/E] - k OL J'_{k-1} - (k-1) Ok J'_{k+1}
        // - (k-2) Or J'_{k+3}, the Or terms iterated (same scheme as the forward d_abs).
        constexpr int KJ = REC_KJ;            // levels k = 3 .. 3 + KJ - 2, solved directly (band_solve)
        T Jp[7], Sp[7];
        Jp[0] = Jp[1] = T(0); Sp[0] = Sp[1] = T(0);
#pragma unroll
        for (int p = 2; p < 5; ++p) {
            T gj[5];
            rows.rowJ(p, gj);
            Jp[p] = gj[0] * R.I0 + gj[1] * R.K + gj[2] * bt0 + gj[3] * bt1 + gj[4] * bt2;
            Sp[p] = kCond ? asum5(gj) : T(0);
        }
        T bk[KJ - 1], vj[KJ - 1], trunc;
        {
            T dk = n3;             // x^k - 1 = x (x^(k-1) - 1) + z, from x^3 - 1: no cancellation at small z
#pragma unroll
            for (int j = 0; j < KJ - 1; ++j) { bk[j] = N::fma_(dk, iE, bt0); dk = N::fma_(x, dk, z); }     // x^k/E - 1 = (x^k - 1)/E + (1/E - 1)
        }
        band_solve<T, KJ - 1, 1, 2, 3, 1>(C.Om, C.OL, C.Or, C.Ok, bk, Jp[4], Jp[3], Jp[2], x, vj, trunc);               // vj[j] = J'_{j+5}
        Jp[5] = vj[0]; Jp[6] = vj[1];
        const T tol = T(sizeof(T) == 8 ? 1e-13 : 1e-6);
        const bool useJ = trunc <= tol * N::abs_(Jp[5]) && trunc <= tol * N::abs_(Jp[6]);
        if (kCond) {      // error bounds of J'_5, J'_6 through the first two levels of the recursion (the Or terms are small where it is used)
            Sp[5] = (N::abs_(bk[0]) + T(3) * C.OL * Sp[2] + T(2) * N::abs_(C.Ok) * Sp[4]) * C.iOm * T(1.0 / 1.5);
            Sp[6] = (N::abs_(bk[1]) + T(4) * C.OL * Sp[3] + T(3) * N::abs_(C.Ok) * Sp[5]) * C.iOm * T(1.0 / 2.5);
        }
        if (useJ) {
#pragma unroll
            for (int t = 0; t < 3; ++t) {
                const int a = t == 0 ? 5 : (t == 1 ? 2 : 6);      // x^2 D_theta = x^5, x^2, x^6 minus x^4
                D.dA[t] = Jp[a] - Jp[4];
                if (kCond) acc.add(Sp[a] + Sp[4], D.dA[t], R.AA);
            }
        } else {
#pragma unroll
            for (int t = 0; t < 3; ++t) {
                T ga[7];
                rows.rowA(t, ga);
                D.dA[t] = ga[0] * R.I0 + ga[1] * R.K + ga[2] * bt0 + ga[3] * bt1 + ga[4] * bt2 + ga[5] * btA + ga[6] * R.AA;
                if (kCond) acc.add(N::fma_(N::abs_(ga[5]), N::abs_(btA), N::fma_(N::abs_(ga[6]), N::abs_(R.AA), asum5(ga))), D.dA[t], R.AA);
            }
        }
    }
    if (kCond == 2) *cond = acc.cmax;
    if (kCond == 1) *cond = acc.over ? T(INFINITY) : T(0);
}

// The same nine integrals by Gauss-Legendre quadrature of their definition (Leibniz' rule on eqs. (2.3)-(2.5), the
// route PAPER.md:285 fn.23 names), for the elements where grad_basis() is ill-conditioned: E^2 has (nearly) repeated roots away
// from the path, or the range is tiny.  There the integrand is smooth on the path: with panels that grow geometrically (ratio <= 2) in
// the distance x - c from the root pair (c = its right end when it lies left of the path, else 0: every other root is at x <= 0) a
// panel of ratio q sees no singularity inside the Bernstein ellipse of parameter rho = ((q+1) + 2 sqrt(q))/(q-1), so n nodes leave
// ~ rho^-2n times a constant that grows with the order of the singularity (x^-9/2 at Einstein-de Sitter): 4 nodes for q <= 1.02
// (rho = 202), 6 for q <= 1.2 (rho = 22), 12 for q <= 2 (rho = 5.8); measured against the oracle <= 4e-14 wherever grad_basis() gives
// way to it.  E^2 is evaluated as printed, eq. (2.2), so
// every root structure -- Einstein-de Sitter's triple root included -- takes the same code.  FP64 in every variant; never inlined
// (rare path).  x0, d2: centre of the root pair of Q2 and (half its gap)^2 (d2 < 0: conjugate pair x0 +- i sqrt(-d2)).
// Returns 0, or ST_GRAD_ILLCOND when the pair sits next to the path without the panels being graded towards it (peaked integrand).
template <int NG, typename T>
CB_HD void grad_quad_panel(const double (&XI)[NG], const double (&WI)[NG], T Om, T OL, T Or, T Ok, T tlo, T wd, bool wantT, bool wantA,
                           T (&acc)[9]) {
    using N = Num<T>;
    T dm[NG], dl[NG], dr[NG], xs[NG];
#pragma unroll
    for (int i = 0; i < NG; ++i) {              // NG independent chains: the rare path is latency-bound, not throughput-bound
        const T t = N::fma_(wd, T(XI[i]), tlo), x = T(1) + t;        // t = x - 1 is formed directly: D_theta has the factor (x - 1)
        const T e2 = N::fma_(N::fma_(N::fma_(Or, x, Om), x, Ok), x * x, OL);
        const T ie = N::rsqrt_(e2), f = (T(WI[i]) * wd) * (ie * ie) * (ie * t);
        xs[i] = x;
        dm[i] = f * (x * x); dl[i] = -f * (x + T(1)); dr[i] = dm[i] * (x + T(1));       // w D_theta / E^3, theta = Om, OL, Or
    }
#pragma unroll
    for (int i = 0; i < NG; ++i) { acc[0] += dm[i]; acc[1] += dl[i]; acc[2] += dr[i]; }
    if (wantT) {
#pragma unroll
        for (int i = 0; i < NG; ++i) { const T ix = N::rcp_(xs[i]); acc[3] = N::fma_(dm[i], ix, acc[3]); acc[4] = N::fma_(dl[i], ix, acc[4]); acc[5] = N::fma_(dr[i], ix, acc[5]); }
    }
    if (wantA) {
#pragma unroll
        for (int i = 0; i < NG; ++i) { const T x2 = xs[i] * xs[i]; acc[6] = N::fma_(dm[i], x2, acc[6]); acc[7] = N::fma_(dl[i], x2, acc[7]); acc[8] = N::fma_(dr[i], x2, acc[8]); }
    }
}

CB_HD_NOINLINE unsigned grad_quad(double Om, double OL, double Or, double x0, double d2, double z1, double dz, bool wantT, bool wantA,
                                  double out[9]) {
    const double X4[4] = {0.0694318442029737124, 0.330009478207571868, 0.669990521792428132, 0.930568155797026288};
    const double W4[4] = {0.173927422568726929, 0.326072577431273071, 0.326072577431273071, 0.173927422568726929};
    const double X6[6] = {0.0337652428984239861, 0.169395306766867743, 0.380690406958401546, 0.619309593041598454, 
                           0.830604693233132257, 0.966234757101576014};
    const double W6[6] = {0.0856622461895851725, 0.180380786524069304, 0.233956967286345524, 0.233956967286345524, 
                           0.180380786524069304, 0.0856622461895851725};
    const double X12[12] = {0.00921968287664037465, 0.0479413718147625717, 0.115048662902847656, 0.206341022856691276, 
                           0.316084250500909903, 0.437383295744265542, 0.562616704255734458, 0.683915749499090097, 
                           0.793658977143308724, 0.884951337097152344, 0.952058628185237428, 0.990780317123359625};
    const double W12[12] = {0.0235876681932559136, 0.0534696629976592155, 0.0800391642716731132, 0.101583713361532961, 
                           0.116746268269177404, 0.124573522906701393, 0.124573522906701393, 0.116746268269177404, 
                           0.101583713361532961, 0.0800391642716731132, 0.0534696629976592155, 0.0235876681932559136};
    double acc[9] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    for (int i = 0; i < 9; ++i) out[i] = 0.0;
    const double Ok = 1.0 - Om - OL - Or, X1 = 1.0 + z1, X2 = X1 + dz;
    const double lo = fmin(X1, X2), hi = fmax(X1, X2);
    unsigned st = 0u;
    if (!(lo > 0.0) || dz == 0.0) return st;
    const double xr = x0 + (d2 > 0.0 ? sqrt(d2) : 0.0);              // right end of the pair (its centre for a conjugate pair)
    const double c = (xr > 0.0 && xr < lo) ? xr : 0.0;
    const double q = (X2 - c) / (X1 - c);                             // overall ratio (< 1 when z2 < z1)
    const double qa = q >= 1.0 ? q : 1.0 / q;
    int np = 1;
    double r = q;
    if (qa > 2.0) {
        const double lr = log(q);
        np = (int)ceil(fabs(lr) * 1.4426950408889634);                // panels of ratio <= 2
        if (np > 64) np = 64;
        r = exp(lr / np);
    }
    double rho = 1e300;
    if (!(xr < lo)) {
        // the pair is not left of the path, so the panels are not graded towards it.  Bernstein parameter of the panel next to its
        // nearest member s = xs + i y0: rho = a + sqrt(a^2 - 1), a = (|w + 1| + |w - 1|)/2, w = (s - centre)/half-width; a pair whose
        // real part lies on the path is taken over the centre of a panel (the worst case)
        const double y0 = d2 < 0.0 ? sqrt(-d2) : 0.0, hg = d2 > 0.0 ? sqrt(d2) : 0.0;
        const double rr = r >= 1.0 ? r : 1.0 / r;                       // panel ratio, >= 1
        double wre, h;
        if (x0 + hg < lo) { h = 0.5 * lo * (rr - 1.0); wre = (lo - (x0 + hg)) / h + 1.0; }                 // first panel [lo, lo rr]
        else if (x0 - hg > hi) { h = 0.5 * hi * (1.0 - 1.0 / rr); wre = ((x0 - hg) - hi) / h + 1.0; }       // last panel [hi/rr, hi]
        else { h = 0.5 * fmin(fmax(x0, lo), hi) * (rr - 1.0); wre = 0.0; }
        const double wim = y0 / h;
        const double a = 0.5 * (hypot(wre + 1.0, wim) + hypot(wre - 1.0, wim));
        rho = a + sqrt(fmax(a * a - 1.0, 0.0));
        if (!(rho >= 3.5)) st = (unsigned)ST_GRAD_ILLCOND;           // 12 nodes: 3.5^-24 = 9e-14
    }
    double wd = (np == 1) ? dz : dz * (r - 1.0) / (q - 1.0);            // widths sum to dz; one panel: dz itself
    double tlo = z1;                                                   // x - 1 at the panel's lower end
    if (np == 1 && qa <= 1.02 && rho >= 60.0) grad_quad_panel<4, double>(X4, W4, Om, OL, Or, Ok, tlo, wd, wantT, wantA, acc);
    else if (np == 1 && qa <= 1.2 && rho >= 12.0) grad_quad_panel<6, double>(X6, W6, Om, OL, Or, Ok, tlo, wd, wantT, wantA, acc);
    else {
        for (int k = 0; k < np; ++k) {
            grad_quad_panel<12, double>(X12, W12, Om, OL, Or, Ok, tlo, wd, wantT, wantA, acc);
            tlo += wd;
            wd *= r;
        }
    }
    for (int i = 0; i < 9; ++i) out[i] = acc[i];
    return st;
}

// FP32 variant: the gradient integrals of EVERY element by the same quadrature in FP32 arithmetic (6 nodes per panel of ratio <= 2:
// rho^-12 = 6e-10).  The gradient bases lose cond x 6e-8 in FP32 and cond reaches 1e3-1e5 at small z, while the quadrature sums terms of
// one sign pattern and is as accurate as FP32 allows (~1e-6) at every z; it is also FP32 work, which the bases' FP64 rows are not.
// x0, d2 as grad_quad.  Inlined (it is this variant's main path).
CB_HD unsigned grad_quad_f32(float Om, float OL, float Or, float x0, float d2, float z, bool wantT, bool wantA, float (&acc)[9]) {
    const double X6[6] = {0.0337652428984239861, 0.169395306766867743, 0.380690406958401546, 0.619309593041598454, 0.830604693233132257,
                          0.966234757101576014};
    const double W6[6] = {0.0856622461895851725, 0.180380786524069303, 0.233956967286345524, 0.233956967286345524, 0.180380786524069303,
                          0.0856622461895851725};
#pragma unroll
    for (int i = 0; i < 9; ++i) acc[i] = 0.0f;
    const float Ok = 1.0f - Om - OL - Or, X2 = 1.0f + z;
    if (!(X2 > 0.0f) || z == 0.0f) return 0u;
    const float lo = fminf(1.0f, X2), hi = fmaxf(1.0f, X2);
    const float hg = d2 > 0.0f ? sqrtf(d2) : 0.0f, xr = x0 + hg;
    const float c = (xr > 0.0f && xr < lo) ? xr : 0.0f;
    const float q = (X2 - c) / (1.0f - c), qa = q >= 1.0f ? q : 1.0f / q;
    int np = 1;
    float r = q;
    if (qa > 2.0f) {
        const float lr = logf(q);
        np = (int)ceilf(fabsf(lr) * 1.44269504f);
        if (np > 64) np = 64;
        r = expf(lr / (float)np);
    }
    unsigned st = 0u;
    if (!(xr < lo)) {       // pair not left of the path: Bernstein parameter of the panel next to it (see grad_quad); 6 nodes need rho >= 5
        const float y0 = d2 < 0.0f ? sqrtf(-d2) : 0.0f, rr = r >= 1.0f ? r : 1.0f / r;
        float wre, h;
        if (x0 + hg < lo) { h = 0.5f * lo * (rr - 1.0f); wre = (lo - (x0 + hg)) / h + 1.0f; }
        else if (x0 - hg > hi) { h = 0.5f * hi * (1.0f - 1.0f / rr); wre = ((x0 - hg) - hi) / h + 1.0f; }
        else { h = 0.5f * fminf(fmaxf(x0, lo), hi) * (rr - 1.0f); wre = 0.0f; }
        const float wim = y0 / h;
        const float a = 0.5f * (hypotf(wre + 1.0f, wim) + hypotf(wre - 1.0f, wim));
        if (!(a + sqrtf(fmaxf(a * a - 1.0f, 0.0f)) >= 5.0f)) st = (unsigned)ST_GRAD_ILLCOND;
    }
    float wd = (np == 1) ? z : z * (r - 1.0f) / (q - 1.0f), tlo = 0.0f;
    for (int k = 0; k < np; ++k) {
        grad_quad_panel<6, float>(X6, W6, Om, OL, Or, Ok, tlo, wd, wantT, wantA, acc);
        tlo += wd;
        wd *= r;
    }
    return st;
}

// Above this cancellation factor the gradient integrals are taken from grad_quad() instead of grad_basis() (FP64: basis error
// ~ 2e-16 x 1e6; measured on config 5: basis <= 4e-10 below it, quadrature <= 4e-14 above it)
template <typename T>
CB_HD unsigned grad_robust_fix(const Cosmo<T>& C, T z, bool wantT, bool wantA, T cond, GradInt<T>& D) {
    const T limit = T(sizeof(T) == 8 ? GRAD_COND_LIMIT : GRAD_COND_LIMIT_F32);
    if (cond <= limit) return 0u;
    double q[9];
    const double b = (double)C.b;
    const unsigned st = grad_quad((double)C.Om, (double)C.OL, (double)C.Or, -0.5 * b, 0.25 * b * b - (double)C.c, 0.0, (double)z, wantT, wantA, q);
#pragma unroll
    for (int t = 0; t < 3; ++t) { D.dI[t] = (T)q[t]; D.dT[t] = (T)q[3 + t]; D.dA[t] = (T)q[6 + t]; }
    return st;
}

// ---- S8, second half.  VJP of one element: g[N_PLANES] upstream (entries outside `which` must be 0); D = its gradient integrals.
// Adds to gz and gp[0..3] = (Om, OL, Or, H0).
// `which`: planes that can carry a non-zero upstream gradient; where the caller knows it at compile time the terms of the
// other planes fold away (x * 0 is not foldable in IEEE arithmetic, so a zero g alone does not remove them).
template <typename T, bool kT, bool kA>
CB_HD void backward_chain(const Cosmo<T>& C, T z, const Core<T>& R, const Obs<T>& O, const GradInt<T>& D, const T g[N_PLANES], T& gz,
                          T gp[4], unsigned which = W_ALL) {
    using N = Num<T>;
    const T x = T(1) + z;
    const T iE = R.iE;
    T ix, xiDL;                                            // 1/x and x/D_L = 1/D_M
    if (which & W_MU) {                                    // one reciprocal serves 1/x and 1/D_M
        const T rxd = N::rcp_(x * O.v[1]);
        ix = O.v[1] * rxd;
        xiDL = x * rxd;
        // z = 0: D_M = 0 and mu is undefined (status 4), but the other planes' gradients are finite and must not see 0 * inf
        if (which != W_MU && O.v[1] == T(0)) ix = N::rcp_(x);
    } else {
        ix = N::rcp_(x);
        xiDL = T(0);
    }
    T gM = T(0);
    if (which & W_DM) gM = g[1];
    if (which & W_DL) gM = N::fma_(x, g[2], gM);
    if ((which & W_MU) && g[3] != T(0)) gM = N::fma_(T(CB_KT.five_over_ln10) * g[3], xiDL, gM);
    if ((which & W_DA) && g[6] != T(0)) gM = N::fma_(g[6], ix, gM);     // D_A = D_M / (1+z)
    T aI = C.dH * ((which & W_DC) ? N::fma_(gM, O.Fi, g[0]) : gM * O.Fi);
    T aK = -gM * C.dH * O.Fk;
    if ((which & W_VC) && g[7] != T(0)) {                                                 // V_C = 4 pi dH^3 v(Ok, I0): dv = F^2 dI0 + v_k dOk
        const T c4pi = T(12.566370614359172954) * C.dH * C.dH * C.dH * g[7];
        aI = N::fma_(c4pi, O.F * O.F, aI);
        aK = N::fma_(-c4pi, O.Vk, aK);
    }
    const T aIh = T(-0.5) * aI;
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        T acc = N::fma_(aIh, D.dI[t], aK);
        if (kT) {
            acc = N::fma_((g[4] - g[8]) * C.tH, T(-0.5) * D.dT[t], acc);       // t_L = tH T, age = tH (Tinf - T)
            acc = N::fma_(g[8] * C.tH, C.dTinf[t], acc);
        }
        if (kA) acc = N::fma_(g[5] * C.dH, T(-0.5) * D.dA[t], acc);
        gp[t] += acc;
    }
    T h = T(0);
    if (which & W_DC) h = g[0] * O.v[0];
    if (which & W_DM) h = N::fma_(g[1], O.v[1], h);
    if (which & W_DL) h = N::fma_(g[2], O.v[2], h);
    if (which & W_MU) h = N::fma_(g[3], T(CB_KT.five_over_ln10), h);
    if (kT) h += g[4] * O.v[4] + g[8] * O.v[8];
    if (kA) h += g[5] * O.v[5];
    if (which & W_DA) h = N::fma_(g[6], O.v[6], h);
    if (which & W_VC) h = N::fma_(T(3) * g[7], O.v[7], h);
    gp[3] = N::fma_(-h * C.dH, T(1.0 / C_KM_S), gp[3]);        // / H0
    T dz = aI * iE;
    if (which & W_DL) dz = N::fma_(g[2], O.v[1], dz);
    if ((which & W_MU) && g[3] != T(0)) dz = N::fma_(T(CB_KT.five_over_ln10) * g[3], ix, dz);
    if (kT) dz += (g[4] - g[8]) * C.tH * iE * ix;
    if ((which & W_DA) && g[6] != T(0)) dz -= g[6] * O.v[6] * ix;
    if (kA) dz += g[5] * C.dH * x * x * iE;
    gz += dz;
}

// VJP of one element from the gradient bases alone (the hot OUTER loop: its cosmologies are screened by cosmo_prep, Cosmo::cubic
// bits 2, 3); kCond as grad_basis.
template <typename T, bool kT, bool kA, bool kCond = false>
CB_HD void backward(const Cosmo<T>& C, T z, const Core<T>& R, const Obs<T>& O, const T g[N_PLANES], T& gz, T gp[4], T* cond = nullptr,
                    unsigned which = W_ALL) {
    GradInt<T> D;
    const RowsStored<T> rows{C};
    grad_basis<T, kT, kA, kCond ? 2 : 0, RowsStored<T>>(C, rows, z, R, D, cond);
    backward_chain<T, kT, kA>(C, z, R, O, D, g, gz, gp, which);
}

// VJP of one element with the conditioning check: bases where they are accurate, quadrature elsewhere.  Returns status bits to OR in.
// kSolve: the basis rows are solved on the spot from the factorisation (ELEMENTWISE kernels) instead of read from the Cosmo block.
// kDefer: do not run the quadrature here; return ST_INTERNAL_REDO for an element that needs it (the ELEMENTWISE kernels collect
// those few per cent of elements and a second, dense pass redoes them: a divergent call inside the main kernel costs it a third
// of its time, measured).
// (G: the upstream gradients as an array, or an IO object whose get_grads() fetches them only now -- elem_one_io)
template <typename T>
CB_HD void fetch_grads(const T* g, T (&go)[N_PLANES]) {
#pragma unroll
    for (int w = 0; w < N_PLANES; ++w) go[w] = g[w];
}
template <typename T, typename IO>
CB_HD void fetch_grads(const IO& io, T (&go)[N_PLANES]) { io.get_grads(go); }
// kQuadOnly (second pass of the FP64 ELEMENTWISE kernel): an element with the real root structure is on the work list because its bases
// are singular or cancel beyond the limit -- the main pass has established that -- so the bases are not formed again and the
// quadrature is taken straight away (a third of the second pass's instructions).
template <typename T, bool kT, bool kA, bool kSolve = false, bool kDefer = false, typename G = const T*, bool kQuadOnly = false>
CB_HD unsigned backward_robust(const Cosmo<T>& C, T z, const Core<T>& R, const Obs<T>& O, const G& gsrc, T& gz, T gp[4],
                               unsigned which = W_ALL) {
    GradInt<T> D;
    T cond = T(0);
    const T limit = T(sizeof(T) == 8 ? GRAD_COND_LIMIT : GRAD_COND_LIMIT_F32);
    bool singular = (C.cubic & 4u) != 0;
    if (kQuadOnly && !(C.cubic & 2u)) {
        for (int t = 0; t < 3; ++t) { D.dI[t] = D.dT[t] = D.dA[t] = T(0); }
        unsigned st = 0u;
        if (!(R.status & (ST_ROOT_ON_PATH | ST_UNSUPPORTED)))
            st = grad_robust_fix<T>(C, z, kT && (which & (W_TL | W_AGE)), kA && (which & W_DABS), T(INFINITY), D);
        T g[N_PLANES];
        fetch_grads<T>(gsrc, g);
        backward_chain<T, kT, kA>(C, z, R, O, D, g, gz, gp, which);
        return st;
    }
    if (kSolve) {
        Cosmo<double> Cd;
        Cd.Om = (double)C.Om; Cd.OL = (double)C.OL; Cd.Or = (double)C.Or; Cd.Ok = (double)C.Ok;
        Cd.m = (double)C.m; Cd.rn = (double)C.rn; Cd.b = (double)C.b; Cd.c = (double)C.c; Cd.cubic = C.cubic;
        GradSolve S;
        S.init(Cd);
        singular = S.singular;
        const RowsSolved<T> rows{S};
        grad_basis<T, kT, kA, 1, RowsSolved<T>>(C, rows, z, R, D, &cond, limit);
    } else {
        const RowsStored<T> rows{C};
        grad_basis<T, kT, kA, 1, RowsStored<T>>(C, rows, z, R, D, &cond, limit);
    }
    const bool valid = !(R.status & (ST_ROOT_ON_PATH | ST_UNSUPPORTED));
    unsigned st = 0u;
    if (valid) {
        if (kDefer) {
            if (singular || !(cond <= limit)) st = ST_INTERNAL_REDO;
        } else {
            st = grad_robust_fix<T>(C, z, kT && (which & (W_TL | W_AGE)), kA && (which & W_DABS), singular ? T(INFINITY) : cond, D);
        }
    }
    T g[N_PLANES];
    fetch_grads<T>(gsrc, g);
    backward_chain<T, kT, kA>(C, z, R, O, D, g, gz, gp, which);
    return st;
}

// ---- one element of the ELEMENTWISE calls with its own cosmology: S1-S8.  Out: values v[N_PLANES], status; with kG also
// dz and gp[4] for the upstream gradients g[N_PLANES].  No gradient bases are stored: backward_robust<.., kSolve> produces each row
// where it is consumed, and the constants are formed a second time after the duplication loop (kRecon), so that little more than
// the factorisation crosses the loop (registers decide how many warps fit).
// kDefer: the main pass of the ELEMENTWISE kernels -- elements that need a slow path (complex root structure, ill-conditioned
// gradient bases: backward_robust) are only marked ST_INTERNAL_REDO; the second pass runs them again without kDefer.
// kAge: the age plane may be asked for (its T_inf costs a second pass of eq. (3.8) per element: kept out of the other instantiations)
// IO: where the values go and the upstream gradients come from.  put_values() is called as soon as the observables exist and
// get_grads() only when the backward chain needs them, so that in the kernel neither set occupies registers through the other
// half of the element (ArrayIO: plain arrays, for the second pass and the host checks).
template <typename T>
struct ArrayIO {
    const T* g; T* v;
    CB_HD void put_values(const T (&o)[N_PLANES]) const {
#pragma unroll
        for (int w = 0; w < N_PLANES; ++w) v[w] = o[w];
    }
    CB_HD void get_grads(T (&go)[N_PLANES]) const {
#pragma unroll
        for (int w = 0; w < N_PLANES; ++w) go[w] = g[w];
    }
};
template <typename T, bool kT, bool kA, bool kG, typename Vote, bool kDefer = false, bool kAge = true, typename IO = ArrayIO<T>, bool kRedo = false>
CB_HD unsigned elem_one_io(T zv, double Om, double OL, double Or, double H0, unsigned which, const Vote& vote, const IO& io, T& dz, T gp[4]) {
    Cosmo<T> C0{}, C{};
    {
        Cosmo<double> Cd{};
        cosmo_factor(Om, OL, Or, H0, Cd);
        cosmo_constants(Cd);
        if (kT && kAge && (which & W_AGE)) prep_age(Cd, kG);
        convert_cosmo<T>(Cd, C0);
    }
    Core<T> R;
    R.K = T(0); R.TT = T(0); R.AA = T(0);
    eval_core<T, kT, kA, kG, Vote, true>(C0, zv, vote, R, &C);
    // E^2 without a real negative root: complex slow path (cosmo_c4.cuh), a never-inlined call that costs the kernel a fifth of its
    // time where it diverges (measured on config 2) -- with kDefer such elements go to the second pass instead
    unsigned redo = 0u;
    if (kDefer && kG) redo = (C.cubic & 2u) ? (unsigned)ST_INTERNAL_REDO : 0u;      // (the forward kernels have no second pass)
    else apply_c4<T, kT, kA, kG>(C, zv, R);
    Obs<T> O;
    observables<T, kT, kA>(C, zv, R, which, O);
    io.put_values(O.v);
    unsigned st = O.status | redo;
    if (kG) {
        dz = T(0); gp[0] = gp[1] = gp[2] = gp[3] = T(0);
        if (sizeof(T) == 4) {       // FP32 variant: gradient integrals by FP32 quadrature (grad_quad_f32), no bases
            float q[9];
            GradInt<T> D;
            const float b = (float)C.b;
            const unsigned sq = grad_quad_f32((float)C.Om, (float)C.OL, (float)C.Or, -0.5f * b, 0.25f * b * b - (float)C.c, (float)zv,
                                              kT && (which & (W_TL | W_AGE)), kA && (which & W_DABS), q);
#pragma unroll
            for (int t = 0; t < 3; ++t) { D.dI[t] = (T)q[t]; D.dT[t] = (T)q[3 + t]; D.dA[t] = (T)q[6 + t]; }
            const bool peaked = sq != 0u && !(R.status & (ST_ROOT_ON_PATH | ST_UNSUPPORTED));
            // a root pair next to the path (peaked integrand: the 6-node panels do not resolve it; loitering models, where FP32 cannot
            // even hold the pair's gap): such elements are evaluated by the FP64 path, values included (second pass of the kernel when kDefer)
            if (peaked && kDefer) st |= ST_INTERNAL_REDO;
            if (peaked && !kDefer) {
                T g[N_PLANES], v[N_PLANES];
                io.get_grads(g);
                double gd[N_PLANES], vd[N_PLANES], dzd = 0.0, gpd[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
                for (int w = 0; w < N_PLANES; ++w) gd[w] = (double)g[w];
                const ArrayIO<double> iod{gd, vd};
                st = elem_one_io<double, kT, kA, kG, VoteNone, false, kAge, ArrayIO<double>>((double)zv, Om, OL, Or, H0, which, VoteNone(), iod, dzd, gpd);
#pragma unroll
                for (int w = 0; w < N_PLANES; ++w) v[w] = (T)vd[w];
                io.put_values(v);
                dz = (T)dzd;
#pragma unroll
                for (int j = 0; j < 4; ++j) gp[j] = (T)gpd[j];
            } else {
                T g[N_PLANES];
                io.get_grads(g);
                backward_chain<T, kT, kA>(C, zv, R, O, D, g, dz, gp, which);
            }
        } else {
            st |= backward_robust<T, kT, kA, true, kDefer, IO, kRedo>(C, zv, R, O, io, dz, gp, which);
        }
    }
    return st;
}
template <typename T, bool kT, bool kA, bool kG, typename Vote, bool kDefer = false, bool kAge = true, bool kRedo = false>
CB_HD unsigned elem_one(T zv, double Om, double OL, double Or, double H0, unsigned which, const Vote& vote, const T* g, T* v, T& dz, T gp[4]) {
    const ArrayIO<T> io{g, v};
    return elem_one_io<T, kT, kA, kG, Vote, kDefer, kAge, ArrayIO<T>, kRedo>(zv, Om, OL, Or, H0, which, vote, io, dz, gp);
}

}  // namespace cb
