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
    eval_c4((double)C.Or, (double)C.m, (double)C.rn, (double)C.b, (double)C.c, 1.0, 1.0 + (double)z, kT, kA, I0, TT, AA, KK);
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
    } else {
        for (int k = 0; k < K; ++k) sinn<T>(C.Ok, I0[k], O[k].F, O[k].Fi, O[k].Fk);
    }
#pragma unroll
    for (int k = 0; k < K; ++k) {
        const T x = T(1) + z[k];
        unsigned st = R[k].status | ((C.cubic & 4u) << 2);      // ST_GRAD_ILLCOND of the cosmology (set by cosmo_prep with want_grad)
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
        if (kT && (which & W_AGE)) O[k].v[8] = C.tH * (C.Tinf - TT);
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
    if (!with_grad) return;
    const double iE = R.iE;
    const double bt0 = -R.Em1 * iE, bt1 = (z - R.Em1) * iE, bt2 = (z * (X + 1.0) - R.Em1) * iE;
    for (int t = 0; t < 3; ++t)
        C.dTinf[t] = -0.5 * (C.GT[t][0] * R.I0 + C.GT[t][1] * R.K + C.GT[t][2] * bt0 + C.GT[t][3] * bt1 + C.GT[t][4] * bt2
                             + C.GT[t][5] * R.TT);
    // remainder beyond X of the Or-derivative, -1/2 int_X^inf (x^3 - x)/E^3 dx with E^2 ~ x^3 (Or x + Om): it decays only like
    // X^(-1/2) while matter dominates at X (2e-5/Om^1.5 at Or = 0); the Om and OL remainders are O(X^-3/2) and dropped.
    double rem;
    if (C.Or * X > 1.0e3 * C.Om) rem = 0.5 / (C.Or * sqrt(C.Or) * X * X);
    else rem = 2.0 * (2.0 * C.Or * X + C.Om) / (C.Om * C.Om * sqrt(X) * sqrt(C.Or * X + C.Om)) - 4.0 * sqrt(C.Or) / (C.Om * C.Om);
    C.dTinf[2] -= 0.5 * rem;
}

// VJP of one element: g[N_PLANES] upstream (entries outside `which` must be 0).  Adds to gz and gp[0..3] = (Om, OL, Or, H0).
// kCond: also return in *cond the cancellation factor max_theta sum_j |G_j basis_j| / max(|dI0/dtheta|, 1e-3 |I0|) of the
// chi-family gradient (status bit 16 of the ELEMENTWISE calls is derived from it).
// `which`: planes that can carry a non-zero upstream gradient; where the caller knows it at compile time the terms of the
// other planes fold away (x * 0 is not foldable in IEEE arithmetic, so a zero g alone does not remove them).
template <typename T, bool kT, bool kA, bool kCond = false>
CB_HD void backward(const Cosmo<T>& C, T z, const Core<T>& R, const Obs<T>& O, const T g[N_PLANES], T& gz, T gp[4], T* cond = nullptr,
                    unsigned which = W_ALL) {
    using N = Num<T>;
    const T x = T(1) + z;
    const T iE = R.iE;
    const T rxd = N::rcp_(x * O.v[1]);                   // 1/(x D_M): one reciprocal serves 1/x and 1/D_M
    const T ix = O.v[1] * rxd;
    // boundary terms b_k = x^k / E - 1 (cancellation-free)
    const T xp1 = x + T(1);
    const T n1 = z, n2 = z * xp1, n3 = z * N::fma_(xp1, x, T(1)), n4 = n2 * N::fma_(x, x, T(1));
    const T bt0 = -R.Em1 * iE, bt1 = (n1 - R.Em1) * iE, bt2 = (n2 - R.Em1) * iE;
    T gM = T(0);
    if (which & W_DM) gM = g[1];
    if (which & W_DL) gM = N::fma_(x, g[2], gM);
    if ((which & W_MU) && g[3] != T(0)) gM = N::fma_(T(CB_KT.five_over_ln10) * g[3], x * rxd, gM);
    if ((which & W_DA) && g[6] != T(0)) gM = N::fma_(g[6], ix, gM);     // D_A = D_M / (1+z)
    T aI = C.dH * ((which & W_DC) ? N::fma_(gM, O.Fi, g[0]) : gM * O.Fi);
    T aK = -gM * C.dH * O.Fk;
    if ((which & W_VC) && g[7] != T(0)) {                                                 // V_C = 4 pi dH^3 v(Ok, I0): dv = F^2 dI0 + v_k dOk
        const T c4pi = T(12.566370614359172954) * C.dH * C.dH * C.dH * g[7];
        aI = N::fma_(c4pi, O.F * O.F, aI);
        aK = N::fma_(-c4pi, O.Vk, aK);
    }
    T btA = T(0);
    if (kA) btA = (((C.cubic & 1u) ? n4 : n3) - R.Em1) * iE;
    // d_abs gradient where radiation is a perturbation: the exact basis above then multiplies the forward A by ~3/Or
    // (the x^5, x^6 rows), which loses Om/Or digits.  Instead J'_p = int x^p dx/E^3, p <= 4, come from the basis and
    // J'_5.. follow from d(x^k / E) = N_k / E^3:  Om (k - 3/2) J'_{k+2} = [x^k/E] - k OL J'_{k-1} - (k-1) Ok J'_{k+1}
    // - (k-2) Or J'_{k+3}, the Or terms iterated (same scheme as the forward d_abs).
    bool useJ = false;
    T Jp[17];
    if (kA) {
        constexpr int KJ = 12;                // levels k = 3 .. 3 + KJ - 1
#pragma unroll
        for (int p = 0; p < 5; ++p)
            Jp[p] = C.GJ[p][0] * R.I0 + C.GJ[p][1] * R.K + C.GJ[p][2] * bt0 + C.GJ[p][3] * bt1 + C.GJ[p][4] * bt2;
#pragma unroll
        for (int p = 5; p < 17; ++p) Jp[p] = T(0);
        T bk[KJ];
        {
            T xk = x * x * x;
#pragma unroll
            for (int j = 0; j < KJ; ++j) { bk[j] = N::fma_(xk - T(1), iE, bt0); xk *= x; }     // x^k/E - 1 = (x^k - 1)/E + (1/E - 1)
        }
        T prev5 = T(0), prev6 = T(0);
#pragma unroll
        for (int sw = 0; sw < KJ - 1; ++sw) {
            if (sw == KJ - 2) { prev5 = Jp[5]; prev6 = Jp[6]; }
#pragma unroll
            for (int j = 0; j < KJ - 1 - sw; ++j) {
                const int k = 3 + j;
                const T a = bk[j] - T(k) * C.OL * Jp[k - 1] - T(k - 1) * C.Ok * Jp[k + 1] - T(k - 2) * C.Or * Jp[k + 3];
                Jp[k + 2] = a * C.iOm * T(1.0 / (k - 1.5));
            }
        }
        const T tol = T(sizeof(T) == 8 ? 1e-12 : 1e-5);
        useJ = N::abs_(Jp[5] - prev5) <= tol * N::abs_(Jp[5]) && N::abs_(Jp[6] - prev6) <= tol * N::abs_(Jp[6]);
    }
    const T aIh = T(-0.5) * aI;
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        T dI = C.GI[t][0] * R.I0 + C.GI[t][1] * R.K + C.GI[t][2] * bt0 + C.GI[t][3] * bt1 + C.GI[t][4] * bt2;
        if (kCond) {
            const T sa = N::abs_(C.GI[t][0] * R.I0) + N::abs_(C.GI[t][1] * R.K) + N::abs_(C.GI[t][2] * bt0) + N::abs_(C.GI[t][3] * bt1)
                         + N::abs_(C.GI[t][4] * bt2);
            const T c = sa / N::max_(N::abs_(dI), T(1e-3) * N::abs_(R.I0));
            if (t == 0 || c > *cond) *cond = c;
        }
        T acc = N::fma_(aIh, dI, aK);
        if (kT) {
            T dT = C.GT[t][0] * R.I0 + C.GT[t][1] * R.K + C.GT[t][2] * bt0 + C.GT[t][3] * bt1 + C.GT[t][4] * bt2 + C.GT[t][5] * R.TT;
            acc = N::fma_((g[4] - g[8]) * C.tH, T(-0.5) * dT, acc);       // t_L = tH T, age = tH (Tinf - T)
            acc = N::fma_(g[8] * C.tH, C.dTinf[t], acc);
        }
        if (kA) {
            T dA = C.GA[t][0] * R.I0 + C.GA[t][1] * R.K + C.GA[t][2] * bt0 + C.GA[t][3] * bt1 + C.GA[t][4] * bt2 + C.GA[t][5] * btA
                   + C.GA[t][6] * R.AA;
            if (useJ) dA = (t == 0 ? Jp[5] : (t == 1 ? Jp[2] : Jp[6])) - Jp[4];      // x^2 D_theta = x^5, x^2, x^6 minus x^4
            acc = N::fma_(g[5] * C.dH, T(-0.5) * dA, acc);
        }
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

}  // namespace cb
