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
    T v[6];            // DC, DM, DL, MU, TL, DABS
    T F, Fi, Fk;       // curvature transform and its partials
    unsigned status;
};

// Rows whose E^2 has no real negative root (Cosmo::cubic bit 1): replace the fused real path's result by the complex
// slow path (cosmo_c4.cuh).  Forward values only: K, 1/E are poisoned so that every gradient of such a row is NaN.
template <typename T, bool kT, bool kA, bool kGrad>
CB_HD void apply_c4(const Cosmo<T>& C, T z, Core<T>& R) {
    if (!(C.cubic & 2u)) return;
    double I0, TT, AA;
    eval_c4((double)C.Or, (double)C.m, (double)C.rn, (double)C.b, (double)C.c, (double)z, kT, kA, I0, TT, AA);
    R.I0 = (T)I0; R.TT = (T)TT; R.AA = (T)AA;
    R.K = T(NAN); R.iE = T(NAN);
    R.status = C.status | ((T(1) + z > T(0)) ? 0u : (unsigned)ST_UNSUPPORTED) | (kGrad ? (unsigned)ST_GRAD_ILLCOND : 0u);
}

template <typename T, bool kT, bool kA>
CB_HD void observables(const Cosmo<T>& C, T z, const Core<T>& R, unsigned which, Obs<T>& O) {
    using N = Num<T>;
    const T x = T(1) + z;
    unsigned st = R.status;
    sinn<T>(C.Ok, R.I0, O.F, O.Fi, O.Fk);
    O.v[0] = C.dH * R.I0;
    O.v[1] = C.dH * O.F;
    O.v[2] = x * O.v[1];
    O.v[3] = T(0);
    if (which & W_MU) {
        if (O.v[2] > T(0)) O.v[3] = N::fma_(T(CB_KT.five_over_ln10), N::log_(O.v[2]), T(25));
        else { O.v[3] = T(NAN); st |= ST_DL_NONPOS; }
    }
    O.v[4] = kT ? C.tH * R.TT : T(0);
    O.v[5] = kA ? C.dH * R.AA : T(0);
    if (st & (ST_ROOT_ON_PATH | ST_UNSUPPORTED)) {
#pragma unroll
        for (int i = 0; i < 6; ++i) O.v[i] = T(NAN);
    }
    O.status = st;
}

// VJP of one element: g[6] upstream (entries outside `which` must be 0).  Adds to gz and gp[0..3] = (Om, OL, Or, H0).
// kCond: also return in *cond the cancellation factor max_theta sum_j |G_j basis_j| / max(|dI0/dtheta|, 1e-3 |I0|) of the
// chi-family gradient (status bit 16 of the ELEMENTWISE calls is derived from it).
template <typename T, bool kT, bool kA, bool kCond = false>
CB_HD void backward(const Cosmo<T>& C, T z, const Core<T>& R, const Obs<T>& O, const T g[6], T& gz, T gp[4], T* cond = nullptr) {
    using N = Num<T>;
    const T x = T(1) + z;
    const T iE = R.iE;
    const T rxd = N::rcp_(x * O.v[1]);                   // 1/(x D_M): one reciprocal serves 1/x and 1/D_M
    const T ix = O.v[1] * rxd;
    // boundary terms b_k = x^k / E - 1 (cancellation-free)
    const T xp1 = x + T(1);
    const T n1 = z, n2 = z * xp1, n3 = z * N::fma_(xp1, x, T(1)), n4 = n2 * N::fma_(x, x, T(1));
    const T bt0 = -R.Em1 * iE, bt1 = (n1 - R.Em1) * iE, bt2 = (n2 - R.Em1) * iE;
    T gM = g[1] + x * g[2];
    if (g[3] != T(0)) gM += T(CB_KT.five_over_ln10) * g[3] * (x * rxd);
    const T aI = C.dH * N::fma_(gM, O.Fi, g[0]);
    const T aK = -gM * C.dH * O.Fk;
    T btA = T(0);
    if (kA) btA = (((C.cubic & 1u) ? n4 : n3) - R.Em1) * iE;
    // d_abs gradient where radiation is a perturbation: the exact basis above then multiplies the forward A by ~3/Or
    // (the x^5, x^6 rows), which loses Om/Or digits.  Instead J'_p = int x^p dx/E^3, p <= 4, come from the basis and
    // J'_5.. follow from d(x^k / E) = N_k / E^3:  Om (k - 3/2) J'_{k+2} = [x^k/E] - k OL J'_{k-1} - (k-1) Ok J'_{k+1}
    // - (k-2) Or J'_{k+3}, the Or terms iterated (same scheme as the forward d_abs).
    bool useJ = false;
    T Jp[17];
    if (kA && !(C.cubic & 2u)) {
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
#pragma unroll
    for (int t = 0; t < 3; ++t) {
        T dI = C.GI[t][0] * R.I0 + C.GI[t][1] * R.K + C.GI[t][2] * bt0 + C.GI[t][3] * bt1 + C.GI[t][4] * bt2;
        if (kCond) {
            const T sa = N::abs_(C.GI[t][0] * R.I0) + N::abs_(C.GI[t][1] * R.K) + N::abs_(C.GI[t][2] * bt0) + N::abs_(C.GI[t][3] * bt1)
                         + N::abs_(C.GI[t][4] * bt2);
            const T c = sa / N::max_(N::abs_(dI), T(1e-3) * N::abs_(R.I0));
            if (t == 0 || c > *cond) *cond = c;
        }
        T acc = N::fma_(aI, T(-0.5) * dI, aK);
        if (kT) {
            T dT = C.GT[t][0] * R.I0 + C.GT[t][1] * R.K + C.GT[t][2] * bt0 + C.GT[t][3] * bt1 + C.GT[t][4] * bt2 + C.GT[t][5] * R.TT;
            acc = N::fma_(g[4] * C.tH, T(-0.5) * dT, acc);
        }
        if (kA) {
            T dA = C.GA[t][0] * R.I0 + C.GA[t][1] * R.K + C.GA[t][2] * bt0 + C.GA[t][3] * bt1 + C.GA[t][4] * bt2 + C.GA[t][5] * btA
                   + C.GA[t][6] * R.AA;
            if (useJ) dA = (t == 0 ? Jp[5] : (t == 1 ? Jp[2] : Jp[6])) - Jp[4];      // x^2 D_theta = x^5, x^2, x^6 minus x^4
            acc = N::fma_(g[5] * C.dH, T(-0.5) * dA, acc);
        }
        gp[t] += acc;
    }
    T h = g[0] * O.v[0] + g[1] * O.v[1] + g[2] * O.v[2] + g[3] * T(CB_KT.five_over_ln10);
    if (kT) h += g[4] * O.v[4];
    if (kA) h += g[5] * O.v[5];
    gp[3] -= h * C.dH * T(1.0 / C_KM_S);        // / H0
    T dz = aI * iE + g[2] * O.v[1];
    if (g[3] != T(0)) dz += T(CB_KT.five_over_ln10) * g[3] * ix;
    if (kT) dz += g[4] * C.tH * iE * ix;
    if (kA) dz += g[5] * C.dH * x * x * iE;
    gz += dz;
}

}  // namespace cb
