// cosmo_two.cuh -- the TWO-LIMIT forms chi(z1,z2), t(z1,z2), d_abs(z1,z2) of eqs. (2.3)-(2.5) by
// eqs. (3.7)-(3.9) / (B.1)-(B.3) as printed (they are two-limit: Y_n = sqrt(z1 - r_n)), with analytic
// gradients wrt (z1, z2, Om, OL, Or, H0).  ELEMENTWISE only and kept apart from the z1 = 0 hot path (cosmo_eval.cuh), whose
// per-cosmology constants bake x1 = 1 in; it reuses the same Carlson device functions and the same gradient bases.
// Observables: D_C12, D_M12 = d_H sinn(sqrt|Ok| I0(z1,z2))/sqrt|Ok| (the transverse distance between two redshifts, as used
// for lensing), t12, d_abs12, D_A12 = D_M12/(1+z2).   FP64.
#pragma once
#include "cosmo_obs.cuh"

namespace cb {

struct Two {
    double v[5];            // DC, DM, TL, DABS, DA
    double gz1[5], gz2[5], gp[5][4];   // d v / d z1, d z2, d (Om, OL, Or, H0)
    unsigned status;
};

// kDefer (main pass of k_two's VJP): an element that needs a slow path -- complex root structure (cosmo_c4.cuh) or quadrature of the
// gradient integrals -- is only marked ST_INTERNAL_REDO; the second pass runs it again without kDefer (as the ELEMENTWISE kernels do).
template <typename Vote, bool kDefer = false>
CB_HD void eval_two(const Cosmo<double>& C, double z1, double z2, bool with_grad, const Vote& vote, Two& O) {
    const double x1 = 1.0 + z1, x2 = 1.0 + z2, dz = z2 - z1, dz2 = dz * dz;
    unsigned st[1] = {C.status};
    if (!(x1 > 0.0) || !(x2 > 0.0)) st[0] |= ST_UNSUPPORTED;
    if (fmax(x1, x2) >= C.xlim && fmin(x1, x2) < C.xlim) st[0] |= ST_ROOT_ON_PATH;
    double I0, K, TT, AA, E1, E2, dE;
    if (kDefer && (C.cubic & 2u)) {
        I0 = K = TT = AA = E1 = E2 = dE = NAN;
        st[0] |= ST_INTERNAL_REDO;
    } else if (C.cubic & 2u) {
        // two complex pairs (C.m, C.rn carry g1, h1): eqs. (3.7)-(3.9) as printed with a complex r_i, cosmo_c4.cuh
        eval_c4(C.Or, C.m, C.rn, C.b, C.c, x1, x2, dz, true, true, I0, TT, AA, K);
        E1 = sqrt(fma(fma(C.Or, x1, C.m), x1, C.rn) * fma(x1 + C.b, x1, C.c));
        E2 = sqrt(fma(fma(C.Or, x2, C.m), x2, C.rn) * fma(x2 + C.b, x2, C.c));
        const double s12 = x1 + x2, p12 = x1 * x2, sq = fma(x2, x2, x1 * x1);
        dE = dz * (C.Or * s12 * sq + C.Om * (sq + p12) + C.Ok * s12) / (E1 + E2);
    } else {
        const bool quartA = !(C.cubic & 1u);
        // ---- S4 radicands with both limits
        const double L1 = fma(C.Or, x1, C.m), L2 = fma(C.Or, x2, C.m), xm1 = x1 - C.rn, xm2 = x2 - C.rn;
        const double q21 = fma(x1 + C.b, x1, C.c), q22 = fma(x2 + C.b, x2, C.c);
        const double a1 = L2 * xm2 * q21, a2 = L1 * xm1 * q22;
        const double ra = cb_sqrt0(a1), rb = cb_sqrt0(a2), U12 = ra + rb;
        double xa[1] = {U12 * U12}, mp[1], s[1], p5[1], p0[1];
        const double hd = 0.5 * dz2 * C.theta, hs = dz2 * C.sDr;
        mp[0] = xa[0] - hd;
        s[0] = dz2 * dz2 * C.sD;
        const double xa0 = xa[0], m0 = mp[0], s0 = s[0];
        p5[0] = fma(dz2, C.p5c, xa0);
        p0[0] = quartA ? fma(-C.Or * dz2, C.Q2n, xa0) : xa0;
        const double p5_0 = p5[0], p0_0 = p0[0];
        const double pm5 = p5_0 - m0, pm0 = p0_0 - m0;
        const double dl5[1] = {(p5_0 - xa0) * fma(pm5, pm5, -s0)}, dl0[1] = {(p0_0 - xa0) * fma(pm0, pm0, -s0)};
        const double Qc[1] = {carlson_Qc<double>(hd, hs, true)}, Q5v[1] = {carlson_Qj<double>(xa0, m0, hs, p5_0)},
                     Q0v[1] = {carlson_Qj<double>(xa0, m0, hs, p0_0)};
        double f, tailD[1], sum5[1], sum0[1];
        carlson_dup<double, true, true, true, 1, Vote>(xa, mp, s, p5, p0, dl5, dl0, Qc, Q5v, Q0v, st, vote, f, tailD, sum5, sum0);
        const double RF = carlson_rf_series<double>(xa[0], mp[0], f, hd, s0);
        const double RD = carlson_rd_series<double>(xa[0], mp[0], f, hd, s0, tailD[0]);
        const double RJ5 = carlson_rj_series<double>(xa[0], mp[0], p5[0], f, xa0, m0, s0, p5_0, sum5[0]);
        const double RJ0 = carlson_rj_series<double>(xa[0], mp[0], p0[0], f, xa0, m0, s0, p0_0, sum0[0]);
        // E at both limits; E2 - E1 without cancellation
        E1 = cb_sqrt0(L1 * xm1 * q21); E2 = ra * rb * cb_rcp(E1);
        const double s12 = x1 + x2, p12 = x1 * x2, sq = fma(x2, x2, x1 * x1);          // x1+x2, x1 x2, x1^2+x2^2
        dE = dz * (C.Or * s12 * sq + C.Om * (sq + p12) + C.Ok * s12) * cb_rcp(E1 + E2);
        const double rx12 = cb_rcp(xm1 * xm2), rL12 = cb_rcp(L1 * L2), rU = cb_rcp(U12);
        // ---- S6 reductions
        I0 = 2.0 * dz * RF;                                                // eq. (3.7)
        K = 2.0 * dz * fma(dz2 * CB_KT.third * C.W, RD, cb_sqrt0(L1 * L2 * rx12) * rU);
        const double qh = p12 * p5_0 * C.m * C.m * rL12;
        TT = 2.0 * dz * (dz2 * CB_KT.third * C.Gp * RJ5 + rc<double>(fma(dz2, C.OL, qh), qh) - C.OrM * RF);   // eq. (3.8)
        const double bnd = cb_sqrt0(xm1 * xm2) * rU;
        if (quartA) {                                                                   // eq. (3.9), (i,j,k,l) = (rn, pair, pair, big)
            const double q0 = p0_0 * rx12;
            const double B0 = fma(dz2 * CB_KT.third * C.Q2n * C.mOrn, RJ0, rc<double>(fma(C.Or, dz2, q0), q0));
            const double F1 = cb_sqrt0(xm1 * q21 * L2 * rL12), F2 = cb_sqrt0(xm2 * q22 * L1 * rL12);
            const double c2 = C.b - C.rn, c1 = fma(-C.rn, C.b, C.c);
            const double dC = (sq + p12) + fma(c2, s12, c1);                            // (C(x2) - C(x1)) / dz, C = (x - rn) Q2
            const double t1 = dz * fma(L1, dC, -xm1 * q21 * C.Or) * rL12 * cb_rcp(F1 + F2);
            const double t2 = dz * C.aF * RF;
            const double t3 = dz * C.WoOr * fma(dz2 * CB_KT.third * C.Q2n, RD, bnd * cb_sqrt0(rL12));
            const double t4 = dz * C.sig * B0;
            const double A39 = (t1 + t2) + (t3 + t4);
            // radiation-perturbative assembly (see eval_core_k): u_j = int x^j dx/E between the limits
            constexpr int KS = REC_KS;
            double bk[KS + 1], u2[KS + 1], trunc;
            const double u1 = fma(2.0 * dz, B0, C.rn * I0);
            double xk1 = 1.0, dk = 0.0;      // dk = x2^j - x1^j = x2 (x2^(j-1) - x1^(j-1)) + x1^(j-1) dz: no cancellation as z2 -> z1
            for (int j = 0; j <= KS; ++j) { bk[j] = fma(dk, E2, xk1 * dE); dk = fma(x2, dk, xk1 * dz); xk1 *= x1; }    // x2^j E2 - x1^j E1
            band_solve<double, KS + 1, 2, 1, 0, 0>(C.Om, C.OL, C.Or, C.Ok, bk, u1, I0, 0.0, fmax(x1, x2), u2, trunc);    // u2[j] = u_{j+2}
            AA = (trunc <= 1e-15 * fabs(u2[0])) ? u2[0] : A39;
        } else {                                                                        // eq. (B.3), i = rn
            AA = CB_KT.two_thirds * dz * (dE * cb_rcp(C.m * dz) + C.aF * RF + 2.0 * C.sig * fma(dz2 * CB_KT.third * C.Q2n * C.m, RD, bnd));
            if (dz == 0.0) AA = 0.0;
        }
    }
    // ---- S7
    double F, Fi, Fk;
    sinn<double>(C.Ok, I0, F, Fi, Fk);
    const double ix1 = cb_rcp(x1), ix2 = cb_rcp(x2);
    O.v[0] = C.dH * I0; O.v[1] = C.dH * F; O.v[2] = C.tH * TT; O.v[3] = C.dH * AA; O.v[4] = O.v[1] * ix2;
    O.status = st[0];
    if (st[0] & (ST_ROOT_ON_PATH | ST_UNSUPPORTED)) {
        for (int i = 0; i < 5; ++i) O.v[i] = NAN;
    }
    if (!with_grad) return;
    // ---- S8: the same bases (GI, GT, GA/GJ) on two-limit basis values; b_k = x2^k/E2 - x1^k/E1
    const double iE1 = cb_rcp(E1), iE2 = cb_rcp(E2), diE = -dE * iE1 * iE2;            // 1/E2 - 1/E1
    double btv[REC_KJ + 2];
    {
        double xk1 = 1.0, dk = 0.0;
        for (int k = 0; k < REC_KJ + 2; ++k) { btv[k] = fma(dk, iE2, xk1 * diE); dk = fma(x2, dk, xk1 * dz); xk1 *= x1; }
    }
    // raw gradient integrals int D_theta p_X / E^3 dx between the limits (cosmo_obs.cuh, GradInt) with their cancellation factor
    double rI[3], rT[3], rA[3];
    bool over = false;                   // cancellation factor above GRAD_COND_LIMIT somewhere (a NaN counts)
    auto worse = [&](double sa, double val, double fwd) { over = over | !(sa <= GRAD_COND_LIMIT * fmax(fabs(val), 1e-3 * fabs(fwd))); };
    // basis rows solved on the spot from the factorisation (cosmo_prep.cuh, GradSolve): nothing stored per cosmology
    GradSolve S;
    S.init(C);
    const double aI0 = fabs(I0), aK = fabs(K), a0 = fabs(btv[0]), a1 = fabs(btv[1]), a2 = fabs(btv[2]);
    auto dot5 = [&](const double* g) { return g[0] * I0 + g[1] * K + g[2] * btv[0] + g[3] * btv[1] + g[4] * btv[2]; };
    auto abs5 = [&](const double* g) { return fabs(g[0]) * aI0 + fabs(g[1]) * aK + fabs(g[2]) * a0 + fabs(g[3]) * a1 + fabs(g[4]) * a2; };
    double Jp[7], Sp[7];
    bool useJ = false;
    {
        constexpr int KJ = REC_KJ;
        Jp[0] = Jp[1] = 0.0; Sp[0] = Sp[1] = 0.0;
        for (int p = 2; p < 5; ++p) {
            double g[5];
            S.rowJ(p, g);
            Jp[p] = dot5(g); Sp[p] = abs5(g);
        }
        double bj[KJ - 1], vj[KJ - 1], trunc;
#pragma unroll
        for (int j = 0; j < KJ - 1; ++j) bj[j] = btv[3 + j];
        band_solve<double, KJ - 1, 1, 2, 3, 1>(C.Om, C.OL, C.Or, C.Ok, bj, Jp[4], Jp[3], Jp[2], fmax(x1, x2), vj, trunc);    // vj[j] = J'_{j+5}
        Jp[5] = vj[0]; Jp[6] = vj[1];
        useJ = trunc <= 1e-13 * fabs(Jp[5]) && trunc <= 1e-13 * fabs(Jp[6]);
        Sp[5] = (fabs(btv[3]) + 3.0 * C.OL * Sp[2] + 2.0 * fabs(C.Ok) * Sp[4]) * C.iOm / 1.5;
        Sp[6] = (fabs(btv[4]) + 4.0 * C.OL * Sp[3] + 3.0 * fabs(C.Ok) * Sp[5]) * C.iOm / 2.5;
    }
    const double btA = (C.cubic & 1u) ? btv[4] : btv[3];
    for (int t = 0; t < 3; ++t) {
        double g[7];
        S.rowI(t, g);
        rI[t] = dot5(g);
        worse(abs5(g), rI[t], I0);
        S.rowT(t, g);
        rT[t] = dot5(g) + g[5] * TT;
        worse(abs5(g) + fabs(g[5] * TT), rT[t], TT);
        const int ia = t == 0 ? 5 : (t == 1 ? 2 : 6);
        if (useJ) {
            rA[t] = Jp[ia] - Jp[4];
            worse(Sp[ia] + Sp[4], rA[t], AA);
        } else {
            S.rowA(t, g);
            rA[t] = dot5(g) + g[5] * btA + g[6] * AA;
            worse(abs5(g) + fabs(g[5] * btA) + fabs(g[6] * AA), rA[t], AA);
        }
    }
    // ill-conditioned bases (near-repeated roots away from the path, tiny ranges): quadrature of the same integrals (grad_quad)
    if (kDefer) {
        if ((over || S.singular) && !(st[0] & (ST_ROOT_ON_PATH | ST_UNSUPPORTED))) O.status |= ST_INTERNAL_REDO;
    } else if ((over || S.singular) && !(st[0] & (ST_ROOT_ON_PATH | ST_UNSUPPORTED))) {
        double q[9];
        O.status |= grad_quad(C.Om, C.OL, C.Or, -0.5 * C.b, 0.25 * C.b * C.b - C.c, z1, dz, true, true, q);
        for (int t = 0; t < 3; ++t) { rI[t] = q[t]; rT[t] = q[3 + t]; rA[t] = q[6 + t]; }
    }
    for (int t = 0; t < 3; ++t) {
        const double dI = -0.5 * rI[t], dT = -0.5 * rT[t], dA = -0.5 * rA[t];
        O.gp[0][t] = C.dH * dI;
        O.gp[1][t] = C.dH * (Fi * dI - Fk);
        O.gp[2][t] = C.tH * dT;
        O.gp[3][t] = C.dH * dA;
        O.gp[4][t] = O.gp[1][t] * ix2;
    }
    const double iH0 = C.dH * (1.0 / C_KM_S);
    for (int o = 0; o < 5; ++o) O.gp[o][3] = -O.v[o] * iH0;
    O.gz1[0] = -C.dH * iE1;            O.gz2[0] = C.dH * iE2;
    O.gz1[1] = -C.dH * Fi * iE1;       O.gz2[1] = C.dH * Fi * iE2;
    O.gz1[2] = -C.tH * iE1 * ix1;      O.gz2[2] = C.tH * iE2 * ix2;
    O.gz1[3] = -C.dH * x1 * x1 * iE1;  O.gz2[3] = C.dH * x2 * x2 * iE2;
    O.gz1[4] = O.gz1[1] * ix2;         O.gz2[4] = O.gz2[1] * ix2 - O.v[1] * (ix2 * ix2);
}

}  // namespace cb
