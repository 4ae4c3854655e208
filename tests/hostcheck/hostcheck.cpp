// hostcheck.cpp -- TEST HELPER ONLY (never loaded by the product path).
// Compiles the per-element math headers of the CUDA path (paper_2212_01937_b200/csrc/*.cuh) with plain g++ so that
// `-m "not gpu"` tests can check that host-compiled arithmetic against the oracle before any GPU time is spent.
// The product runs these same headers inside CUDA kernels only; there is no CPU fallback (see binding.py).
#include <stdint.h>
#include "../../paper_2212_01937_b200/csrc/cosmo_prep.cuh"
#include "../../paper_2212_01937_b200/csrc/cosmo_obs.cuh"
#include "../../paper_2212_01937_b200/csrc/cosmo_two.cuh"
#include "../../paper_2212_01937_b200/csrc/cosmo_w.cuh"

using namespace cb;

template <typename T>
static void run(int64_t n, const double* z, const double* Om, const double* OL, const double* Or, const double* H0,
                unsigned which, const double* gup, double* out, double* gz, double* gp, uint8_t* status) {
    for (int64_t i = 0; i < n; ++i) {
        Cosmo<double> Cd;
        cosmo_prep(Om[i], OL[i], Or[i], H0[i], gup ? 2 : 0, Cd);
        if (which & W_AGE) prep_age(Cd, gup != nullptr);
        else { Cd.Tinf = 0; Cd.dTinf[0] = Cd.dTinf[1] = Cd.dTinf[2] = 0; }
        Cosmo<T> C;
        convert_cosmo<T>(Cd, C);
        Core<T> R;
        R.K = 0; R.TT = 0; R.AA = 0;
        eval_core<T, true, true, true, VoteNone>(C, (T)z[i], VoteNone(), R);
        if (gup) apply_c4<T, true, true, true>(C, (T)z[i], R); else apply_c4<T, true, true, false>(C, (T)z[i], R);
        Obs<T> O;
        observables<T, true, true>(C, (T)z[i], R, which, O);
        for (int w = 0; w < N_PLANES; ++w) out[w * n + i] = (double)O.v[w];
        status[i] = (uint8_t)O.status;
        if (gup) {
            T g[N_PLANES], a = 0, p[4] = {0, 0, 0, 0};
            for (int w = 0; w < N_PLANES; ++w) g[w] = (which >> w & 1) ? (T)gup[w * n + i] : T(0);
            // what the OUTER kernels' checked row does: bases where accurate, quadrature elsewhere
            status[i] |= (uint8_t)backward_robust<T, true, true>(C, (T)z[i], R, O, g, a, p, which);
            gz[i] = (double)a;
            for (int t = 0; t < 4; ++t) gp[t * n + i] = (double)p[t];
        }
    }
}

extern "C" void hostcheck_f64(int64_t n, const double* z, const double* Om, const double* OL, const double* Or, const double* H0,
                              unsigned which, const double* gup, double* out, double* gz, double* gp, uint8_t* status) {
    run<double>(n, z, Om, OL, Or, H0, which, gup, out, gz, gp, status);
}
extern "C" void hostcheck_f32(int64_t n, const double* z, const double* Om, const double* OL, const double* Or, const double* H0,
                              unsigned which, const double* gup, double* out, double* gz, double* gp, uint8_t* status) {
    run<float>(n, z, Om, OL, Or, H0, which, gup, out, gz, gp, status);
}
// exactly what the ELEMENTWISE kernel k_elem runs per element (cosmo_obs.cuh, elem_one): no stored bases, constants re-formed after the loop
template <typename T>
static void run_elem(int64_t n, const double* z, const double* Om, const double* OL, const double* Or, const double* H0, unsigned which,
                     const double* gup, double* out, double* gz, double* gp, uint8_t* status) {
    for (int64_t i = 0; i < n; ++i) {
        T g[N_PLANES], v[N_PLANES], dz = 0, p[4] = {0, 0, 0, 0};
        for (int w = 0; w < N_PLANES; ++w) g[w] = (gup && (which >> w & 1)) ? (T)gup[w * n + i] : T(0);
        unsigned st = gup ? elem_one<T, true, true, true, VoteNone>((T)z[i], Om[i], OL[i], Or[i], H0[i], which, VoteNone(), g, v, dz, p)
                          : elem_one<T, true, true, false, VoteNone>((T)z[i], Om[i], OL[i], Or[i], H0[i], which, VoteNone(), g, v, dz, p);
        for (int w = 0; w < N_PLANES; ++w) out[w * n + i] = (double)v[w];
        status[i] = (uint8_t)st;
        if (gup) { gz[i] = (double)dz; for (int t = 0; t < 4; ++t) gp[t * n + i] = (double)p[t]; }
    }
}
extern "C" void hostcheck_elem_f64(int64_t n, const double* z, const double* Om, const double* OL, const double* Or, const double* H0,
                                   unsigned which, const double* gup, double* out, double* gz, double* gp, uint8_t* status) {
    run_elem<double>(n, z, Om, OL, Or, H0, which, gup, out, gz, gp, status);
}
extern "C" void hostcheck_elem_f32(int64_t n, const double* z, const double* Om, const double* OL, const double* Or, const double* H0,
                                   unsigned which, const double* gup, double* out, double* gz, double* gp, uint8_t* status) {
    run_elem<float>(n, z, Om, OL, Or, H0, which, gup, out, gz, gp, status);
}
extern "C" void hostcheck_factor(double Om, double OL, double Or, double* out5) {
    Cosmo<double> C;
    cosmo_prep(Om, OL, Or, 70.0, 0, C);
    out5[0] = C.m; out5[1] = C.rn; out5[2] = C.b; out5[3] = C.c; out5[4] = (double)C.status;
}

// two-limit path: val[5][n], gz1[5][n], gz2[5][n], gp[5][4][n]
extern "C" void hostcheck_two(int64_t n, const double* z1, const double* z2, const double* Om, const double* OL, const double* Or,
                              const double* H0, double* val, double* gz1, double* gz2, double* gp, uint8_t* status) {
    for (int64_t i = 0; i < n; ++i) {
        Cosmo<double> C{};
        cosmo_factor(Om[i], OL[i], Or[i], H0[i], C);
        cosmo_constants(C);
        Two O;
        eval_two<VoteNone>(C, z1[i], z2[i], true, VoteNone(), O);
        for (int o = 0; o < 5; ++o) {
            val[o * n + i] = O.v[o]; gz1[o * n + i] = O.gz1[o]; gz2[o * n + i] = O.gz2[o];
            for (int t = 0; t < 4; ++t) gp[(o * 4 + t) * n + i] = O.gp[o][t];
        }
        status[i] = (uint8_t)O.status;
    }
}

// extra constant-w components (cosmo_w.cuh): val[4][n], dz[4][n]
extern "C" void hostcheck_w(int64_t n, const double* z, const double* Om, const double* OL, const double* Or, const double* Ow13,
                            const double* Ow23, const double* H0, double* val, double* dz, uint8_t* status) {
    for (int64_t i = 0; i < n; ++i) {
        WCosmo W;
        w_prep(Om[i], OL[i], Or[i], Ow13[i], Ow23[i], H0[i], W);
        double v[4], d[4];
        status[i] = (uint8_t)w_eval<VoteNone>(W, z[i], VoteNone(), v, d);
        for (int o = 0; o < 4; ++o) { val[o * n + i] = v[o]; dz[o * n + i] = d[o]; }
    }
}

// the w family in full (cosmo_w.cuh, w_eval_full): val[6][n], dz[6][n], gp[6][6][n] (observable, parameter, element)
extern "C" void hostcheck_w_full(int64_t n, const double* z, const double* Om, const double* OL, const double* Or, const double* Ow13,
                                 const double* Ow23, const double* H0, double* val, double* dz, double* gp, uint8_t* status) {
    for (int64_t i = 0; i < n; ++i) {
        WCosmo W;
        w_prep(Om[i], OL[i], Or[i], Ow13[i], Ow23[i], H0[i], W);
        double v[6], d[6], g[6][6];
        status[i] = (uint8_t)w_eval_full<VoteNone>(W, z[i], VoteNone(), true, true, true, v, d, g);
        for (int o = 0; o < 6; ++o) {
            val[o * n + i] = v[o]; dz[o * n + i] = d[o];
            for (int t = 0; t < 6; ++t) gp[(o * 6 + t) * n + i] = g[o][t];
        }
    }
}

// the curvature transform on its own (cosmo_eval.cuh, sinn): F = I0 S(w), Fi = C(w), Fk = I0^3 S'(w), w = k I0^2
extern "C" void hostcheck_sinn(int64_t n, const double* k, const double* I0, double* F, double* Fi, double* Fk) {
    for (int64_t i = 0; i < n; ++i) sinn<double>(k[i], I0[i], F[i], Fi[i], Fk[i]);
}

// the banded solve of the d_abs moment recurrences on its own (cosmo_eval.cuh, band_solve), in the two shapes the path uses:
// shape 0: value (rows k = 0..8: SO, AO, CO = 2, 1, 0), shape 1: gradient (rows k = 3..13: 1, 2, 3; error bound from row 1 on)
extern "C" void hostcheck_band(int shape, double Om, double OL, double Or, double Ok, const double* b, double km1, double km2, double km3,
                               double x, double* v, double* trunc) {
    if (shape == 0) {
        double bb[REC_KS + 1], vv[REC_KS + 1];
        for (int j = 0; j <= REC_KS; ++j) bb[j] = b[j];
        band_solve<double, REC_KS + 1, 2, 1, 0, 0>(Om, OL, Or, Ok, bb, km1, km2, km3, x, vv, *trunc);
        for (int j = 0; j <= REC_KS; ++j) v[j] = vv[j];
    } else {
        double bb[REC_KJ - 1], vv[REC_KJ - 1];
        for (int j = 0; j < REC_KJ - 1; ++j) bb[j] = b[j];
        band_solve<double, REC_KJ - 1, 1, 2, 3, 1>(Om, OL, Or, Ok, bb, km1, km2, km3, x, vv, *trunc);
        for (int j = 0; j < REC_KJ - 1; ++j) v[j] = vv[j];
    }
}
