// tu_w.cu -- the kernels of the extra-w family (cosmo_w.cuh; PAPER.md:82 fn.4) and their launcher.  A translation unit of its own
// because complex arithmetic is this family's MAIN path: CB_CX_FAST selects the MUFU-seeded complex division / modulus / square root
// (cosmo_c4.cuh), which the hot path's rare complex rows do not use.
#define CB_CX_FAST 1
#include "cosmo_kernels.cuh"
#include "cosmo_w.cuh"

namespace cb {

// Extra constant-w components (cosmo_w.cuh), one thread per (z, cosmology); n_cosmo in {1, n}.  which: DC, DM, DL, MU, TL, DABS.
// out[n_which][n]; dout[n_which][n] = d out / dz (nullable); with gout the VJP: gz[n], gparams[6][n] (Om, OL, Or, Ow13, Ow23, H0).
// A shared cosmology is factored ONCE per call by k_w_prep (into the workspace), not once per thread or block.
__global__ void k_w_prep(const double* Om, const double* OL, const double* Or, const double* Ow13, const double* Ow23, const double* H0,
                         WCosmo* out) {
    if (blockIdx.x == 0 && threadIdx.x == 0) w_prep(Om[0], OL[0], Or[0], Ow13[0], Ow23[0], H0[0], *out);
}

template <bool kG, bool kTA>
__global__ void __launch_bounds__(ELEM_THREADS) k_w(const double* __restrict__ z, const double* __restrict__ Om,
                                                    const double* __restrict__ OL, const double* __restrict__ Or,
                                                    const double* __restrict__ Ow13, const double* __restrict__ Ow23,
                                                    const double* __restrict__ H0, int64_t n, int64_t n_cosmo, unsigned which,
                                                    const WCosmo* __restrict__ shared_cosmo, const double* __restrict__ gout,
                                                    double* __restrict__ out, double* __restrict__ dout, double* __restrict__ gz,
                                                    double* __restrict__ gparams, uint8_t* __restrict__ status) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool live = i < n;
    const int64_t ii = live ? i : n - 1;
    WCosmo W;
    if (n_cosmo == 1) W = *shared_cosmo;
    else w_prep(Om[ii], OL[ii], Or[ii], Ow13[ii], Ow23[ii], H0[ii], W);
    const unsigned bits[6] = {W_DC, W_DM, W_DL, W_MU, W_TL, W_DABS};
    double v[6], dz[6], gp[6][6];
    unsigned st;
    if (kTA || kG) {
        st = w_eval_full<VoteWarp>(W, z[ii], VoteWarp(), kTA && (which & W_TL), kTA && (which & W_DABS), kG, v, dz, gp);
    } else {          // chi family, forward: the lean path (no complex arithmetic, no quadrature compiled in)
        st = w_eval<VoteWarp>(W, z[ii], VoteWarp(), v, dz);
        v[4] = v[5] = dz[4] = dz[5] = NAN;
    }
    if (!live) return;
    double az = 0.0, ap[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    int pl = 0;
    for (int o = 0; o < 6; ++o) {
        if (!(which & bits[o])) continue;
        if (out != nullptr) out[(int64_t)pl * n + i] = v[o];
        if (dout != nullptr) dout[(int64_t)pl * n + i] = dz[o];
        if (kG) {
            const double g = gout[(int64_t)pl * n + i];
            if (g != 0.0) {                    // (a plane that is NaN for this element must not poison the others: 0 x NaN)
                az = fma(g, dz[o], az);
                for (int t = 0; t < 6; ++t) ap[t] = fma(g, gp[o][t], ap[t]);
            }
        }
        ++pl;
    }
    if (status != nullptr) status[i] = (uint8_t)st;
    if (kG) {
        gz[i] = az;
        for (int t = 0; t < 6; ++t) gparams[(int64_t)t * n + i] = ap[t];
    }
}

size_t w_cosmo_bytes() { return sizeof(WCosmo); }
void launch_w(const double* z, const double* Om, const double* OL, const double* Or, const double* Ow13, const double* Ow23,
              const double* H0, int64_t n, int64_t n_cosmo, unsigned which, const double* gout, double* out, double* dout, double* gz,
              double* gparams, uint8_t* status, void* ws, cudaStream_t st) {
    WCosmo* shared = static_cast<WCosmo*>(ws);
    if (n_cosmo == 1) k_w_prep<<<1, 32, 0, st>>>(Om, OL, Or, Ow13, Ow23, H0, shared);
    const unsigned grid = (unsigned)cdiv64(n, ELEM_THREADS);
    const bool ta = (which & (W_TL | W_DABS)) != 0;
    if (gout && ta) k_w<true, true><<<grid, ELEM_THREADS, 0, st>>>(z, Om, OL, Or, Ow13, Ow23, H0, n, n_cosmo, which, shared, gout, out, dout, gz, gparams, status);
    else if (gout) k_w<true, false><<<grid, ELEM_THREADS, 0, st>>>(z, Om, OL, Or, Ow13, Ow23, H0, n, n_cosmo, which, shared, gout, out, dout, gz, gparams, status);
    else if (ta) k_w<false, true><<<grid, ELEM_THREADS, 0, st>>>(z, Om, OL, Or, Ow13, Ow23, H0, n, n_cosmo, which, shared, nullptr, out, dout, nullptr, nullptr, status);
    else k_w<false, false><<<grid, ELEM_THREADS, 0, st>>>(z, Om, OL, Or, Ow13, Ow23, H0, n, n_cosmo, which, shared, nullptr, out, dout, nullptr, nullptr, status);
}
}  // namespace cb
