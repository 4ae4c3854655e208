// tu_w.cu -- the kernels of the extra-w family (cosmo_w.cuh; PAPER.md:82 fn.4) and their launcher.  A translation unit of its own
// because complex arithmetic is this family's MAIN path: CB_CX_FAST selects the MUFU-seeded complex division / modulus / square root
// (cosmo_c4.cuh), which the hot path's rare complex rows do not use.
#define CB_CX_FAST 1
#include "cosmo_kernels.cuh"
#include "cosmo_w.cuh"

namespace cb {

// Extra constant-w components (cosmo_w.cuh), one thread per (z, cosmology); n_cosmo in {1, n}.  which: DC, DM, DL, MU, TL, DABS.
// out[n_which][n]; dout[n_which][n] = d out / dz (nullable); with gout the VJP: gz[n], gparams[6][n] (Om, OL, Or, Ow13, Ow23, H0).
// A shared cosmology is factored ONCE per call by k_w_prep (into the workspace), not once per thread or block.  Per-element
// cosmologies: two passes as k_elem -- the structured root solve for every element, the general one (a few per cent of a mixed batch,
// but enough to stall every warp) for the listed rest.
__global__ void k_w_prep(const double* Om, const double* OL, const double* Or, const double* Ow13, const double* Ow23, const double* H0,
                         WCosmo* out) {
    if (blockIdx.x == 0 && threadIdx.x == 0) w_prep(Om[0], OL[0], Or[0], Ow13[0], Ow23[0], H0[0], *out);
}

struct WArgs {
    const double *z, *Om, *OL, *Or, *Ow13, *Ow23, *H0;
    int64_t n, n_cosmo; unsigned which;
    const WCosmo* shared_cosmo; const double* gout; double *out, *dout, *gz, *gparams; uint8_t* status;
    unsigned *redo_count, *redo_list;       // per-element cosmologies: work list of the second pass (workspace)
};

// one element.  kDefer: main pass -- an element whose E^2 needs the general root solve is not evaluated, only reported (returns
// ST_INTERNAL_REDO, writes nothing); the second pass runs it with kDefer = false.
template <bool kG, bool kTA, bool kDefer, typename Vote>
__device__ __forceinline__ unsigned w_one(const WArgs& a, int64_t i, bool live, const Vote& vote) {
    const int64_t n = a.n, ii = live ? i : n - 1;
    WCosmo W;
    if (a.n_cosmo == 1) W = *a.shared_cosmo;
    else w_prep<kDefer>(a.Om[ii], a.OL[ii], a.Or[ii], a.Ow13[ii], a.Ow23[ii], a.H0[ii], W);
    const bool redo = kDefer && (W.status & ST_INTERNAL_REDO);
    const unsigned bits[6] = {W_DC, W_DM, W_DL, W_MU, W_TL, W_DABS};
    double v[6], dz[6], gp[6][6];
    unsigned st;
    if (kTA || kG) {
        st = w_eval_full<Vote>(W, a.z[ii], vote, kTA && (a.which & W_TL), kTA && (a.which & W_DABS), kG, v, dz, gp);
    } else {          // chi family, forward: the lean path (no complex arithmetic, no quadrature compiled in)
        st = w_eval<Vote>(W, a.z[ii], vote, v, dz);
        v[4] = v[5] = dz[4] = dz[5] = NAN;
    }
    if (!live) return 0u;
    if (redo) return (unsigned)ST_INTERNAL_REDO;
    double az = 0.0, ap[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    int pl = 0;
    for (int o = 0; o < 6; ++o) {
        if (!(a.which & bits[o])) continue;
        if (a.out != nullptr) a.out[(int64_t)pl * n + i] = v[o];
        if (a.dout != nullptr) a.dout[(int64_t)pl * n + i] = dz[o];
        if (kG) {
            const double g = a.gout[(int64_t)pl * n + i];
            if (g != 0.0) {                    // (a plane that is NaN for this element must not poison the others: 0 x NaN)
                az = fma(g, dz[o], az);
                for (int t = 0; t < 6; ++t) ap[t] = fma(g, gp[o][t], ap[t]);
            }
        }
        ++pl;
    }
    if (a.status != nullptr) a.status[i] = (uint8_t)st;
    if (kG) {
        a.gz[i] = az;
        for (int t = 0; t < 6; ++t) a.gparams[(int64_t)t * n + i] = ap[t];
    }
    return 0u;
}

template <bool kG, bool kTA, bool kDefer>
__global__ void __launch_bounds__(ELEM_THREADS) k_w(WArgs a) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool live = i < a.n;
    const unsigned st = w_one<kG, kTA, kDefer, VoteWarp>(a, i, live, VoteWarp());
    if (kDefer) {       // work list of the second pass: one atomic per warp
        const bool redo = live && (st & ST_INTERNAL_REDO);
        const unsigned active = __activemask();
        const unsigned m = __ballot_sync(active, redo);
        if (m) {
            const int lane = threadIdx.x & 31, leader = __ffs(m) - 1;
            unsigned base = 0;
            if (lane == leader) base = atomicAdd(a.redo_count, (unsigned)__popc(m));
            base = __shfl_sync(active, base, leader);
            if (redo) a.redo_list[base + __popc(m & ((1u << lane) - 1u))] = (unsigned)i;
        }
    }
}
// second pass: the listed elements with the general root solve (Aberth's iteration, cosmo_w.cuh), densely packed
template <bool kG, bool kTA>
__global__ void __launch_bounds__(ELEM_THREADS) k_w_redo(WArgs a) {
    const unsigned count = *a.redo_count;
    for (unsigned j = blockIdx.x * blockDim.x + threadIdx.x; j < count; j += gridDim.x * blockDim.x)
        w_one<kG, kTA, false, VoteNone>(a, (int64_t)a.redo_list[j], true, VoteNone());
}

size_t w_cosmo_bytes() { return sizeof(WCosmo); }
template <bool kG, bool kTA>
static void launch_w_variant(const WArgs& a, cudaStream_t st) {
    const unsigned grid = (unsigned)cdiv64(a.n, ELEM_THREADS);
    if (a.n_cosmo == 1) { k_w<kG, kTA, false><<<grid, ELEM_THREADS, 0, st>>>(a); return; }
    cudaMemsetAsync(a.redo_count, 0, sizeof(unsigned), st);
    k_w<kG, kTA, true><<<grid, ELEM_THREADS, 0, st>>>(a);
    k_w_redo<kG, kTA><<<148 * 4, ELEM_THREADS, 0, st>>>(a);
}

void launch_w(const double* z, const double* Om, const double* OL, const double* Or, const double* Ow13, const double* Ow23,
              const double* H0, int64_t n, int64_t n_cosmo, unsigned which, const double* gout, double* out, double* dout, double* gz,
              double* gparams, uint8_t* status, void* ws, cudaStream_t st) {
    WCosmo* shared = static_cast<WCosmo*>(ws);
    unsigned* wl = static_cast<unsigned*>(ws);
    if (n_cosmo == 1) k_w_prep<<<1, 32, 0, st>>>(Om, OL, Or, Ow13, Ow23, H0, shared);
    WArgs a{z, Om, OL, Or, Ow13, Ow23, H0, n, n_cosmo, which, shared, gout, out, dout, gz, gparams, status, wl, wl + 64};
    const bool ta = (which & (W_TL | W_DABS)) != 0;
    if (gout && ta) launch_w_variant<true, true>(a, st);
    else if (gout) launch_w_variant<true, false>(a, st);
    else if (ta) launch_w_variant<false, true>(a, st);
    else launch_w_variant<false, false>(a, st);
}
}  // namespace cb
