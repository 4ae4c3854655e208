// tu_misc.cu -- instantiates the small kernels of cosmo_kernels.cuh: per-cosmology prep, the reductions, the two-limit ELEMENTWISE
// kernels, the stand-alone Carlson functions and the ALU probes.
#include "cosmo_kernels.cuh"
#include "cosmo_two.cuh"

namespace cb {

// S1-S3, one thread per cosmology
__global__ void k_prep(const double* __restrict__ Om, const double* __restrict__ OL, const double* __restrict__ Or,
                       const double* __restrict__ H0, int64_t S, int want_grad, Cosmo<double>* __restrict__ out) {
    int64_t s = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    if (s >= S) return;
    Cosmo<double> C;
    cosmo_prep(Om[s], OL[s], Or[s], H0[s], want_grad & 3, C);
    if (want_grad & 4) prep_age(C, (want_grad & 3) != 0);
    else { C.Tinf = 0.0; C.dTinf[0] = C.dTinf[1] = C.dTinf[2] = 0.0; }
    if ((want_grad & 3) < 2) {
        for (int t = 0; t < 3; ++t) {
            for (int j = 0; j < 7; ++j) C.GA[t][j] = 0.0;
            for (int j = 0; j < 5; ++j) C.GJ[t][j] = C.GJ[t + 2][j] = 0.0;
            if ((want_grad & 3) < 1) { for (int j = 0; j < 5; ++j) C.GI[t][j] = 0.0; for (int j = 0; j < 6; ++j) C.GT[t][j] = 0.0; }
        }
    }
    out[s] = C;
}

// Two-limit evaluation (cosmo_two.cuh), one thread per (z1, z2, cosmology); n_cosmo in {1, n}.  which: DC, DM, TL, DABS, DA.
// (128-register cap as for k_elem.)  kG: with the VJP; its slow paths go to the second pass k_two<.., kRedo> through a work list, as in
// k_elem; the forward kernel keeps the complex path inline.
#ifndef CB_TWO_BLOCK
#define CB_TWO_BLOCK 256      // as k_elem: 256-thread blocks measured a few per cent faster than 128 at the same occupancy
#endif
#ifndef CB_TWO_DEFER_MIN
#define CB_TWO_DEFER_MIN 3000000
#endif
constexpr int64_t TWO_DEFER_MIN = CB_TWO_DEFER_MIN;
struct TwoArgs {
    const double *z1, *z2, *Om, *OL, *Or, *H0;
    int64_t n, n_cosmo; unsigned which;
    const double* gout; double *out, *gz1, *gz2, *gparams; uint8_t* status;
    unsigned *redo_count, *redo_list;
};

template <bool kG, bool kDefer, bool kRedo>
__device__ __forceinline__ unsigned two_one(const TwoArgs& a, int64_t i, bool live) {
    const int64_t n = a.n, ii = live ? i : n - 1, ic = a.n_cosmo == 1 ? 0 : ii;
    Cosmo<double> C{};
    cosmo_factor(a.Om[ic], a.OL[ic], a.Or[ic], a.H0[ic], C);
    cosmo_constants(C);
    Two O;
    if (kRedo) eval_two<VoteNone, false>(C, a.z1[ii], a.z2[ii], kG, VoteNone(), O);
    else eval_two<VoteWarp, kDefer>(C, a.z1[ii], a.z2[ii], kG, VoteWarp(), O);
    if (!live) return 0u;
    const unsigned bits[5] = {W_DC, W_DM, W_TL, W_DABS, W_DA};
    double a1 = 0.0, a2 = 0.0, ap[4] = {0.0, 0.0, 0.0, 0.0};
    int pl = 0;
    for (int o = 0; o < 5; ++o) {
        if (!(a.which & bits[o])) continue;
        if (a.out != nullptr) a.out[(int64_t)pl * n + i] = O.v[o];
        if (kG) {
            const double g = a.gout[(int64_t)pl * n + i];
            a1 = fma(g, O.gz1[o], a1); a2 = fma(g, O.gz2[o], a2);
            for (int t = 0; t < 4; ++t) ap[t] = fma(g, O.gp[o][t], ap[t]);
        }
        ++pl;
    }
    if (a.status != nullptr) a.status[i] = (uint8_t)(O.status & ~(unsigned)ST_INTERNAL_REDO);
    if (kG) {
        a.gz1[i] = a1; a.gz2[i] = a2;
        for (int t = 0; t < 4; ++t) a.gparams[(int64_t)t * n + i] = ap[t];
    }
    return O.status;
}

template <bool kG, bool kDefer>
__global__ void __launch_bounds__(CB_TWO_BLOCK, kG ? 2 : 3) k_two(TwoArgs a) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool live = i < a.n;
    const unsigned st = two_one<kG, kDefer, false>(a, i, live);
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
__global__ void __launch_bounds__(ELEM_THREADS, 4) k_two_redo(TwoArgs a) {
    const unsigned count = *a.redo_count;
    for (unsigned j = blockIdx.x * blockDim.x + threadIdx.x; j < count; j += gridDim.x * blockDim.x) two_one<true, false, true>(a, (int64_t)a.redo_list[j], true);
}

// The device Carlson functions on their own (same code as the hot path): R_F(x, m+h, m-h), R_D(m+h, m-h, x) and
// R_J(x, m+h, m-h, p) with h^2 = s (s < 0: complex-conjugate pair), positive x and p.
__global__ void k_carlson_pair(const double* __restrict__ x, const double* __restrict__ m, const double* __restrict__ s,
                               const double* __restrict__ p, int64_t n, double* __restrict__ rf, double* __restrict__ rd,
                               double* __restrict__ rj) {
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const int64_t ii = i < n ? i : n - 1;
    double xa[1] = {x[ii]}, mp[1] = {m[ii]}, ss[1] = {s[ii]}, p5[1] = {p[ii]}, p0[1] = {0.0};
    const double xa0 = xa[0], m0 = mp[0], s0 = ss[0], pp0 = p5[0];
    const double hd = xa0 - m0, hs = sqrt(fabs(s0));
    const double pm = pp0 - m0;
    const double dl5[1] = {(pp0 - xa0) * fma(pm, pm, -s0)}, dl0[1] = {0.0};
    const double Qc[1] = {carlson_Qc<double>(hd, hs, true)}, Q5v[1] = {carlson_Qj<double>(xa0, m0, hs, pp0)}, Q0v[1] = {0.0};
    unsigned st[1] = {0u};
    double f, tailD[1], sum5[1], sum0[1];
    carlson_dup<double, true, true, false, 1, VoteWarp>(xa, mp, ss, p5, p0, dl5, dl0, Qc, Q5v, Q0v, st, VoteWarp(), f, tailD, sum5, sum0);
    if (i >= n) return;
    rf[i] = carlson_rf_series<double>(xa[0], mp[0], f, hd, s0);
    rd[i] = carlson_rd_series<double>(xa[0], mp[0], f, hd, s0, tailD[0]);
    rj[i] = carlson_rj_series<double>(xa[0], mp[0], p5[0], f, xa0, m0, s0, pp0, sum5[0]);
}


void launch_prep(const double* Om, const double* OL, const double* Or, const double* H0, int64_t S, int want_grad, Cosmo<double>* out,
                 cudaStream_t st) {
    k_prep<<<(unsigned)cdiv64(S, 64), 64, 0, st>>>(Om, OL, Or, H0, S, want_grad, out);
}
void launch_reduce_params(int np, const double* part, int64_t ntiles, int64_t S, double* logL, double* grad, cudaStream_t st) {
    if (np == 5) launch_pdl(k_reduce_params<5>, dim3((unsigned)cdiv64(S * 5 * 32, 256)), dim3(256), st, part, ntiles, S, logL, grad);
    else launch_pdl(k_reduce_params<4>, dim3((unsigned)cdiv64(S * 4 * 32, 256)), dim3(256), st, part, ntiles, S, (double*)nullptr, grad);
}
void launch_reduce_vjp(bool f32, const double* part, int64_t ntiles, int64_t S, double* grad, const void* gzpart, int ny, int64_t N, void* gz,
                       cudaStream_t st) {
    const unsigned nb_gz = gzpart ? (unsigned)cdiv64(N, 256) : 0u, nb_p = (unsigned)cdiv64(S * 4 * 32, 256);
    if (f32) launch_pdl(k_reduce_vjp<float>, dim3(nb_gz + nb_p), dim3(256), st, part, ntiles, S, grad, static_cast<const float*>(gzpart), ny, N, static_cast<float*>(gz), nb_gz);
    else launch_pdl(k_reduce_vjp<double>, dim3(nb_gz + nb_p), dim3(256), st, part, ntiles, S, grad, static_cast<const double*>(gzpart), ny, N, static_cast<double*>(gz), nb_gz);
}
void launch_two(const double* z1, const double* z2, const double* Om, const double* OL, const double* Or, const double* H0, int64_t n,
                int64_t n_cosmo, unsigned which, const double* gout, double* out, double* gz1, double* gz2, double* gparams,
                uint8_t* status, unsigned* ws, cudaStream_t st) {
    TwoArgs a{z1, z2, Om, OL, Or, H0, n, n_cosmo, which, gout, out, gz1, gz2, gparams, status, ws, ws ? ws + 64 : nullptr};
    const unsigned grid = (unsigned)cdiv64(n, CB_TWO_BLOCK);
    if (gout == nullptr) { k_two<false, false><<<grid, CB_TWO_BLOCK, 0, st>>>(a); return; }
    // The second pass costs the latency of one slow element (tens of microseconds) whatever the batch size, the inline slow paths
    // ~10 % of the main kernel: two passes from a few million elements on (measured, profiles/)
    if (n < TWO_DEFER_MIN) { k_two<true, false><<<grid, CB_TWO_BLOCK, 0, st>>>(a); return; }
    cudaMemsetAsync(a.redo_count, 0, sizeof(unsigned), st);
    k_two<true, true><<<grid, CB_TWO_BLOCK, 0, st>>>(a);
    k_two_redo<<<148 * 4, ELEM_THREADS, 0, st>>>(a);
}
void launch_carlson_pair(const double* x, const double* m, const double* s, const double* p, int64_t n, double* rf, double* rd, double* rj,
                         cudaStream_t st) {
    k_carlson_pair<<<(unsigned)cdiv64(n, 128), 128, 0, st>>>(x, m, s, p, n, rf, rd, rj);
}
void launch_probe_fma(bool f32, int blocks, int iters, void* sink, cudaStream_t st) {
    if (f32) k_probe_fma<float><<<blocks, 256, 0, st>>>(iters, static_cast<float*>(sink));
    else k_probe_fma<double><<<blocks, 256, 0, st>>>(iters, static_cast<double*>(sink));
}

}  // namespace cb
