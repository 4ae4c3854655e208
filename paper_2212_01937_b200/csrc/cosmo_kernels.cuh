// cosmo_kernels.cuh -- the CUDA kernels of the hot path (sm_100a).  Launchers and the C ABI are in cosmo_b200.cu.
//
// Layout in HBM: SoA everywhere; z[N]; parameters Om/OL/Or/H0[S]; outputs and upstream
// gradients as planes [plane][row][N] with N fastest, so that a warp reads/writes contiguous 512-byte runs per plane row
// (two or four consecutive elements per thread, 128-bit accesses in FP64).  Per-cosmology constants (Cosmo<T>) are
// computed once by k_prep and staged in shared memory by the OUTER kernels, one block = one tile of redshifts
// looping over a chunk of cosmologies, so the only per-eval HBM traffic is grad_out (8 B) and, if asked, out.
#pragma once
#include <cuda_runtime.h>
#include "cosmo_launch.cuh"
#include "cosmo_prep.cuh"
#include "cosmo_obs.cuh"

namespace cb {

__device__ __forceinline__ double warp_sum(double v) {
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) v += __shfl_xor_sync(0xffffffffu, v, off);
    return v;
}

// Sum of four values over the warp with 6 shuffles instead of 20: the exchange halves the number of values a lane
// carries at each of the first two steps.  On return the lanes 0, 8, 16, 24 hold the totals of v[0], v[1], v[2], v[3].
__device__ __forceinline__ double warp_sum4(const double (&v)[4], int lane) {
    const bool hi = lane & 16;
    double a = hi ? v[2] : v[0], b = hi ? v[3] : v[1];
    a += __shfl_xor_sync(0xffffffffu, hi ? v[0] : v[2], 16);
    b += __shfl_xor_sync(0xffffffffu, hi ? v[1] : v[3], 16);
    const bool h3 = lane & 8;
    double k = h3 ? b : a;
    k += __shfl_xor_sync(0xffffffffu, h3 ? a : b, 8);
#pragma unroll
    for (int off = 4; off > 0; off >>= 1) k += __shfl_xor_sync(0xffffffffu, k, off);
    return k;
}

template <typename T> struct Vec2;
template <> struct Vec2<double> { using type = double2; };
template <> struct Vec2<float> { using type = float2; };

template <typename T, int KZ>
__device__ __forceinline__ void load2(const T* __restrict__ p, int64_t i, int64_t n, bool vec, T (&v)[KZ]) {
#pragma unroll
    for (int k = 0; k < KZ; k += 2) {
        if (vec && i + k + 1 < n) {
            typename Vec2<T>::type t = *reinterpret_cast<const typename Vec2<T>::type*>(p + i + k);
            v[k] = t.x; v[k + 1] = t.y;
        } else {
            v[k] = p[i + k < n ? i + k : n - 1];
            v[k + 1] = p[i + k + 1 < n ? i + k + 1 : n - 1];
        }
    }
}
template <typename T, int KZ>
__device__ __forceinline__ void store2(T* __restrict__ p, int64_t i, int64_t n, bool vec, const T (&v)[KZ]) {
#pragma unroll
    for (int k = 0; k < KZ; k += 2) {
        if (vec && i + k + 1 < n) {
            typename Vec2<T>::type t; t.x = v[k]; t.y = v[k + 1];
            *reinterpret_cast<typename Vec2<T>::type*>(p + i + k) = t;
        } else {
            if (i + k < n) p[i + k] = v[k];
            if (i + k + 1 < n) p[i + k + 1] = v[k + 1];
        }
    }
}

// One cosmology row of the OUTER kernels that cannot take the fused loop: E^2 without a real negative root (Cosmo::cubic bit 1:
// complex slow path, cosmo_c4.cuh) or gradient bases that need the per-element conditioning check (bits 2, 3: backward_robust).
// One element at a time.  Never inlined and called at the top of the per-cosmology iteration, where almost nothing is live, so
// that these rare cases cost the hot loop no registers.
template <typename T, bool kT, bool kA, int MODE>
__device__ __noinline__ void outer_slow_row(const OuterArgs& a, const Cosmo<T>& C, int64_t row, int64_t n0, const T* zv, const T* mo,
                                            const T* isig2, const T* lnorm, const T* zo, unsigned which, double* sacc_row, int lane,
                                            T* gzacc) {
    constexpr bool kLike = MODE == MODE_SNIA || MODE == MODE_JOINT;
    constexpr bool kG = MODE != MODE_FWD;
    constexpr int NP = kLike ? 5 : 4;
    constexpr int KZ = outer_kz(kT, kA);
    const int64_t N = a.N, S = a.S;
    T pacc[5] = {T(0), T(0), T(0), T(0), T(0)};
    for (int k = 0; k < KZ; ++k) {
        const bool live = n0 + k < N;
        const int64_t col = live ? n0 + k : N - 1;
        Core<T> R;
        R.I0 = R.TT = R.AA = R.K = R.E = R.iE = R.Em1 = T(0);
        R.status = C.status;
        if (C.cubic & 2u) apply_c4<T, kT, kA, kG>(C, zv[k], R);
        else eval_core<T, kT, kA, kG, VoteWarp>(C, zv[k], VoteWarp(), R);
        Obs<T> O;
        observables<T, kT, kA>(C, zv[k], R, which, O);
        if (kLike) {
            const T resid = mo[k] - O.v[3];
            T gg[N_PLANES] = {T(0), T(0), T(0), resid * isig2[k], T(0), T(0), T(0), T(0), T(0)};
            T dz = T(0), gp[4] = {T(0), T(0), T(0), T(0)};
            backward_robust<T, false, false>(C, zv[k], R, O, gg, dz, gp, W_MU);
            T ll = Num<T>::fma_(T(-0.5) * resid, resid * isig2[k], lnorm[k]);
            if (MODE == MODE_JOINT) {       // same photometric-redshift and prior terms as the fused row of k_outer
                const T x = T(1) + zv[k], ix = Num<T>::rcp_(x);
                const T isz = ix * T(1.0 / a.sigma_z);
                const T rz = (zo[k] - zv[k]) * isz;
                ll += Num<T>::fma_(T(-0.5) * rz, rz, -Num<T>::log_(x));
                ll += T(a.prior_norm) + T(a.shape_m1) * Num<T>::log_(zv[k]) - T(a.beta) * zv[k];
                dz += rz * isz + (rz * rz - T(1)) * ix + T(a.shape_m1) * Num<T>::rcp_(zv[k]) - T(a.beta);
                if (live && a.gz != nullptr) static_cast<T*>(a.gz)[row * N + col] = dz;
            }
            if (live) {
                pacc[0] += ll;
                for (int j = 0; j < 4; ++j) pacc[1 + j] += gp[j];
            }
        } else {
            unsigned stg = 0u;
            if (MODE == MODE_VJP) {
                T g[N_PLANES];
                int pl = 0;
                for (int w = 0; w < N_PLANES; ++w) {
                    g[w] = T(0);
                    if (!(which >> w & 1)) continue;
                    if (live) g[w] = static_cast<const T*>(a.gout)[((int64_t)pl * S + row) * N + col];
                    ++pl;
                }
                T dz = T(0);
                stg = backward_robust<T, kT, kA>(C, zv[k], R, O, g, dz, pacc, which);
                if (live) gzacc[k] += dz;
            }
            if (live) {
                if (a.out != nullptr) {
                    int pl = 0;
                    for (int w = 0; w < N_PLANES; ++w) {
                        if (!(which >> w & 1)) continue;
                        static_cast<T*>(a.out)[((int64_t)pl * S + row) * N + col] = O.v[w];
                        ++pl;
                    }
                }
                if (a.status != nullptr) a.status[row * N + col] = (uint8_t)(O.status | stg);
            }
        }
    }
    if (MODE != MODE_FWD) {
        for (int j = 0; j < NP; ++j) {
            const double v = warp_sum((double)pacc[j]);
            if (lane == 0) sacc_row[j] = v;
        }
    }
}

// OUTER forward / fused forward+VJP / fused likelihood.  grid = (tiles of TILE redshifts, S-chunk groups).
#ifndef CB_MINBLOCKS
#define CB_MINBLOCKS 3     // chi-family kernels: 160 registers, 12 warps/SM (measured best with KZ = 4, profiles/)
#endif
// The VJP kernels that also carry the R_J tracks (t_L, d_abs, age) hold ~60 doubles of per-element state for two elements in lock-step
// besides the loop state and spill 1.4 KB per thread at any register cap.  They take the one-element-at-a-time row function for every
// cosmology instead (with 255 registers, 8 warps/SM): 3.07 -> 2.37 ms on 10^6 x 16, all six planes (profiles/, bench_calls.py outer6).
__host__ __device__ constexpr bool outer_sequential(bool kT, bool kA, int mode) { return mode == MODE_VJP && (kT || kA); }

template <typename T, bool kT, bool kA, int MODE, unsigned WCT>
// (forward-only chi-family kernels need 128 registers as they stand: the fourth block per SM is asked for so that a few registers more
// after an unrelated change cannot silently cost a quarter of the occupancy -- 0.581 -> 0.609 ms on config 3 forward when that happened)
#ifndef CB_SEQ_MINB
#define CB_SEQ_MINB 2
#endif
__global__ void __launch_bounds__(OUTER_THREADS, outer_sequential(kT, kA, MODE) ? CB_SEQ_MINB : ((MODE == MODE_FWD && !kT && !kA) ? 4 : CB_MINBLOCKS)) k_outer(OuterArgs a) {
    constexpr int KZ = outer_kz(kT, kA), TILE = outer_tile(kT, kA);
    const unsigned which = WCT ? WCT : a.which;      // WCT != 0: output set known at compile time (drops dead planes)
    constexpr bool kG = MODE != MODE_FWD;
    constexpr bool kLike = MODE == MODE_SNIA || MODE == MODE_JOINT;
    constexpr int NP = kLike ? 5 : 4;
    __shared__ Cosmo<T> sc[S_CHUNK];
    __shared__ double sacc[kG ? NWARP : 1][kG ? S_CHUNK : 1][NP];
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int64_t N = a.N, S = a.S, SN = S * N;
    const int64_t n0 = (int64_t)blockIdx.x * TILE + (int64_t)tid * KZ;
    const bool vec = a.vec != 0;
    const T* zp = static_cast<const T*>(a.z);
    T zv[KZ];
    load2(zp, n0, N, vec, zv);
    bool live[KZ];
#pragma unroll
    for (int k = 0; k < KZ; ++k) live[k] = n0 + k < N;
    T mo[KZ], isig2[KZ], lnorm[KZ], zo[KZ];
    if (MODE == MODE_JOINT) load2(static_cast<const T*>(a.z_obs), n0, N, vec, zo);
    if (kLike) {
        T sg[KZ];
        load2(static_cast<const T*>(a.mu_obs), n0, N, vec, mo);
        load2(static_cast<const T*>(a.sigma), n0, N, vec, sg);
#pragma unroll
        for (int k = 0; k < KZ; ++k) {
            isig2[k] = T(1) / (sg[k] * sg[k]);
            lnorm[k] = -Num<T>::log_(sg[k]) - T(CB_KT.half_ln_2pi);   // - ln sigma - ln(2 pi)/2
        }
    }
    T gzacc[KZ];
#pragma unroll
    for (int k = 0; k < KZ; ++k) gzacc[k] = T(0);
    const VoteWarp vote;

    cudaGridDependencySynchronize();          // PDL: k_prep's constants (everything above only read the caller's inputs)
    for (int64_t c0 = (int64_t)blockIdx.y * S_CHUNK; c0 < S; c0 += (int64_t)gridDim.y * S_CHUNK) {
        const int ns = (int)((S - c0 < S_CHUNK) ? (S - c0) : S_CHUNK);
        __syncthreads();
        for (int i = tid; i < ns * COSMO_NFIELDS; i += OUTER_THREADS) {
            int sl = i / COSMO_NFIELDS, f = i - sl * COSMO_NFIELDS;
            reinterpret_cast<T*>(&sc[sl])[f] = (T) reinterpret_cast<const double*>(&a.consts[c0 + sl])[f];
        }
        for (int sl = tid; sl < ns; sl += OUTER_THREADS) {
            sc[sl].status = a.consts[c0 + sl].status;
            sc[sl].cubic = a.consts[c0 + sl].cubic;
        }
        __syncthreads();
        int64_t roff = c0 * N;                                   // row * N, advanced by N per cosmology (no 64-bit multiplies)
        for (int sl = 0; sl < ns; ++sl, roff += N) {
            const Cosmo<T>& C = sc[sl];
            const int64_t row = c0 + sl;
            if (MODE == MODE_JOINT) load2(zp + roff, n0, N, vec, zv);      // latent redshifts: one row per sample
            // two complex root pairs, or (with gradients) bases that need the per-element conditioning check: whole row apart; so do
            // the variants whose per-element state does not fit two elements in lock-step (outer_sequential)
            if ((C.cubic & 2u) || (kG && (C.cubic & 12u)) || outer_sequential(kT, kA, MODE)) {
                outer_slow_row<T, kT, kA, MODE>(a, C, row, n0, zv, mo, isig2, lnorm, zo, kLike ? (unsigned)W_MU : which,
                                                kG ? &sacc[warp][sl][0] : nullptr, lane, gzacc);
                continue;
            }
            T pacc[NP];
#pragma unroll
            for (int j = 0; j < NP; ++j) pacc[j] = T(0);
            T g[KZ][N_PLANES];
            if (MODE == MODE_VJP) {
#pragma unroll
                for (int k = 0; k < KZ; ++k)
#pragma unroll
                    for (int w = 0; w < N_PLANES; ++w) g[k][w] = T(0);
                int pl = 0;
                for (int w = 0; w < N_PLANES; ++w) {
                    if (!(which >> w & 1)) continue;
                    T t[KZ];
                    load2(static_cast<const T*>(a.gout) + ((int64_t)pl * SN + roff), n0, N, vec, t);
#pragma unroll
                    for (int k = 0; k < KZ; ++k) g[k][w] = live[k] ? t[k] : T(0);
                    ++pl;
                }
            }
            T ov[N_PLANES][KZ];
            uint8_t stv[KZ];
            Core<T> R[KZ];
            eval_core_k<T, kT, kA, kG, KZ, VoteWarp>(C, zv, vote, R);
            Obs<T> Ok[KZ];
            observables_k<T, kT, kA, KZ>(C, zv, R, kLike ? (unsigned)W_MU : which, Ok);
#pragma unroll
            for (int k = 0; k < KZ; ++k) {
                const Obs<T>& O = Ok[k];
#pragma unroll
                for (int w = 0; w < N_PLANES; ++w) ov[w][k] = O.v[w];
                stv[k] = (uint8_t)O.status;
                if (kLike) {
                    const T resid = mo[k] - O.v[3];
                    T gg[N_PLANES] = {T(0), T(0), T(0), resid * isig2[k], T(0), T(0), T(0), T(0), T(0)};
                    T dz = T(0), gp[4] = {T(0), T(0), T(0), T(0)};
                    backward<T, false, false>(C, zv[k], R[k], O, gg, dz, gp);
                    T ll = Num<T>::fma_(T(-0.5) * resid, resid * isig2[k], lnorm[k]);
                    if (MODE == MODE_JOINT) {
                        // photometric-redshift term N(z_obs | z, (1+z)^2 sigma_z^2) and gamma prior on the latent redshift
                        const T x = T(1) + zv[k], ix = Num<T>::rcp_(x);
                        const T isz = ix * T(1.0 / a.sigma_z);
                        const T rz = (zo[k] - zv[k]) * isz;
                        ll += Num<T>::fma_(T(-0.5) * rz, rz, -Num<T>::log_(x));
                        ll += T(a.prior_norm) + T(a.shape_m1) * Num<T>::log_(zv[k]) - T(a.beta) * zv[k];
                        dz += rz * isz + (rz * rz - T(1)) * ix + T(a.shape_m1) * Num<T>::rcp_(zv[k]) - T(a.beta);
                        gzacc[k] = dz;
                    }
                    if (live[k]) {
                        pacc[0] += ll;
#pragma unroll
                        for (int j = 0; j < 4; ++j) pacc[1 + j] += gp[j];
                    }
                }
                // straight into the accumulators: elements past N carry zero upstream gradients (see the load) and their
                // grad_z is never stored
                if (MODE == MODE_VJP) {
                    // the chi-family bases of a screened cosmology run unchecked (cosmo_prep, Cosmo::cubic bit 3); the larger t_L / d_abs
                    // bases are checked element by element
                    if (kT || kA) stv[k] |= (uint8_t)backward_robust<T, kT, kA>(C, zv[k], R[k], O, g[k], gzacc[k], pacc, which);
                    else backward<T, kT, kA>(C, zv[k], R[k], O, g[k], gzacc[k], pacc, nullptr, which);
                }
            }
            if (MODE == MODE_JOINT && a.gz != nullptr) store2(static_cast<T*>(a.gz) + roff, n0, N, vec, gzacc);
            if (!kLike && a.out != nullptr) {
                int pl = 0;
                for (int w = 0; w < N_PLANES; ++w) {
                    if (!(which >> w & 1)) continue;
                    store2(static_cast<T*>(a.out) + ((int64_t)pl * SN + roff), n0, N, vec, ov[w]);
                    ++pl;
                }
            }
            if (!kLike && a.status != nullptr) {
#pragma unroll
                for (int k = 0; k < KZ; ++k)
                    if (live[k]) a.status[roff + n0 + k] = stv[k];
            }
            if (kG) {
                const double v4[4] = {(double)pacc[NP - 4], (double)pacc[NP - 3], (double)pacc[NP - 2], (double)pacc[NP - 1]};
                const double tot = warp_sum4(v4, lane);
                if ((lane & 7) == 0) sacc[warp][sl][NP - 4 + (lane >> 3)] = tot;
                if (NP == 5) {
                    const double l = warp_sum((double)pacc[0]);
                    if (lane == 0) sacc[warp][sl][0] = l;
                }
            }
        }
        if (kG) {
            __syncthreads();
            for (int i = tid; i < ns * NP; i += OUTER_THREADS) {
                int sl = i / NP, j = i - sl * NP;
                double v = 0.0;
#pragma unroll
                for (int w = 0; w < NWARP; ++w) v += sacc[w][sl][j];
                a.part[((c0 + sl) * NP + j) * (int64_t)gridDim.x + blockIdx.x] = v;    // [S][NP][ntiles]: the reduction reads contiguously
            }
        }
    }
    if (MODE == MODE_VJP) {
        T* gzp = static_cast<T*>(a.gz) + (a.gz_accumulate ? (int64_t)blockIdx.y * N : 0);
        store2(gzp, n0, N, vec, gzacc);
    }
}

// partial parameter sums [S][NP][ntiles] -> dst planes: dst_first[S] (snia logL) and dst_grad[4][S]; fixed order => deterministic
template <int NP>
__global__ void k_reduce_params(const double* __restrict__ part, int64_t ntiles, int64_t S, double* __restrict__ logL,
                                double* __restrict__ grad) {
    cudaGridDependencySynchronize();          // PDL: the OUTER kernel's partial sums
    // one warp per (s, j)
    const int64_t wid = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wid >= S * NP) return;
    const int64_t s = wid / NP;
    const int j = (int)(wid - s * NP);
    double v = 0.0;
    const double* __restrict__ row = part + (s * NP + j) * ntiles;
    for (int64_t t = lane; t < ntiles; t += 32) v += row[t];
    v = warp_sum(v);
    if (lane == 0) {
        if (NP == 5) {
            if (j == 0) logL[s] = v;
            else if (grad) grad[(int64_t)(j - 1) * S + s] = v;
        } else {
            grad[(int64_t)j * S + s] = v;
        }
    }
}

// the two reductions of an OUTER VJP in ONE launch: blocks [0, nb_gz) sum the grad_z partials of the cosmology groups (if any),
// the others the per-tile parameter sums (as k_reduce_params<4>)
template <typename T>
__global__ void k_reduce_vjp(const double* __restrict__ part, int64_t ntiles, int64_t S, double* __restrict__ grad,
                             const T* __restrict__ gzpart, int ny, int64_t N, T* __restrict__ gz, unsigned nb_gz) {
    cudaGridDependencySynchronize();          // PDL: the OUTER kernel's partial sums
    if (blockIdx.x < nb_gz) {
        const int64_t n = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
        if (n >= N) return;
        T v = T(0);
        for (int y = 0; y < ny; ++y) v += gzpart[(int64_t)y * N + n];
        gz[n] = v;
        return;
    }
    const int64_t wid = ((blockIdx.x - nb_gz) * (int64_t)blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (wid >= S * 4) return;
    const int64_t s = wid >> 2;
    const int j = (int)(wid & 3);
    double v = 0.0;
    const double* __restrict__ row = part + (s * 4 + j) * ntiles;
    for (int64_t t = lane; t < ntiles; t += 32) v += row[t];
    v = warp_sum(v);
    if (lane == 0) grad[(int64_t)j * S + s] = v;
}

// ELEMENTWISE with one cosmology per redshift: S1-S8 per thread (cosmo_obs.cuh, elem_one), no reductions.
// Register budget: left alone the all-outputs variants take 255 registers (8 warps/SM) and wait on latency at a third of the
// FP64 pipe; capped at 128 (VJP) / 80 (forward) registers they run 16 / 24 warps per SM (profiles/).  Blocks of 256 threads measured 7-10 %
// faster than 128 at the same occupancy (2.79 vs 3.09 ms on config 5); block-wide barriers between the phases of an element did not help.
// Two passes.  k_elem is the fast path for every element; the few that need a slow path -- E^2 without a real negative root
// (complex arithmetic, cosmo_c4.cuh), gradient bases too ill-conditioned (quadrature, cosmo_obs.cuh) -- are only listed
// (redo_count, redo_list in the workspace) and k_elem_redo runs them again, densely packed, with the slow paths compiled in.
// A never-inlined call inside the main kernel costs it 15-30 % even where it is not taken (profiles/).
#ifndef CB_ELEM_BLOCK
#define CB_ELEM_BLOCK 256
#endif
#ifndef CB_ELEM_MINB_G
#define CB_ELEM_MINB_G 2
#endif
#ifndef CB_ELEM_MINB_F
#define CB_ELEM_MINB_F 3
#endif
// values out as soon as they exist, upstream gradients in only when the backward chain starts (elem_one_io): neither set is held in
// registers through the other half of the element.  The present planes follow one another, N apart.
template <typename T>
struct PlaneIO {
    const T* gpl; T* opl; int64_t N; unsigned which; bool live;
    __device__ __forceinline__ void put_values(const T (&o)[N_PLANES]) const {
        if (!live || opl == nullptr) return;
        T* p = opl;
#pragma unroll
        for (int w = 0; w < N_PLANES; ++w) {
            const bool on = which >> w & 1;
            if (on) *p = o[w];
            p += on ? N : 0;
        }
    }
    __device__ __forceinline__ void get_grads(T (&go)[N_PLANES]) const {
        const T* p = gpl;
        if (sizeof(T) == 8) asm volatile("" : "+l"(p));              // FP64: keeps the loads below the forward pass (registers)
#pragma unroll
        for (int w = 0; w < N_PLANES; ++w) {
            const bool on = which >> w & 1;
            go[w] = on ? *p : T(0);
            p += on ? N : 0;
        }
    }
};
template <typename T, bool kT, bool kA, bool kG, bool kAge>
__global__ void __launch_bounds__(CB_ELEM_BLOCK, kG ? CB_ELEM_MINB_G : CB_ELEM_MINB_F) k_elem(ElemArgs a) {
    const int64_t N = a.N;
    const unsigned which = a.which;
    const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
    const bool live = i < N;
    const int64_t ii = live ? i : N - 1;
    const PlaneIO<T> io{kG ? static_cast<const T*>(a.gout) + ii : nullptr, a.out != nullptr ? static_cast<T*>(a.out) + ii : nullptr, N, which, live};
    T dz = T(0), gp[4] = {T(0), T(0), T(0), T(0)};
    unsigned st;
    if constexpr (sizeof(T) == 8) {
        st = elem_one_io<T, kT, kA, kG, VoteWarp, true, kAge, PlaneIO<T>>(static_cast<const T*>(a.z)[ii], a.Om[ii], a.OL[ii], a.Or[ii], a.H0[ii],
                                                                         which, VoteWarp(), io, dz, gp);
    } else {                        // FP32: registers are not what limits it, and it measures 3 % faster with the loads up front
        T g[N_PLANES], v[N_PLANES];
        if (kG) io.get_grads(g);
        st = elem_one<T, kT, kA, kG, VoteWarp, true, kAge>(static_cast<const T*>(a.z)[ii], a.Om[ii], a.OL[ii], a.Or[ii], a.H0[ii], which,
                                                           VoteWarp(), g, v, dz, gp);
        io.put_values(v);
    }
    if (live && a.status != nullptr) a.status[i] = (uint8_t)(st & ~(unsigned)ST_INTERNAL_REDO);
    if (kG && live) {
        static_cast<T*>(a.gz)[i] = dz;
#pragma unroll
        for (int j = 0; j < 4; ++j) a.gparams[(int64_t)j * N + i] = (double)gp[j];
    }
    if (kG) {   // work list of the second pass: one atomic per warp (no lane has returned early)
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

// second pass: the listed elements again with every slow path available (elem_one without kDefer).  Dense: consecutive threads take
// consecutive list entries, whatever their position in the batch.
template <typename T, bool kT, bool kA, bool kG>      // (kG = true: only the VJP has a second pass)
#ifndef CB_REDO_MINB
#define CB_REDO_MINB 2      // 254 registers, no spills (at 4 blocks: 128 registers, 800 B of spills per thread; measured 2.177 -> 2.135 ms on config 5)
#endif
#ifndef CB_REDO_GRID
#define CB_REDO_GRID 8      // blocks per SM of the persistent grid (finer tail)
#endif
__global__ void __launch_bounds__(ELEM_THREADS, CB_REDO_MINB) k_elem_redo(ElemArgs a) {
    const int64_t N = a.N;
    const unsigned which = a.which;
    const unsigned count = *a.redo_count;
    const T* __restrict__ gout = static_cast<const T*>(a.gout);
    for (unsigned j = blockIdx.x * blockDim.x + threadIdx.x; j < count; j += gridDim.x * blockDim.x) {
        const int64_t i = a.redo_list[j];
        T g[N_PLANES], v[N_PLANES];
        if (kG) {
            int pl = 0;
            for (int w = 0; w < N_PLANES; ++w) {
                g[w] = T(0);
                if (!(which >> w & 1)) continue;
                g[w] = gout[(int64_t)pl * N + i];
                ++pl;
            }
        }
        T dz = T(0), gp[4] = {T(0), T(0), T(0), T(0)};
        const unsigned st = elem_one<T, kT, kA, kG, VoteNone, false, true, sizeof(T) == 8>(static_cast<const T*>(a.z)[i], a.Om[i], a.OL[i], a.Or[i], a.H0[i], which,
                                                                     VoteNone(), g, v, dz, gp);
        if (a.out != nullptr) {
            T* __restrict__ out = static_cast<T*>(a.out);
            int pl = 0;
            for (int w = 0; w < N_PLANES; ++w) {
                if (!(which >> w & 1)) continue;
                out[(int64_t)pl * N + i] = v[w];
                ++pl;
            }
        }
        if (a.status != nullptr) a.status[i] = (uint8_t)st;
        if (kG) {
            static_cast<T*>(a.gz)[i] = dz;
#pragma unroll
            for (int k = 0; k < 4; ++k) a.gparams[(int64_t)k * N + i] = (double)gp[k];
        }
    }
}

// ALU roofline probes: 8 independent FMA chains per thread
template <typename T>
__global__ void __launch_bounds__(256) k_probe_fma(int iters, T* __restrict__ sink) {
    T a0 = T(threadIdx.x) * T(1e-3), a1 = a0 + T(1), a2 = a0 + T(2), a3 = a0 + T(3), a4 = a0 + T(4), a5 = a0 + T(5), a6 = a0 + T(6),
      a7 = a0 + T(7);
    const T m = T(0.999999), c = T(1e-7);
    for (int i = 0; i < iters; ++i) {
        a0 = Num<T>::fma_(a0, m, c); a1 = Num<T>::fma_(a1, m, c); a2 = Num<T>::fma_(a2, m, c); a3 = Num<T>::fma_(a3, m, c);
        a4 = Num<T>::fma_(a4, m, c); a5 = Num<T>::fma_(a5, m, c); a6 = Num<T>::fma_(a6, m, c); a7 = Num<T>::fma_(a7, m, c);
    }
    sink[blockIdx.x * (int64_t)blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

}  // namespace cb
