// tu_outer_f64.cu -- instantiates the OUTER kernels (cosmo_kernels.cuh: k_outer) for double, forward and fused forward + VJP and exports their launcher.
#include "cosmo_kernels.cuh"

namespace cb {

template <int MODE>
static void outer_dispatch_f64(const OuterArgs& a, dim3 grid, cudaStream_t st) {
    using T = double;
    const bool kT = a.which & (W_TL | W_AGE), kA = a.which & W_DABS;
    if (MODE == MODE_SNIA || MODE == MODE_JOINT) launch_pdl(k_outer<T, false, false, MODE, W_MU>, grid, dim3(OUTER_THREADS), st, a);
    else if (kT && kA) launch_pdl(k_outer<T, true, true, MODE, 0>, grid, dim3(OUTER_THREADS), st, a);
    else if (kT) launch_pdl(k_outer<T, true, false, MODE, 0>, grid, dim3(OUTER_THREADS), st, a);
    else if (kA) launch_pdl(k_outer<T, false, true, MODE, 0>, grid, dim3(OUTER_THREADS), st, a);
    else if (a.which == W_MU) launch_pdl(k_outer<T, false, false, MODE, W_MU>, grid, dim3(OUTER_THREADS), st, a);
    else launch_pdl(k_outer<T, false, false, MODE, 0>, grid, dim3(OUTER_THREADS), st, a);
}

void launch_outer_f64_like(int mode, const OuterArgs& a, dim3 grid, cudaStream_t st);      // tu_outer_f64_like.cu

void launch_outer_f64(int mode, const OuterArgs& a, dim3 grid, cudaStream_t st) {
    switch (mode) {
        case MODE_FWD: outer_dispatch_f64<MODE_FWD>(a, grid, st); break;
        case MODE_VJP: outer_dispatch_f64<MODE_VJP>(a, grid, st); break;
        default: launch_outer_f64_like(mode, a, grid, st); break;
    }
}

}  // namespace cb
