// tu_outer_f64_like.cu -- instantiates the fused likelihood kernels (k_outer in MODE_SNIA / MODE_JOINT) for double.
#include "cosmo_kernels.cuh"

namespace cb {

void launch_outer_f64_like(int mode, const OuterArgs& a, dim3 grid, cudaStream_t st) {
    if (mode == MODE_SNIA) launch_pdl(k_outer<double, false, false, MODE_SNIA, W_MU>, grid, dim3(OUTER_THREADS), st, a);
    else launch_pdl(k_outer<double, false, false, MODE_JOINT, W_MU>, grid, dim3(OUTER_THREADS), st, a);
}

}  // namespace cb
