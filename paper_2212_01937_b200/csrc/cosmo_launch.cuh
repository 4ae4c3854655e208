// cosmo_launch.cuh -- what the translation units of libcosmo_b200.so share on the HOST side: tile constants, the argument block of the
// OUTER kernels and the launchers each kernel family's translation unit exports (the kernels themselves are in cosmo_kernels.cuh and
// are instantiated once, in tu_*.cu; splitting them lets nvcc compile the families in parallel).
#pragma once
#include <cuda_runtime.h>
#include "cosmo_types.cuh"

namespace cb {

#ifndef CB_THREADS
#define CB_THREADS 128
#endif
constexpr int OUTER_THREADS = CB_THREADS;
// consecutive redshifts per thread (even), advanced in lock-step.  Per-thread overhead (staging, address arithmetic, the
// warp reduction, constant and shared-memory loads) is paid once per KZ elements, so the chi family -- whose working set
// fits -- takes 4; the kernels that also carry the R_J tracks (t_L, d_abs) stay at 2 (4 spills).  Measured: profiles/.
#ifndef CB_KZ_CHI
#define CB_KZ_CHI 4
#endif
#ifndef CB_KZ_TA
#define CB_KZ_TA 2
#endif
__host__ __device__ constexpr int outer_kz(bool kT, bool kA) { return (kT || kA) ? CB_KZ_TA : CB_KZ_CHI; }
__host__ __device__ constexpr int outer_tile(bool kT, bool kA) { return OUTER_THREADS * outer_kz(kT, kA); }   // redshifts per block
#ifndef CB_SCHUNK
#define CB_SCHUNK 16
#endif
constexpr int S_CHUNK = CB_SCHUNK;                         // cosmologies staged in shared memory at a time
constexpr int NWARP = OUTER_THREADS / 32;
constexpr int ELEM_THREADS = 128;

enum { MODE_FWD = 0, MODE_VJP = 1, MODE_SNIA = 2, MODE_JOINT = 3 };   // JOINT: SNIA + latent redshifts z[S][N]

struct OuterArgs {
    const void* z; const void* gout; const void* mu_obs; const void* sigma; const void* z_obs;
    double sigma_z, beta, shape_m1, prior_norm;   // MODE_JOINT: photo-z scatter, gamma prior rate, shape - 1, and the constant
                                                  // shape ln(beta) - lnGamma(shape) - ln(sigma_z) - ln(2 pi)/2
    void* out; void* gz; uint8_t* status;
    const Cosmo<double>* consts;
    double* part;            // [S][NP][ntiles] partial parameter sums (NP = 4 vjp, 5 snia)
    int64_t N, S;
    unsigned which;
    int gz_accumulate;       // gridDim.y > 1: gz holds [gridDim.y][N] partials
    int vec;                 // N even and pointers 16-byte aligned
};

struct ElemArgs {            // ELEMENTWISE with one cosmology per redshift
    const void* z; const double *Om, *OL, *Or, *H0;
    int64_t N; unsigned which;
    const void* gout; void* out; void* gz; double* gparams; uint8_t* status;
    unsigned* redo_count; unsigned* redo_list;     // VJP: work list of the second pass (workspace), see k_elem
};

// launchers (one translation unit per kernel family); every one only enqueues on `st`
void launch_prep(const double* Om, const double* OL, const double* Or, const double* H0, int64_t S, int want_grad, Cosmo<double>* out,
                 cudaStream_t st);
void launch_outer_f64(int mode, const OuterArgs& a, dim3 grid, cudaStream_t st);
void launch_outer_f32(int mode, const OuterArgs& a, dim3 grid, cudaStream_t st);
void launch_elem_f64(bool with_grad, const ElemArgs& a, cudaStream_t st);
void launch_elem_f32(bool with_grad, const ElemArgs& a, cudaStream_t st);
void launch_reduce_params(int np, const double* part, int64_t ntiles, int64_t S, double* logL, double* grad, cudaStream_t st);
void launch_reduce_vjp(bool f32, const double* part, int64_t ntiles, int64_t S, double* grad, const void* gzpart, int ny, int64_t N, void* gz,
                       cudaStream_t st);
void launch_two(const double* z1, const double* z2, const double* Om, const double* OL, const double* Or, const double* H0, int64_t n,
                int64_t n_cosmo, unsigned which, const double* gout, double* out, double* gz1, double* gz2, double* gparams,
                uint8_t* status, unsigned* ws, cudaStream_t st);
size_t w_cosmo_bytes();
void launch_w(const double* z, const double* Om, const double* OL, const double* Or, const double* Ow13, const double* Ow23,
              const double* H0, int64_t n, int64_t n_cosmo, unsigned which, const double* gout, double* out, double* dout, double* gz,
              double* gparams, uint8_t* status, void* ws, cudaStream_t st);
void launch_carlson_pair(const double* x, const double* m, const double* s, const double* p, int64_t n, double* rf, double* rd, double* rj,
                         cudaStream_t st);
void launch_probe_fma(bool f32, int blocks, int iters, void* sink, cudaStream_t st);

inline int64_t cdiv64(int64_t a, int64_t b) { return (a + b - 1) / b; }

#ifdef __CUDACC__
// Launch with programmatic dependent launch (PDL): the kernel may start while its predecessor in the stream is still draining; it
// must call cudaGridDependencySynchronize() before touching anything the predecessor wrote.  Closes most of the gap that a chain of
// short launches (prep -> outer -> reduce) otherwise leaves between kernels.
template <typename... KArgs, typename... Args>
inline void launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, cudaStream_t st, Args... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = 0; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#endif

}  // namespace cb
