// tu_static.cu -- cosmo_snia_loglike_static: the fused SN-Ia likelihood (cosmo_snia_loglike) for callers that cannot
// allocate device memory or hand over a workspace (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
// Same kernels, same arithmetic, same order of summation as cosmo_snia_loglike; the only difference is where the scratch lives: a
// file-scope device array of fixed size instead of the caller's workspace.
//
// Scratch layout (as the workspace of cosmo_snia_loglike): Cosmo<double>[S] | partial sums [S][5][ntiles].  Every byte a call reads it
// has written before in the same call (k_prep writes the S blocks, every block of k_outer writes its (s, j, tile) partials), so nothing
// needs to start at zero and stale contents of an earlier call are never read.  ALL calls on a GPU share the array: calls that may
// overlap on the device (different streams without ordering, different host threads) race on it -- serialise them.
#include <mutex>
#include "../../include/cosmo_b200.h"
#include "cosmo_launch.cuh"

namespace {

using namespace cb;

// 24 MiB per GPU that loads the library, held until the process exits: enough for BASELINE.json config 4 at full size
// (S = 256 samples x N = 10^6 supernovae: 0.24 MB of per-cosmology blocks + 20.0 MB of partial sums)
static __device__ __align__(256) unsigned char g_static_scratch[COSMO_STATIC_SCRATCH_BYTES];

// In HOST code the name g_static_scratch is a stand-in, not a device address: the address is asked for once per device, with
// that device current, and cached.
constexpr int MAX_DEVICES = 64;
std::mutex g_mu;
void* g_scratch_ptr[MAX_DEVICES] = {};

int scratch_address(unsigned char** out) {
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= MAX_DEVICES) return COSMO_E_CUDA;
    std::lock_guard<std::mutex> lk(g_mu);
    if (!g_scratch_ptr[dev]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);
        if (e != cudaSuccess || !p) { cudaGetLastError(); return COSMO_E_CUDA; }
        g_scratch_ptr[dev] = p;
    }
    *out = static_cast<unsigned char*>(g_scratch_ptr[dev]);
    return COSMO_OK;
}

inline size_t align256(size_t b) { return (b + 255) & ~size_t(255); }

// bytes of the static scratch a call with (N, S) needs; ntiles as cosmo_snia_loglike lays its grid out
size_t static_need(int64_t N, int64_t S, int64_t* ntiles) {
    *ntiles = cdiv64(N > 0 ? N : 1, outer_tile(false, false));
    return align256((size_t)S * sizeof(Cosmo<double>)) + align256((size_t)*ntiles * (size_t)S * 5 * sizeof(double));
}

}  // namespace

extern "C" {

size_t cosmo_static_scratch_bytes(void) { return COSMO_STATIC_SCRATCH_BYTES; }

int cosmo_snia_loglike_static(const double* z, const double* mu_obs, const double* sigma, int64_t N, cosmo_params p, int64_t S,
                              double* logL, double* grad, void* stream) {
    if (N < 0 || S < 0) return COSMO_E_SIZE;
    if (S > 0 && (!p.Om || !p.OL || !p.Or || !p.H0 || !logL)) return COSMO_E_NULL;
    if (N > 0 && (!z || !mu_obs || !sigma)) return COSMO_E_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (S == 0) return COSMO_OK;
    int64_t ntiles = 0;
    if (static_need(N, S, &ntiles) > (size_t)COSMO_STATIC_SCRATCH_BYTES) return COSMO_E_STATIC_LIMIT;      // nothing launched
    if (N == 0) {
        cudaMemsetAsync(logL, 0, sizeof(double) * S, st);
        if (grad) cudaMemsetAsync(grad, 0, sizeof(double) * 4 * S, st);
        return cudaGetLastError() == cudaSuccess ? COSMO_OK : COSMO_E_CUDA;
    }
    unsigned char* w = nullptr;
    int rc = scratch_address(&w);
    if (rc) return rc;
    Cosmo<double>* consts = reinterpret_cast<Cosmo<double>*>(w);
    launch_prep(p.Om, p.OL, p.Or, p.H0, S, 1, consts, st);
    if (cudaGetLastError() != cudaSuccess) return COSMO_E_CUDA;
    OuterArgs a{};
    a.z = z; a.mu_obs = mu_obs; a.sigma = sigma; a.consts = consts; a.N = N; a.S = S; a.which = W_MU;
    a.part = reinterpret_cast<double*>(w + align256((size_t)S * sizeof(Cosmo<double>)));
    a.vec = (N % 2 == 0) && ((reinterpret_cast<uintptr_t>(z) | reinterpret_cast<uintptr_t>(mu_obs) | reinterpret_cast<uintptr_t>(sigma)) & 15) == 0;
    int ny = (int)cdiv64(S, S_CHUNK);                       // as cosmo_snia_loglike: cosmology chunks spread over gridDim.y
    int64_t cap = cdiv64((int64_t)16 * 148 * 5, ntiles);
    if (cap < 1) cap = 1;
    if (ny > cap) ny = (int)cap;
    launch_outer_f64(MODE_SNIA, a, dim3((unsigned)ntiles, (unsigned)ny), st);
    if (cudaGetLastError() != cudaSuccess) return COSMO_E_CUDA;
    launch_reduce_params(5, a.part, ntiles, S, logL, grad, st);
    return cudaGetLastError() == cudaSuccess ? COSMO_OK : COSMO_E_CUDA;
}

}  // extern "C"
