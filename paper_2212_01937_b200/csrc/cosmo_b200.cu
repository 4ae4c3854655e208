// cosmo_b200.cu -- launchers and the C ABI declared in include/cosmo_b200.h.  sm_100a only; no CPU path.
#include <atomic>
#include <cstdlib>
#include <mutex>
#include "../../include/cosmo_b200.h"
#include "../../include/cosmo_b200_diag.h"
#include "cosmo_launch.cuh"

using namespace cb;

namespace {

std::atomic<int64_t> g_launches{0};
std::atomic<int> g_last_cuda{0};

// optional timing of the dominant kernel (k_outer / k_elem) with CUDA events on the launching stream
bool g_prof_on = false;
cudaEvent_t g_prof_ev[2] = {nullptr, nullptr};
double g_prof_ms_sum = 0.0;
int64_t g_prof_n = 0;
bool g_prof_pending = false;

void prof_begin(cudaStream_t st) {
    if (!g_prof_on) return;
    if (g_prof_pending) {   // fold the previous launch in before reusing the events
        float ms = 0.f;
        if (cudaEventSynchronize(g_prof_ev[1]) == cudaSuccess && cudaEventElapsedTime(&ms, g_prof_ev[0], g_prof_ev[1]) == cudaSuccess) {
            g_prof_ms_sum += ms; ++g_prof_n;
        }
        g_prof_pending = false;
    }
    cudaEventRecord(g_prof_ev[0], st);
}
void prof_end(cudaStream_t st) {
    if (!g_prof_on) return;
    cudaEventRecord(g_prof_ev[1], st);
    g_prof_pending = true;
}

inline size_t align256(size_t b) { return (b + 255) & ~size_t(255); }
inline int64_t cdiv(int64_t a, int64_t b) { return (a + b - 1) / b; }

int check_launch() {
    ++g_launches;
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) { g_last_cuda = (int)e; return COSMO_E_CUDA; }
    return COSMO_OK;
}

// S-chunk groups in gridDim.y.  The chip holds 148 SMs x 5 resident blocks; with fewer than ~16 blocks per slot the last
// partial wave costs up to 10 % (measured, profiles/), so cosmology chunks are spread over gridDim.y until there are
// enough blocks; grad_z is then accumulated through [ny][N] partials and a tiny reduction kernel.
int grid_y(int64_t ntiles, int64_t S) {
    const int64_t nchunks = cdiv(S, S_CHUNK);
    const int64_t want = cdiv((int64_t)16 * 148 * 5, ntiles);
    return (int)(want < nchunks ? (want < 1 ? 1 : want) : nchunks);
}

struct WsLayout { size_t consts, part, gzpart, total; int ny; int64_t ntiles; };

WsLayout ws_layout(int64_t n_z, int64_t n_cosmo, int mode, uint32_t which, int with_grad, size_t elt) {
    WsLayout L{};
    const bool per_elem = (mode == COSMO_ELEMENTWISE && n_cosmo != 1);
    if (per_elem) {     // VJP: the work list of the second pass (k_elem_redo): a counter and up to n_z 32-bit indices
        L.total = with_grad ? 256 + align256((size_t)(n_z > 0 ? n_z : 1) * sizeof(unsigned)) : 0;
        L.ny = 1; L.ntiles = 0;
        return L;
    }
    L.ntiles = cdiv(n_z > 0 ? n_z : 1, outer_tile(which & (W_TL | W_AGE), which & W_DABS));   // as launch_outer dispatches
    L.ny = grid_y(L.ntiles, n_cosmo);
    L.consts = 0;
    size_t off = align256((size_t)n_cosmo * sizeof(Cosmo<double>));
    if (with_grad) {
        L.part = off;
        off += align256((size_t)L.ntiles * n_cosmo * 5 * sizeof(double));
        L.gzpart = off;
        if (L.ny > 1) off += align256((size_t)L.ny * n_z * elt);
    }
    L.total = off;
    return L;
}

int check_common(const void* z, int64_t n_z, const cosmo_params& p, int64_t n_cosmo, int mode, uint32_t which) {
    if (n_z < 0 || n_cosmo < 0) return COSMO_E_SIZE;
    if (mode != COSMO_ELEMENTWISE && mode != COSMO_OUTER) return COSMO_E_MODE;
    if (which == 0 || (which & ~uint32_t(W_ALL))) return COSMO_E_WHICH;
    if (mode == COSMO_ELEMENTWISE && !(n_cosmo == 1 || n_cosmo == n_z)) return COSMO_E_SIZE;
    if (n_z > 0 && n_cosmo == 0) return COSMO_E_SIZE;
    if (n_z > 0 && (!z || !p.Om || !p.OL || !p.Or || !p.H0)) return COSMO_E_NULL;
    return COSMO_OK;
}

template <typename T>
int launch_outer(int mode, OuterArgs& a, dim3 grid, cudaStream_t st) {
    prof_begin(st);
    if (sizeof(T) == 8) launch_outer_f64(mode, a, grid, st);
    else launch_outer_f32(mode, a, grid, st);
    prof_end(st);
    return check_launch();
}

template <typename T>
int launch_elem(bool with_grad, const T* z, const cosmo_params& p, int64_t N, unsigned which, const T* gout, T* out, T* gz, double* gparams,
                uint8_t* status, unsigned* ws, cudaStream_t st) {
    ElemArgs a{z, p.Om, p.OL, p.Or, p.H0, N, which, gout, out, gz, gparams, status, ws, ws ? ws + 64 : nullptr};
    prof_begin(st);
    if (sizeof(T) == 8) launch_elem_f64(with_grad, a, st);
    else launch_elem_f32(with_grad, a, st);
    prof_end(st);
    if (with_grad) g_launches += 1;      // the second pass
    return check_launch();
}

// forward (gout == nullptr) or fused forward+VJP
template <typename T>
int run_eval(const T* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which, const T* gout, T* out, T* gz,
             double* gparams, uint8_t* status, void* ws, size_t ws_bytes, void* stream, bool with_grad) {
    int rc = check_common(z, n_z, p, n_cosmo, mode, which);
    if (rc) return rc;
    if (with_grad && n_z > 0 && (!gout || !gz || !gparams)) return COSMO_E_NULL;
    if (!with_grad && n_z > 0 && !out) return COSMO_E_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (n_z == 0) {
        if (with_grad && gparams && n_cosmo > 0 && mode == COSMO_OUTER) {
            cudaMemsetAsync(gparams, 0, sizeof(double) * 4 * n_cosmo, st);
        }
        return COSMO_OK;
    }
    const bool per_elem = (mode == COSMO_ELEMENTWISE && n_cosmo != 1);
    if (per_elem) {
        if (!with_grad) return launch_elem<T>(false, z, p, n_z, which, nullptr, out, nullptr, nullptr, status, nullptr, st);
        if (n_z > (int64_t)0xffffffffll) return COSMO_E_SIZE;            // 32-bit work list
        WsLayout L = ws_layout(n_z, n_cosmo, mode, which, with_grad, sizeof(T));
        if (ws_bytes < L.total || !ws) return ws ? COSMO_E_WORKSPACE : COSMO_E_NULL;
        return with_grad ? launch_elem<T>(true, z, p, n_z, which, gout, out, gz, gparams, status, static_cast<unsigned*>(ws), st)
                         : launch_elem<T>(false, z, p, n_z, which, nullptr, out, nullptr, nullptr, status, static_cast<unsigned*>(ws), st);
    }
    WsLayout L = ws_layout(n_z, n_cosmo, mode, which, with_grad, sizeof(T));
    if (ws_bytes < L.total || !ws) return ws ? COSMO_E_WORKSPACE : COSMO_E_NULL;
    char* w = static_cast<char*>(ws);
    Cosmo<double>* consts = reinterpret_cast<Cosmo<double>*>(w + L.consts);
    const bool kT = which & (W_TL | W_AGE), kA = which & W_DABS;
    launch_prep(p.Om, p.OL, p.Or, p.H0, n_cosmo, (with_grad ? ((kT || kA) ? 2 : 1) : 0) | ((which & W_AGE) ? 4 : 0), consts, st);
    if ((rc = check_launch())) return rc;
    OuterArgs a{};
    a.z = z; a.gout = gout; a.out = out; a.status = status; a.consts = consts;
    a.N = n_z; a.S = n_cosmo; a.which = which;
    {
        const uintptr_t m = sizeof(T) == 8 ? 15 : 7;
        a.vec = (n_z % 2 == 0) && ((reinterpret_cast<uintptr_t>(z) | reinterpret_cast<uintptr_t>(out) |
                                    reinterpret_cast<uintptr_t>(gout) | reinterpret_cast<uintptr_t>(gz)) & m) == 0;
    }
    dim3 grid((unsigned)L.ntiles, (unsigned)L.ny);
    if (!with_grad) return launch_outer<T>(MODE_FWD, a, grid, st);
    a.part = reinterpret_cast<double*>(w + L.part);
    a.gz_accumulate = L.ny > 1;
    a.gz = a.gz_accumulate ? static_cast<void*>(w + L.gzpart) : static_cast<void*>(gz);
    if ((rc = launch_outer<T>(MODE_VJP, a, grid, st))) return rc;
    launch_reduce_vjp(sizeof(T) == 4, a.part, L.ntiles, n_cosmo, gparams, a.gz_accumulate ? a.gz : nullptr, L.ny, n_z, gz, st);
    if ((rc = check_launch())) return rc;
    return COSMO_OK;
}

template <typename T>
int run_snia(const T* z, const T* mu_obs, const T* sigma, int64_t N, cosmo_params p, int64_t S, double* logL, double* grad,
             void* ws, size_t ws_bytes, void* stream) {
    if (N < 0 || S < 0) return COSMO_E_SIZE;
    if (S > 0 && (!p.Om || !p.OL || !p.Or || !p.H0 || !logL)) return COSMO_E_NULL;
    if (N > 0 && (!z || !mu_obs || !sigma)) return COSMO_E_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (S == 0) return COSMO_OK;
    if (N == 0) {
        cudaMemsetAsync(logL, 0, sizeof(double) * S, st);
        if (grad) cudaMemsetAsync(grad, 0, sizeof(double) * 4 * S, st);
        return COSMO_OK;
    }
    WsLayout L = ws_layout(N, S, COSMO_OUTER, W_MU, 1, sizeof(T));
    if (!ws) return COSMO_E_NULL;
    if (ws_bytes < L.total) return COSMO_E_WORKSPACE;
    char* w = static_cast<char*>(ws);
    Cosmo<double>* consts = reinterpret_cast<Cosmo<double>*>(w + L.consts);
    int rc;
    launch_prep(p.Om, p.OL, p.Or, p.H0, S, 1, consts, st);
    if ((rc = check_launch())) return rc;
    OuterArgs a{};
    a.z = z; a.mu_obs = mu_obs; a.sigma = sigma; a.consts = consts; a.N = N; a.S = S; a.which = W_MU;
    a.part = reinterpret_cast<double*>(w + L.part);
    const uintptr_t m = sizeof(T) == 8 ? 15 : 7;
    a.vec = (N % 2 == 0) && ((reinterpret_cast<uintptr_t>(z) | reinterpret_cast<uintptr_t>(mu_obs) | reinterpret_cast<uintptr_t>(sigma)) & m) == 0;
    // the likelihood has no per-redshift output, so cosmology chunks can always spread over gridDim.y
    int ny = (int)cdiv(S, S_CHUNK);
    int64_t cap = cdiv((int64_t)16 * 148 * 5, L.ntiles);
    if (cap < 1) cap = 1;
    if (ny > cap) ny = (int)cap;
    dim3 grid((unsigned)L.ntiles, (unsigned)ny);
    if ((rc = launch_outer<T>(MODE_SNIA, a, grid, st))) return rc;
    launch_reduce_params(5, a.part, L.ntiles, S, logL, grad, st);
    return check_launch();
}

// log-joint with latent redshifts z[S][N] (MODE_JOINT)
template <typename T>
int run_joint(const T* z, const T* z_obs, const T* mu_obs, const T* sigma_mu, double sigma_z, double beta, double shape, int64_t N,
              cosmo_params p, int64_t S, double* logp, double* grad, T* grad_z, void* ws, size_t ws_bytes, void* stream) {
    if (N < 0 || S < 0 || !(sigma_z > 0.0) || !(beta > 0.0) || !(shape > 0.0)) return COSMO_E_SIZE;
    if (S > 0 && (!p.Om || !p.OL || !p.Or || !p.H0 || !logp)) return COSMO_E_NULL;
    if (N > 0 && S > 0 && (!z || !z_obs || !mu_obs || !sigma_mu)) return COSMO_E_NULL;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (S == 0) return COSMO_OK;
    if (N == 0) {
        cudaMemsetAsync(logp, 0, sizeof(double) * S, st);
        if (grad) cudaMemsetAsync(grad, 0, sizeof(double) * 4 * S, st);
        return COSMO_OK;
    }
    WsLayout L = ws_layout(N, S, COSMO_OUTER, W_MU, 1, sizeof(T));
    if (!ws) return COSMO_E_NULL;
    if (ws_bytes < L.total) return COSMO_E_WORKSPACE;
    char* w = static_cast<char*>(ws);
    Cosmo<double>* consts = reinterpret_cast<Cosmo<double>*>(w + L.consts);
    int rc;
    launch_prep(p.Om, p.OL, p.Or, p.H0, S, 1, consts, st);
    if ((rc = check_launch())) return rc;
    OuterArgs a{};
    a.z = z; a.z_obs = z_obs; a.mu_obs = mu_obs; a.sigma = sigma_mu; a.gz = grad_z; a.consts = consts; a.N = N; a.S = S; a.which = W_MU;
    a.sigma_z = sigma_z; a.beta = beta; a.shape_m1 = shape - 1.0;
    a.prior_norm = shape * log(beta) - lgamma(shape) - log(sigma_z) - 0.91893853320467274178;
    a.part = reinterpret_cast<double*>(w + L.part);
    const uintptr_t m = sizeof(T) == 8 ? 15 : 7;
    a.vec = (N % 2 == 0) && ((reinterpret_cast<uintptr_t>(z) | reinterpret_cast<uintptr_t>(z_obs) | reinterpret_cast<uintptr_t>(mu_obs) |
                              reinterpret_cast<uintptr_t>(sigma_mu) | reinterpret_cast<uintptr_t>(grad_z)) & m) == 0;
    int ny = (int)cdiv(S, S_CHUNK);
    int64_t cap = cdiv((int64_t)16 * 148 * 5, L.ntiles);
    if (cap < 1) cap = 1;
    if (ny > cap) ny = (int)cap;
    dim3 grid((unsigned)L.ntiles, (unsigned)ny);
    if ((rc = launch_outer<T>(MODE_JOINT, a, grid, st))) return rc;
    launch_reduce_params(5, a.part, L.ntiles, S, logp, grad, st);
    return check_launch();
}

// staging of the host-buffer call cosmo_eval_host: device scratch (grow-only until cosmo_host_release), a pinned block for the per-chunk
// parameter sums, HOST_SETS streams and one event
constexpr int HOST_SETS = 3;
std::mutex g_host_mu;
void* g_host_buf = nullptr;
size_t g_host_cap = 0;
void* g_host_pin = nullptr;
size_t g_host_pin_cap = 0;
cudaStream_t g_host_streams[HOST_SETS] = {};
cudaEvent_t g_host_ev = nullptr;

}  // namespace

extern "C" {

size_t cosmo_eval2_workspace_bytes(int64_t n, int with_grad) {
    if (n < 0 || !with_grad) return 0;
    return 256 + align256((size_t)(n > 0 ? n : 1) * sizeof(unsigned));       // counter + work list of the second pass
}

size_t cosmo_workspace_bytes(int64_t n_z, int64_t n_cosmo, int mode, uint32_t which, int with_grad) {
    if (n_z < 0 || n_cosmo < 0) return 0;
    WsLayout L = ws_layout(n_z, n_cosmo, mode, which, with_grad, sizeof(double));
    return L.total;
}

int cosmo_eval(const double* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which, double* out,
               uint8_t* status, void* workspace, size_t ws_bytes, void* stream) {
    return run_eval<double>(z, n_z, p, n_cosmo, mode, which, nullptr, out, nullptr, nullptr, status, workspace, ws_bytes, stream, false);
}
int cosmo_vjp(const double* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which, const double* grad_out,
              double* out, double* grad_z, double* grad_params, uint8_t* status, void* workspace, size_t ws_bytes, void* stream) {
    return run_eval<double>(z, n_z, p, n_cosmo, mode, which, grad_out, out, grad_z, grad_params, status, workspace, ws_bytes, stream, true);
}
int cosmo_snia_loglike(const double* z, const double* mu_obs, const double* sigma, int64_t N, cosmo_params p, int64_t S,
                       double* logL, double* grad, void* workspace, size_t ws_bytes, void* stream) {
    return run_snia<double>(z, mu_obs, sigma, N, p, S, logL, grad, workspace, ws_bytes, stream);
}
int cosmo_snia_logjoint(const double* z, const double* z_obs, const double* mu_obs, const double* sigma_mu, double sigma_z,
                        double beta, double shape, int64_t N, cosmo_params p, int64_t S, double* logp, double* grad, double* grad_z,
                        void* workspace, size_t ws_bytes, void* stream) {
    return run_joint<double>(z, z_obs, mu_obs, sigma_mu, sigma_z, beta, shape, N, p, S, logp, grad, grad_z, workspace, ws_bytes, stream);
}
int cosmo_eval_f32(const float* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which, float* out,
                   uint8_t* status, void* workspace, size_t ws_bytes, void* stream) {
    return run_eval<float>(z, n_z, p, n_cosmo, mode, which, nullptr, out, nullptr, nullptr, status, workspace, ws_bytes, stream, false);
}
int cosmo_vjp_f32(const float* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which, const float* grad_out,
                  float* out, float* grad_z, double* grad_params, uint8_t* status, void* workspace, size_t ws_bytes, void* stream) {
    return run_eval<float>(z, n_z, p, n_cosmo, mode, which, grad_out, out, grad_z, grad_params, status, workspace, ws_bytes, stream, true);
}
int cosmo_snia_loglike_f32(const float* z, const float* mu_obs, const float* sigma, int64_t N, cosmo_params p, int64_t S,
                           double* logL, double* grad, void* workspace, size_t ws_bytes, void* stream) {
    return run_snia<float>(z, mu_obs, sigma, N, p, S, logL, grad, workspace, ws_bytes, stream);
}

// Host-buffer call: the redshift axis is cut into chunks that travel through three streams with three sets of device staging buffers,
// so that the H2D copy of chunk i+1, the kernels of chunk i and the D2H copy of chunk i-1 overlap (PCIe is full duplex; the path is
// PCIe-bound: 8 B of grad_out per eval against ~20 ps of kernel time).  Three sets, not two: with two, the H2D copy of chunk i+2 waits
// in its stream behind the D2H copy of chunk i, and where as much comes back as goes in (per-element cosmologies with the VJP:
// 88 B each way per element) the two directions then run one after the other instead of together.  Pinned host memory is needed for the overlap; pageable
// memory still gives the right result.  Per-chunk parameter-gradient sums are added on the host in chunk order (deterministic).
int cosmo_eval_host(const double* z, int64_t n_z, cosmo_params p, int64_t n_cosmo, int mode, uint32_t which,
                    const double* grad_out, double* out, double* grad_z, double* grad_params, uint8_t* status) {
    int rc = check_common(z, n_z, p, n_cosmo, mode, which);
    if (rc) return rc;
    if (n_z == 0) return COSMO_OK;
    const bool with_grad = grad_out != nullptr;
    if (with_grad && (!grad_z || !grad_params)) return COSMO_E_NULL;
    if (!with_grad && !out) return COSMO_E_NULL;
    const bool outer = (mode == COSMO_OUTER), per_elem = (mode == COSMO_ELEMENTWISE && n_cosmo != 1);
    const int64_t rows = outer ? n_cosmo : 1;
    const int np = __builtin_popcount(which);
    const int64_t n_par = per_elem ? 0 : n_cosmo;             // parameters copied once (shared) or chunked with z (per element)
    // chunk length: ~32 MB of traffic per chunk (COSMO_HOST_CHUNK_MB), at least 64 Ki redshifts, even (128-bit accesses); a job of more
    // than 16 such chunks is cut into 16, up to 256 MB each: every copy call costs ~10 us of set-up, which at 32 MB was a quarter of
    // the time of a per-element VJP call (10 copies per chunk; measured 26.9 -> 22.6 ms on config 5)
    const int64_t bytes_per_z = (int64_t)sizeof(double) * ((int64_t)np * rows * ((with_grad ? 1 : 0) + (out ? 1 : 0)) + 2 + (per_elem ? 8 : 0)) + rows;
    static const int64_t chunk_mb = []() { const char* e = getenv("COSMO_HOST_CHUNK_MB"); const long v = e ? atol(e) : 0; return (int64_t)(v > 0 ? v : 32); }();
    int64_t nc = (chunk_mb << 20) / bytes_per_z;
    if (nc < 65536) nc = 65536;
    if (nc * 16 < n_z) {
        const int64_t nmax = (int64_t(256) << 20) / bytes_per_z;
        nc = cdiv(n_z, 16);
        if (nc > nmax && nmax >= 65536) nc = nmax;
    }
    nc = (nc + 1) & ~int64_t(1);
    if (nc > n_z) nc = n_z;
    const int64_t nchunks = cdiv(n_z, nc);
    const size_t b_z = align256(sizeof(double) * nc), b_pc = per_elem ? align256(sizeof(double) * nc) : 0;
    const size_t b_pl = align256(sizeof(double) * np * rows * nc);
    const size_t b_gp = align256(sizeof(double) * 4 * (per_elem ? nc : n_cosmo)), b_st = align256((size_t)rows * nc);
    const size_t b_ws = align256(cosmo_workspace_bytes(nc, per_elem ? nc : n_cosmo, mode, which, with_grad));
    const size_t per_set = b_z + 4 * b_pc + (out ? b_pl : 0) + (with_grad ? b_pl + b_z + b_gp : 0) + (status ? b_st : 0) + b_ws;
    const size_t b_par = align256(sizeof(double) * (n_par > 0 ? n_par : 1));
    const size_t total = 4 * b_par + HOST_SETS * per_set;
    std::lock_guard<std::mutex> lk(g_host_mu);
    if (!g_host_streams[0]) {
        for (int i = 0; i < HOST_SETS; ++i)
            if (cudaStreamCreateWithFlags(&g_host_streams[i], cudaStreamNonBlocking) != cudaSuccess) { g_last_cuda = (int)cudaGetLastError(); return COSMO_E_CUDA; }
        if (cudaEventCreateWithFlags(&g_host_ev, cudaEventDisableTiming) != cudaSuccess) { g_last_cuda = (int)cudaGetLastError(); return COSMO_E_CUDA; }
    }
    if (total > g_host_cap) {
        if (g_host_buf) cudaFree(g_host_buf);
        g_host_buf = nullptr; g_host_cap = 0;
        cudaError_t e = cudaMalloc(&g_host_buf, total);
        if (e != cudaSuccess) { g_last_cuda = (int)e; return COSMO_E_CUDA; }
        g_host_cap = total;
    }
    const size_t hp_bytes = with_grad && !per_elem ? sizeof(double) * 4 * n_cosmo * nchunks : 0;     // per-chunk parameter sums (pinned)
    if (hp_bytes > g_host_pin_cap) {
        if (g_host_pin) cudaFreeHost(g_host_pin);
        g_host_pin = nullptr; g_host_pin_cap = 0;
        if (cudaMallocHost(&g_host_pin, hp_bytes) != cudaSuccess) { g_last_cuda = (int)cudaGetLastError(); return COSMO_E_CUDA; }
        g_host_pin_cap = hp_bytes;
    }
    char* base = static_cast<char*>(g_host_buf);
    size_t off = 0;
    auto take = [&](size_t b) { char* q = base + off; off += b; return q; };
    double* d_par[4];
    for (int i = 0; i < 4; ++i) d_par[i] = (double*)take(b_par);
    struct Set { double *z, *pc[4], *out, *gout, *gz, *gp; uint8_t* st; void* ws; } S[HOST_SETS];
    for (int k = 0; k < HOST_SETS; ++k) {
        S[k].z = (double*)take(b_z);
        for (int i = 0; i < 4; ++i) S[k].pc[i] = per_elem ? (double*)take(b_pc) : d_par[i];
        S[k].out = out ? (double*)take(b_pl) : nullptr;
        S[k].gout = with_grad ? (double*)take(b_pl) : nullptr;
        S[k].gz = with_grad ? (double*)take(b_z) : nullptr;
        S[k].gp = with_grad ? (double*)take(b_gp) : nullptr;
        S[k].st = status ? (uint8_t*)take(b_st) : nullptr;
        S[k].ws = take(b_ws);
    }
    const double* hp[4] = {p.Om, p.OL, p.Or, p.H0};
    cudaStream_t s0 = g_host_streams[0];
    if (!per_elem) {
        for (int i = 0; i < 4; ++i) cudaMemcpyAsync(d_par[i], hp[i], sizeof(double) * n_cosmo, cudaMemcpyHostToDevice, s0);
        cudaEventRecord(g_host_ev, s0);
        for (int k = 1; k < HOST_SETS; ++k) cudaStreamWaitEvent(g_host_streams[k], g_host_ev, 0);
    }
    const size_t hpitch = sizeof(double) * n_z;               // host planes [np][rows][n_z]: row pitch n_z
    double* hsum = static_cast<double*>(g_host_pin);
    for (int64_t c = 0; c < nchunks && rc == COSMO_OK; ++c) {
        const int k = (int)(c % HOST_SETS);
        cudaStream_t st = g_host_streams[k];
        const int64_t n0 = c * nc, n = (n0 + nc <= n_z) ? nc : (n_z - n0);
        cudaMemcpyAsync(S[k].z, z + n0, sizeof(double) * n, cudaMemcpyHostToDevice, st);
        if (per_elem)
            for (int i = 0; i < 4; ++i) cudaMemcpyAsync(S[k].pc[i], hp[i] + n0, sizeof(double) * n, cudaMemcpyHostToDevice, st);
        if (with_grad)
            cudaMemcpy2DAsync(S[k].gout, sizeof(double) * n, grad_out + n0, hpitch, sizeof(double) * n, (size_t)np * rows, cudaMemcpyHostToDevice, st);
        cosmo_params dp{S[k].pc[0], S[k].pc[1], S[k].pc[2], S[k].pc[3]};
        const int64_t ncos = per_elem ? n : n_cosmo;
        rc = with_grad ? cosmo_vjp(S[k].z, n, dp, ncos, mode, which, S[k].gout, S[k].out, S[k].gz, S[k].gp, S[k].st, S[k].ws, b_ws, st)
                       : cosmo_eval(S[k].z, n, dp, ncos, mode, which, S[k].out, S[k].st, S[k].ws, b_ws, st);
        if (rc) break;
        if (out) cudaMemcpy2DAsync(out + n0, hpitch, S[k].out, sizeof(double) * n, sizeof(double) * n, (size_t)np * rows, cudaMemcpyDeviceToHost, st);
        if (status) cudaMemcpy2DAsync(status + n0, (size_t)n_z, S[k].st, (size_t)n, (size_t)n, (size_t)rows, cudaMemcpyDeviceToHost, st);
        if (with_grad) {
            cudaMemcpyAsync(grad_z + n0, S[k].gz, sizeof(double) * n, cudaMemcpyDeviceToHost, st);
            if (per_elem) cudaMemcpy2DAsync(grad_params + n0, hpitch, S[k].gp, sizeof(double) * n, sizeof(double) * n, 4, cudaMemcpyDeviceToHost, st);
            else cudaMemcpyAsync(hsum + c * 4 * n_cosmo, S[k].gp, sizeof(double) * 4 * n_cosmo, cudaMemcpyDeviceToHost, st);
        }
    }
    cudaError_t es = cudaSuccess;
    for (int k = 0; k < HOST_SETS; ++k) { const cudaError_t e = cudaStreamSynchronize(g_host_streams[k]); if (es == cudaSuccess) es = e; }
    if (rc) return rc;
    if (es != cudaSuccess) { g_last_cuda = (int)es; return COSMO_E_CUDA; }
    if (with_grad && !per_elem) {
        for (int64_t i = 0; i < 4 * n_cosmo; ++i) {
            double v = 0.0;
            for (int64_t c = 0; c < nchunks; ++c) v += hsum[c * 4 * n_cosmo + i];
            grad_params[i] = v;
        }
    }
    return COSMO_OK;
}

void cosmo_host_release(void) {
    std::lock_guard<std::mutex> lk(g_host_mu);
    if (g_host_buf) cudaFree(g_host_buf);
    if (g_host_pin) cudaFreeHost(g_host_pin);
    g_host_buf = nullptr; g_host_cap = 0; g_host_pin = nullptr; g_host_pin_cap = 0;
}

int cosmo_eval2(const double* z1, const double* z2, int64_t n, cosmo_params p, int64_t n_cosmo, uint32_t which, const double* grad_out,
                double* out, double* grad_z1, double* grad_z2, double* grad_params, uint8_t* status, void* workspace, size_t ws_bytes,
                void* stream) {
    if (n < 0 || !(n_cosmo == 1 || n_cosmo == n)) return COSMO_E_SIZE;
    if (which == 0 || (which & ~uint32_t(W_DC | W_DM | W_TL | W_DABS | W_DA))) return COSMO_E_WHICH;
    if (n == 0) return COSMO_OK;
    if (!z1 || !z2 || !p.Om || !p.OL || !p.Or || !p.H0) return COSMO_E_NULL;
    if (grad_out ? (!grad_z1 || !grad_z2 || !grad_params) : !out) return COSMO_E_NULL;
    if (grad_out) {
        if (n > (int64_t)0xffffffffll) return COSMO_E_SIZE;              // 32-bit work list
        if (!workspace) return COSMO_E_NULL;
        if (ws_bytes < cosmo_eval2_workspace_bytes(n, 1)) return COSMO_E_WORKSPACE;
    }
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    prof_begin(st);
    launch_two(z1, z2, p.Om, p.OL, p.Or, p.H0, n, n_cosmo, which, grad_out, out, grad_z1, grad_z2, grad_params, status,
               grad_out ? static_cast<unsigned*>(workspace) : nullptr, st);
    prof_end(st);
    if (grad_out) g_launches += 1;
    return check_launch();
}

size_t cosmo_eval_w_workspace_bytes(int64_t n_cosmo) {
    if (n_cosmo <= 0) return 0;
    // a shared cosmology's factored block, or (per-element cosmologies) the counter + work list of the second pass
    return n_cosmo == 1 ? align256(w_cosmo_bytes()) : 256 + align256((size_t)n_cosmo * sizeof(unsigned));
}

int cosmo_eval_w(const double* z, int64_t n, const double* Om, const double* OL, const double* Or, const double* Ow13,
                 const double* Ow23, const double* H0, int64_t n_cosmo, uint32_t which, const double* grad_out, double* out,
                 double* dout_dz, double* grad_z, double* grad_params, uint8_t* status, void* workspace, size_t ws_bytes, void* stream) {
    if (n < 0 || !(n_cosmo == 1 || n_cosmo == n)) return COSMO_E_SIZE;
    if (which == 0 || (which & ~uint32_t(W_DC | W_DM | W_DL | W_MU | W_TL | W_DABS))) return COSMO_E_WHICH;
    if (n == 0) return COSMO_OK;
    if (!z || !Om || !OL || !Or || !Ow13 || !Ow23 || !H0) return COSMO_E_NULL;
    if (grad_out ? (!grad_z || !grad_params) : !out) return COSMO_E_NULL;
    if (n > (int64_t)0xffffffffll) return COSMO_E_SIZE;                  // 32-bit work list
    if (!workspace) return COSMO_E_NULL;
    if (ws_bytes < cosmo_eval_w_workspace_bytes(n_cosmo)) return COSMO_E_WORKSPACE;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    prof_begin(st);
    launch_w(z, Om, OL, Or, Ow13, Ow23, H0, n, n_cosmo, which, grad_out, out, dout_dz, grad_z, grad_params, status, workspace, st);
    prof_end(st);
    g_launches += (n_cosmo == 1) ? 1 : 2;          // prep kernel, or memset-free second pass (+ its list reset)
    return check_launch();
}

int cosmo_carlson_pair(const double* x, const double* m, const double* s, const double* p, int64_t n, double* rf, double* rd,
                       double* rj, void* stream) {
    if (n < 0) return COSMO_E_SIZE;
    if (n == 0) return COSMO_OK;
    if (!x || !m || !s || !p || !rf || !rd || !rj) return COSMO_E_NULL;
    launch_carlson_pair(x, m, s, p, n, rf, rd, rj, static_cast<cudaStream_t>(stream));
    return check_launch();
}

int cosmo_probe_fma_f64(int blocks, int iters, double* sink, void* stream) {
    if (blocks <= 0 || iters < 0) return COSMO_E_SIZE;
    if (!sink) return COSMO_E_NULL;
    launch_probe_fma(false, blocks, iters, sink, static_cast<cudaStream_t>(stream));
    return check_launch();
}
int cosmo_probe_fma_f32(int blocks, int iters, float* sink, void* stream) {
    if (blocks <= 0 || iters < 0) return COSMO_E_SIZE;
    if (!sink) return COSMO_E_NULL;
    launch_probe_fma(true, blocks, iters, sink, static_cast<cudaStream_t>(stream));
    return check_launch();
}

int cosmo_profile(int on) {
    if (on && !g_prof_ev[0]) {
        if (cudaEventCreate(&g_prof_ev[0]) != cudaSuccess || cudaEventCreate(&g_prof_ev[1]) != cudaSuccess) {
            g_last_cuda = (int)cudaGetLastError();
            return COSMO_E_CUDA;
        }
    }
    g_prof_on = on != 0;
    g_prof_ms_sum = 0.0; g_prof_n = 0; g_prof_pending = false;
    return COSMO_OK;
}
double cosmo_profile_mean_ms(int64_t* n_launches) {
    if (g_prof_pending) {
        float ms = 0.f;
        if (cudaEventSynchronize(g_prof_ev[1]) == cudaSuccess && cudaEventElapsedTime(&ms, g_prof_ev[0], g_prof_ev[1]) == cudaSuccess) {
            g_prof_ms_sum += ms; ++g_prof_n;
        }
        g_prof_pending = false;
    }
    if (n_launches) *n_launches = g_prof_n;
    return g_prof_n ? g_prof_ms_sum / (double)g_prof_n : 0.0;
}

int64_t cosmo_launch_count(void) { return g_launches.load(); }
int cosmo_last_cuda_error(void) { return g_last_cuda.load(); }
const char* cosmo_strerror(int code) {
    switch (code) {
        case COSMO_OK: return "ok";
        case COSMO_E_NULL: return "a required pointer is NULL";
        case COSMO_E_SIZE: return "bad size (negative, or n_cosmo incompatible with mode)";
        case COSMO_E_WHICH: return "bad `which` bitmask";
        case COSMO_E_MODE: return "unknown mode";
        case COSMO_E_WORKSPACE: return "workspace too small (see cosmo_workspace_bytes)";
        case COSMO_E_CUDA: return "CUDA launch or runtime error (see cosmo_last_cuda_error)";
        case COSMO_E_STATIC_LIMIT: return "problem too large for the fixed static scratch (COSMO_STATIC_SCRATCH_BYTES): use the workspace call";
        default: return "unknown error code";
    }
}
const char* cosmo_version(void) { return "cosmo_b200 0.1.0 (sm_100a)"; }

}  // extern "C"
