// C-ABI layer of the batched small-grid integrator (include/cavmag.h "Batched sweeps of small grids").
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include "../../include/cavmag.h"
#include "batch_kernel.cuh"

using namespace cavmag;

struct cav_batch {
    cav_grid grid;
    cav_params prm;
    int n_rep = 0, N = 0, nc = 0, esize = 4;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    double* d_B0 = nullptr;
    void* d_u = nullptr;
    double* d_modep = nullptr;
    std::vector<double> h_modep;   // host mirror of d_modep
    double* d_drive = nullptr;     // [5][N] or NULL: no drive
    double* d_pol = nullptr;       // [N][6] polarisation + quadrature axes or NULL: x^, y^
    int split_nllg = 0;            // 0: unified RK45; n >= 1: operator-split loop with n LLG sub-steps per cavity step
    double* d_spec = nullptr;      // [n_rep][spec_K][2N + n_sub][2] Fourier sums or NULL
    long long* d_spec_n = nullptr; // [n_rep]
    int spec_K = 0;
    double spec_w0 = 0.0, spec_dw = 0.0;
    int modep_per_rep = 0;
    void* d_m = nullptr;
    double* d_a = nullptr;
    BatchCtl* d_ctl = nullptr;
    double* d_trace = nullptr;
    double sample_dt = 0.0, trace_t0 = 0.0;
    int trace_cap = 0;
    bool m_set = false;
    size_t smem_optin = 0;
    int n_sm = 148;
    char cuda_err[256] = {0};
};

namespace {

#define CKB(call)                                                                     \
    do {                                                                              \
        cudaError_t e_ = (call);                                                      \
        if (e_ != cudaSuccess) {                                                      \
            snprintf(b->cuda_err, sizeof(b->cuda_err), "%s: %s", #call, cudaGetErrorString(e_)); \
            cudaGetLastError();                                                       \
            return (e_ == cudaErrorMemoryAllocation) ? CAV_E_NOMEM : CAV_E_CUDA;      \
        }                                                                             \
    } while (0)

template <typename T>
__global__ void k_batch_normalize(T* m, int nc, int n_sub, int n_rep) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)nc * n_sub * n_rep) return;
    const long long rs = i / nc, r = i - rs * nc;
    T* p = m + rs * 3 * nc + r;
    const T x = p[0], y = p[nc], z = p[2 * nc];
    const T n2 = x * x + y * y + z * z;
    const T inv = n2 > (T)0 ? (T)1 / sqrt(n2) : (T)0;
    p[0] = x * inv; p[nc] = y * inv; p[2 * nc] = z * inv;
}

int row_len_of(const cav_batch* b) { return 1 + 4 * b->N + 3 * b->prm.n_sub; }

template <typename T, int NSUB>
const void* batch_fn(int threads, bool two_per_sm) {
    if (threads <= 128) return (const void*)k_batch<T, NSUB, 128, 1>;
    if (threads <= 256) return (const void*)k_batch<T, NSUB, 256, 1>;
    if (threads <= 512) {
        if constexpr (NSUB == 1) { if (two_per_sm) return (const void*)k_batch<T, NSUB, 512, 2>; }
        return (const void*)k_batch<T, NSUB, 512, 1>;
    }
    return (const void*)k_batch<T, NSUB, 1024, 1>;
}

int pull_ctl(cav_batch* b, std::vector<BatchCtl>& h) {
    h.resize(b->n_rep);
    CKB(cudaMemcpyAsync(h.data(), b->d_ctl, sizeof(BatchCtl) * b->n_rep, cudaMemcpyDeviceToHost, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

}  // namespace

namespace cavmag {

// [N][6] = (p_n, q_n): p_n normalised; q_n as given, or z^ x p_n (reading G32).  CAV_E_ARG for a zero vector.
int pack_polarisation(int N, const double* pol, const double* quad, double* out) {
    for (int n = 0; n < N; ++n) {
        const double* p = pol + 3 * n;
        const double len = std::sqrt(p[0] * p[0] + p[1] * p[1] + p[2] * p[2]);
        if (!(len > 0.0)) return CAV_E_ARG;
        double* o = out + 6 * n;
        for (int i = 0; i < 3; ++i) o[i] = p[i] / len;
        if (quad) { for (int i = 0; i < 3; ++i) o[3 + i] = quad[3 * n + i]; }
        else { o[3] = -o[1]; o[4] = o[0]; o[5] = 0.0; }
    }
    return CAV_OK;
}

// Launches k_batch for A.n_rep replicas (also used by cav_run for a single tiny grid: CAV_PATH_BLOCK).
int launch_batch_kernel(BatchArgs& A, bool f32, int n_sub, bool two_per_sm, size_t smem_optin, cudaStream_t stream,
                        cudaError_t* cuda_err) {
    auto fail = [&](cudaError_t e) { *cuda_err = e; cudaGetLastError(); return e == cudaErrorMemoryAllocation ? CAV_E_NOMEM : CAV_E_CUDA; };
    const size_t esize = f32 ? 4 : 8;
    int threads = (A.nc + 31) / 32 * 32;
    if (threads < 64) threads = 64;
    const size_t ms_bytes = (size_t)n_sub * 3 * A.nc * esize, u_bytes = (size_t)A.N * A.nc * esize;
    const void* fn = f32 ? (n_sub == 1 ? batch_fn<float, 1>(threads, two_per_sm) : batch_fn<float, 2>(threads, two_per_sm))
                         : (n_sub == 1 ? batch_fn<double, 1>(threads, two_per_sm) : batch_fn<double, 2>(threads, two_per_sm));
    cudaFuncAttributes fa;
    cudaError_t e = cudaFuncGetAttributes(&fa, fn);
    if (e != cudaSuccess) return fail(e);
    const size_t room = smem_optin > fa.sharedSizeBytes ? smem_optin - fa.sharedSizeBytes : 0;
    if (ms_bytes > room) return CAV_E_UNSUPPORTED;
    A.u_in_smem = (A.N > 0 && ms_bytes + u_bytes <= room && ms_bytes + u_bytes <= 96 * 1024) ? 1 : 0;
    const size_t smem = ms_bytes + (A.u_in_smem ? u_bytes : 0);
    e = cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)room);
    if (e != cudaSuccess) return fail(e);
    void* params[] = {&A};
    e = cudaLaunchKernel(fn, dim3(A.n_rep), dim3(threads), params, smem, stream);
    if (e != cudaSuccess) return fail(e);
    return CAV_OK;
}

// Launches the cooperative variant (COOP) for ONE simulation of A.nc cells on ceil(nc / 512) co-resident blocks.
int launch_coop_kernel(BatchArgs& A, bool f32, int n_sub, cudaStream_t stream, cudaError_t* cuda_err) {
    auto fail = [&](cudaError_t e) { *cuda_err = e; cudaGetLastError(); return e == cudaErrorMemoryAllocation ? CAV_E_NOMEM : CAV_E_CUDA; };
    const int threads = 512;
    A.nblk = (A.nc + threads - 1) / threads;
    A.n_rep = 1; A.u_in_smem = 0;
    const void* fn = f32 ? (n_sub == 1 ? (const void*)k_batch<float, 1, 512, 1, true> : (const void*)k_batch<float, 2, 512, 1, true>)
                         : (n_sub == 1 ? (const void*)k_batch<double, 1, 512, 1, true> : (const void*)k_batch<double, 2, 512, 1, true>);
    int per_sm = 0, dev = 0, n_sm = 0;
    cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, fn, threads, 0);
    if (e != cudaSuccess) return fail(e);
    cudaGetDevice(&dev);
    cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev);
    if (A.nblk > per_sm * n_sm) return CAV_E_UNSUPPORTED;          // the grid barrier needs every block resident
    e = cudaMemsetAsync(A.bar, 0, sizeof(unsigned long long), stream);
    if (e != cudaSuccess) return fail(e);
    void* params[] = {&A};
    e = cudaLaunchCooperativeKernel(fn, dim3(A.nblk), dim3(threads), params, 0, stream);
    if (e != cudaSuccess) return fail(e);
    return CAV_OK;
}

}  // namespace cavmag

extern "C" {

int cav_batch_create(const cav_grid* grid, const cav_params* prm, int n_rep, cav_batch** out) {
    if (!grid || !prm || !out || n_rep < 1) return CAV_E_ARG;
    *out = nullptr;
    if (grid->nx < 1 || grid->ny < 1 || grid->nz < 1 || !(grid->dx > 0) || !(grid->dy > 0) || !(grid->dz > 0)) return CAV_E_ARG;
    const long long nc = (long long)grid->nx * grid->ny * grid->nz;
    if (nc > kBatchMaxCells) return CAV_E_ARG;
    if (!(prm->Ms > 0) || prm->Aex < 0 || !(prm->gamma > 0) || prm->alpha < 0) return CAV_E_ARG;
    if (prm->n_sub != 1 && prm->n_sub != 2) return CAV_E_ARG;
    if (prm->precision != CAV_F32 && prm->precision != CAV_F64) return CAV_E_ARG;
    if (prm->overlap_norm != CAV_NORM_NCELLS && prm->overlap_norm != CAV_NORM_SUM_U) return CAV_E_ARG;
    int dev = 0, ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return CAV_E_UNSUPPORTED; }
    cudaDeviceProp dp;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&dp, dev) != cudaSuccess) { cudaGetLastError(); return CAV_E_UNSUPPORTED; }
    if (dp.major != 10) return CAV_E_UNSUPPORTED;
    cav_batch* b = new (std::nothrow) cav_batch();
    if (!b) return CAV_E_NOMEM;
    b->grid = *grid; b->prm = *prm; b->n_rep = n_rep; b->nc = (int)nc;
    b->esize = prm->precision == CAV_F32 ? 4 : 8;
    b->smem_optin = dp.sharedMemPerBlockOptin;
    b->n_sm = dp.multiProcessorCount;
    auto fail = [&](int code) { cav_batch_destroy(b); return code; };
    if (cudaStreamCreateWithFlags(&b->stream, cudaStreamNonBlocking) != cudaSuccess) return fail(CAV_E_CUDA);
    b->own_stream = true;
    const size_t mbytes = (size_t)n_rep * prm->n_sub * 3 * nc * b->esize;
    if (cudaMalloc(&b->d_B0, sizeof(double) * 3 * n_rep) != cudaSuccess || cudaMalloc(&b->d_m, mbytes) != cudaSuccess ||
        cudaMalloc(&b->d_ctl, sizeof(BatchCtl) * n_rep) != cudaSuccess ||
        cudaMalloc(&b->d_a, sizeof(double) * 2 * CAV_MAX_MODES * n_rep) != cudaSuccess ||
        cudaMalloc(&b->d_modep, sizeof(double) * 7 * CAV_MAX_MODES * n_rep) != cudaSuccess) {
        cudaGetLastError();
        return fail(CAV_E_NOMEM);
    }
    std::vector<double> B0(3 * (size_t)n_rep);
    for (int r = 0; r < n_rep; ++r) for (int i = 0; i < 3; ++i) B0[3 * r + i] = prm->B0[i];
    std::vector<BatchCtl> ctl(n_rep);
    for (auto& c : ctl) { memset(&c, 0, sizeof(c)); c.dt_min = INFINITY; }
    if (cudaMemcpy(b->d_B0, B0.data(), sizeof(double) * B0.size(), cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemcpy(b->d_ctl, ctl.data(), sizeof(BatchCtl) * n_rep, cudaMemcpyHostToDevice) != cudaSuccess ||
        cudaMemset(b->d_a, 0, sizeof(double) * 2 * CAV_MAX_MODES * n_rep) != cudaSuccess)
        return fail(CAV_E_CUDA);
    *out = b;
    return CAV_OK;
}

int cav_batch_destroy(cav_batch* b) {
    if (!b) return CAV_E_ARG;
    if (b->stream) cudaStreamSynchronize(b->stream);
    cudaFree(b->d_B0); cudaFree(b->d_u); cudaFree(b->d_modep); cudaFree(b->d_drive); cudaFree(b->d_m); cudaFree(b->d_a);
    cudaFree(b->d_pol); cudaFree(b->d_spec); cudaFree(b->d_spec_n);
    cudaFree(b->d_ctl); cudaFree(b->d_trace);
    if (b->own_stream && b->stream) cudaStreamDestroy(b->stream);
    cudaGetLastError();
    delete b;
    return CAV_OK;
}

int cav_batch_set_stream(cav_batch* b, void* stream) {
    if (!b) return CAV_E_ARG;
    CKB(cudaStreamSynchronize(b->stream));
    if (b->own_stream && b->stream) cudaStreamDestroy(b->stream);
    b->stream = (cudaStream_t)stream;
    b->own_stream = false;
    return CAV_OK;
}

int cav_batch_set_field(cav_batch* b, const double* B0) {
    if (!b || !B0) return CAV_E_ARG;
    CKB(cudaMemcpyAsync(b->d_B0, B0, sizeof(double) * 3 * b->n_rep, cudaMemcpyHostToDevice, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_set_modes(cav_batch* b, int N, const void* u, const double* omega, const double* kappa, const double* g,
                        const double* Gamma, const double* Phi, int per_replica) {
    if (!b || N < 0 || N > CAV_MAX_MODES) return CAV_E_ARG;
    if (N > 0 && (!u || !omega || !kappa || !g)) return CAV_E_ARG;
    // overlap normalisation W_n (G4) first, from the caller's host array: N_cells, or sum_r u_n (fixed-order host sum).
    // CAV_E_SINGULAR_NORM is returned before anything in the handle has changed.
    std::vector<double> invW(N > 0 ? N : 1, 1.0 / (double)b->nc);
    if (N > 0 && b->prm.overlap_norm == CAV_NORM_SUM_U) {
        for (int n = 0; n < N; ++n) {
            double sum = 0.0;
            for (int r = 0; r < b->nc; ++r)
                sum += b->esize == 4 ? (double)((const float*)u)[(size_t)n * b->nc + r] : ((const double*)u)[(size_t)n * b->nc + r];
            if (std::fabs(sum) < 1e-6 * (double)b->nc) return CAV_E_SINGULAR_NORM;
            invW[n] = 1.0 / sum;
        }
    }
    CKB(cudaStreamSynchronize(b->stream));
    // a CUDA failure below leaves the batch with no modes (consistent), not with a half-uploaded table
    struct Guard {
        cav_batch* b; bool ok;
        ~Guard() { if (!ok) { b->N = 0; cudaFree(b->d_u); b->d_u = nullptr; b->h_modep.clear(); b->modep_per_rep = 0; cudaGetLastError(); } }
    } guard{b, false};
    cudaFree(b->d_u);
    b->d_u = nullptr;
    cudaFree(b->d_drive);
    b->d_drive = nullptr;                  // a new mode set clears the drive,
    cudaFree(b->d_pol);
    b->d_pol = nullptr;                    // the polarisation (back to x^)
    cudaFree(b->d_spec); cudaFree(b->d_spec_n);
    b->d_spec = nullptr; b->d_spec_n = nullptr; b->spec_K = 0;      // and the spectrum (its layout depends on N)
    b->N = N;
    b->modep_per_rep = per_replica ? 1 : 0;
    if (N > 0) {
        const size_t ub = (size_t)N * b->nc * b->esize;
        CKB(cudaMalloc(&b->d_u, ub));
        CKB(cudaMemcpyAsync(b->d_u, u, ub, cudaMemcpyHostToDevice, b->stream));
        const int reps = per_replica ? b->n_rep : 1;
        std::vector<double> mp((size_t)reps * 7 * N);
        for (int r = 0; r < reps; ++r)
            for (int n = 0; n < N; ++n) {
                const size_t i = (size_t)r * N + n;
                const double Gm = Gamma ? Gamma[i] : 0.0, Ph = Phi ? Phi[i] : 0.0;
                double* q = mp.data() + (size_t)r * 7 * N;
                q[n] = omega[i]; q[N + n] = kappa[i];
                q[2 * N + n] = g[i] + Gm * std::cos(Ph); q[3 * N + n] = Gm * std::sin(Ph); q[4 * N + n] = invW[n];
                q[5 * N + n] = q[2 * N + n]; q[6 * N + n] = q[3 * N + n];          // reciprocal until cav_batch_set_backaction
            }
        b->h_modep = mp;
        CKB(cudaMemcpyAsync(b->d_modep, mp.data(), sizeof(double) * mp.size(), cudaMemcpyHostToDevice, b->stream));
        CKB(cudaStreamSynchronize(b->stream));
    }
    CKB(cudaMemsetAsync(b->d_a, 0, sizeof(double) * 2 * CAV_MAX_MODES * b->n_rep, b->stream));
    cudaFree(b->d_trace);
    b->d_trace = nullptr; b->trace_cap = 0; b->sample_dt = 0.0;      // the row length changed
    CKB(cudaStreamSynchronize(b->stream));
    guard.ok = true;
    return CAV_OK;
}

int cav_batch_set_backaction(cav_batch* b, const double* g_b, const double* Gamma_b, const double* Phi_b) {
    if (!b) return CAV_E_ARG;
    const int N = b->N;
    if (N == 0) return CAV_OK;
    const int reps = b->modep_per_rep ? b->n_rep : 1;
    for (int r = 0; r < reps; ++r) {
        double* q = b->h_modep.data() + (size_t)r * 7 * N;
        for (int n = 0; n < N; ++n) {
            if (g_b) {
                const double Gm = Gamma_b ? Gamma_b[n] : 0.0, Ph = Phi_b ? Phi_b[n] : 0.0;
                q[5 * N + n] = g_b[n] + Gm * std::cos(Ph); q[6 * N + n] = Gm * std::sin(Ph);
            } else {
                q[5 * N + n] = q[2 * N + n]; q[6 * N + n] = q[3 * N + n];
            }
        }
    }
    CKB(cudaMemcpyAsync(b->d_modep, b->h_modep.data(), sizeof(double) * b->h_modep.size(), cudaMemcpyHostToDevice, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_set_drive(cav_batch* b, const double* amp, const double* t0, const double* sigma, const double* omega_d) {
    if (!b) return CAV_E_ARG;
    CKB(cudaStreamSynchronize(b->stream));
    cudaFree(b->d_drive);
    b->d_drive = nullptr;
    if (!amp || b->N == 0) return CAV_OK;
    if (!t0 || !sigma) return CAV_E_ARG;
    const int N = b->N;
    std::vector<double> d(5 * (size_t)N);
    for (int n = 0; n < N; ++n) {
        if (!(sigma[n] > 0.0)) return CAV_E_ARG;
        d[n] = amp[2 * n]; d[N + n] = amp[2 * n + 1]; d[2 * N + n] = t0[n];
        d[3 * N + n] = 1.0 / (2.0 * sigma[n] * sigma[n]); d[4 * N + n] = omega_d ? omega_d[n] : 0.0;
    }
    CKB(cudaMalloc(&b->d_drive, sizeof(double) * d.size()));
    CKB(cudaMemcpyAsync(b->d_drive, d.data(), sizeof(double) * d.size(), cudaMemcpyHostToDevice, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_set_m(cav_batch* b, const void* m, int per_replica) {
    if (!b || !m) return CAV_E_ARG;
    const size_t one = (size_t)b->prm.n_sub * 3 * b->nc * b->esize;
    if (per_replica) CKB(cudaMemcpyAsync(b->d_m, m, one * b->n_rep, cudaMemcpyHostToDevice, b->stream));
    else
        for (int r = 0; r < b->n_rep; ++r)
            CKB(cudaMemcpyAsync((char*)b->d_m + one * r, m, one, cudaMemcpyHostToDevice, b->stream));
    const long long n = (long long)b->nc * b->prm.n_sub * b->n_rep;
    const int blocks = (int)((n + 255) / 256);
    if (b->esize == 4) k_batch_normalize<float><<<blocks, 256, 0, b->stream>>>((float*)b->d_m, b->nc, b->prm.n_sub, b->n_rep);
    else k_batch_normalize<double><<<blocks, 256, 0, b->stream>>>((double*)b->d_m, b->nc, b->prm.n_sub, b->n_rep);
    CKB(cudaGetLastError());
    std::vector<BatchCtl> h;
    int rc = pull_ctl(b, h);
    if (rc) return rc;
    for (auto& c : h) c.status = 0;
    CKB(cudaMemcpyAsync(b->d_ctl, h.data(), sizeof(BatchCtl) * b->n_rep, cudaMemcpyHostToDevice, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    b->m_set = true;
    return CAV_OK;
}

int cav_batch_set_a(cav_batch* b, const double* a, int per_replica) {
    if (!b || (!a && b->N > 0)) return CAV_E_ARG;
    if (b->N == 0) return CAV_OK;
    const size_t one = sizeof(double) * 2 * b->N;
    if (per_replica) CKB(cudaMemcpyAsync(b->d_a, a, one * b->n_rep, cudaMemcpyHostToDevice, b->stream));
    else
        for (int r = 0; r < b->n_rep; ++r)
            CKB(cudaMemcpyAsync((char*)b->d_a + one * r, a, one, cudaMemcpyHostToDevice, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_trace_row_len(cav_batch* b, int* row_len) {
    if (!b || !row_len) return CAV_E_ARG;
    *row_len = row_len_of(b);
    return CAV_OK;
}

int cav_batch_set_trace(cav_batch* b, double sample_dt, int capacity) {
    if (!b || capacity < 0) return CAV_E_ARG;
    std::vector<BatchCtl> h;
    int rc = pull_ctl(b, h);
    if (rc) return rc;
    cudaFree(b->d_trace);
    b->d_trace = nullptr;
    b->sample_dt = (sample_dt > 0.0 && capacity > 0) ? sample_dt : 0.0;
    b->trace_cap = b->sample_dt > 0.0 ? capacity : 0;
    b->trace_t0 = h[0].t;                  // trace origin: the time of replica 0 now
    for (auto& c : h) { c.trace_n = 0; c.trace_acc0 = c.accepted; }
    if (b->trace_cap > 0) {
        const size_t bytes = sizeof(double) * (size_t)b->n_rep * b->trace_cap * row_len_of(b);
        CKB(cudaMalloc(&b->d_trace, bytes));
        CKB(cudaMemsetAsync(b->d_trace, 0, bytes, b->stream));
    }
    CKB(cudaMemcpyAsync(b->d_ctl, h.data(), sizeof(BatchCtl) * b->n_rep, cudaMemcpyHostToDevice, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_run(cav_batch* b, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps) {
    if (!b) return CAV_E_ARG;
    if (!b->m_set) return CAV_E_STATE;
    if ((tol > 0.0) == (fixed_dt > 0.0)) return CAV_E_ARG;
    if (!(t_end == t_end) || (std::isinf(t_end) && max_steps <= 0)) return CAV_E_ARG;
    const cav_params& p = b->prm;
    BatchArgs A;
    memset(&A, 0, sizeof(A));
    A.nx = b->grid.nx; A.ny = b->grid.ny; A.nz = b->grid.nz; A.nc = b->nc; A.N = b->N; A.n_rep = b->n_rep;
    const double pe = 2.0 * p.Aex / p.Ms;
    A.ex_wx = pe / (b->grid.dx * b->grid.dx); A.ex_wy = pe / (b->grid.dy * b->grid.dy); A.ex_wz = pe / (b->grid.dz * b->grid.dz);
    A.an_pref = 2.0 * p.Ku / p.Ms;
    const double an = std::sqrt(p.ku_axis[0] * p.ku_axis[0] + p.ku_axis[1] * p.ku_axis[1] + p.ku_axis[2] * p.ku_axis[2]);
    for (int i = 0; i < 3; ++i) A.axis[i] = an > 0.0 ? p.ku_axis[i] / an : (i == 2 ? 1.0 : 0.0);
    A.alpha = p.alpha; A.llg = -p.gamma / (1.0 + p.alpha * p.alpha);
    A.B_exch_inter = p.n_sub == 2 ? p.B_exch_inter : 0.0;
    A.two_over_gamma = 2.0 / p.gamma; A.inv_nc = 1.0 / (double)b->nc;
    A.renormalize = p.renormalize;
    A.B0 = b->d_B0; A.u = b->d_u; A.modep = b->d_modep; A.modep_per_rep = b->modep_per_rep;
    A.m = b->d_m; A.a = b->d_a; A.ctl = b->d_ctl;
    A.t_end = t_end; A.tol = tol > 0.0 ? tol : 0.0; A.fixed_dt = fixed_dt > 0.0 ? fixed_dt : 0.0; A.dt_init = dt_init;
    A.max_steps = max_steps;
    A.sample_dt = b->sample_dt; A.trace_t0 = b->trace_t0; A.trace_cap = b->trace_cap; A.row_len = row_len_of(b);
    A.trace = b->d_trace;
    A.drive = b->d_drive;
    A.pol = b->d_pol;
    A.spec = b->d_spec; A.spec_n = b->d_spec_n; A.spec_K = b->spec_K; A.spec_w0 = b->spec_w0; A.spec_dw = b->spec_dw;
    if (b->split_nllg > 0) {
        // the comparison integrator is the paper's fixed-step co-simulation loop: fixed_dt is the co-simulation step;
        // the kernel counts LLG sub-steps
        if (!(fixed_dt > 0.0)) return CAV_E_ARG;
        A.split_nllg = b->split_nllg;
        A.fixed_dt = fixed_dt / (double)b->split_nllg;
        A.max_steps = max_steps > 0 ? max_steps * b->split_nllg : 0;
    }

    cudaError_t ce = cudaSuccess;
    int rc = cavmag::launch_batch_kernel(A, p.precision == CAV_F32, p.n_sub, b->n_rep > b->n_sm, b->smem_optin, b->stream, &ce);
    if (rc == CAV_E_CUDA || rc == CAV_E_NOMEM) snprintf(b->cuda_err, sizeof(b->cuda_err), "k_batch launch: %s", cudaGetErrorString(ce));
    return rc;
}

int cav_batch_set_polarisation(cav_batch* b, const double* pol, const double* quad) {
    if (!b) return CAV_E_ARG;
    CKB(cudaStreamSynchronize(b->stream));
    cudaFree(b->d_pol);
    b->d_pol = nullptr;
    if (!pol || b->N == 0) return CAV_OK;
    std::vector<double> h(6 * (size_t)b->N);
    int rc = cavmag::pack_polarisation(b->N, pol, quad, h.data());
    if (rc) return rc;
    CKB(cudaMalloc(&b->d_pol, sizeof(double) * h.size()));
    CKB(cudaMemcpyAsync(b->d_pol, h.data(), sizeof(double) * h.size(), cudaMemcpyHostToDevice, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_set_integrator(cav_batch* b, int integrator, int n_llg) {
    if (!b || (integrator != CAV_INTEGRATOR_UNIFIED && integrator != CAV_INTEGRATOR_SPLIT)) return CAV_E_ARG;
    if (integrator == CAV_INTEGRATOR_SPLIT && n_llg < 1) return CAV_E_ARG;
    b->split_nllg = integrator == CAV_INTEGRATOR_SPLIT ? n_llg : 0;
    return CAV_OK;
}

int cav_batch_set_spectrum(cav_batch* b, int n_bins, double omega_lo, double omega_hi) {
    if (!b || n_bins < 0 || (n_bins > 1 && !(omega_hi > omega_lo))) return CAV_E_ARG;
    CKB(cudaStreamSynchronize(b->stream));
    cudaFree(b->d_spec); cudaFree(b->d_spec_n);
    b->d_spec = nullptr; b->d_spec_n = nullptr; b->spec_K = 0;
    if (n_bins == 0) return CAV_OK;
    const size_t bytes = sizeof(double) * (size_t)b->n_rep * n_bins * 2 * (2 * b->N + b->prm.n_sub);
    CKB(cudaMalloc(&b->d_spec, bytes));
    CKB(cudaMalloc(&b->d_spec_n, sizeof(long long) * b->n_rep));
    CKB(cudaMemsetAsync(b->d_spec, 0, bytes, b->stream));
    CKB(cudaMemsetAsync(b->d_spec_n, 0, sizeof(long long) * b->n_rep, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    b->spec_K = n_bins; b->spec_w0 = omega_lo; b->spec_dw = n_bins > 1 ? (omega_hi - omega_lo) / (double)(n_bins - 1) : 0.0;
    return CAV_OK;
}

int cav_batch_get_spectrum(cav_batch* b, double* out, long long* n_samples) {
    if (!b || !out) return CAV_E_ARG;
    if (!b->d_spec) return CAV_E_STATE;
    CKB(cudaMemcpyAsync(out, b->d_spec, sizeof(double) * (size_t)b->n_rep * b->spec_K * 2 * (2 * b->N + b->prm.n_sub), cudaMemcpyDeviceToHost, b->stream));
    if (n_samples) CKB(cudaMemcpyAsync(n_samples, b->d_spec_n, sizeof(long long) * b->n_rep, cudaMemcpyDeviceToHost, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_get_m(cav_batch* b, void* m_out) {
    if (!b || !m_out) return CAV_E_ARG;
    CKB(cudaMemcpyAsync(m_out, b->d_m, (size_t)b->n_rep * b->prm.n_sub * 3 * b->nc * b->esize, cudaMemcpyDeviceToHost, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_get_a(cav_batch* b, double* a_out) {
    if (!b || (!a_out && b->N > 0)) return CAV_E_ARG;
    if (b->N > 0) CKB(cudaMemcpyAsync(a_out, b->d_a, sizeof(double) * 2 * b->N * b->n_rep, cudaMemcpyDeviceToHost, b->stream));
    CKB(cudaStreamSynchronize(b->stream));
    return CAV_OK;
}

int cav_batch_get_stats(cav_batch* b, cav_stats* out) {
    if (!b || !out) return CAV_E_ARG;
    std::vector<BatchCtl> h;
    int rc = pull_ctl(b, h);
    if (rc) return rc;
    int status = CAV_OK;
    for (int r = 0; r < b->n_rep; ++r) {
        out[r].accepted = h[r].accepted; out[r].rejected = h[r].rejected; out[r].rhs_evals = h[r].rhs_evals;
        out[r].dt_min = h[r].dt_min; out[r].dt_max = h[r].dt_max; out[r].dt_next = h[r].dt; out[r].t = h[r].t;
        out[r].last_err = h[r].last_err;
        if (status == CAV_OK && h[r].status != 0) status = h[r].status;
    }
    return status;
}

int cav_batch_get_trace(cav_batch* b, double* out, int* n_samples) {
    if (!b || !n_samples) return CAV_E_ARG;
    std::vector<BatchCtl> h;
    int rc = pull_ctl(b, h);
    if (rc) return rc;
    for (int r = 0; r < b->n_rep; ++r) n_samples[r] = h[r].trace_n;
    if (b->trace_cap > 0 && out) {
        CKB(cudaMemcpyAsync(out, b->d_trace, sizeof(double) * (size_t)b->n_rep * b->trace_cap * row_len_of(b),
                            cudaMemcpyDeviceToHost, b->stream));
        CKB(cudaStreamSynchronize(b->stream));
    }
    return CAV_OK;
}

}  // extern "C"
