// C-ABI layer of the cavity-magnonics hot path (include/cavmag.h): device buffers, the
// CUDA graph whose body is a device-side WHILE loop over the six stage kernels, and the
// small single-block kernels around it.  No torch types, no CPU fallback: every step of the
// path runs in the kernels of stage_kernel.cuh.
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

#include <cuda.h>      // CUtensorMap types only; the encoder is fetched with cudaGetDriverEntryPoint

#include "../../include/cavmag.h"
#include "stage_tma.cuh"
#include "batch_kernel.cuh"
#include "demag.cuh"

using namespace cavmag;

struct cav_sim {
    cav_grid grid;
    cav_params prm;
    long long nc = 0, nvec = 0;
    int vecw = 1;            // cells per thread (4 float / 2 double / 1)
    int vec = 0;             // 1: vectorised kernels
    size_t esize = 4;
    size_t field_bytes = 0;  // n_sub*3*ncp*esize (device buffers; rows padded when `padded`)
    int pitch = 0;           // elements per row in device memory (>= nx)
    long long ncp = 0;       // pitch*ny*nz
    bool padded = false;     // pitch > nx: only the TMA kernels run on this handle (cavmag_types.cuh)
    void* Y[2] = {nullptr, nullptr};
    void* MS[2] = {nullptr, nullptr};
    void* K[7] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    void* u = nullptr;
    size_t u_bytes = 0;
    unsigned long long u_hash = 0;   // FNV-1a of the profile bytes given to cav_set_modes from the host (0: unknown / device source)
    double* partial = nullptr;
    double* partial_max = nullptr;
    int pstride = 0;
    Ctrl* d_ctrl = nullptr;      // canonical instance
    Ctrl* d_ctrl0 = nullptr;     // step-boundary copy (cavmag_types.cuh)
    Ctrl* h_ctrl = nullptr;      // pinned mirror
    double* d_trace = nullptr;
    int trace_cap = 0;
    int N = 0, nb = 0;
    bool m_set = false;
    bool h_fresh = false;        // h_ctrl equals the device's Ctrl (nothing that writes Ctrl has been enqueued since the last pull / push)
    int iters = 1, nblocks = 1, user_block_cells = 0, serpentine = 1;
    int launch_mode = CAV_LAUNCH_GRAPH;
    cudaStream_t stream = nullptr;
    bool own_stream = false;
    // two run graphs: [0] one step per iteration of the device-side WHILE loop, [1] kLoopUnroll steps per iteration (long
    // runs on the TMA path: the step boundary inside the body is a programmatic edge like the stage boundaries)
    cudaGraph_t graph[2] = {nullptr, nullptr};
    cudaGraphExec_t exec[2] = {nullptr, nullptr};
    bool graph_dirty = true;
    long long host_launches = 0;
    int* h_flag = nullptr;       // pinned
    char cuda_err[256] = {0};
    // ---- TMA-pipelined path ----
    int kernel_path = CAV_PATH_AUTO;
    int n_sm = 148;
    size_t smem_optin = 0;
    unsigned char* d_maps = nullptr;   // [MAP_COUNT][128] CUtensorMap table
#ifdef CAVMAG_PROBE
    unsigned long long* d_probe = nullptr;
#endif
    bool maps_ok = false;              // cell-field maps encoded
    bool tma_eligible = false;         // alignment + shared-memory budget allow the TMA kernels
    bool use_tma = false;              // decision for the current graph / launches
    TmaArgs targs[8];
    size_t tsmem[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int tgrid = 1;
    bool last_run_block = false;       // h_ctrl->ycur is known to be current (no stage-kernel run since the last pull)
    bool use_coop = false;             // CAV_PATH_COOP: one cooperative launch per run, grid barriers instead of kernel boundaries
    unsigned char* d_coop = nullptr;   // COOP scratch: block partials x2, block maxima x2, barrier counter
    bool use_block = false;            // CAV_PATH_BLOCK: the whole run in one thread block (k_batch with one replica)
    unsigned char* d_blk = nullptr;    // bridge buffers of the block path: BatchCtl, a, mode parameters, drive, B0
    bool want_pdl = true;              // cav_set_stage_overlap
    // ---- SURVEY.md 8(f3) / 8(f2) variants ----
    double* d_pol = nullptr;           // [N][6] polarisation + quadrature axes, or NULL: x^, y^
    int split_nllg = 0;                // 0: unified RK45; n >= 1: operator-split comparison integrator, n LLG sub-steps per cavity step
    double* d_spec = nullptr;          // [spec_K][2N + n_sub][2] Fourier sums, or NULL
    DemagPlan* demag = nullptr;        // dipolar field by FFT convolution, or NULL: off (the paper's setting)
    void* d_bdem = nullptr;            // [3][nc] dipolar field of the stage about to be evaluated
    bool graph_pdl = false;            // loop-body edges of the current graph are programmatic dependencies
};

namespace {

#define CK(call)                                                                              \
    do {                                                                                      \
        cudaError_t e_ = (call);                                                              \
        if (e_ != cudaSuccess) {                                                              \
            snprintf(s->cuda_err, sizeof(s->cuda_err), "%s at %s:%d: %s", #call, __FILE__, __LINE__, \
                     cudaGetErrorString(e_));                                                 \
            return (e_ == cudaErrorMemoryAllocation) ? CAV_E_NOMEM : CAV_E_CUDA;              \
        }                                                                                     \
    } while (0)

// ---- small kernels around the stage kernels -------------------------------------------------

__device__ void setrun_body(Ctrl* c, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps);
__global__ void k_setrun(Ctrl* c, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps) {
    setrun_body(c, t_end, tol, fixed_dt, dt_init, max_steps);
}
__device__ void setrun_body(Ctrl* c, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps) {
    c->t_end = t_end;
    c->tol = tol;
    c->adaptive = tol > 0.0 ? 1 : 0;
    c->fixed_dt = fixed_dt;
    c->max_steps = max_steps;
    c->steps_run = 0;
    if (c->adaptive) {
        if (dt_init > 0.0) c->dt = dt_init;
        else if (!(c->dt > 0.0)) c->dt = 1e-14;
    } else {
        c->dt = fixed_dt;
        long long st = llround(c->sample_dt / fixed_dt);
        c->trace_stride = st < 1 ? 1 : st;
    }
}

// First node of the run graph: decides whether there is anything to do, fixes h for the first
// step and the mode amplitudes / RF weights of the first kernel, arms the WHILE condition.
__device__ void begin_body(Ctrl* c, Ctrl* c0, unsigned long long handle);

__global__ void k_begin(Ctrl* c, Ctrl* c0, unsigned long long handle) { begin_body(c, c0, handle); }

// joint launch: one block per simulation, then the WHILE condition = "any simulation has something to do"
__global__ void k_sweep_setrun(const RepPtrs* reps, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps);
__global__ void k_sweep_begin(const RepPtrs* reps) { begin_body(reps[blockIdx.x].ctrl, reps[blockIdx.x].ctrl0, 0ull); }
__global__ void k_sweep_cond(const RepPtrs* reps, int R, unsigned int* live, unsigned long long handle) {
    // one thread per simulation (strided): the two dependent loads per member run side by side, not one after the other
    unsigned int mine = 0u;
    for (int r = threadIdx.x; r < R; r += blockDim.x) mine |= reps[r].ctrl->done ? 0u : 1u;
    const int any = __syncthreads_or((int)mine);
    if (threadIdx.x == 0) {
        *live = 0u;
        cudaGraphSetConditional((cudaGraphConditionalHandle)handle, any ? 1u : 0u);
    }
}

// (One block of kBeginThreads threads.  The control block is fetched with one batch of independent loads into shared
// memory, worked on there, and written to both instances with one batch of stores: three L2 round trips instead of one
// per dependent field - this kernel heads every run, so its latency is all of a one-step run's overhead.)
constexpr int kBeginThreads = 128;
constexpr int kBeginWords = (kCtrlWords + kBeginThreads - 1) / kBeginThreads;

__device__ void begin_body(Ctrl* gc, Ctrl* c0, unsigned long long handle) {
    __shared__ __align__(16) unsigned long long sw[kCtrlWords];
    const int tid = threadIdx.x;
    const unsigned long long* const src = reinterpret_cast<const unsigned long long*>(gc);
    unsigned long long v[kBeginWords];
#pragma unroll
    for (int k = 0; k < kBeginWords; ++k) {
        const int i = tid + k * kBeginThreads;
        v[k] = i < kCtrlWords ? __ldcg(src + i) : 0ull;
    }
#pragma unroll
    for (int k = 0; k < kBeginWords; ++k) {
        const int i = tid + k * kBeginThreads;
        if (i < kCtrlWords) sw[i] = v[k];
    }
    __syncthreads();
    Ctrl* const c = reinterpret_cast<Ctrl*>(sw);
    if (tid == 0) {
        c->done = (!(c->t < c->t_end) || c->status != 0) ? 1 : 0;
        c->arrive = 0u;
        c->pend7 = 0;
        prepare_h(c);
    }
    __syncthreads();
    if (tid < c->N) {
        if (!c->k1_valid) {      // stage 1 evaluates f(m_0, a_0)
            c->as[1][tid][0] = c->a[tid][0]; c->as[1][tid][1] = c->a[tid][1];
            c->c[tid] = c->two_over_gamma * (c->Gbre[tid] * c->a[tid][0] - c->Gbim[tid] * c->a[tid][1]);
        } else {
            mode_stage_state<1>(c, tid);
        }
    }
    if (tid == 0 && handle != 0ull) cudaGraphSetConditional((cudaGraphConditionalHandle)handle, c->done ? 0u : 1u);
    __syncthreads();
    // the canonical instance, and the step-boundary copy the TMA stage-2 kernel starts from (cavmag_types.cuh)
    unsigned long long* const d1 = reinterpret_cast<unsigned long long*>(gc);
    unsigned long long* const d0 = reinterpret_cast<unsigned long long*>(c0);
#pragma unroll
    for (int k = 0; k < kBeginWords; ++k) {
        const int i = tid + k * kBeginThreads;
        if (i < kCtrlWords) { const unsigned long long x = sw[i]; d1[i] = x; d0[i] = x; }
    }
}

template <typename T>
__global__ void k_normalize(const T* __restrict__ src, T* __restrict__ dst, long long nc, int n_sub) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nc * n_sub) return;
    const long long s = i / nc, r = i - s * nc;
    const T* p = src + s * 3 * nc + r;
    const T x = p[0], y = p[nc], z = p[2 * nc];
    const T n2 = x * x + y * y + z * z;
    const T inv = n2 > (T)0 ? (T)1 / sqrt(n2) : (T)0;
    T* q = dst + s * 3 * nc + r;
    q[0] = x * inv; q[nc] = y * inv; q[2 * nc] = z * inv;
}

// sum_r u_n(r) for CAV_NORM_SUM_U: 256 fixed-order block sums per mode, finished on the host.
template <typename T>
__global__ void k_sum_u(const T* __restrict__ u, long long nc, double* __restrict__ out /*[N][256]*/) {
    const int n = blockIdx.y;
    const T* p = u + (long long)n * nc;
    const long long chunk = (nc + gridDim.x - 1) / gridDim.x;
    const long long lo = (long long)blockIdx.x * chunk, hi = (lo + chunk < nc) ? lo + chunk : nc;
    double acc = 0.0;
    for (long long i = lo + threadIdx.x; i < hi; i += blockDim.x) acc += (double)p[i];
    __shared__ double sh[256];
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
        if ((int)threadIdx.x < o) sh[threadIdx.x] += sh[threadIdx.x + o];
        __syncthreads();
    }
    if (threadIdx.x == 0) out[n * gridDim.x + blockIdx.x] = sh[0];
}

__global__ void k_sweep_setrun(const RepPtrs* reps, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps) {
    setrun_body(reps[blockIdx.x].ctrl, t_end, tol, fixed_dt, dt_init, max_steps);
}

const void* stage_tma_fn(const cav_sim* s, int stage) {
    const bool f32 = s->prm.precision == CAV_F32;
    if (s->d_pol) {          // the instantiation with per-mode polarisation (mode buckets up to 8; NULL beyond)
        if (s->prm.n_sub == 1) return f32 ? stage_tma_pol_kernel_f32_fm(stage, s->nb) : stage_tma_pol_kernel_f64_fm(stage, s->nb);
        return f32 ? stage_tma_pol_kernel_f32_afm(stage, s->nb) : stage_tma_pol_kernel_f64_afm(stage, s->nb);
    }
    if (s->prm.n_sub == 1) return f32 ? stage_tma_kernel_f32_fm(stage, s->nb) : stage_tma_kernel_f64_fm(stage, s->nb);
    return f32 ? stage_tma_kernel_f32_afm(stage, s->nb) : stage_tma_kernel_f64_afm(stage, s->nb);
}

const void* stage_fn(const cav_sim* s, int stage) {
    const bool f32 = s->prm.precision == CAV_F32;
    if (s->d_pol) {          // the instantiation with per-mode polarisation
        if (s->prm.n_sub == 1) return f32 ? stage_kernel_pol_f32_fm(s->vec, stage, s->nb) : stage_kernel_pol_f64_fm(s->vec, stage, s->nb);
        return f32 ? stage_kernel_pol_f32_afm(s->vec, stage, s->nb) : stage_kernel_pol_f64_afm(s->vec, stage, s->nb);
    }
    if (s->demag) {          // the instantiation that adds the dipolar field
        if (s->prm.n_sub == 1) return f32 ? stage_kernel_demag_f32_fm(s->vec, stage, s->nb) : stage_kernel_demag_f64_fm(s->vec, stage, s->nb);
        return f32 ? stage_kernel_demag_f32_afm(s->vec, stage, s->nb) : stage_kernel_demag_f64_afm(s->vec, stage, s->nb);
    }
    if (s->prm.n_sub == 1) return f32 ? stage_kernel_f32_fm(s->vec, stage, s->nb) : stage_kernel_f64_fm(s->vec, stage, s->nb);
    return f32 ? stage_kernel_f32_afm(s->vec, stage, s->nb) : stage_kernel_f64_afm(s->vec, stage, s->nb);
}

int bucket(int N) { return N == 0 ? 0 : N == 1 ? 1 : N <= 2 ? 2 : N <= 8 ? 8 : 32; }

// ---- TMA path: tensor maps, ring depths, shared-memory budget -----------------------------------

typedef CUresult (*encode_tiled_fn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                    const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                    CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

encode_tiled_fn get_encoder() {
    static encode_tiled_fn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (encode_tiled_fn)p;
        else
            cudaGetLastError();
    }
    return fn;
}

// 4-D map over [C][nz][ny][nx] (x fastest) with box [C][1][by][bx].
bool encode_map(const cav_sim* s, CUtensorMap* out, void* base, int C, int bx, int by, int boxC = 0) {
    encode_tiled_fn enc = get_encoder();
    if (!enc || !base || C < 1) return false;
    const cuuint64_t es = s->esize;
    cuuint64_t dims[4] = {(cuuint64_t)s->grid.nx, (cuuint64_t)s->grid.ny, (cuuint64_t)s->grid.nz, (cuuint64_t)C};
    const cuuint64_t row = (cuuint64_t)s->pitch * es;           // rows padded to a multiple of 16 bytes when nx is not
    cuuint64_t strides[3] = {row, row * dims[1], (cuuint64_t)s->ncp * es};
    cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1u, (cuuint32_t)(boxC > 0 ? boxC : C)};
    cuuint32_t estr[4] = {1u, 1u, 1u, 1u};
    const CUtensorMapDataType dt = s->prm.precision == CAV_F32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64;
    return enc(out, dt, 4, base, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
               CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

int tma_stage_naux(int stage) { return stage <= 2 ? 0 : stage == 7 ? 1 : stage == 6 ? 5 : stage; }

// Encodes the maps of the fixed cell-field buffers (once) and of u (whenever the mode set changes), then sizes
// the rings of every stage for the current N.  Leaves tma_eligible = false if anything does not fit.
int plan_tma(cav_sim* s) {
    s->tma_eligible = false;
    const int es = (int)s->esize;
    if (((long long)s->pitch * es) % 16 != 0) return CAV_OK;           // TMA global strides must be multiples of 16 B
    if (!get_encoder() || !s->d_maps) return CAV_OK;
    const int TX = kTmaRowBytes / es, HX = kTmaHaloBytes / es, C = 3 * s->prm.n_sub;
    CUtensorMap h[MAP_COUNT];
    memset(h, 0, sizeof(h));
    bool ok = true;
    ok = ok && encode_map(s, &h[MAP_H_Y0], s->Y[0], C, TX + 2 * HX, kTmaTY + 2);
    ok = ok && encode_map(s, &h[MAP_H_Y1], s->Y[1], C, TX + 2 * HX, kTmaTY + 2);
    ok = ok && encode_map(s, &h[MAP_H_MS0], s->MS[0], C, TX + 2 * HX, kTmaTY + 2);
    ok = ok && encode_map(s, &h[MAP_H_MS1], s->MS[1], C, TX + 2 * HX, kTmaTY + 2);
    ok = ok && encode_map(s, &h[MAP_H_K0], s->K[0], C, TX + 2 * HX, kTmaTY + 2);
    ok = ok && encode_map(s, &h[MAP_H_K6], s->K[6], C, TX + 2 * HX, kTmaTY + 2);
    ok = ok && encode_map(s, &h[MAP_P_Y0], s->Y[0], C, TX, kTmaTY);
    ok = ok && encode_map(s, &h[MAP_P_Y1], s->Y[1], C, TX, kTmaTY);
    ok = ok && encode_map(s, &h[MAP_P_MS0], s->MS[0], C, TX, kTmaTY);
    for (int j = 0; j < 7; ++j) ok = ok && encode_map(s, &h[MAP_P_K0 + j], s->K[j], C, TX, kTmaTY);
    if (s->N > 0) ok = ok && encode_map(s, &h[MAP_P_U], s->u, s->N, TX, kTmaTY, s->nb < kTmaUChunk ? s->nb : kTmaUChunk);
    if (!ok) return CAV_OK;
    CK(cudaMemcpyAsync(s->d_maps, h, sizeof(h), cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream));

    const unsigned hbox_tx = (unsigned)(kTmaHaloRowBytes * (kTmaTY + 2) * C);
    const unsigned hbox = (hbox_tx + 127u) & ~127u;
    const int ntx = (s->grid.nx + TX - 1) / TX, nty = (s->grid.ny + kTmaTY - 1) / kTmaTY;
    const long long Q = (long long)ntx * nty * s->grid.nz;
    s->tgrid = (int)(Q < s->n_sm ? Q : s->n_sm);
    // Prefetching k_2..k_{s-2} before griddepcontrol.wait is only ordered after kernel s-2 when a block of kernel s
    // cannot be resident beside a block of kernel s-1 that has not passed its own wait (stage_tma.cuh): one CTA per SM
    // for every stage kernel (each asks for more than half an SM's shared memory) and a grid that fills every SM.
    int smem_sm = 0, dev = 0;
    cudaGetDevice(&dev);
    if (cudaDeviceGetAttribute(&smem_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, dev) != cudaSuccess) { cudaGetLastError(); smem_sm = 0; }
    bool all_big = true;
    for (int stage = 1; stage <= 7; ++stage) {
        const void* fn = stage_tma_fn(s, stage);
        if (!fn) return CAV_OK;
        cudaFuncAttributes fa;
        CK(cudaFuncGetAttributes(&fa, fn));
        // dynamic budget = opt-in limit - the kernel's static shared memory - a little slack
        const size_t budget = s->smem_optin > fa.sharedSizeBytes + 256 ? s->smem_optin - fa.sharedSizeBytes - 256 : 0;
        TmaArgs& t = s->targs[stage];
        memset(&t, 0, sizeof(t));
        t.maps = s->d_maps;
        t.ntx = ntx; t.nty = nty; t.Q = Q;
        t.hbox_bytes = hbox; t.hbox_tx = hbox_tx;
        t.ms_slot_bytes = (stage == 2 ? 2u : 1u) * hbox;
        t.aux_slot_bytes = (unsigned)(tma_stage_naux(stage) * C) * (unsigned)(kTmaRowBytes * kTmaTY);
        t.n_uchunks = (s->nb + kTmaUChunk - 1) / kTmaUChunk;      // the kernel streams the whole mode bucket; modes >= N are TMA zero fill
        t.u_slot_bytes = (unsigned)(s->nb < kTmaUChunk ? s->nb : kTmaUChunk) * (unsigned)(kTmaRowBytes * kTmaTY);
        // ring depths: maximise the smallest look-ahead (in planes) of the rings the stage uses
        const bool has_a = t.aux_slot_bytes > 0, has_u = t.u_slot_bytes > 0;
        double best = -1e9;
        int bDa = 0, bDu = 0, bDm = 0;
        for (int Da = has_a ? 1 : 0; Da <= (has_a ? 4 : 0); ++Da)       // (one aux slot - no look-ahead - only where two do not fit)
            for (int Du = has_u ? 2 : 0; Du <= (has_u ? kTmaMaxDepth : 0); ++Du)
                for (int Dm = 4; Dm <= 8; ++Dm) {
                    const size_t bytes = (size_t)Da * t.aux_slot_bytes + (size_t)Du * t.u_slot_bytes + (size_t)Dm * t.ms_slot_bytes + 128;
                    if (bytes > budget) continue;
                    const double la_m = Dm - 3, la_a = has_a ? Da - 1 : 1e3, la_u = has_u ? (double)Du / t.n_uchunks - 1.0 : 1e3;
                    const double mn = la_m < la_a ? (la_m < la_u ? la_m : la_u) : (la_a < la_u ? la_a : la_u);
                    const double score = 100.0 * mn + (has_a ? la_a : 0) + (has_u ? la_u : 0) + 0.5 * la_m;
                    if (score > best) { best = score; bDa = Da; bDu = Du; bDm = Dm; }
                }
        if (bDm == 0) return CAV_OK;             // does not fit: stay on the generic kernels
        t.Da = bDa > 0 ? bDa : 1; t.Du = bDu > 0 ? bDu : 1; t.Dm = bDm;
        s->tsmem[stage] = (size_t)bDa * t.aux_slot_bytes + (size_t)bDu * t.u_slot_bytes + (size_t)bDm * t.ms_slot_bytes + 128;
        const size_t half = (size_t)smem_sm / 2 + 1024;
        if (s->tsmem[stage] < half && half <= budget) s->tsmem[stage] = half;      // shallow rings: still one CTA per SM
        if (2 * s->tsmem[stage] <= (size_t)smem_sm) all_big = false;
        // the attribute is per function, not per simulation: always raise it to the device limit
        CK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(s->smem_optin - fa.sharedSizeBytes)));
    }
    const bool one_cta = smem_sm > 0 && s->tgrid == s->n_sm;
    for (int stage = 1; stage <= 7; ++stage) {
        s->targs[stage].pre_k = (one_cta && all_big) ? 1 : 0;
        // Ctrl (buffer indices, done) is rewritten by block 0 of this step's stage-2 kernel: stage 3 reads it after
        // its wait, later stages may read it earlier under the same one-CTA-per-SM argument
        s->targs[stage].pre_ctrl = (one_cta && all_big && stage >= 4) ? 1 : 0;
        s->targs[stage].N = s->N;
    }
    s->tma_eligible = true;
    return CAV_OK;
}

StageArgs make_args(const cav_sim* s, unsigned long long handle);
int sync_pull(cav_sim* s);

// Dense ABI array [ncomp][nz][ny][nx]  <->  device buffer with rows of s->pitch elements (a plain copy when not padded).
int copy_in(cav_sim* s, void* dst, const void* src, int ncomp, bool src_is_device) {
    const cudaMemcpyKind kind = src_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
    if (!s->padded) { CK(cudaMemcpyAsync(dst, src, (size_t)ncomp * s->nc * s->esize, kind, s->stream)); return CAV_OK; }
    const size_t w = (size_t)s->grid.nx * s->esize;
    CK(cudaMemcpy2DAsync(dst, (size_t)s->pitch * s->esize, src, w, w, (size_t)ncomp * s->grid.ny * s->grid.nz, kind, s->stream));
    return CAV_OK;
}
int copy_out(cav_sim* s, void* dst, const void* src, int ncomp, bool dst_is_device) {
    const cudaMemcpyKind kind = dst_is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost;
    if (!s->padded) { CK(cudaMemcpyAsync(dst, src, (size_t)ncomp * s->nc * s->esize, kind, s->stream)); return CAV_OK; }
    const size_t w = (size_t)s->grid.nx * s->esize;
    CK(cudaMemcpy2DAsync(dst, w, src, (size_t)s->pitch * s->esize, w, (size_t)ncomp * s->grid.ny * s->grid.nz, kind, s->stream));
    return CAV_OK;
}

constexpr int kCoopThreads = 512;

void decide_path(cav_sim* s) {
    const bool block_ok = s->nc <= kBatchMaxCells;
    const bool coop_ok = !block_ok && s->nc <= (long long)s->n_sm * kCoopThreads;
    // the operator-split comparison integrator exists in the small-grid kernel only; a non-default polarisation in the
    // small-grid kernel and in the generic stage kernels (their own instantiation), not in the TMA kernels
    const bool small_only = s->split_nllg > 0;
    s->use_block = block_ok && (s->kernel_path == CAV_PATH_BLOCK || s->kernel_path == CAV_PATH_AUTO || small_only);
    s->use_coop = coop_ok && (s->kernel_path == CAV_PATH_COOP || s->kernel_path == CAV_PATH_AUTO || small_only);
    if (s->demag) { s->use_block = s->use_coop = s->use_tma = false; return; }                 // dipolar field: generic stage kernels
    const bool pol_tma = s->d_pol && s->tma_eligible && stage_tma_fn(s, 2) != nullptr;         // polarisation: TMA kernels for up to 8 modes
    if (s->d_pol && !pol_tma) { s->use_tma = false; return; }                                  // else small-grid or generic kernels
    if (s->padded) { s->use_block = s->use_coop = false; s->use_tma = s->tma_eligible; }       // padded rows: TMA kernels only
    else if (s->kernel_path == CAV_PATH_GENERIC || s->use_block || s->use_coop) s->use_tma = false;
    else if (s->kernel_path == CAV_PATH_TMA) s->use_tma = s->tma_eligible;
    else s->use_tma = s->tma_eligible && s->targs[1].Q >= (long long)s->n_sm;
}

// ---- CAV_PATH_BLOCK: a grid of <= 1024 cells is integrated by ONE thread block for the whole run (k_batch with a
//      single replica, batch_kernel.cuh): no kernel launch per stage.  Two tiny kernels copy the controller / mode state
//      between Ctrl and the batch kernel's arguments on the stream, so cav_run stays asynchronous. ----
constexpr size_t kBlkCtl = 0, kBlkA = 256, kBlkModep = kBlkA + 16 * kMaxModes, kBlkDrive = kBlkModep + 8 * 7 * kMaxModes,
                 kBlkB0 = kBlkDrive + 8 * 5 * kMaxModes, kBlkBytes = kBlkB0 + 64;
static_assert(sizeof(BatchCtl) <= kBlkA, "bridge layout");

__global__ void k_block_in(const Ctrl* c, unsigned char* blk, double B0x, double B0y, double B0z) {
    BatchCtl* bc = reinterpret_cast<BatchCtl*>(blk + kBlkCtl);
    double* a = reinterpret_cast<double*>(blk + kBlkA);
    double* mp = reinterpret_cast<double*>(blk + kBlkModep);
    double* dr = reinterpret_cast<double*>(blk + kBlkDrive);
    double* B0 = reinterpret_cast<double*>(blk + kBlkB0);
    const int n = threadIdx.x, N = c->N;
    if (n < N) {
        a[2 * n] = c->a[n][0]; a[2 * n + 1] = c->a[n][1];
        mp[n] = c->omega[n]; mp[N + n] = c->kappa[n]; mp[2 * N + n] = c->Gre[n]; mp[3 * N + n] = c->Gim[n];
        mp[4 * N + n] = c->invW[n]; mp[5 * N + n] = c->Gbre[n]; mp[6 * N + n] = c->Gbim[n];
        dr[n] = c->eta_re[n]; dr[N + n] = c->eta_im[n]; dr[2 * N + n] = c->eta_t0[n];
        dr[3 * N + n] = c->eta_i2s2[n]; dr[4 * N + n] = c->eta_wd[n];
    }
    if (n == 0) {
        bc->t = c->t; bc->dt = c->dt; bc->dt_min = c->dt_min; bc->dt_max = c->dt_max; bc->last_err = c->last_err;
        bc->accepted = c->accepted; bc->rejected = c->rejected; bc->rhs_evals = c->rhs_evals;
        bc->trace_acc0 = c->trace_acc0; bc->status = c->status; bc->trace_n = c->trace_n;
        B0[0] = B0x; B0[1] = B0y; B0[2] = B0z;
    }
}

__global__ void k_block_out(Ctrl* c, const unsigned char* blk) {
    const BatchCtl* bc = reinterpret_cast<const BatchCtl*>(blk + kBlkCtl);
    const double* a = reinterpret_cast<const double*>(blk + kBlkA);
    const int n = threadIdx.x;
    if (n < c->N) { c->a[n][0] = a[2 * n]; c->a[n][1] = a[2 * n + 1]; }
    if (n == 0) {
        c->t = bc->t; c->dt = bc->dt; c->dt_min = bc->dt_min; c->dt_max = bc->dt_max; c->last_err = bc->last_err;
        c->accepted = bc->accepted; c->rejected = bc->rejected; c->rhs_evals = bc->rhs_evals;
        c->status = bc->status; c->trace_n = bc->trace_n;
        c->k1_valid = 0;             // the block path keeps its slopes in registers: nothing cached for the stage kernels
        c->done = 1;
    }
}

int run_block_path(cav_sim* s, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps) {
    if (!s->d_blk) CK(cudaMalloc(&s->d_blk, kBlkBytes));
    const size_t coop_part = sizeof(double) * (size_t)kMaxSums * s->n_sm, coop_max = sizeof(double) * (size_t)s->n_sm;
    if (s->use_coop && !s->d_coop) CK(cudaMalloc(&s->d_coop, 2 * coop_part + 2 * coop_max + 64));
    // (cav_run_steps has pulled Ctrl if a stage-kernel run may have flipped ycur on the device since the last pull)
    const cav_params& p = s->prm;
    const Ctrl* hc = s->h_ctrl;                          // host-set fields only (N, trace and drive settings)
    k_block_in<<<1, 32, 0, s->stream>>>(s->d_ctrl, s->d_blk, p.B0[0], p.B0[1], p.B0[2]);
    CK(cudaGetLastError());
    BatchArgs A;
    memset(&A, 0, sizeof(A));
    const StageArgs S = make_args(s, 0ull);
    A.nx = s->grid.nx; A.ny = s->grid.ny; A.nz = s->grid.nz; A.nc = (int)s->nc; A.N = s->N; A.n_rep = 1;
    A.ex_wx = S.ex_wx; A.ex_wy = S.ex_wy; A.ex_wz = S.ex_wz; A.an_pref = S.an_pref;
    for (int i = 0; i < 3; ++i) A.axis[i] = S.axis[i];
    A.alpha = S.alpha; A.llg = S.llg; A.B_exch_inter = S.B_exch_inter;
    A.two_over_gamma = 2.0 / p.gamma; A.inv_nc = S.inv_nc; A.renormalize = p.renormalize;
    A.B0 = reinterpret_cast<const double*>(s->d_blk + kBlkB0);
    A.u = s->u;
    A.modep = reinterpret_cast<const double*>(s->d_blk + kBlkModep); A.modep_per_rep = 0;
    A.m = s->Y[hc->ycur];                                // ycur only changes in the stage kernels' controller: the host copy
    A.a = reinterpret_cast<double*>(s->d_blk + kBlkA);   // is current after any setter, and the block path never flips it
    A.ctl = reinterpret_cast<BatchCtl*>(s->d_blk + kBlkCtl);
    A.t_end = t_end; A.tol = tol; A.fixed_dt = fixed_dt; A.dt_init = dt_init; A.max_steps = max_steps;
    A.sample_dt = hc->sample_dt; A.trace_t0 = hc->trace_t0; A.trace_cap = hc->trace_cap;
    A.row_len = 1 + 4 * s->N + 3 * p.n_sub; A.trace = s->d_trace;
    A.drive = hc->drive_on ? reinterpret_cast<const double*>(s->d_blk + kBlkDrive) : nullptr;
    A.pol = s->d_pol;
    if (s->split_nllg > 0) {
        if (!(fixed_dt > 0.0)) return CAV_E_ARG;         // the co-simulation loop is a fixed-step scheme
        A.split_nllg = s->split_nllg;
        A.fixed_dt = fixed_dt / (double)s->split_nllg;   // the kernel counts LLG sub-steps
        A.max_steps = max_steps > 0 ? max_steps * s->split_nllg : 0;
    }
    if (s->d_spec && hc->spec_K > 0) {
        A.spec = s->d_spec; A.spec_K = hc->spec_K; A.spec_w0 = hc->spec_w0; A.spec_dw = hc->spec_dw;
        A.spec_n = &s->d_ctrl->spec_n;                   // counted straight into Ctrl (the bridge kernels do not touch it)
    }
    cudaError_t ce = cudaSuccess;
    int rc;
    if (s->use_coop) {
        A.gms[0] = s->MS[0]; A.gms[1] = s->MS[1];
        A.cpart[0] = reinterpret_cast<double*>(s->d_coop); A.cpart[1] = reinterpret_cast<double*>(s->d_coop + coop_part);
        A.cmax[0] = reinterpret_cast<double*>(s->d_coop + 2 * coop_part); A.cmax[1] = reinterpret_cast<double*>(s->d_coop + 2 * coop_part + coop_max);
        A.bar = reinterpret_cast<unsigned long long*>(s->d_coop + 2 * coop_part + 2 * coop_max);
        rc = launch_coop_kernel(A, p.precision == CAV_F32, p.n_sub, s->stream, &ce);
    } else {
        rc = launch_batch_kernel(A, p.precision == CAV_F32, p.n_sub, false, s->smem_optin, s->stream, &ce);
    }
    if (rc == CAV_E_CUDA || rc == CAV_E_NOMEM) snprintf(s->cuda_err, sizeof(s->cuda_err), "k_batch launch: %s", cudaGetErrorString(ce));
    if (rc) return rc;
    k_block_out<<<1, 32, 0, s->stream>>>(s->d_ctrl, s->d_blk);
    CK(cudaGetLastError());
    s->host_launches += 3;
    return CAV_OK;
}

void choose_grid(cav_sim* s) {
    const long long biters = (s->nvec + kBlock - 1) / kBlock;      // block-iterations in total
    long long iters;
    if (s->user_block_cells > 0) {
        iters = s->user_block_cells / (kBlock * s->vecw);
        if (iters < 1) iters = 1;
    } else {
        const long long target = 148 * 8;
        iters = (biters + target - 1) / target;
        if (iters < 1) iters = 1;
    }
    long long nb = (biters + iters - 1) / iters;
    while (nb > s->pstride) { iters++; nb = (biters + iters - 1) / iters; }
    s->iters = (int)iters;
    s->nblocks = (int)nb;
}

StageArgs make_args(const cav_sim* s, unsigned long long handle) {
    StageArgs A;
    memset(&A, 0, sizeof(A));
    A.ctrl = s->d_ctrl;
    A.ctrl0 = s->d_ctrl0;
    for (int i = 0; i < 2; ++i) { A.Y[i] = s->Y[i]; A.MS[i] = s->MS[i]; }
    for (int i = 0; i < 7; ++i) A.K[i] = s->K[i];
    A.u = s->u;
    A.partial = s->partial;
    A.partial_max = s->partial_max;
    A.spec = s->d_spec;
    A.bdem = s->demag ? s->d_bdem : nullptr;
    A.pol = s->d_pol;
    A.cond_handle = handle;
    A.pstride = s->pstride;
    A.nx = s->grid.nx; A.ny = s->grid.ny; A.nz = s->grid.nz;
    A.iters = s->iters;
    A.serpentine = s->serpentine;
    A.nc = s->nc;
    A.pitch = s->pitch;
    A.ncp = s->ncp;
    A.inv_nc = 1.0 / (double)s->nc;
    A.nvec = s->nvec;
    const cav_params& p = s->prm;
    for (int i = 0; i < 3; ++i) A.B0[i] = p.B0[i];
    const double pe = (p.Ms > 0.0) ? 2.0 * p.Aex / p.Ms : 0.0;
    A.ex_wx = pe / (s->grid.dx * s->grid.dx);
    A.ex_wy = pe / (s->grid.dy * s->grid.dy);
    A.ex_wz = pe / (s->grid.dz * s->grid.dz);
    A.an_pref = (p.Ms > 0.0) ? 2.0 * p.Ku / p.Ms : 0.0;
    double ax[3] = {p.ku_axis[0], p.ku_axis[1], p.ku_axis[2]};
    const double an = std::sqrt(ax[0] * ax[0] + ax[1] * ax[1] + ax[2] * ax[2]);
    for (int i = 0; i < 3; ++i) A.axis[i] = an > 0.0 ? ax[i] / an : (i == 2 ? 1.0 : 0.0);
    A.alpha = p.alpha;
    A.llg = -p.gamma / (1.0 + p.alpha * p.alpha);
    A.B_exch_inter = p.n_sub == 2 ? p.B_exch_inter : 0.0;
    A.renormalize = p.renormalize;
#ifdef CAVMAG_PROBE
    A.probe = s->d_probe;
#endif
    return A;
}

int sync_pull(cav_sim* s) {
    if (s->h_fresh) return CAV_OK;       // setters and getters in a row (upload m, upload a, ... ) need one pull, not one each
    CK(cudaStreamSynchronize(s->stream));
    CK(cudaMemcpyAsync(s->h_ctrl, s->d_ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    s->h_fresh = true;
    return CAV_OK;
}

int push_ctrl(cav_sim* s) {
    CK(cudaMemcpyAsync(s->d_ctrl, s->h_ctrl, sizeof(Ctrl), cudaMemcpyHostToDevice, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    return CAV_OK;
}

constexpr int kLoopUnroll = 4;            // steps per WHILE iteration of the long-run graph
constexpr long long kUnrollMinSteps = 8;  // runs bounded to fewer steps use the one-step body (when max_steps is not a multiple of
                                          // kLoopUnroll, or the run ends at t_end, up to 6 kLoopUnroll - 1 empty kernels follow the last step)

void destroy_graph(cav_sim* s) {
    for (int i = 0; i < 2; ++i) {
        if (s->exec[i]) { cudaGraphExecDestroy(s->exec[i]); s->exec[i] = nullptr; }
        if (s->graph[i]) { cudaGraphDestroy(s->graph[i]); s->graph[i] = nullptr; }
    }
    s->graph_dirty = true;
}

// programmatic = true: the edge dep -> node is a programmatic dependency (the node may be scheduled once every
// block of dep has executed griddepcontrol.launch_dependents; it synchronises with griddepcontrol.wait).
int add_kernel(cav_sim* s, cudaGraph_t g, cudaGraphNode_t* node, const cudaGraphNode_t* dep, const void* fn,
               dim3 grid, dim3 block, void** params, size_t smem, bool programmatic = false) {
    cudaKernelNodeParams kp;
    memset(&kp, 0, sizeof(kp));
    kp.func = const_cast<void*>(fn);
    kp.gridDim = grid;
    kp.blockDim = block;
    kp.sharedMemBytes = (unsigned)smem;
    kp.kernelParams = params;
    kp.extra = nullptr;
    if (dep && programmatic) {
        CK(cudaGraphAddKernelNode(node, g, nullptr, 0, &kp));
        cudaGraphEdgeData ed;
        memset(&ed, 0, sizeof(ed));
        ed.type = cudaGraphDependencyTypeProgrammatic;
        ed.from_port = cudaGraphKernelNodePortProgrammatic;
        CK(cudaGraphAddDependencies_v2(g, dep, node, &ed, 1));
    } else {
        CK(cudaGraphAddKernelNode(node, g, dep, dep ? 1 : 0, &kp));
    }
    return CAV_OK;
}

// begin -> K1 -> WHILE { K2 -> K3 -> K4 -> K5 -> K6 -> K7 [-> K2 -> ... -> K7] x (unroll - 1) }
// On the TMA path the edges between consecutive stage kernels inside the loop body are programmatic dependencies: the
// next stage kernel's blocks become resident (barrier init, tensor-map prefetch, early profile loads) as the SMs drain
// and only then wait for the previous kernel to complete.  The step controller runs in the prologue of every stage-2
// kernel, so a body may hold several steps: the WHILE condition is then evaluated once per `unroll` steps (one loop
// iteration costs ~6 us of idle GPU between K7 and the next K2), and the kernels after the step that ends the run
// return at once.
int launch_stage(cav_sim* s, int stage, StageArgs& A, cudaStream_t stream);

// With the dipolar field a stage is a chain of launches, cuFFT's among them, which only cuFFT can enqueue: those are
// recorded by stream capture INTO the run graph (stage 1 behind k_begin, stages 2..7 into the body of the WHILE node) from
// a private stream, so the run is the same single graph launch as without the field.
int capture_stages(cav_sim* s, cudaGraph_t into, const cudaGraphNode_t* dep, int first, int last, StageArgs& A,
                   cudaGraphNode_t* tail, size_t* n_tail) {
    cudaStream_t cs = nullptr;
    CK(cudaStreamCreateWithFlags(&cs, cudaStreamNonBlocking));
    cudaError_t e = cudaStreamBeginCaptureToGraph(cs, into, dep, nullptr, dep ? 1 : 0, cudaStreamCaptureModeThreadLocal);
    int rc = CAV_OK;
    if (e == cudaSuccess) {
        for (int stage = first; stage <= last && rc == CAV_OK; ++stage) rc = launch_stage(s, stage, A, cs);
        if (rc == CAV_OK && tail) {
            cudaStreamCaptureStatus st;
            const cudaGraphNode_t* deps = nullptr;
            size_t nd = 0;
            e = cudaStreamGetCaptureInfo(cs, &st, nullptr, nullptr, &deps, &nd);
            if (e == cudaSuccess && nd >= 1 && nd <= 4) { for (size_t i = 0; i < nd; ++i) tail[i] = deps[i]; *n_tail = nd; }
            else rc = CAV_E_CUDA;
        }
        cudaGraph_t g = nullptr;
        const cudaError_t e2 = cudaStreamEndCapture(cs, &g);
        if (e == cudaSuccess) e = e2;
    }
    cudaStreamDestroy(cs);
    if (rc == CAV_OK && e != cudaSuccess) {
        snprintf(s->cuda_err, sizeof(s->cuda_err), "capture of the dipolar-field stages: %s", cudaGetErrorString(e));
        rc = CAV_E_CUDA;
    }
    return rc;
}

int build_graph_impl(cav_sim* s, int which, bool pdl, int unroll) {
    choose_grid(s);
    decide_path(s);
    CK(cudaGraphCreate(&s->graph[which], 0));
    cudaGraph_t graph = s->graph[which];
    cudaGraphConditionalHandle handle;
    CK(cudaGraphConditionalHandleCreate(&handle, graph, 0, cudaGraphCondAssignDefault));
    unsigned long long h64 = (unsigned long long)handle;
    StageArgs A = make_args(s, h64);
    double* trace = s->d_trace;
    Ctrl* ctrl = s->d_ctrl;
    Ctrl* ctrl0 = s->d_ctrl0;

    cudaGraphNode_t n_begin, n_k1, n_while;
    {
        void* params[] = {&ctrl, &ctrl0, &h64};
        int rc = add_kernel(s, graph, &n_begin, nullptr, (const void*)k_begin, dim3(1), dim3(kBeginThreads), params, 0);
        if (rc) return rc;
    }
    cudaGraphNode_t tail[4];
    size_t n_tail = 1;
    if (s->demag) {
        int rc = capture_stages(s, graph, &n_begin, 1, 1, A, tail, &n_tail);
        if (rc) return rc;
    } else {
        void* params[] = {&A, &trace};
        void* tparams[] = {&A, &s->targs[1], &trace};
        int rc = s->use_tma ? add_kernel(s, graph, &n_k1, &n_begin, stage_tma_fn(s, 1), dim3(s->tgrid), dim3(kTmaThreads), tparams, s->tsmem[1])
                            : add_kernel(s, graph, &n_k1, &n_begin, stage_fn(s, 1), dim3(s->nblocks), dim3(kBlock), params, 0);
        if (rc) return rc;
        tail[0] = n_k1;
    }
    cudaGraphNodeParams cp = {};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = handle;
    cp.conditional.type = cudaGraphCondTypeWhile;
    cp.conditional.size = 1;
    CK(cudaGraphAddNode(&n_while, graph, tail, n_tail, &cp));
    cudaGraph_t body = cp.conditional.phGraph_out[0];
    cudaGraphNode_t prev;
    if (s->demag) {
        int rc = capture_stages(s, body, nullptr, 2, 7, A, nullptr, nullptr);
        if (rc) return rc;
    } else
    for (int u = 0; u < unroll; ++u)
        for (int stage = 2; stage <= 7; ++stage) {
            void* params[] = {&A, &trace};
            void* tparams[] = {&A, &s->targs[stage], &trace};
            cudaGraphNode_t node;
            const cudaGraphNode_t* dep = (u == 0 && stage == 2) ? nullptr : &prev;
            int rc = s->use_tma ? add_kernel(s, body, &node, dep, stage_tma_fn(s, stage), dim3(s->tgrid), dim3(kTmaThreads), tparams, s->tsmem[stage], pdl)
                                : add_kernel(s, body, &node, dep, stage_fn(s, stage), dim3(s->nblocks), dim3(kBlock), params, 0);
            if (rc) return rc;
            prev = node;
        }
    if (s->use_tma) {
        // after the loop: one more stage-2 kernel, which finishes stage 7 of the last step (controller, trace, statistics)
        // and returns; when the loop has already seen `done` it returns at once
        void* tparams[] = {&A, &s->targs[2], &trace};
        cudaGraphNode_t n_fin;
        int rc = add_kernel(s, graph, &n_fin, &n_while, stage_tma_fn(s, 2), dim3(s->tgrid), dim3(kTmaThreads), tparams, s->tsmem[2]);
        if (rc) return rc;
    }
    CK(cudaGraphInstantiate(&s->exec[which], graph, 0));
    CK(cudaGraphUpload(s->exec[which], s->stream));      // not inside the first (possibly timed) launch
    return CAV_OK;
}

int build_graph(cav_sim* s) {
    destroy_graph(s);
    decide_path(s);
    // the generic kernels finish a step in the last block of K7 and set the condition there: one step per iteration
    const int unroll1 = s->use_tma ? kLoopUnroll : 1;
    if (s->use_tma && s->want_pdl) {
        if (build_graph_impl(s, 0, true, 1) == CAV_OK && build_graph_impl(s, 1, true, unroll1) == CAV_OK) {
            s->graph_pdl = true;
            s->graph_dirty = false;
            return CAV_OK;
        }
        cudaGetLastError();          // programmatic edges refused here: fall back to full dependencies
        destroy_graph(s);
    }
    s->graph_pdl = false;
    int rc = build_graph_impl(s, 0, false, 1);
    if (rc == CAV_OK) rc = build_graph_impl(s, 1, false, unroll1);
    if (rc == CAV_OK) s->graph_dirty = false;
    return rc;
}

int launch_stage(cav_sim* s, int stage, StageArgs& A, cudaStream_t stream) {
    double* trace = s->d_trace;
    if (s->demag) {          // dipolar field of the state this stage is evaluated at, then the stage kernel that adds it
        int rc = demag_apply(s->demag, A, stage, s->d_bdem, stream);
        if (rc) { snprintf(s->cuda_err, sizeof(s->cuda_err), "demag_apply failed at stage %d", stage); return rc; }
        if (stream == s->stream) s->host_launches += 5;
    }
    if (s->use_tma) {
        void* tparams[] = {&A, &s->targs[stage], &trace};
        CK(cudaLaunchKernel(stage_tma_fn(s, stage), dim3(s->tgrid), dim3(kTmaThreads), tparams, s->tsmem[stage], stream));
    } else {
        void* params[] = {&A, &trace};
        CK(cudaLaunchKernel(stage_fn(s, stage), dim3(s->nblocks), dim3(kBlock), params, 0, stream));
    }
    return CAV_OK;
}

int run_stream_mode(cav_sim* s) {
    choose_grid(s);
    decide_path(s);
    StageArgs A = make_args(s, 0ull);
    k_begin<<<1, kBeginThreads, 0, s->stream>>>(s->d_ctrl, s->d_ctrl0, 0ull);
    CK(cudaGetLastError());
    int rc = launch_stage(s, 1, A, s->stream);
    if (rc) return rc;
    const int chunk = 16;
    for (;;) {
        for (int i = 0; i < chunk; ++i)
            for (int stage = 2; stage <= 7; ++stage) {
                rc = launch_stage(s, stage, A, s->stream);
                if (rc) return rc;
            }
        CK(cudaMemcpyAsync(s->h_flag, &s->d_ctrl->done, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        if (*s->h_flag) break;
    }
    return CAV_OK;
}

}  // namespace

extern "C" {

const char* cav_version(void) { return "cavmag-b200 0.1 (sm_100a)"; }

const char* cav_strerror(int st) {
    switch (st) {
        case CAV_OK: return "ok";
        case CAV_E_ARG: return "invalid argument";
        case CAV_E_STATE: return "invalid call order / state";
        case CAV_E_CUDA: return "CUDA runtime error";
        case CAV_E_NOMEM: return "out of memory";
        case CAV_E_NONFINITE: return "non-finite error norm";
        case CAV_E_DT_UNDERFLOW: return "step size underflow";
        case CAV_E_SINGULAR_NORM: return "sum of mode profile is ~0 (CAV_NORM_SUM_U)";
        case CAV_E_UNSUPPORTED: return "unsupported: no sm_100 CUDA device, or the requested kernel path does not fit this problem";
        default: return "unknown status";
    }
}

const char* cav_last_cuda_error(cav_sim* s) { return s ? s->cuda_err : ""; }

int cav_create(const cav_grid* grid, const cav_params* prm, cav_sim** out) {
    if (!grid || !prm || !out) return CAV_E_ARG;
    *out = nullptr;
    if (grid->nx < 1 || grid->ny < 1 || grid->nz < 1 || !(grid->dx > 0) || !(grid->dy > 0) || !(grid->dz > 0)) return CAV_E_ARG;
    if (!(prm->Ms > 0) || prm->Aex < 0 || !(prm->gamma > 0) || prm->alpha < 0) return CAV_E_ARG;
    if (prm->n_sub != 1 && prm->n_sub != 2) return CAV_E_ARG;
    if (prm->precision != CAV_F32 && prm->precision != CAV_F64) return CAV_E_ARG;
    if (prm->overlap_norm != CAV_NORM_NCELLS && prm->overlap_norm != CAV_NORM_SUM_U) return CAV_E_ARG;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return CAV_E_UNSUPPORTED; }
    int dev = 0;
    cudaDeviceProp dp;
    if (cudaGetDevice(&dev) != cudaSuccess || cudaGetDeviceProperties(&dp, dev) != cudaSuccess) return CAV_E_UNSUPPORTED;
    if (dp.major != 10) return CAV_E_UNSUPPORTED;      // built for sm_100a only

    cav_sim* s = new (std::nothrow) cav_sim();
    if (!s) return CAV_E_NOMEM;
    s->grid = *grid;
    s->prm = *prm;
    s->nc = (long long)grid->nx * grid->ny * grid->nz;
    s->esize = prm->precision == CAV_F32 ? 4 : 8;
    const int vw = prm->precision == CAV_F32 ? 4 : 2;
    s->vec = (grid->nx % vw == 0) ? 1 : 0;
    s->vecw = s->vec ? vw : 1;
    s->nvec = s->nc / s->vecw;
    // Row pitch.  The TMA path needs 16-byte row strides; a large grid whose nx * sizeof(T) is not a multiple of 16 is
    // stored with padded rows (the ABI stays dense: strided copies in and out) instead of falling back to the generic
    // kernels at half the throughput.  Grids in the range of the single-block / cooperative kernel stay dense.
    s->pitch = grid->nx;
    {
        const int per16 = 16 / (int)s->esize, per128 = 128 / (int)s->esize;
        const bool small = s->nc <= (long long)dp.multiProcessorCount * 512;
        // padded rows start on 128-byte lines (a 16-byte pitch measured 16 % slower on cfg3 with nx = 250: every 256-byte
        // tile row then straddles one more 32-byte sector and the stores split sectors)
        if (grid->nx % per16 != 0 && !small) { s->pitch = (grid->nx + per128 - 1) / per128 * per128; s->padded = true; }
    }
    s->ncp = (long long)s->pitch * grid->ny * grid->nz;
    s->field_bytes = (size_t)prm->n_sub * 3 * s->ncp * s->esize;
    const long long biters = (s->nvec + kBlock - 1) / kBlock;
    long long pmax = biters < kMaxBlocks ? biters : kMaxBlocks;       // generic kernel: one partial per block
    if (pmax < dp.multiProcessorCount) pmax = dp.multiProcessorCount;  // TMA kernel: one partial per SM
    s->pstride = (int)((pmax + 31) / 32 * 32);
    int rc = CAV_OK;
    auto fail = [&](int code) { cav_destroy(s); return code; };
#define CKC(call)                                                                                         \
    do {                                                                                                  \
        cudaError_t e_ = (call);                                                                          \
        if (e_ != cudaSuccess) {                                                                          \
            cudaGetLastError();                                                                           \
            return fail(e_ == cudaErrorMemoryAllocation ? CAV_E_NOMEM : CAV_E_CUDA);                      \
        }                                                                                                 \
    } while (0)
    CKC(cudaStreamCreateWithFlags(&s->stream, cudaStreamNonBlocking));
    s->own_stream = true;
    for (int i = 0; i < 2; ++i) { CKC(cudaMalloc(&s->Y[i], s->field_bytes)); CKC(cudaMalloc(&s->MS[i], s->field_bytes)); }
    for (int i = 0; i < 7; ++i) CKC(cudaMalloc(&s->K[i], s->field_bytes));
    CKC(cudaMalloc(&s->partial, sizeof(double) * 2 * (size_t)kMaxSums * s->pstride));      // two buffers: stage parity
    CKC(cudaMalloc(&s->partial_max, sizeof(double) * (size_t)s->pstride));
    CKC(cudaMalloc(&s->d_ctrl, sizeof(Ctrl)));
    CKC(cudaMalloc(&s->d_ctrl0, sizeof(Ctrl)));
    CKC(cudaMemset(s->d_ctrl0, 0, sizeof(Ctrl)));
    CKC(cudaMallocHost(&s->h_ctrl, sizeof(Ctrl)));
    CKC(cudaMallocHost(&s->h_flag, sizeof(int)));
    CKC(cudaMalloc(&s->d_maps, 128 * MAP_COUNT));
#ifdef CAVMAG_PROBE
    CKC(cudaMalloc(&s->d_probe, 8 * 256 * 32 * sizeof(unsigned long long)));
    CKC(cudaMemset(s->d_probe, 0, 8 * 256 * 32 * sizeof(unsigned long long)));
#endif
#undef CKC
    s->n_sm = dp.multiProcessorCount;
    s->smem_optin = dp.sharedMemPerBlockOptin;
    memset(s->h_ctrl, 0, sizeof(Ctrl));
    s->h_ctrl->gamma = prm->gamma;
    s->h_ctrl->two_over_gamma = 2.0 / prm->gamma;
    s->h_ctrl->dt_min = INFINITY;
    s->h_ctrl->t_end = 0.0;
    s->h_ctrl->trace_stride = 1;
    rc = push_ctrl(s);
    if (rc) return fail(rc);
    choose_grid(s);
    rc = plan_tma(s);
    if (rc) return fail(rc);
    *out = s;
    return CAV_OK;
}

int cav_destroy(cav_sim* s) {
    if (!s) return CAV_E_ARG;
    if (s->stream) cudaStreamSynchronize(s->stream);
    destroy_graph(s);
    for (int i = 0; i < 2; ++i) { cudaFree(s->Y[i]); cudaFree(s->MS[i]); }
    for (int i = 0; i < 7; ++i) cudaFree(s->K[i]);
    cudaFree(s->u);
    cudaFree(s->partial);
    cudaFree(s->partial_max);
    cudaFree(s->d_ctrl);
    cudaFree(s->d_ctrl0);
    cudaFree(s->d_trace);
    cudaFree(s->d_maps);
    cudaFree(s->d_blk);
    cudaFree(s->d_coop);
    cudaFree(s->d_pol);
    cudaFree(s->d_spec);
    demag_destroy(s->demag);
    cudaFree(s->d_bdem);
    if (s->h_ctrl) cudaFreeHost(s->h_ctrl);
    if (s->h_flag) cudaFreeHost(s->h_flag);
    if (s->own_stream && s->stream) cudaStreamDestroy(s->stream);
    cudaGetLastError();
    delete s;
    return CAV_OK;
}

int cav_set_stream(cav_sim* s, void* stream) {
    if (!s) return CAV_E_ARG;
    CK(cudaStreamSynchronize(s->stream));
    if (s->own_stream) { cudaStreamDestroy(s->stream); s->own_stream = false; }
    s->stream = (cudaStream_t)stream;
    return CAV_OK;
}

int cav_set_launch_mode(cav_sim* s, int mode) {
    if (!s || (mode != CAV_LAUNCH_GRAPH && mode != CAV_LAUNCH_STREAM)) return CAV_E_ARG;
    s->launch_mode = mode;
    return CAV_OK;
}

int cav_set_block_cells(cav_sim* s, int cells) {
    if (!s || cells < 0) return CAV_E_ARG;
    s->user_block_cells = cells;
    s->graph_dirty = true;
    choose_grid(s);
    return CAV_OK;
}

int cav_set_kernel_path(cav_sim* s, int path) {
    if (!s || (path != CAV_PATH_AUTO && path != CAV_PATH_GENERIC && path != CAV_PATH_TMA && path != CAV_PATH_BLOCK && path != CAV_PATH_COOP)) return CAV_E_ARG;
    if (path == CAV_PATH_TMA && !s->tma_eligible) return CAV_E_UNSUPPORTED;
    if (s->padded && path != CAV_PATH_TMA && path != CAV_PATH_AUTO) return CAV_E_UNSUPPORTED;      // rows padded for the TMA path
    if (path == CAV_PATH_BLOCK && s->nc > kBatchMaxCells) return CAV_E_UNSUPPORTED;
    if (path == CAV_PATH_COOP && (s->nc <= kBatchMaxCells || s->nc > (long long)s->n_sm * kCoopThreads)) return CAV_E_UNSUPPORTED;
    s->kernel_path = path;
    s->graph_dirty = true;
    return CAV_OK;
}

int cav_get_kernel_path(cav_sim* s, int* path) {
    if (!s || !path) return CAV_E_ARG;
    decide_path(s);
    *path = s->use_block ? CAV_PATH_BLOCK : s->use_coop ? CAV_PATH_COOP : s->use_tma ? CAV_PATH_TMA : CAV_PATH_GENERIC;
    return CAV_OK;
}

int cav_set_stage_overlap(cav_sim* s, int on) {
    if (!s) return CAV_E_ARG;
    s->want_pdl = on != 0;
    s->graph_dirty = true;
    return CAV_OK;
}

int cav_get_stage_overlap(cav_sim* s, int* active) {
    if (!s || !active) return CAV_E_ARG;
    *active = (s->exec[0] && !s->graph_dirty && s->graph_pdl) ? 1 : 0;
    return CAV_OK;
}

int cav_set_sweep_order(cav_sim* s, int serpentine) {
    if (!s) return CAV_E_ARG;
    s->serpentine = serpentine ? 1 : 0;
    s->graph_dirty = true;
    return CAV_OK;
}

int cav_set_modes(cav_sim* s, int N, const void* u, int u_is_device, const double* omega, const double* kappa,
                  const double* g, const double* Gamma, const double* Phi) {
    if (!s || N < 0 || N > CAV_MAX_MODES) return CAV_E_ARG;
    if (N > 0 && (!u || !omega || !kappa || !g)) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    // Any failure below leaves the handle in a consistent state with NO modes: the old graph and the u tensor map
    // may point at a buffer that has been freed or overwritten, so they are dropped, not kept.
    auto fail = [&](int code, cudaError_t e = cudaSuccess) {
        if (e != cudaSuccess) {
            snprintf(s->cuda_err, sizeof(s->cuda_err), "cav_set_modes: %s", cudaGetErrorString(e));
            cudaGetLastError();
        }
        s->N = 0; s->nb = 0;
        Ctrl* c = s->h_ctrl;
        c->N = 0; c->k1_valid = 0; c->drive_on = 0;
        cudaFree(s->d_pol); s->d_pol = nullptr;          // no modes: nothing to polarise
        destroy_graph(s);
        plan_tma(s);
        push_ctrl(s);
        return code;
    };
    auto cuda_fail = [&](cudaError_t e) { return fail(e == cudaErrorMemoryAllocation ? CAV_E_NOMEM : CAV_E_CUDA, e); };
    const size_t bytes = (size_t)N * s->ncp * s->esize;
    cudaError_t e;
    if (bytes > s->u_bytes) {
        cudaFree(s->u);
        s->u = nullptr;
        s->u_bytes = 0;
        if ((e = cudaMalloc(&s->u, bytes)) != cudaSuccess) return cuda_fail(e);
        s->u_bytes = bytes;
    }
    s->u_hash = 0;
    if (N > 0 && !u_is_device) {          // lets a sweep recognise members with identical profiles
        unsigned long long hsh = 1469598103934665603ull;
        const unsigned char* pb = (const unsigned char*)u;
        const size_t nb8 = (size_t)N * s->nc * s->esize;
        for (size_t i = 0; i < nb8; i += 8) {
            unsigned long long w8 = 0;
            memcpy(&w8, pb + i, nb8 - i >= 8 ? 8 : nb8 - i);
            hsh = (hsh ^ w8) * 1099511628211ull;
        }
        s->u_hash = hsh ? hsh : 1ull;
    }
    if (N > 0) {
        if (s->padded && (e = cudaMemsetAsync(s->u, 0, bytes, s->stream)) != cudaSuccess) return cuda_fail(e);     // pad cells: u = 0
        if (copy_in(s, s->u, u, N, u_is_device != 0) != CAV_OK) return fail(CAV_E_CUDA);
    }
    // overlap normalisation W_n into a temporary first: CAV_E_SINGULAR_NORM must not leave half-set mode tables behind
    double invW[kMaxModes];
    for (int n = 0; n < N; ++n) invW[n] = 1.0 / (double)s->nc;
    if (N > 0 && s->prm.overlap_norm == CAV_NORM_SUM_U) {
        double* d_out = nullptr;
        if ((e = cudaMalloc(&d_out, sizeof(double) * 256 * N)) != cudaSuccess) return cuda_fail(e);
        if (s->prm.precision == CAV_F32) k_sum_u<float><<<dim3(256, N), 256, 0, s->stream>>>((const float*)s->u, s->ncp, d_out);
        else k_sum_u<double><<<dim3(256, N), 256, 0, s->stream>>>((const double*)s->u, s->ncp, d_out);
        s->host_launches++;
        double* h = new (std::nothrow) double[256 * (size_t)N];
        if (!h) { cudaFree(d_out); return fail(CAV_E_NOMEM); }
        e = cudaMemcpyAsync(h, d_out, sizeof(double) * 256 * N, cudaMemcpyDeviceToHost, s->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(s->stream);
        cudaFree(d_out);
        if (e != cudaSuccess) { delete[] h; return cuda_fail(e); }
        bool singular = false;
        for (int n = 0; n < N; ++n) {
            double sum = 0.0;
            for (int b = 0; b < 256; ++b) sum += h[n * 256 + b];
            if (std::fabs(sum) < 1e-6 * (double)s->nc) singular = true;
            else invW[n] = 1.0 / sum;
        }
        delete[] h;
        if (singular) return fail(CAV_E_SINGULAR_NORM);
    }
    Ctrl* c = s->h_ctrl;
    c->N = N;
    for (int n = 0; n < N; ++n) {
        const double Gm = Gamma ? Gamma[n] : 0.0, Ph = Phi ? Phi[n] : 0.0;
        c->omega[n] = omega[n];
        c->kappa[n] = kappa[n];
        c->Gre[n] = g[n] + Gm * std::cos(Ph);
        c->Gim[n] = Gm * std::sin(Ph);
        c->Gbre[n] = c->Gre[n]; c->Gbim[n] = c->Gim[n];      // reciprocal until cav_set_backaction
        c->invW[n] = invW[n];
        c->a[n][0] = c->a[n][1] = 0.0;
    }
    c->drive_on = 0;                     // a new mode set clears the drive,
    cudaFree(s->d_pol); s->d_pol = nullptr;          // the polarisation (back to x^)
    cudaFree(s->d_spec); s->d_spec = nullptr;        // and the spectrum (its layout depends on N)
    c->spec_K = 0; c->spec_n = 0;
    c->k1_valid = 0;
    s->N = N;
    s->nb = bucket(N);
    destroy_graph(s);                    // the old graph's kernels were instantiated for the old mode bucket / u pointer
    rc = plan_tma(s);
    if (rc) return fail(rc);
    return push_ctrl(s);
}

int cav_set_backaction(cav_sim* s, const double* g_b, const double* Gamma_b, const double* Phi_b) {
    if (!s) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    Ctrl* c = s->h_ctrl;
    for (int n = 0; n < c->N; ++n) {
        if (g_b) {
            const double Gm = Gamma_b ? Gamma_b[n] : 0.0, Ph = Phi_b ? Phi_b[n] : 0.0;
            c->Gbre[n] = g_b[n] + Gm * std::cos(Ph);
            c->Gbim[n] = Gm * std::sin(Ph);
        } else {
            c->Gbre[n] = c->Gre[n]; c->Gbim[n] = c->Gim[n];
        }
    }
    c->k1_valid = 0;                     // dm/dt of the current state changes
    return push_ctrl(s);
}

int cav_set_polarisation(cav_sim* s, const double* pol, const double* quad) {
    if (!s) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    cudaFree(s->d_pol);
    s->d_pol = nullptr;
    s->graph_dirty = true;
    s->h_ctrl->k1_valid = 0;             // dm/dt and da/dt of the current state change
    if (pol && s->N > 0) {
        double h[6 * CAV_MAX_MODES];
        rc = pack_polarisation(s->N, pol, quad, h);
        if (rc) return rc;
        CK(cudaMalloc(&s->d_pol, sizeof(double) * 6 * s->N));
        CK(cudaMemcpyAsync(s->d_pol, h, sizeof(double) * 6 * s->N, cudaMemcpyHostToDevice, s->stream));
        CK(cudaStreamSynchronize(s->stream));
        // the dipolar-field kernels know x^ only; rows padded inside the library need the TMA kernels, which take
        // a polarisation for up to 8 modes
        if (s->demag || (s->padded && stage_tma_fn(s, 2) == nullptr)) {
            cudaFree(s->d_pol);
            s->d_pol = nullptr;
            plan_tma(s);
            push_ctrl(s);
            return CAV_E_UNSUPPORTED;
        }
    }
    rc = plan_tma(s);                    // the polarised TMA kernels are other functions: their own shared-memory budget
    if (rc) return rc;
    return push_ctrl(s);
}

int cav_set_integrator(cav_sim* s, int integrator, int n_llg) {
    if (!s || (integrator != CAV_INTEGRATOR_UNIFIED && integrator != CAV_INTEGRATOR_SPLIT)) return CAV_E_ARG;
    if (integrator == CAV_INTEGRATOR_SPLIT && n_llg < 1) return CAV_E_ARG;
    const int old = s->split_nllg;
    s->split_nllg = integrator == CAV_INTEGRATOR_SPLIT ? n_llg : 0;
    if (s->split_nllg > 0) {
        decide_path(s);
        if (!s->use_block && !s->use_coop) { s->split_nllg = old; return CAV_E_UNSUPPORTED; }
    }
    s->graph_dirty = true;
    return CAV_OK;
}

int cav_set_demag(cav_sim* s, int on) {
    if (!s) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    if (!on) {
        demag_destroy(s->demag);
        s->demag = nullptr;
    } else if (!s->demag) {
        if (s->padded) return CAV_E_UNSUPPORTED;             // rows padded for the TMA path; the dipolar field runs on the generic kernels
        if (s->d_pol != nullptr || s->split_nllg > 0) return CAV_E_UNSUPPORTED;      // those live in the small-grid kernel
        if (!s->d_bdem) CK(cudaMalloc(&s->d_bdem, (size_t)3 * s->nc * s->esize));
        rc = demag_create(&s->demag, s->grid.nx, s->grid.ny, s->grid.nz, s->grid.dx, s->grid.dy, s->grid.dz, s->prm.Ms,
                          s->prm.n_sub, s->prm.precision == CAV_F32, s->stream, s->cuda_err, (int)sizeof(s->cuda_err));
        if (rc) return rc;
    }
    s->graph_dirty = true;
    s->h_ctrl->k1_valid = 0;             // dm/dt of the current state changes
    s->last_run_block = false;
    return push_ctrl(s);
}

int cav_set_spectrum(cav_sim* s, int n_bins, double omega_lo, double omega_hi) {
    if (!s || n_bins < 0 || (n_bins > 1 && !(omega_hi > omega_lo))) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    cudaFree(s->d_spec);
    s->d_spec = nullptr;
    s->graph_dirty = true;               // the pointer is a kernel argument
    Ctrl* c = s->h_ctrl;
    c->spec_K = 0; c->spec_n = 0;
    if (n_bins > 0) {
        const size_t bytes = sizeof(double) * (size_t)n_bins * 2 * (2 * s->N + s->prm.n_sub);
        CK(cudaMalloc(&s->d_spec, bytes));
        CK(cudaMemsetAsync(s->d_spec, 0, bytes, s->stream));
        c->spec_K = n_bins; c->spec_w0 = omega_lo; c->spec_dw = n_bins > 1 ? (omega_hi - omega_lo) / (double)(n_bins - 1) : 0.0;
    }
    return push_ctrl(s);
}

int cav_get_spectrum(cav_sim* s, double* out, long long* n_samples) {
    if (!s || !out) return CAV_E_ARG;
    if (!s->d_spec) return CAV_E_STATE;
    int rc = sync_pull(s);
    if (rc) return rc;
    CK(cudaMemcpyAsync(out, s->d_spec, sizeof(double) * (size_t)s->h_ctrl->spec_K * 2 * (2 * s->N + s->prm.n_sub), cudaMemcpyDeviceToHost, s->stream));
    CK(cudaStreamSynchronize(s->stream));
    if (n_samples) *n_samples = s->h_ctrl->spec_n;
    return s->h_ctrl->status;
}

int cav_set_drive(cav_sim* s, const double* amp, const double* t0, const double* sigma, const double* omega_d) {
    if (!s) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    Ctrl* c = s->h_ctrl;
    if (!amp || c->N == 0) {
        c->drive_on = 0;
    } else {
        if (!t0 || !sigma) return CAV_E_ARG;
        for (int n = 0; n < c->N; ++n)
            if (!(sigma[n] > 0.0)) return CAV_E_ARG;
        for (int n = 0; n < c->N; ++n) {
            c->eta_re[n] = amp[2 * n]; c->eta_im[n] = amp[2 * n + 1];
            c->eta_t0[n] = t0[n];
            c->eta_i2s2[n] = 1.0 / (2.0 * sigma[n] * sigma[n]);
            c->eta_wd[n] = omega_d ? omega_d[n] : 0.0;
        }
        c->drive_on = 1;
    }
    c->k1_valid = 0;                     // da/dt of the current state changes
    return push_ctrl(s);
}

int cav_set_m(cav_sim* s, const void* m, int is_device) {
    if (!s || !m) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    const void* src = m;
    if (!is_device || s->padded) {       // staged through MS[1] (host source, or rows to be padded)
        rc = copy_in(s, s->MS[1], m, 3 * s->prm.n_sub, is_device != 0);
        if (rc) return rc;
        src = s->MS[1];
    }
    void* dst = s->Y[s->h_ctrl->ycur];
    const long long n = s->ncp * s->prm.n_sub;        // pad cells included: they are never read back as cells
    const int blocks = (int)((n + 255) / 256);
    if (s->prm.precision == CAV_F32) k_normalize<float><<<blocks, 256, 0, s->stream>>>((const float*)src, (float*)dst, s->ncp, s->prm.n_sub);
    else k_normalize<double><<<blocks, 256, 0, s->stream>>>((const double*)src, (double*)dst, s->ncp, s->prm.n_sub);
    CK(cudaGetLastError());
    s->host_launches++;
    s->h_ctrl->k1_valid = 0;
    s->h_ctrl->status = 0;
    s->m_set = true;
    return push_ctrl(s);
}

int cav_get_m(cav_sim* s, void* out, int is_device) {
    if (!s || !out) return CAV_E_ARG;
    if (!s->m_set) return CAV_E_STATE;
    int rc = sync_pull(s);
    if (rc) return rc;
    rc = copy_out(s, out, s->Y[s->h_ctrl->ycur], 3 * s->prm.n_sub, is_device != 0);
    if (rc) return rc;
    CK(cudaStreamSynchronize(s->stream));
    return s->h_ctrl->status;
}

int cav_set_a(cav_sim* s, const double* a) {
    if (!s || (!a && s->N > 0)) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    for (int n = 0; n < s->N; ++n) { s->h_ctrl->a[n][0] = a[2 * n]; s->h_ctrl->a[n][1] = a[2 * n + 1]; }
    s->h_ctrl->k1_valid = 0;
    return push_ctrl(s);
}

int cav_get_a(cav_sim* s, double* out) {
    if (!s || (!out && s->N > 0)) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    for (int n = 0; n < s->N; ++n) { out[2 * n] = s->h_ctrl->a[n][0]; out[2 * n + 1] = s->h_ctrl->a[n][1]; }
    return s->h_ctrl->status;
}

static int ensure_k1(cav_sim* s) {
    if (!s->m_set) return CAV_E_STATE;
    int rc = sync_pull(s);
    if (rc) return rc;
    if (!s->h_ctrl->k1_valid) {
        choose_grid(s);
        decide_path(s);
        if (s->padded && !s->use_tma) return CAV_E_UNSUPPORTED;
        StageArgs A = make_args(s, 0ull);
        s->h_fresh = false;
        k_begin<<<1, kBeginThreads, 0, s->stream>>>(s->d_ctrl, s->d_ctrl0, 0ull);
        CK(cudaGetLastError());
        s->host_launches++;
        rc = launch_stage(s, 1, A, s->stream);
        if (rc) return rc;
        rc = sync_pull(s);
    }
    return rc;
}

int cav_get_dmdt(cav_sim* s, void* out, int is_device) {
    if (!s || !out) return CAV_E_ARG;
    int rc = ensure_k1(s);
    if (rc) return rc;
    rc = copy_out(s, out, s->K[s->h_ctrl->k1slot], 3 * s->prm.n_sub, is_device != 0);
    if (rc) return rc;
    CK(cudaStreamSynchronize(s->stream));
    return s->h_ctrl->status;
}

int cav_get_dadt(cav_sim* s, double* out) {
    if (!s || (!out && s->N > 0)) return CAV_E_ARG;
    int rc = ensure_k1(s);
    if (rc) return rc;
    for (int n = 0; n < s->N; ++n) { out[2 * n] = s->h_ctrl->ka[0][n][0]; out[2 * n + 1] = s->h_ctrl->ka[0][n][1]; }
    return s->h_ctrl->status;
}

int cav_get_overlaps(cav_sim* s, double* out) {
    if (!s || (!out && s->N > 0)) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    for (int n = 0; n < s->N; ++n) { out[2 * n] = s->h_ctrl->S[n][0]; out[2 * n + 1] = s->h_ctrl->S[n][1]; }
    return s->h_ctrl->status;
}

int cav_run_steps(cav_sim* s, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps) {
    if (!s) return CAV_E_ARG;
    if (!s->m_set) return CAV_E_STATE;
    const bool adaptive = tol > 0.0;
    if (adaptive == (fixed_dt > 0.0)) return CAV_E_ARG;        // exactly one of the two
    if (std::isnan(t_end) || max_steps < 0) return CAV_E_ARG;
    if (std::isinf(t_end) && max_steps == 0) return CAV_E_ARG;
    decide_path(s);
    if (!s->last_run_block && (s->use_block || s->use_coop)) { int rc0 = sync_pull(s); if (rc0) return rc0; s->last_run_block = true; }
    s->h_fresh = false;                                        // the run rewrites Ctrl on the device
    if (s->use_block || s->use_coop) return run_block_path(s, t_end, adaptive ? tol : 0.0, adaptive ? 0.0 : fixed_dt, dt_init, max_steps);
    if (s->split_nllg > 0) return CAV_E_UNSUPPORTED;                            // grid beyond the small-grid kernel (cavmag.h)
    if (s->padded && !s->use_tma) return CAV_E_UNSUPPORTED;                     // padded rows are only understood by the TMA kernels
    s->last_run_block = false;
    k_setrun<<<1, 1, 0, s->stream>>>(s->d_ctrl, t_end, adaptive ? tol : 0.0, adaptive ? 0.0 : fixed_dt, dt_init, max_steps);
    CK(cudaGetLastError());
    s->host_launches++;
    if (s->launch_mode == CAV_LAUNCH_GRAPH) {
        if (s->graph_dirty || !s->exec[0] || !s->exec[1]) {
            int rc = build_graph(s);
            if (rc && s->demag) {                    // cuFFT's launches could not be captured here: enqueue from the host
                cudaGetLastError();
                destroy_graph(s);
                s->host_launches++;
                return run_stream_mode(s);
            }
            if (rc) return rc;
        }
        const int which = (max_steps == 0 || max_steps >= kUnrollMinSteps) ? 1 : 0;
        CK(cudaGraphLaunch(s->exec[which], s->stream));
        s->host_launches += s->use_tma ? 2 : 1;   // k_begin (+ the stage-2 kernel after the loop that finishes the last step)
        return CAV_OK;
    }
    s->host_launches++;
    return run_stream_mode(s);
}

int cav_run(cav_sim* s, double t_end, double tol, double fixed_dt, double dt_init) {
    if (!(t_end < INFINITY)) return CAV_E_ARG;
    return cav_run_steps(s, t_end, tol, fixed_dt, dt_init, 0);
}

int cav_sync(cav_sim* s) {
    if (!s) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    return s->h_ctrl->status;
}

int cav_get_time(cav_sim* s, double* t, double* dt) {
    if (!s) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    if (t) *t = s->h_ctrl->t;
    if (dt) *dt = s->h_ctrl->dt;
    return s->h_ctrl->status;
}

int cav_set_time(cav_sim* s, double t) {
    if (!s || std::isnan(t)) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    s->h_ctrl->t = t;
    return push_ctrl(s);
}

int cav_get_stats(cav_sim* s, cav_stats* o) {
    if (!s || !o) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    const Ctrl* c = s->h_ctrl;
    o->accepted = c->accepted; o->rejected = c->rejected; o->rhs_evals = c->rhs_evals;
    o->dt_min = c->dt_min; o->dt_max = c->dt_max; o->dt_next = c->dt; o->t = c->t; o->last_err = c->last_err;
    return c->status;
}

int cav_set_trace(cav_sim* s, double sample_dt, int capacity) {
    if (!s || capacity < 0) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    Ctrl* c = s->h_ctrl;
    if (!(sample_dt > 0.0) || capacity == 0) {
        c->sample_dt = 0.0; c->trace_cap = 0; c->trace_n = 0;
        return push_ctrl(s);
    }
    const int row = 1 + 4 * s->N + 3 * s->prm.n_sub;
    if (capacity > s->trace_cap) {
        cudaFree(s->d_trace);
        s->d_trace = nullptr;
        s->trace_cap = 0;
        CK(cudaMalloc(&s->d_trace, sizeof(double) * (size_t)capacity * (1 + 4 * CAV_MAX_MODES + 6)));
        s->trace_cap = capacity;
        s->graph_dirty = true;
    }
    (void)row;
    c->sample_dt = sample_dt;
    c->trace_cap = capacity;
    c->trace_n = 0;
    c->trace_t0 = c->t;
    c->trace_acc0 = c->accepted;
    c->trace_stride = 1;
    return push_ctrl(s);
}

int cav_trace_row_len(cav_sim* s, int* row_len) {
    if (!s || !row_len) return CAV_E_ARG;
    *row_len = 1 + 4 * s->N + 3 * s->prm.n_sub;
    return CAV_OK;
}

int cav_get_trace(cav_sim* s, double* out, int* n_samples) {
    if (!s || !n_samples) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    const int n = s->h_ctrl->trace_n;
    *n_samples = n;
    const int row = 1 + 4 * s->N + 3 * s->prm.n_sub;
    if (out && n > 0) {
        CK(cudaMemcpyAsync(out, s->d_trace, sizeof(double) * (size_t)n * row, cudaMemcpyDeviceToHost, s->stream));
        CK(cudaStreamSynchronize(s->stream));
    }
    return s->h_ctrl->status;
}

int cav_get_launch_count(cav_sim* s, long long* n) {
    if (!s || !n) return CAV_E_ARG;
    int rc = sync_pull(s);
    if (rc) return rc;
    *n = s->host_launches + s->h_ctrl->rhs_evals;
    return CAV_OK;
}

/* ---------------------------------------------------------------------------------------------------------
 * Joint launch of several simulations of the same shape (cavmag.h "Sweeps of mid-size grids")
 * --------------------------------------------------------------------------------------------------------- */
struct cav_sweep {
    std::vector<cav_sim*> sims;
    cudaStream_t stream = nullptr;
    RepPtrs* d_reps = nullptr;
    unsigned int* d_live = nullptr;
    std::vector<RepPtrs> h_reps;
    cudaGraph_t graph[2] = {nullptr, nullptr};
    cudaGraphExec_t exec[2] = {nullptr, nullptr};
    TmaArgs targs[8];
    size_t tsmem[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    int tgrid = 0;
    char cuda_err[256] = {0};
};

namespace {

void sweep_fill_reps(cav_sweep* w) {
    w->h_reps.resize(w->sims.size());
    bool same_u = w->sims[0]->u_hash != 0;
    for (cav_sim* q : w->sims) same_u = same_u && q->u_hash == w->sims[0]->u_hash && q->N == w->sims[0]->N;
    for (size_t r = 0; r < w->sims.size(); ++r) {
        cav_sim* q = w->sims[r];
        RepPtrs& p = w->h_reps[r];
        memset(&p, 0, sizeof(p));
        p.ctrl = q->d_ctrl; p.ctrl0 = q->d_ctrl0;
        for (int i = 0; i < 2; ++i) { p.Y[i] = q->Y[i]; p.MS[i] = q->MS[i]; }
        for (int i = 0; i < 7; ++i) p.K[i] = q->K[i];
        p.u = q->u; p.partial = q->partial; p.partial_max = q->partial_max; p.spec = q->d_spec; p.trace = q->d_trace;
        p.maps = q->d_maps;
        p.umap = (same_u ? w->sims[0]->d_maps : q->d_maps) + 128 * MAP_P_U;
        for (int i = 0; i < 3; ++i) p.B0[i] = q->prm.B0[i];
    }
}

void sweep_destroy_graphs(cav_sweep* w) {
    for (int i = 0; i < 2; ++i) {
        if (w->exec[i]) { cudaGraphExecDestroy(w->exec[i]); w->exec[i] = nullptr; }
        if (w->graph[i]) { cudaGraphDestroy(w->graph[i]); w->graph[i] = nullptr; }
    }
}

const void* stage_tma_sweep_fn(const cav_sim* q, int stage) {
    return q->prm.precision == CAV_F32 ? stage_tma_sweep_kernel_f32(q->prm.n_sub, stage, q->nb)
                                       : stage_tma_sweep_kernel_f64(q->prm.n_sub, stage, q->nb);
}

// k_sweep_begin -> K1 of every simulation (ordinary launches; they return at once when FSAL's k1 is valid) -> k_sweep_cond
//   -> WHILE { joint K2 .. K7 [x unroll] } -> joint K2 (finishes the last step)
int sweep_build_graph(cav_sweep* w, int which, int unroll) {
    cav_sim* s = w->sims[0];                 // CK() reports into the first simulation's error text
    const int R = (int)w->sims.size();
    CK(cudaGraphCreate(&w->graph[which], 0));
    cudaGraph_t graph = w->graph[which];
    cudaGraphConditionalHandle handle;
    CK(cudaGraphConditionalHandleCreate(&handle, graph, 0, cudaGraphCondAssignDefault));
    unsigned long long h64 = (unsigned long long)handle;
    const RepPtrs* reps = w->d_reps;
    unsigned int* live = w->d_live;
    cudaGraphNode_t prev, node;
    {
        void* params[] = {(void*)&reps};
        int rc = add_kernel(s, graph, &prev, nullptr, (const void*)k_sweep_begin, dim3(R), dim3(kBeginThreads), params, 0);
        if (rc) return rc;
    }
    std::vector<StageArgs> A1(R);
    for (int r = 0; r < R; ++r) {
        cav_sim* q = w->sims[r];
        A1[r] = make_args(q, 0ull);
        double* trace = q->d_trace;
        void* tparams[] = {&A1[r], &q->targs[1], &trace};
        int rc = add_kernel(s, graph, &node, &prev, stage_tma_fn(q, 1), dim3(q->tgrid), dim3(kTmaThreads), tparams, q->tsmem[1]);
        if (rc) return rc;
        prev = node;
    }
    {
        int Rv = R;
        void* params[] = {(void*)&reps, &Rv, &live, &h64};
        int rc = add_kernel(s, graph, &node, &prev, (const void*)k_sweep_cond, dim3(1), dim3(128), params, 0);
        if (rc) return rc;
        prev = node;
    }
    cudaGraphNodeParams cp = {};
    cp.type = cudaGraphNodeTypeConditional;
    cp.conditional.handle = handle;
    cp.conditional.type = cudaGraphCondTypeWhile;
    cp.conditional.size = 1;
    cudaGraphNode_t n_while;
    CK(cudaGraphAddNode(&n_while, graph, &prev, 1, &cp));
    cudaGraph_t body = cp.conditional.phGraph_out[0];
    StageArgs A = make_args(s, 0ull);
    SweepArgs SW;
    SW.reps = w->d_reps; SW.R = R; SW.live = w->d_live; SW.cond_handle = h64;
    const bool pdl = s->want_pdl;
    for (int u = 0; u < unroll; ++u)
        for (int stage = 2; stage <= 7; ++stage) {
            void* tparams[] = {&A, &w->targs[stage], &SW};
            const cudaGraphNode_t* dep = (u == 0 && stage == 2) ? nullptr : &prev;
            int rc = add_kernel(s, body, &node, dep, stage_tma_sweep_fn(s, stage), dim3(w->tgrid), dim3(kTmaThreads), tparams, w->tsmem[stage], pdl);
            if (rc) return rc;
            prev = node;
        }
    {
        void* tparams[] = {&A, &w->targs[2], &SW};
        int rc = add_kernel(s, graph, &node, &n_while, stage_tma_sweep_fn(s, 2), dim3(w->tgrid), dim3(kTmaThreads), tparams, w->tsmem[2]);
        if (rc) return rc;
    }
    CK(cudaGraphInstantiate(&w->exec[which], graph, 0));
    CK(cudaGraphUpload(w->exec[which], w->stream));
    return CAV_OK;
}

}  // namespace

int cav_sweep_create(cav_sim* const* sims, int n, cav_sweep** out) {
    if (!sims || !out || n < 1) return CAV_E_ARG;
    *out = nullptr;
    cav_sim* s = sims[0];
    if (!s) return CAV_E_ARG;
    for (int r = 0; r < n; ++r) {
        cav_sim* q = sims[r];
        if (!q || !q->m_set) return q ? CAV_E_STATE : CAV_E_ARG;
        if (q->grid.nx != s->grid.nx || q->grid.ny != s->grid.ny || q->grid.nz != s->grid.nz || q->prm.precision != s->prm.precision ||
            q->N != s->N || q->stream != s->stream || q->prm.renormalize != s->prm.renormalize || q->prm.n_sub != s->prm.n_sub ||
            q->prm.B_exch_inter != s->prm.B_exch_inter)
            return CAV_E_ARG;
        // the joint kernels take the material and cell constants from simulation 0: only B0, the modes and the state may differ
        if (q->grid.dx != s->grid.dx || q->grid.dy != s->grid.dy || q->grid.dz != s->grid.dz || q->prm.Ms != s->prm.Ms ||
            q->prm.Aex != s->prm.Aex || q->prm.Ku != s->prm.Ku || q->prm.alpha != s->prm.alpha || q->prm.gamma != s->prm.gamma ||
            memcmp(q->prm.ku_axis, s->prm.ku_axis, sizeof(s->prm.ku_axis)) != 0)
            return CAV_E_ARG;
        if (!q->tma_eligible || q->demag || q->d_pol || q->split_nllg > 0 || q->nb > (q->prm.n_sub == 1 ? 8 : 2)) return CAV_E_UNSUPPORTED;
        for (int r2 = 0; r2 < r; ++r2) if (sims[r2] == q) return CAV_E_ARG;
    }
    if (s->targs[1].Q * (long long)n < (long long)s->n_sm) return CAV_E_UNSUPPORTED;      // not enough plane-tiles for a persistent grid
    cav_sweep* w = new (std::nothrow) cav_sweep();
    if (!w) return CAV_E_NOMEM;
    w->sims.assign(sims, sims + n);
    w->stream = s->stream;
    w->tgrid = s->n_sm;
    for (int stage = 1; stage <= 7; ++stage) {
        w->targs[stage] = s->targs[stage];
        w->targs[stage].pre_k = 0;           // a joint launch fetches nothing before the dependency wait
        w->targs[stage].pre_ctrl = 0;
        w->tsmem[stage] = s->tsmem[stage];
        if (stage >= 2) {
            const void* fn = stage_tma_sweep_fn(s, stage);
            if (!fn) { delete w; return CAV_E_UNSUPPORTED; }
            cudaFuncAttributes fa;
            if (cudaFuncGetAttributes(&fa, fn) != cudaSuccess ||
                cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(s->smem_optin - fa.sharedSizeBytes)) != cudaSuccess ||
                w->tsmem[stage] + fa.sharedSizeBytes > s->smem_optin) {
                cudaGetLastError();
                delete w;
                return CAV_E_UNSUPPORTED;
            }
        }
    }
    if (cudaMalloc(&w->d_reps, sizeof(RepPtrs) * n) != cudaSuccess || cudaMalloc(&w->d_live, sizeof(unsigned int)) != cudaSuccess) {
        cudaGetLastError(); cudaFree(w->d_reps); cudaFree(w->d_live); delete w;
        return CAV_E_NOMEM;
    }
    *out = w;
    return CAV_OK;
}

int cav_sweep_destroy(cav_sweep* w) {
    if (!w) return CAV_E_ARG;
    if (w->stream) cudaStreamSynchronize(w->stream);
    sweep_destroy_graphs(w);
    cudaFree(w->d_reps); cudaFree(w->d_live);
    cudaGetLastError();
    delete w;
    return CAV_OK;
}

int cav_sweep_run(cav_sweep* w, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps) {
    if (!w) return CAV_E_ARG;
    const bool adaptive = tol > 0.0;
    if (adaptive == (fixed_dt > 0.0)) return CAV_E_ARG;
    if (std::isnan(t_end) || max_steps < 0 || (std::isinf(t_end) && max_steps == 0)) return CAV_E_ARG;
    cav_sim* s = w->sims[0];
    // what cav_sweep_create refuses must not have been switched on in a member since (the joint kernels know none of it)
    for (cav_sim* q : w->sims)
        if (q->d_pol || q->demag || q->split_nllg > 0) return CAV_E_UNSUPPORTED;
    // per-simulation pointers may have changed since the last run (trace, spectrum, mode profiles): refresh, and rebuild
    // the graphs when anything the graph nodes hold by value did
    std::vector<RepPtrs> old = w->h_reps;
    sweep_fill_reps(w);
    const bool changed = old.size() != w->h_reps.size() || memcmp(old.data(), w->h_reps.data(), sizeof(RepPtrs) * old.size()) != 0;
    CK(cudaMemcpyAsync(w->d_reps, w->h_reps.data(), sizeof(RepPtrs) * w->h_reps.size(), cudaMemcpyHostToDevice, w->stream));
    CK(cudaStreamSynchronize(w->stream));
    if (changed || !w->exec[0] || !w->exec[1]) {
        sweep_destroy_graphs(w);
        int rc = sweep_build_graph(w, 0, 1);
        if (rc == CAV_OK) rc = sweep_build_graph(w, 1, kLoopUnroll);
        if (rc) { sweep_destroy_graphs(w); return rc; }
    }
    const int R = (int)w->sims.size();
    k_sweep_setrun<<<R, 1, 0, w->stream>>>(w->d_reps, t_end, adaptive ? tol : 0.0, adaptive ? 0.0 : fixed_dt, dt_init, max_steps);
    CK(cudaGetLastError());
    const int which = (max_steps == 0 || max_steps >= kUnrollMinSteps) ? 1 : 0;
    CK(cudaGraphLaunch(w->exec[which], w->stream));
    for (cav_sim* q : w->sims) { q->last_run_block = false; q->h_fresh = false; q->host_launches += 2; }
    return CAV_OK;
}

#ifdef CAVMAG_PROBE
// profiling builds only (-DCAVMAG_PROBE; not declared in cavmag.h): the per-block timestamps of the last launches
int cav_debug_probe(cav_sim* s, unsigned long long* out /*[8][256][32]*/, int while_running) {
    if (!s || !out) return CAV_E_ARG;
    if (!while_running) CK(cudaStreamSynchronize(s->stream));
    cudaStream_t side;                      // a snapshot while the run graph is still looping (marks of the empty last iteration would overwrite a finished run's)
    CK(cudaStreamCreateWithFlags(&side, cudaStreamNonBlocking));
    CK(cudaMemcpyAsync(out, s->d_probe, 8 * 256 * 32 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, side));
    CK(cudaStreamSynchronize(side));
    cudaStreamDestroy(side);
    return CAV_OK;
}
#endif

}  // extern "C"
