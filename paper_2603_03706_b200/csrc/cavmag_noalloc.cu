// cav_overlaps_noalloc: the overlap reduction (Eq. 18) as a stand-alone call that
// allocates nothing - for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
// harnesses that forbid it).  See include/cavmag.h for the contract.
//
// The block partials of the two-pass, fixed-order reduction - which the handle-based path keeps in buffers that
// cav_create allocates - live in a file-scope __device__ array of a stated maximum size.  In host code the array's name
// is a host-side stand-in, not a device address: the address the kernel gets comes from cudaGetSymbolAddress, once per
// device, with that device current.
#include <atomic>
#include <cmath>
#include <cstdio>
#include <cuda_runtime.h>

#include "../../include/cavmag.h"

namespace {

constexpr int kThreads = 256;
constexpr int kCellsPerThread = 32;
constexpr int kChunk = kThreads * kCellsPerThread;                                   // cells per block: 8192
constexpr int kMaxBlocks = (int)(CAV_NOALLOC_MAX_CELLS / kChunk);                      // 2048
constexpr int kMaxSums = 2 * CAV_MAX_MODES;                                          // Re and Im sum per mode
constexpr size_t kHeaderBytes = 256;                                                 // ticket counter (must start at zero)
constexpr size_t kScratchBytes = kHeaderBytes + sizeof(double) * (size_t)kMaxBlocks * kMaxSums;
static_assert(kScratchBytes == CAV_NOALLOC_SCRATCH_BYTES, "cavmag.h states the size of the scratch array");
static_assert(CAV_NOALLOC_MAX_CELLS % kChunk == 0, "whole chunks");

// [0, 256): unsigned ticket counter; then double partial[block][2 N].  Held by every GPU that loads the library, until exit.
static __device__ __align__(256) unsigned char g_noalloc_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::atomic<unsigned char*> g_scratch_ptr[kMaxDevices];     // device address of g_noalloc_scratch per device (set-up below), or NULL

thread_local char t_err[256] = "";

int fail(int code, const char* fmt, long long a = 0, long long b = 0) {
    snprintf(t_err, sizeof(t_err), fmt, a, b);
    return code;
}

// Block b sums u_n (m_c,x, m_c,y) over its chunk of cells [b kChunk, (b+1) kChunk) for every mode, in a fixed order
// (thread-strided cells, fp64 accumulators, warp shuffle tree, warps in order), and writes 2N partials.  The last block
// to arrive (ticket) adds the partials in block order and writes S_n = (1/N_cells) sum u_n (m_c,x - i m_c,y).
template <typename T>
__global__ void __launch_bounds__(kThreads) k_overlaps_noalloc(const T* __restrict__ m, const T* __restrict__ u, long long nc,
                                                               int n_sub, int N, unsigned char* scratch, double* __restrict__ S_out) {
    __shared__ double s_w[2][kThreads / 32];
    __shared__ int s_last;
    unsigned int* const ticket = reinterpret_cast<unsigned int*>(scratch);
    double* const partial = reinterpret_cast<double*>(scratch + kHeaderBytes);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const long long c0 = (long long)blockIdx.x * kChunk;
    const T half = (T)0.5;
    for (int n = 0; n < N; ++n) {
        const T* const un = u + (long long)n * nc;
        double sx = 0.0, sy = 0.0;
#pragma unroll 4
        for (int i = 0; i < kCellsPerThread; ++i) {
            const long long cell = c0 + (long long)i * kThreads + tid;
            if (cell < nc) {
                T mx = m[cell], my = m[nc + cell];
                if (n_sub == 2) { mx = half * (mx + m[3 * nc + cell]); my = half * (my + m[4 * nc + cell]); }   // m_c: mean over the sublattices
                const T uv = un[cell];
                sx += (double)uv * (double)mx;
                sy += (double)uv * (double)my;
            }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) { sx += __shfl_down_sync(0xffffffffu, sx, o); sy += __shfl_down_sync(0xffffffffu, sy, o); }
        if (lane == 0) { s_w[0][warp] = sx; s_w[1][warp] = sy; }
        __syncthreads();
        if (tid < 2) {
            double acc = 0.0;
            for (int w = 0; w < kThreads / 32; ++w) acc += s_w[tid][w];
            partial[(size_t)blockIdx.x * (2 * N) + 2 * n + tid] = acc;
        }
        __syncthreads();
    }
    if (tid == 0) {
        __threadfence();
        const unsigned int old = atomicAdd(ticket, 1u);
        s_last = (old == gridDim.x - 1) ? 1 : 0;
        if (s_last) __threadfence();
    }
    __syncthreads();
    if (!s_last) return;
    if (tid < 2 * N) {
        double acc = 0.0;
        for (unsigned int b = 0; b < gridDim.x; ++b) acc += __ldcg(partial + (size_t)b * (2 * N) + tid);
        const double inv_W = 1.0 / (double)nc;
        S_out[tid] = (tid & 1) ? -acc * inv_W : acc * inv_W;
    }
    if (tid == 0) *ticket = 0u;                     // leave the counter as the next call needs it
}

// Once per device, with that device current: the device address of the scratch array.
int scratch_address(int dev, unsigned char** out) {
    if (dev < 0 || dev >= kMaxDevices) return fail(CAV_E_UNSUPPORTED, "cav_overlaps_noalloc: device ordinal %lld beyond %lld", dev, kMaxDevices - 1);
    unsigned char* p = g_scratch_ptr[dev].load(std::memory_order_acquire);
    if (!p) {
        const cudaError_t e = cudaGetSymbolAddress((void**)&p, g_noalloc_scratch);
        if (e != cudaSuccess || !p) {
            snprintf(t_err, sizeof(t_err), "cav_overlaps_noalloc: cudaGetSymbolAddress: %s", cudaGetErrorString(e));
            cudaGetLastError();
            return CAV_E_CUDA;
        }
        g_scratch_ptr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return CAV_OK;
}

}  // namespace

extern "C" {

const char* cav_noalloc_last_error(void) { return t_err; }

int cav_overlaps_noalloc(const void* m_dev, const void* u_dev, int precision, int nx, int ny, int nz, int n_sub, int N,
                         double* S_out_dev, void* cuda_stream) {
    t_err[0] = 0;
    if (precision != CAV_F32 && precision != CAV_F64) return fail(CAV_E_ARG, "cav_overlaps_noalloc: precision must be CAV_F32 or CAV_F64");
    if (nx < 1 || ny < 1 || nz < 1) return fail(CAV_E_ARG, "cav_overlaps_noalloc: grid sizes must be positive");
    if (n_sub != 1 && n_sub != 2) return fail(CAV_E_ARG, "cav_overlaps_noalloc: n_sub must be 1 or 2");
    if (N < 0) return fail(CAV_E_ARG, "cav_overlaps_noalloc: N must be >= 0");
    if (N > CAV_MAX_MODES) return fail(CAV_E_UNSUPPORTED, "cav_overlaps_noalloc: %lld modes exceed the maximum of %lld (CAV_MAX_MODES)", N, CAV_MAX_MODES);
    const long long nc = (long long)nx * ny * nz;
    if (nc > CAV_NOALLOC_MAX_CELLS)
        return fail(CAV_E_UNSUPPORTED, "cav_overlaps_noalloc: %lld cells exceed the maximum of %lld (CAV_NOALLOC_MAX_CELLS: the fixed scratch array)", nc, (long long)CAV_NOALLOC_MAX_CELLS);
    if (N == 0) return CAV_OK;
    if (!m_dev || !u_dev || !S_out_dev) return fail(CAV_E_ARG, "cav_overlaps_noalloc: NULL buffer");
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) { snprintf(t_err, sizeof(t_err), "cav_overlaps_noalloc: cudaGetDevice: %s", cudaGetErrorString(e)); cudaGetLastError(); return CAV_E_CUDA; }
    unsigned char* scratch = nullptr;
    int rc = scratch_address(dev, &scratch);
    if (rc) return rc;
    cudaStream_t stream = (cudaStream_t)cuda_stream;
    // the ticket counter must start at zero whatever an earlier (possibly failed) call left there
    e = cudaMemsetAsync(scratch, 0, kHeaderBytes, stream);
    if (e != cudaSuccess) { snprintf(t_err, sizeof(t_err), "cav_overlaps_noalloc: cudaMemsetAsync: %s", cudaGetErrorString(e)); cudaGetLastError(); return CAV_E_CUDA; }
    const unsigned int nblocks = (unsigned int)((nc + kChunk - 1) / kChunk);          // <= kMaxBlocks
    if (precision == CAV_F32)
        k_overlaps_noalloc<float><<<nblocks, kThreads, 0, stream>>>((const float*)m_dev, (const float*)u_dev, nc, n_sub, N, scratch, S_out_dev);
    else
        k_overlaps_noalloc<double><<<nblocks, kThreads, 0, stream>>>((const double*)m_dev, (const double*)u_dev, nc, n_sub, N, scratch, S_out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) { snprintf(t_err, sizeof(t_err), "cav_overlaps_noalloc: launch: %s", cudaGetErrorString(e)); return CAV_E_CUDA; }
    return CAV_OK;
}

}  // extern "C"
