// The fused RK45 stage kernel (hand-written CUDA for sm_100a).
//
// One launch = one evaluation of the coupled right-hand side at stage s of the
// Dormand-Prince step, fused with everything that can ride along on the same pass over HBM:
//
//   (a1) stage state          m_s(r)                    read with its 6-neighbour halo
//   (a4) overlap partials     sum_r u_n(r) m_c(r)       PAPER.md:156 Eq. 18  (of THIS stage's input)
//   (a2) effective field      B0 + exchange + anisotropy + x^ sum_n c_n u_n(r) [- B_E m_other]
//                                                       PAPER.md:121 Eq. 13, :159
//   (a3) LLG slope            k_s = -gamma/(1+alpha^2)[m x B + alpha m x (m x B)]
//   (a1) next stage state     m_{s+1} = m_0 + h sum_j a_{s+1,j} k_j     (materialised for the next launch)
//   (a6) stage 6: y5 -> m_new = y5/|y5| and the partial error field; stage 7: error max-norm
//   (a5,a7) the LAST block to finish reduces the block partials in a fixed order and runs the
//        mode ODEs (PAPER.md:119 Eq. 12, :317 Eq. 19), the mode stage algebra and, after
//        stage 7, the step-size controller — so no separate launch and no host round trip.
//
// Each thread owns VEC consecutive x cells (one 16-byte vector per field component); x
// neighbours come from warp shuffles, y/z neighbours from L1/L2-cached vector loads.  This is
// an HBM-bound streaming stencil: no tensor cores, no shared-memory tile.
#pragma once
#include <math_constants.h>

#include "cavmag_types.cuh"

namespace cavmag {

#ifdef CAVMAG_PROBE
// profiling builds only: globaltimer (slot) and clock64 (16 + slot) of this block at a marked point
template <typename Args>
__device__ __forceinline__ void probe_mark(const Args& A, int stage, int slot) {
    unsigned long long g, c = clock64();
    asm volatile("mov.u64 %0, %globaltimer;" : "=l"(g));
    unsigned long long* p = A.probe + ((size_t)stage * gridDim.x + blockIdx.x) * 32;
    p[slot] = g; p[16 + slot] = c;
}
#define CAVMAG_MARK(slot) probe_mark(A, STAGE, slot)
#define CAVMAG_MARKF(slot) do { if (threadIdx.x == 0) probe_mark(A, stage, slot); } while (0)
#else
#define CAVMAG_MARK(slot) ((void)0)
#define CAVMAG_MARKF(slot) ((void)0)
#endif

__device__ constexpr double kA[7][7] = CAVMAG_DP_A;
__device__ constexpr double kD[7] = CAVMAG_DP_D;
__device__ constexpr double kC[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};   // stage times t + c_s h

// ---------------------------------------------------------------------------------------
// vector load/store of VEC consecutive cells (16 bytes for float4 / double2)
// ---------------------------------------------------------------------------------------
template <typename T, int VEC>
struct alignas(sizeof(T) * VEC) Pack {
    T v[VEC];
};

template <typename T, int VEC>
__device__ __forceinline__ Pack<T, VEC> ldp(const T* __restrict__ p) {
    Pack<T, VEC> r;
    if constexpr (sizeof(T) * VEC == 16) {
        const float4 q = __ldg(reinterpret_cast<const float4*>(p));
        r = *reinterpret_cast<const Pack<T, VEC>*>(&q);
    } else if constexpr (sizeof(T) * VEC == 8) {
        const float2 q = __ldg(reinterpret_cast<const float2*>(p));
        r = *reinterpret_cast<const Pack<T, VEC>*>(&q);
    } else {
        r.v[0] = __ldg(p);
    }
    return r;
}
template <typename T, int VEC>
__device__ __forceinline__ void stp(T* __restrict__ p, const Pack<T, VEC>& x) {
    *reinterpret_cast<Pack<T, VEC>*>(p) = x;
}

template <typename T>
__device__ __forceinline__ T rsqrt_t(T x);
template <>
__device__ __forceinline__ float rsqrt_t<float>(float x) { return 1.0f / sqrtf(x); }
template <>
__device__ __forceinline__ double rsqrt_t<double>(double x) { return 1.0 / sqrt(x); }

// ---------------------------------------------------------------------------------------
// The per-cell arithmetic of one evaluation, shared by the three kernels (k_stage, k_stage_tma, k_batch): what differs
// between them is only where the neighbours and the slopes come from.
// ---------------------------------------------------------------------------------------
// Material part of the effective field of one cell: B0 + exchange (lap = sum over in-grid neighbours of
// (m_nb - m) (2A/Ms)/D^2, formed by the caller) + uniaxial anisotropy (2Ku/Ms)(m.k^)k^.  The RF field, the
// inter-sublattice exchange and the dipolar field are added by the caller in that order.
template <typename T>
__device__ __forceinline__ void material_field(const T mx, const T my, const T mz, const T lapx, const T lapy, const T lapz,
                                               const T B0x, const T B0y, const T B0z, const T anp, const T axx, const T axy,
                                               const T axz, T& Bx, T& By, T& Bz) {
    const T mk = mx * axx + my * axy + mz * axz;
    Bx = B0x + lapx + anp * mk * axx;
    By = B0y + lapy + anp * mk * axy;
    Bz = B0z + lapz + anp * mk * axz;
}
// LLG slope in the explicit Landau-Lifshitz form: k = llg [m x B + alpha m x (m x B)], llg = -gamma/(1+alpha^2)
template <typename T>
__device__ __forceinline__ void llg_slope(const T mx, const T my, const T mz, const T Bx, const T By, const T Bz, const T alpha,
                                          const T llg, T& kx, T& ky, T& kz) {
    const T tx = my * Bz - mz * By, ty = mz * Bx - mx * Bz, tz = mx * By - my * Bx;
    const T dx = my * tz - mz * ty, dy = mz * tx - mx * tz, dz = mx * ty - my * tx;
    kx = llg * (tx + alpha * dx);
    ky = llg * (ty + alpha * dy);
    kz = llg * (tz + alpha * dz);
}
// Stage state of tableau row ROW (0-based: the state stage ROW+1 is evaluated at; ROW = 6: the 5th-order solution b):
// m_0 + h sum_{j < ROW} a_{ROW,j} k_j with k[0..ROW-1] = k_1..k_ROW, zero coefficients (b_2) skipped.
template <int ROW, typename T>
__device__ __forceinline__ T dp_state(const T m0, const T (&k)[ROW], const T h) {
    T acc = (T)kA[ROW][0] * k[0];
#pragma unroll
    for (int j = 1; j < ROW; ++j)
        if (kA[ROW][j] != 0.0) acc += (T)kA[ROW][j] * k[j];
    return m0 + h * acc;
}
// Partial error after stage 6, h sum_{j <= 6} d_j k_j (d_2 = 0), and the full error with the 7th slope.
template <typename T>
__device__ __forceinline__ T dp_error6(const T (&k)[6], const T h) {
    T e = (T)kD[0] * k[0];
    e += (T)kD[2] * k[2];
    e += (T)kD[3] * k[3];
    e += (T)kD[4] * k[4];
    e += (T)kD[5] * k[5];
    return h * e;
}
template <typename T>
__device__ __forceinline__ T dp_error7_sq(const T e6x, const T e6y, const T e6z, const T k7x, const T k7y, const T k7z, const T h) {
    const T hd7 = h * (T)kD[6];
    const T ex = e6x + hd7 * k7x, ey = e6y + hd7 * k7y, ez = e6z + hd7 * k7z;
    const T e2 = ex * ex + ey * ey + ez * ez;
    return (e2 < (T)CUDART_INF) ? e2 : (T)CUDART_INF;      // NaN -> +inf so that max propagates it
}

// ---------------------------------------------------------------------------------------
// Step preparation (single thread): choose h for the step that starts now.
// Mirrors the controller spec in DESIGN.md: clamp onto t_end / the next trace sample.
// ---------------------------------------------------------------------------------------
__device__ __forceinline__ void prepare_h(Ctrl* c) {
    double h = c->dt;
    double target = c->t_end;
    int sample_hit = 0;
    if (c->adaptive && c->sample_dt > 0.0 && c->trace_n < c->trace_cap) {
        const double ts = c->trace_t0 + (double)(c->trace_n + 1) * c->sample_dt;
        if (ts <= target) { target = ts; sample_hit = 1; }
    }
    int clamped = 0;
    if (c->t + h * (1.0 + 1e-12) >= target) { h = target - c->t; clamped = 1; }
    c->h = h; c->target = target; c->clamped = clamped; c->sample_hit = sample_hit;
}

// a_s and the RF weights c_n = (2/gamma) Re[G_n a_s,n] for stage row `row` (0-based: row r gives
// the state of stage r+1), one thread per mode.
template <int ROW>
__device__ __forceinline__ void mode_stage_state(Ctrl* c, int n) {
    double re = 0.0, im = 0.0;
#pragma unroll
    for (int j = 0; j < ROW; ++j) {          // compile-time coefficients: no table loads on the critical path
        re += kA[ROW][j] * c->ka[j][n][0];
        im += kA[ROW][j] * c->ka[j][n][1];
    }
    const double are = c->a[n][0] + c->h * re, aim = c->a[n][1] + c->h * im;
    c->as[(ROW + 1) & 1][n][0] = are; c->as[(ROW + 1) & 1][n][1] = aim;      // the state of stage ROW+1
    c->c[n] = c->two_over_gamma * (c->Gbre[n] * are - c->Gbim[n] * aim);
}

// Mode ODE at stage `stage` for mode n (Eq. 12 / Eq. 19): ka_s = -(i w + kappa) a_s + i G S_s with S_s from the
// reduced overlap sums sred[2n], sred[2n+1]; then the amplitudes / RF weights of the next stage state (stages
// 2..5), the 5th-order candidate (stage 6) or the mode error (stage 7).  c may point to shared memory.
template <int stage>
__device__ __forceinline__ void mode_ode_stage(Ctrl* c, const int n, const double* sred, double* serr) {
    const double Sre = sred[2 * n] * c->invW[n];
    const double Sim = -sred[2 * n + 1] * c->invW[n];
    c->S[n][0] = Sre; c->S[n][1] = Sim;
    const double are = c->as[stage & 1][n][0], aim = c->as[stage & 1][n][1];
    const double Gre = c->Gre[n], Gim = c->Gim[n];
    double kre = (-c->kappa[n] * are + c->omega[n] * aim) - (Gre * Sim + Gim * Sre);
    double kim = (-c->kappa[n] * aim - c->omega[n] * are) + (Gre * Sre - Gim * Sim);
    if (c->drive_on) {          // + eta_n(t + c_s h): Gaussian pulse with carrier (Eq. 1 / Eq. 12)
        const double x = (c->t + kC[stage - 1] * c->h) - c->eta_t0[n];
        const double env = exp(-(x * x) * c->eta_i2s2[n]);
        double sn, cs;
        sincos(c->eta_wd[n] * x, &sn, &cs);
        kre += env * (c->eta_re[n] * cs + c->eta_im[n] * sn);
        kim += env * (c->eta_im[n] * cs - c->eta_re[n] * sn);
    }
    c->ka[stage - 1][n][0] = kre; c->ka[stage - 1][n][1] = kim;
    if constexpr (stage >= 2 && stage <= 5) {
        mode_stage_state<stage>(c, n);              // a_{s+1}, c^{(s+1)}
    } else if constexpr (stage == 6) {
        mode_stage_state<6>(c, n);                  // row 6 = b: the 5th-order candidate
        c->anew[n][0] = c->as[1][n][0]; c->anew[n][1] = c->as[1][n][1];
    } else if constexpr (stage == 7) {
        double ere = 0.0, eim = 0.0;
#pragma unroll
        for (int j = 0; j < 7; ++j) { ere += kD[j] * c->ka[j][n][0]; eim += kD[j] * c->ka[j][n][1]; }
        const double e = fabs(c->h) * sqrt(ere * ere + eim * eim);
        serr[n] = (e < CUDART_INF) ? e : CUDART_INF;
    }
}

// Fixed-order second reduction pass shared by stage_finish and the TMA kernels' deferred finish: warp w of nwarp
// sums components w, w + nwarp, ...; lane l adds blocks l, l+32, ... in order, then a fixed xor tree.  Two
// components per warp are in flight at a time.
__device__ __forceinline__ void reduce_block_partials(const double* partial, const int pstride, const int nsum,
                                                      const int nblk, const int warp, const int nwarp, const int lane,
                                                      double* sred) {
    for (int comp = warp; comp < nsum; comp += 2 * nwarp) {
        const int comp2 = comp + nwarp;
        const bool two = comp2 < nsum;
        const double* p1 = partial + (size_t)comp * pstride;
        const double* p2 = partial + (size_t)(two ? comp2 : comp) * pstride;
        double acc1 = 0.0, acc2 = 0.0;
        for (int b0 = lane; b0 < nblk; b0 += 32 * 8) {
            double v1[8], v2[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const bool in = b0 + 32 * j < nblk;
                v1[j] = in ? __ldcg(p1 + b0 + 32 * j) : 0.0;
                v2[j] = (in && two) ? __ldcg(p2 + b0 + 32 * j) : 0.0;
            }
#pragma unroll
            for (int j = 0; j < 8; ++j) { acc1 += v1[j]; acc2 += v2[j]; }
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            acc1 += __shfl_xor_sync(0xffffffffu, acc1, o);
            acc2 += __shfl_xor_sync(0xffffffffu, acc2, o);
        }
        if (lane == 0) { sred[comp] = acc1; if (two) sred[comp2] = acc2; }
    }
}

// On-device spectroscopy: at a trace sample (time t, amplitudes a_n, overlaps S_n,
// sublattice means <m_s>) every bin k adds x exp(+i w_k t) for the 2N + n_sub signals x = a_1..a_N, S_1..S_N and
// mu_s = <m_s,x> - i <m_s,y> (the paper's m^- of the plain average; (mu_1 - mu_2)/2 is the Neel vector's).
// Thread k owns bin k, k + nthr, ...: no two threads touch the same accumulator, and successive samples are ordered by
// the kernel's own barriers.
__device__ __forceinline__ void dft_accumulate(double* spec, const int K, const double w0, const double dw, const int N,
                                               const double t, const double (*a)[2], const double (*S)[2],
                                               const double* mavg, const int nsub, const int tid, const int nthr) {
    const int nsig = 2 * N + nsub;
    for (int k = tid; k < K; k += nthr) {
        double sn, cs;
        sincos((w0 + (double)k * dw) * t, &sn, &cs);
        double* X = spec + (size_t)k * 2 * nsig;
        for (int sig = 0; sig < nsig; ++sig) {
            double xr, xi;
            if (sig < N) { xr = a[sig][0]; xi = a[sig][1]; }
            else if (sig < 2 * N) { xr = S[sig - N][0]; xi = S[sig - N][1]; }
            else { xr = mavg[3 * (sig - 2 * N)]; xi = -mavg[3 * (sig - 2 * N) + 1]; }
            X[2 * sig] += xr * cs - xi * sn;
            X[2 * sig + 1] += xr * sn + xi * cs;
        }
    }
}

// max over the blocks' error maxima (one warp; the max is order-independent)
__device__ __forceinline__ double reduce_block_max(const double* partial_max, const int nblk, const int lane) {
    double mx = 0.0;
    for (int b0 = lane; b0 < nblk; b0 += 32 * 8) {
        double v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = (b0 + 32 * j < nblk) ? __ldcg(partial_max + b0 + 32 * j) : 0.0;
#pragma unroll
        for (int j = 0; j < 8; ++j) mx = fmax(mx, v[j]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) mx = fmax(mx, __shfl_xor_sync(0xffffffffu, mx, o));
    return mx;
}

__device__ __forceinline__ double fifth_root(double r);

// The step controller (a7), one thread, on a Ctrl in shared memory: error norm = max(cells, modes), accept / reject,
// dt proposal fac = clamp(0.8 (tol/err)^(1/5), 0.5, 2), time, FSAL buffer rotation, statistics, trace sampling.
// smax = max_r |e(r)|^2, serr[n] = |e_a,n|, sred[2N + i] = sum_r m_s,i(r) of the candidate.  `trace` is the device
// trace buffer (nullptr: none); rows are stored only when write_rows (every caller counts them).  Returns accept.
__device__ __forceinline__ int controller_step(Ctrl* c, const double smax, const double* serr, const double* sred, const int N,
                                               const int nsub, const double inv_nc, double* trace, const bool write_rows) {
    double err = sqrt(smax);
    for (int n = 0; n < N; ++n) err = fmax(err, serr[n]);
    const bool finite = err < CUDART_INF;
    const double h = c->h;
    bool accept;
    if (c->adaptive) accept = finite && err <= c->tol;
    else { accept = true; if (!finite) { accept = false; c->status = -5; } }
    double fac;
    if (!finite) fac = 0.5;
    else if (err == 0.0) fac = 2.0;
    else { fac = 0.8 * fifth_root(fmin(fmax(c->tol / err, 1e-2), 1e3)); fac = fmin(fmax(fac, 0.5), 2.0); }
    c->rhs_evals++;
    c->steps_run++;
    c->last_err = err;
    c->took = 0;
    if (accept) {
        c->t = c->clamped ? c->target : c->t + h;
        c->ycur ^= 1;
        c->k1slot = 6 - c->k1slot;
        c->accepted++;
        c->dt_min = fmin(c->dt_min, h);
        c->dt_max = fmax(c->dt_max, h);
        if (c->adaptive) { const double prop = h * fac; c->dt = c->clamped ? fmax(prop, c->dt) : prop; }
        for (int i = 0; i < 3 * nsub; ++i) c->mavg[i] = sred[2 * N + i] * inv_nc;
        const bool take = trace != nullptr && c->sample_dt > 0.0 && c->trace_n < c->trace_cap &&
                          (c->adaptive ? (c->clamped && c->sample_hit)
                                       : ((c->accepted - c->trace_acc0) % c->trace_stride == 0));
        if (take) {
            if (write_rows) {
                double* row = trace + (size_t)c->trace_n * (1 + 4 * N + 3 * nsub);
                row[0] = c->t;
                for (int n = 0; n < N; ++n) {
                    row[1 + 2 * n] = c->anew[n][0]; row[2 + 2 * n] = c->anew[n][1];
                    row[1 + 2 * N + 2 * n] = c->S[n][0]; row[2 + 2 * N + 2 * n] = c->S[n][1];
                }
                for (int i = 0; i < 3 * nsub; ++i) row[1 + 4 * N + i] = c->mavg[i];
            }
            c->trace_n++;
            c->took = 1;
            if (c->spec_K > 0) c->spec_n++;
        }
    } else if (c->status == 0) {
        c->rejected++;
        c->dt = h * fac;
    }
    if (c->adaptive && !(c->dt > 1e-20)) c->status = -6;
    return accept ? 1 : 0;
}

// ---------------------------------------------------------------------------------------
// Tail of every stage kernel, executed by the last block to arrive: deterministic second
// reduction pass, mode ODEs + stage algebra, and (stage 7) the accept/reject controller.
//
// Everything here sits on the critical path between two stage kernels, so global-memory round
// trips are what it costs: the whole Ctrl struct and all block partials are fetched with one
// batch of independent loads, the arithmetic runs on a shared-memory copy of Ctrl, and the copy
// is written back with one batch of coalesced stores.
// ---------------------------------------------------------------------------------------
constexpr int kCtrlWords = (int)(sizeof(Ctrl) / 8);
static_assert(sizeof(Ctrl) % 8 == 0, "Ctrl is copied as 8-byte words");
constexpr int kCtrlWordsPerThread = (kCtrlWords + kBlock - 1) / kBlock;     // stage_finish, 128-thread blocks

// r^(1/5) for r in [1e-2, 1e3]: float seed + one Newton step in fp64 (relative error < 1e-13).  A libm pow()
// in fp64 costs several microseconds of single-thread latency on this part, all of it between two stage kernels.
__device__ __forceinline__ double fifth_root(double r) {
    const double y = (double)powf((float)r, 0.2f);
    const double y2 = y * y;
    return y * (4.0 + r / (y2 * y2 * y)) * 0.2;
}

// The arguments stage_finish needs, by value (a reference to the kernel's StageArgs would sit in local memory
// and cost one more dependent memory round trip before the first load can issue).
struct FinishArgs {
    Ctrl* ctrl;
    Ctrl* ctrl0;             // step-boundary copy (nullptr: none), kept equal to ctrl by every single-block finish
    double* spec;            // Fourier sums [spec_K][2N][2] or nullptr
    const double* partial;
    const double* partial_max;
    unsigned long long cond_handle;
    double inv_nc;
    int pstride;
#ifdef CAVMAG_PROBE
    unsigned long long* probe;
#endif
};
// Block partial sums are double-buffered by stage parity: stage s writes buffer s & 1 and whoever finishes stage s
// (the last block of kernel s, or every block of kernel s+1 in its prologue) reads that buffer.  A block of kernel
// s+1 that starts late (SMs shared with other work) therefore never sees the stage-(s+1) sums another block of
// the same kernel has already written.
__device__ __forceinline__ double* stage_partials(const StageArgs& S, const int stage) {
    return S.partial + (size_t)(stage & 1) * (size_t)kMaxSums * (size_t)S.pstride;
}
__device__ __forceinline__ FinishArgs finish_args(const StageArgs& S, const int stage) {
    FinishArgs F;
    F.ctrl = S.ctrl; F.ctrl0 = S.ctrl0; F.spec = S.spec; F.partial = stage_partials(S, stage); F.partial_max = S.partial_max; F.cond_handle = S.cond_handle;
    F.inv_nc = S.inv_nc; F.pstride = S.pstride;
#ifdef CAVMAG_PROBE
    F.probe = S.probe;
#endif
    return F;
}

template <int stage>
static __device__ __noinline__ void stage_finish(const FinishArgs A, const int nsub, const int N, double* trace) {
    __shared__ __align__(16) unsigned long long sc_words[kCtrlWords];
    __shared__ double sred[kMaxSums];
    __shared__ double smax;
    __shared__ double serr[kMaxModes];
    __shared__ int s_accept;
    Ctrl* const c = reinterpret_cast<Ctrl*>(sc_words);          // shared-memory working copy
    unsigned long long* const gcw = reinterpret_cast<unsigned long long*>(A.ctrl);
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nthr = blockDim.x;
    const int nwarp = nthr >> 5;            // 4 (generic kernel) or 9 (TMA kernel)
    const int nblk = gridDim.x;
    const int nsum = 2 * N + (stage == 7 ? 3 * nsub : 0);
    CAVMAG_MARKF(8);
    // Ctrl -> registers (consumed after the partial sums so that all loads are in flight together)
    unsigned long long cw[kCtrlWordsPerThread];
#pragma unroll
    for (int k = 0; k < kCtrlWordsPerThread; ++k) {
        const int idx = tid + k * nthr;
        cw[k] = idx < kCtrlWords ? __ldcg(gcw + idx) : 0ull;
    }
    reduce_block_partials(A.partial, A.pstride, nsum, nblk, warp, nwarp, lane, sred);
    if (stage == 7 && warp == nwarp - 1) {
        const double mx = reduce_block_max(A.partial_max, nblk, lane);
        if (lane == 0) smax = mx;
    }
#pragma unroll
    for (int k = 0; k < kCtrlWordsPerThread; ++k) {
        const int idx = tid + k * nthr;
        if (idx < kCtrlWords) sc_words[idx] = cw[k];
    }
    __syncthreads();
    CAVMAG_MARKF(9);

    if (tid < N) mode_ode_stage<stage>(c, tid, sred, serr);
    bool set_cond = false;
    if (stage >= 2 && stage <= 6) {
        if (tid == 0) { c->rhs_evals++; c->arrive = 0u; }
    } else {
        __syncthreads();
        if (stage == 7) {
            if (tid == 0) s_accept = controller_step(c, smax, serr, sred, N, nsub, A.inv_nc, trace, true);
            __syncthreads();
            if (A.spec != nullptr && c->spec_K > 0 && c->took)       // Fourier sums of this trace sample
                dft_accumulate(A.spec, c->spec_K, c->spec_w0, c->spec_dw, N, c->t, c->anew, c->S, c->mavg, nsub, tid, nthr);
            if (tid < N && s_accept) {     // y := y_new (modes), FSAL: ka_1 := ka_7
                c->a[tid][0] = c->anew[tid][0]; c->a[tid][1] = c->anew[tid][1];
                c->ka[0][tid][0] = c->ka[6][tid][0]; c->ka[0][tid][1] = c->ka[6][tid][1];
            }
            __syncthreads();
        } else {   // stage 1: k1 of a fresh state
            if (tid == 0) { c->rhs_evals++; c->k1_valid = 1; }
        }

        // start of the next step
        if (tid == 0) {
            const bool done = !(c->t < c->t_end) || (c->max_steps > 0 && c->steps_run >= c->max_steps) || c->status != 0;
            c->done = done ? 1 : 0;
            prepare_h(c);
        }
        __syncthreads();
        if (tid < N) mode_stage_state<1>(c, tid);           // a_2 = a_0 + h a21 ka_1
        if (tid == 0) { c->arrive = 0u; c->pend7 = 0; set_cond = (A.cond_handle != 0ull && stage == 7); }
    }
    // write the working copy back
    __syncthreads();
    CAVMAG_MARKF(10);
    for (int idx = tid; idx < kCtrlWords; idx += nthr) gcw[idx] = sc_words[idx];
    if (A.ctrl0 != nullptr && (stage == 1 || stage == 7)) {      // the TMA stage-2 kernel starts from the boundary copy
        unsigned long long* const g0 = reinterpret_cast<unsigned long long*>(A.ctrl0);
        for (int idx = tid; idx < kCtrlWords; idx += nthr) g0[idx] = sc_words[idx];
    }
    CAVMAG_MARKF(11);
    if (set_cond) cudaGraphSetConditional((cudaGraphConditionalHandle)A.cond_handle, c->done ? 0u : 1u);
    CAVMAG_MARKF(12);
}

// ---------------------------------------------------------------------------------------
// the stage kernel
// ---------------------------------------------------------------------------------------
// VARIANT: 0 = the paper's field; 1 = + dipolar field (A.bdem, demag.cuh); 2 = per-mode polarisation (A.pol, reading G32).
// Separate instantiations: as runtime branches the extra loads cost the plain kernels registers (6 % on CFG3).
template <typename T, int VEC, int STAGE, int NSUB, int NB, int VARIANT = 0>
__global__ void __launch_bounds__(kBlock) k_stage(const StageArgs A, double* __restrict__ trace) {
    constexpr bool POL = VARIANT == 2;
    using P = Pack<T, VEC>;
    Ctrl* ctrl = A.ctrl;
    if (STAGE == 1) { if (ctrl->k1_valid) return; }
    else if (ctrl->done) return;

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = ctrl->N;
    const T h = (T)ctrl->h;
    const int ycur = ctrl->ycur, k1slot = ctrl->k1slot;
    const long long nc = A.nc;
    const int nx = A.nx, ny = A.ny, nz = A.nz;
    const long long plane = (long long)nx * ny;

    const T* __restrict__ y0 = (const T*)(ycur ? A.Y[1] : A.Y[0]);
    T* __restrict__ ynew = (T*)(ycur ? A.Y[0] : A.Y[1]);
    const T* __restrict__ k1 = (const T*)(k1slot ? A.K[6] : A.K[0]);
    const T* __restrict__ uu = (const T*)A.u;
    // stage input (materialised) and outputs
    const T* __restrict__ ms = STAGE == 1 ? y0 : STAGE == 7 ? (const T*)ynew
                              : (STAGE == 3 || STAGE == 5) ? (const T*)A.MS[0] : (const T*)A.MS[1];
    T* __restrict__ kout = STAGE == 1 ? (T*)(k1slot ? A.K[6] : A.K[0]) : STAGE == 7 ? (T*)(k1slot ? A.K[0] : A.K[6]) : (T*)A.K[STAGE - 1];
    T* __restrict__ mnext = STAGE == 6 ? ynew : (STAGE == 2 || STAGE == 4) ? (T*)A.MS[0] : (T*)A.MS[1];
    T* __restrict__ e6 = (T*)A.MS[0];    // written by stage 6, read by stage 7

    const T ha21 = h * (T)kA[1][0];
    const T B0x = (T)A.B0[0], B0y = (T)A.B0[1], B0z = (T)A.B0[2];
    const T wx = (T)A.ex_wx, wy = (T)A.ex_wy, wz = (T)A.ex_wz;
    const T anp = (T)A.an_pref, axx = (T)A.axis[0], axy = (T)A.axis[1], axz = (T)A.axis[2];
    const T alpha = (T)A.alpha, llg = (T)A.llg, BE = (T)A.B_exch_inter;

    T cn[NB > 0 ? NB : 1];
#pragma unroll
    for (int n = 0; n < NB; ++n) cn[n] = (n < N) ? (T)ctrl->c[n] : (T)0;

    // per-thread running sums
    T ox[NB > 0 ? NB : 1], oy[NB > 0 ? NB : 1];
#pragma unroll
    for (int n = 0; n < NB; ++n) { ox[n] = (T)0; oy[n] = (T)0; }
    T sm[NSUB * 3];
#pragma unroll
    for (int i = 0; i < NSUB * 3; ++i) sm[i] = (T)0;
    T emax2 = (T)0;

    const long long nblk = gridDim.x;
    const long long blk = (A.serpentine && (STAGE & 1)) ? (nblk - 1 - blockIdx.x) : blockIdx.x;
    const long long vbase = blk * (long long)A.iters * kBlock;

    for (int it = 0; it < A.iters; ++it) {
        const long long vraw = vbase + (long long)it * kBlock + tid;
        const bool active = vraw < A.nvec;
        const long long cell = (active ? vraw : (A.nvec - 1)) * VEC;
        const int z = (int)(cell / plane);
        const int rem = (int)(cell - (long long)z * plane);
        const int y = rem / nx;
        const int x0 = rem - y * nx;
        const long long iym = (y > 0) ? cell - nx : cell, iyp = (y < ny - 1) ? cell + nx : cell;
        const long long izm = (z > 0) ? cell - plane : cell, izp = (z < nz - 1) ? cell + plane : cell;
        const bool has_l = x0 > 0, has_r = x0 + VEC < nx;

        // ---- stage state at the centre (all sublattices) ----
        P mc[NSUB][3], y0c[NSUB][3], k1c[NSUB][3];
#pragma unroll
        for (int s = 0; s < NSUB; ++s)
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const long long off = (long long)(s * 3 + c) * nc + cell;
                if constexpr (STAGE == 2) {
                    y0c[s][c] = ldp<T, VEC>(y0 + off);
                    k1c[s][c] = ldp<T, VEC>(k1 + off);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) mc[s][c].v[v] = y0c[s][c].v[v] + ha21 * k1c[s][c].v[v];
                } else {
                    mc[s][c] = ldp<T, VEC>(ms + off);
                }
            }

        // ---- mode profiles: RF field weight and overlap partials of THIS stage state ----
        T brf[VEC], brfy[POL ? VEC : 1], brfz[POL ? VEC : 1];
#pragma unroll
        for (int v = 0; v < VEC; ++v) { brf[v] = (T)0; if constexpr (POL) { brfy[v] = (T)0; brfz[v] = (T)0; } }
        if constexpr (NB > 0) {
            T mcx[VEC], mcy[VEC], mcz[POL ? VEC : 1];
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                if constexpr (NSUB == 1) { mcx[v] = mc[0][0].v[v]; mcy[v] = mc[0][1].v[v]; if constexpr (POL) mcz[v] = mc[0][2].v[v]; }
                else {
                    mcx[v] = (T)0.5 * (mc[0][0].v[v] + mc[1][0].v[v]); mcy[v] = (T)0.5 * (mc[0][1].v[v] + mc[1][1].v[v]);
                    if constexpr (POL) mcz[v] = (T)0.5 * (mc[0][2].v[v] + mc[1][2].v[v]);
                }
            }
#pragma unroll
            for (int n = 0; n < NB; ++n) {
                if (n < N) {
                    P un = ldp<T, VEC>(uu + (long long)n * nc + cell);
                    T sx = (T)0, sy = (T)0;
                    if constexpr (!POL) {                  // p = x^, q = y^
#pragma unroll
                        for (int v = 0; v < VEC; ++v) {
                            brf[v] += cn[n] * un.v[v];
                            sx += un.v[v] * mcx[v];
                            sy += un.v[v] * mcy[v];
                        }
                    } else {                               // field along p_n, coupling to m.p_n - i m.q_n (reading G32)
                        const double* pq = A.pol + 6 * n;
                        const double cd = ctrl->c[n];
                        const T cp0 = (T)(cd * pq[0]), cp1 = (T)(cd * pq[1]), cp2 = (T)(cd * pq[2]);
                        const T p0 = (T)pq[0], p1 = (T)pq[1], p2 = (T)pq[2], q0 = (T)pq[3], q1 = (T)pq[4], q2 = (T)pq[5];
#pragma unroll
                        for (int v = 0; v < VEC; ++v) {
                            brf[v] += cp0 * un.v[v]; brfy[v] += cp1 * un.v[v]; brfz[v] += cp2 * un.v[v];
                            sx += un.v[v] * (mcx[v] * p0 + mcy[v] * p1 + mcz[v] * p2);
                            sy += un.v[v] * (mcx[v] * q0 + mcy[v] * q1 + mcz[v] * q2);
                        }
                    }
                    if (active) { ox[n] += sx; oy[n] += sy; }
                }
            }
        }

        // ---- optional dipolar field (off in the paper): computed before this launch by
        //      an FFT convolution of this stage's state (demag.cuh), the same for both sublattices ----
        P bdv[3];                                   // (its own instantiation: a runtime branch costs the others registers)
        constexpr bool has_bd = VARIANT == 1;
        if constexpr (has_bd) {
#pragma unroll
            for (int c = 0; c < 3; ++c) bdv[c] = ldp<T, VEC>((const T*)A.bdem + (long long)c * nc + cell);
        }

#pragma unroll
        for (int s = 0; s < NSUB; ++s) {
            // ---- 6-neighbour exchange: sum over in-grid neighbours of (m_nb - m)/D^2 ----
            T lap[3][VEC];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const long long base = (long long)(s * 3 + c) * nc;
                P nym, nyp, nzm, nzp;
                T xl, xr;
                if constexpr (STAGE == 2) {
                    const P a0 = ldp<T, VEC>(y0 + base + iym), b0 = ldp<T, VEC>(k1 + base + iym);
                    const P a1 = ldp<T, VEC>(y0 + base + iyp), b1 = ldp<T, VEC>(k1 + base + iyp);
                    const P a2 = ldp<T, VEC>(y0 + base + izm), b2 = ldp<T, VEC>(k1 + base + izm);
                    const P a3 = ldp<T, VEC>(y0 + base + izp), b3 = ldp<T, VEC>(k1 + base + izp);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        nym.v[v] = a0.v[v] + ha21 * b0.v[v]; nyp.v[v] = a1.v[v] + ha21 * b1.v[v];
                        nzm.v[v] = a2.v[v] + ha21 * b2.v[v]; nzp.v[v] = a3.v[v] + ha21 * b3.v[v];
                    }
                } else {
                    nym = ldp<T, VEC>(ms + base + iym); nyp = ldp<T, VEC>(ms + base + iyp);
                    nzm = ldp<T, VEC>(ms + base + izm); nzp = ldp<T, VEC>(ms + base + izp);
                }
                xl = __shfl_up_sync(0xffffffffu, mc[s][c].v[VEC - 1], 1);
                xr = __shfl_down_sync(0xffffffffu, mc[s][c].v[0], 1);
                // the two edge lanes of the warp fetch their x neighbour from memory: predicated loads, no divergent branch
                const bool need_l = has_l && lane == 0, need_r = has_r && lane == 31;
                T gl, gr;
                if constexpr (STAGE == 2) {
                    const T a0 = need_l ? __ldg(y0 + base + cell - 1) : (T)0, b0 = need_l ? __ldg(k1 + base + cell - 1) : (T)0;
                    const T a1 = need_r ? __ldg(y0 + base + cell + VEC) : (T)0, b1 = need_r ? __ldg(k1 + base + cell + VEC) : (T)0;
                    gl = a0 + ha21 * b0; gr = a1 + ha21 * b1;
                } else {
                    gl = need_l ? __ldg(ms + base + cell - 1) : (T)0;
                    gr = need_r ? __ldg(ms + base + cell + VEC) : (T)0;
                }
                xl = !has_l ? mc[s][c].v[0] : (need_l ? gl : xl);
                xr = !has_r ? mc[s][c].v[VEC - 1] : (need_r ? gr : xr);
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    const T m0 = mc[s][c].v[v];
                    const T left = (v == 0) ? xl : mc[s][c].v[v > 0 ? v - 1 : 0];
                    const T right = (v == VEC - 1) ? xr : mc[s][c].v[v < VEC - 1 ? v + 1 : VEC - 1];
                    T l = (left - m0) * wx;
                    l += (right - m0) * wx;
                    l += (nym.v[v] - m0) * wy;
                    l += (nyp.v[v] - m0) * wy;
                    l += (nzm.v[v] - m0) * wz;
                    l += (nzp.v[v] - m0) * wz;
                    lap[c][v] = l;
                }
            }

            // ---- effective field and LLG slope ----
            P ks[3];
#pragma unroll
            for (int v = 0; v < VEC; ++v) {
                const T mx = mc[s][0].v[v], my = mc[s][1].v[v], mz = mc[s][2].v[v];
                T Bx, By, Bz;
                material_field(mx, my, mz, lap[0][v], lap[1][v], lap[2][v], B0x, B0y, B0z, anp, axx, axy, axz, Bx, By, Bz);
                Bx += brf[v];
                if constexpr (POL) { By += brfy[v]; Bz += brfz[v]; }
                if constexpr (NSUB == 2) {
                    Bx -= BE * mc[1 - s][0].v[v]; By -= BE * mc[1 - s][1].v[v]; Bz -= BE * mc[1 - s][2].v[v];
                }
                if constexpr (has_bd) { Bx += bdv[0].v[v]; By += bdv[1].v[v]; Bz += bdv[2].v[v]; }
                llg_slope(mx, my, mz, Bx, By, Bz, alpha, llg, ks[0].v[v], ks[1].v[v], ks[2].v[v]);
            }

            // ---- store k_s, then the fused tail: next stage state / candidate / error ----
            if constexpr (STAGE >= 1 && STAGE <= 7) {
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    if (active) stp<T, VEC>(kout + (long long)(s * 3 + c) * nc + cell, ks[c]);
            }
            if constexpr (STAGE >= 2 && STAGE <= 5) {
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const long long off = (long long)(s * 3 + c) * nc + cell;
                    P m0v, q[STAGE];                   // k_1 .. k_STAGE of this component
                    if constexpr (STAGE == 2) {
                        m0v = y0c[s][c];
                        q[0] = k1c[s][c];
                    } else {
                        m0v = ldp<T, VEC>(y0 + off);
                        q[0] = ldp<T, VEC>(k1 + off);
#pragma unroll
                        for (int j = 1; j < STAGE - 1; ++j) q[j] = ldp<T, VEC>((const T*)A.K[j] + off);
                    }
                    q[STAGE - 1] = ks[c];
                    P out;
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        T kv[STAGE];
#pragma unroll
                        for (int j = 0; j < STAGE; ++j) kv[j] = q[j].v[v];
                        out.v[v] = dp_state<STAGE>(m0v.v[v], kv, h);
                    }
                    if (active) stp<T, VEC>(mnext + off, out);
                }
            }
            if constexpr (STAGE == 6) {
                P y5[3], er[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const long long off = (long long)(s * 3 + c) * nc + cell;
                    const P m0v = ldp<T, VEC>(y0 + off);
                    const P q1 = ldp<T, VEC>(k1 + off);
                    const P q3 = ldp<T, VEC>((const T*)A.K[2] + off);
                    const P q4 = ldp<T, VEC>((const T*)A.K[3] + off);
                    const P q5 = ldp<T, VEC>((const T*)A.K[4] + off);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const T kv[6] = {q1.v[v], (T)0, q3.v[v], q4.v[v], q5.v[v], ks[c].v[v]};      // b_2 = d_2 = 0: k_2 is not read
                        y5[c].v[v] = dp_state<6>(m0v.v[v], kv, h);
                        er[c].v[v] = dp_error6(kv, h);
                    }
                }
                if (A.renormalize) {
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const T inv = rsqrt_t<T>(y5[0].v[v] * y5[0].v[v] + y5[1].v[v] * y5[1].v[v] + y5[2].v[v] * y5[2].v[v]);
                        y5[0].v[v] *= inv; y5[1].v[v] *= inv; y5[2].v[v] *= inv;
                    }
                }
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const long long off = (long long)(s * 3 + c) * nc + cell;
                    if (active) { stp<T, VEC>(mnext + off, y5[c]); stp<T, VEC>(e6 + off, er[c]); }
                }
            }
            if constexpr (STAGE == 7) {
                P er[3];
#pragma unroll
                for (int c = 0; c < 3; ++c) er[c] = ldp<T, VEC>(e6 + (long long)(s * 3 + c) * nc + cell);
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    const T e2 = dp_error7_sq(er[0].v[v], er[1].v[v], er[2].v[v], ks[0].v[v], ks[1].v[v], ks[2].v[v], h);
                    if (active) {
                        emax2 = fmax(emax2, e2);
                        sm[s * 3 + 0] += mc[s][0].v[v]; sm[s * 3 + 1] += mc[s][1].v[v]; sm[s * 3 + 2] += mc[s][2].v[v];
                    }
                }
            }
        }
    }

    // ---- pass 1 of the reductions: warp shuffle tree, then fixed-order sum over the block's warps ----
    constexpr int nwarp = kBlock / 32;
    constexpr int NS = 2 * NB + (STAGE == 7 ? 3 * NSUB : 0);
    __shared__ double swarp[nwarp][NS > 0 ? NS : 1];
    __shared__ double swmax[nwarp];
    __shared__ int s_last;
    {
        T vals[NS > 0 ? NS : 1];
#pragma unroll
        for (int n = 0; n < NB; ++n) { vals[2 * n] = ox[n]; vals[2 * n + 1] = oy[n]; }
        if constexpr (STAGE == 7) {
#pragma unroll
            for (int i = 0; i < 3 * NSUB; ++i) vals[2 * NB + i] = sm[i];
        }
#pragma unroll
        for (int i = 0; i < NS; ++i) {
            const bool used = (i < 2 * NB) ? (i < 2 * N) : true;
            if (used) {
                T x = vals[i];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
                if (lane == 0) swarp[warp][i] = (double)x;
            }
        }
        if constexpr (STAGE == 7) {
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) emax2 = fmax(emax2, __shfl_xor_sync(0xffffffffu, emax2, o));
            if (lane == 0) swmax[warp] = (double)emax2;
        }
    }
    __syncthreads();
    if (tid < NS) {
        const int i = tid;
        const bool used = (i < 2 * NB) ? (i < 2 * N) : true;
        if (used) {
            double acc = 0.0;
#pragma unroll
            for (int w = 0; w < nwarp; ++w) acc += swarp[w][i];
            const int comp = (i < 2 * NB) ? i : (2 * N + (i - 2 * NB));
            stage_partials(A, STAGE)[(size_t)comp * A.pstride + blockIdx.x] = acc;
        }
    }
    if (STAGE == 7 && tid == 0) {
        double mx = 0.0;
#pragma unroll
        for (int w = 0; w < nwarp; ++w) mx = fmax(mx, swmax[w]);
        A.partial_max[blockIdx.x] = mx;
    }
    // One fence per block: the barrier orders every thread's stores before thread 0's gpu-scope fence (release),
    // the last block's thread 0 fences again after the ticket (acquire) before the barrier that lets its
    // threads read the other blocks' partials.
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        const unsigned int old = atomicAdd(&ctrl->arrive, 1u);
        s_last = (old == gridDim.x - 1) ? 1 : 0;
        if (s_last) __threadfence();
    }
    __syncthreads();
    if (s_last) stage_finish<STAGE>(finish_args(A, STAGE), NSUB, N, trace);
}

// Kernel lookup, one translation unit per (T, NSUB): returns the device function for
// cudaLaunchKernel / cudaGraphAddKernelNode.  vec: 1 = vectorised (16 B), 0 = scalar.
const void* stage_kernel_f32_fm(int vec, int stage, int nb);
const void* stage_kernel_f32_afm(int vec, int stage, int nb);
const void* stage_kernel_f64_fm(int vec, int stage, int nb);
const void* stage_kernel_f64_afm(int vec, int stage, int nb);
// the same with the dipolar field added (k_stage<..., DEMAG = true>; demag.cuh)
const void* stage_kernel_demag_f32_fm(int vec, int stage, int nb);
const void* stage_kernel_demag_f32_afm(int vec, int stage, int nb);
const void* stage_kernel_demag_f64_fm(int vec, int stage, int nb);
const void* stage_kernel_demag_f64_afm(int vec, int stage, int nb);
// and with per-mode polarisation (k_stage<..., VARIANT = 2>)
const void* stage_kernel_pol_f32_fm(int vec, int stage, int nb);
const void* stage_kernel_pol_f32_afm(int vec, int stage, int nb);
const void* stage_kernel_pol_f64_fm(int vec, int stage, int nb);
const void* stage_kernel_pol_f64_afm(int vec, int stage, int nb);

#define CAVMAG_STAGE_CASES(T, VEC, NSUB, NB)                                       \
    switch (stage) {                                                               \
        case 1: return (const void*)k_stage<T, VEC, 1, NSUB, NB, CAVMAG_VARIANT_INST>; \
        case 2: return (const void*)k_stage<T, VEC, 2, NSUB, NB, CAVMAG_VARIANT_INST>; \
        case 3: return (const void*)k_stage<T, VEC, 3, NSUB, NB, CAVMAG_VARIANT_INST>; \
        case 4: return (const void*)k_stage<T, VEC, 4, NSUB, NB, CAVMAG_VARIANT_INST>; \
        case 5: return (const void*)k_stage<T, VEC, 5, NSUB, NB, CAVMAG_VARIANT_INST>; \
        case 6: return (const void*)k_stage<T, VEC, 6, NSUB, NB, CAVMAG_VARIANT_INST>; \
        case 7: return (const void*)k_stage<T, VEC, 7, NSUB, NB, CAVMAG_VARIANT_INST>; \
        default: return nullptr;                                                   \
    }
#ifndef CAVMAG_VARIANT_INST
#define CAVMAG_VARIANT_INST 0        // translation units that instantiate the dipolar-field / polarisation variants define it to 1 / 2
#endif

#define CAVMAG_DEFINE_LOOKUP(NAME, T, VECW, NSUB)                                  \
    const void* NAME(int vec, int stage, int nb) {                                 \
        if (vec) {                                                                 \
            if (nb == 0) { CAVMAG_STAGE_CASES(T, VECW, NSUB, 0) }                  \
            if (nb == 1) { CAVMAG_STAGE_CASES(T, VECW, NSUB, 1) }                  \
            if (nb == 2) { CAVMAG_STAGE_CASES(T, VECW, NSUB, 2) }                  \
            if (nb == 8) { CAVMAG_STAGE_CASES(T, VECW, NSUB, 8) }                  \
            if (nb == 32) { CAVMAG_STAGE_CASES(T, VECW, NSUB, 32) }                \
        } else {                                                                   \
            if (nb == 0) { CAVMAG_STAGE_CASES(T, 1, NSUB, 0) }                     \
            if (nb == 1) { CAVMAG_STAGE_CASES(T, 1, NSUB, 1) }                     \
            if (nb == 2) { CAVMAG_STAGE_CASES(T, 1, NSUB, 2) }                     \
            if (nb == 8) { CAVMAG_STAGE_CASES(T, 1, NSUB, 8) }                     \
            if (nb == 32) { CAVMAG_STAGE_CASES(T, 1, NSUB, 32) }                   \
        }                                                                          \
        return nullptr;                                                            \
    }

}  // namespace cavmag
