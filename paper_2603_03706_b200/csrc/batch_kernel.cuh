// Batched small-grid integrator (SURVEY.md 8(f1); PAPER.md:217, :229, :335 - the paper's sweeps of a tiny grid).
//
// One thread block per replica, one thread per cell.  The whole adaptive Dormand-Prince loop of the coupled
// LLG + cavity-mode system runs inside the kernel:
//   * the stage state m_s lives in shared memory (neighbours of the 6-point exchange stencil are shared-memory
//     reads), y, k1..k7 and the candidate of a thread's own cell live in registers;
//   * per evaluation: publish m_s, barrier, [field + LLG slope of the own cell] and [warp-shuffle partial sums of
//     u_n m_c^-], barrier, thread n finishes S_n, the mode ODE ka_s (Eq. 12 / Eq. 19) and the amplitudes / RF
//     weights of the next stage state -> 2 block barriers per evaluation, no global memory, no kernel launch;
//   * error norm, accept/reject, dt control, FSAL and trace sampling as in stage_finish<7> (same formulas, same
//     constants: DESIGN.md readings G11-G13).
// Same arithmetic per cell as k_stage (subtract-first exchange stencil, explicit Landau-Lifshitz form), so a
// replica agrees with cav_run on the same inputs to rounding; the overlap sums are added in a different (fixed)
// order.  Mode amplitudes, overlap sums and the controller are fp64 in both precisions.
//
// The same kernel also serves cav_run: with one replica for grids of up to 1024 cells (CAV_PATH_BLOCK), and as a
// cooperative launch over several co-resident blocks for grids of up to 512 cells per SM (CAV_PATH_COOP, template flag
// COOP: stage state and block partial sums through global memory, a grid barrier per evaluation).
#pragma once
#include <type_traits>

#include "stage_kernel.cuh"

namespace cavmag {

constexpr int kBatchMaxCells = 1024;

struct BatchCtl {                 // per replica, persistent across cav_batch_run calls
    double t, dt;
    double dt_min, dt_max, last_err;
    long long accepted, rejected, rhs_evals, trace_acc0;
    int status, trace_n;
};

struct BatchArgs {
    int nx, ny, nz, nc, N, n_rep;
    double ex_wx, ex_wy, ex_wz, an_pref, axis[3], alpha, llg, B_exch_inter, two_over_gamma, inv_nc;
    int renormalize;
    const double* B0;             // [n_rep][3]
    const void* u;                // [N][nc] T
    const double* modep;          // [n_rep or 1][7][N]: omega, kappa, Gre, Gim, invW, Gbre, Gbim
    int modep_per_rep;
    void* m;                      // [n_rep][NSUB][3][nc] T, in/out
    double* a;                    // [n_rep][N][2], in/out
    BatchCtl* ctl;                // [n_rep]
    double t_end, tol, fixed_dt, dt_init;
    long long max_steps;
    double sample_dt, trace_t0;
    int trace_cap, row_len;
    double* trace;                // [n_rep][trace_cap][row_len]
    int u_in_smem;                // profiles staged in dynamic shared memory
    const double* drive;          // [5][N]: eta_re, eta_im, t0, 1/(2 sigma^2), omega_d (common to all replicas) or NULL
    // cooperative variant (COOP: one simulation spread over nblk co-resident blocks, grid barriers between the phases)
    void* gms[2];                 // [NSUB][3][nc] T: stage state in global memory, double-buffered by evaluation parity
    double* cpart[2];             // [2N + 3 NSUB][nblk] block partial sums, double-buffered
    double* cmax[2];              // [nblk] block maxima of |e|^2, double-buffered by step parity
    unsigned long long* bar;      // grid-barrier counter (zeroed before the launch)
    int nblk;
    // SURVEY.md 8(f3) / 8(f2b) variants
    const double* pol;            // [N][6]: polarisation p_n (3) and quadrature axis q_n (3) per mode, or NULL (x^, y^: PAPER.md:52)
    int split_nllg;               // 0: unified RK45 step; n >= 1: the paper's tier-2 operator-split loop, one
                                  // cavity RK4 step per n LLG sub-steps; fixed_dt is then the LLG sub-step and max_steps counts sub-steps
    double* spec;                 // [n_rep][spec_K][2N][2] Fourier sums X(w_k) += x(t_j) exp(+i w_k t_j) of a_n, S_n at the trace samples, or NULL
    long long* spec_n;            // [n_rep] samples accumulated
    int spec_K;
    double spec_w0, spec_dw;      // w_k = spec_w0 + k spec_dw
};

// Shared mode / controller state of one replica.
struct BatchShared {
    double omega[kMaxModes], kappa[kMaxModes], Gre[kMaxModes], Gim[kMaxModes], invW[kMaxModes], Gbre[kMaxModes], Gbim[kMaxModes];
    double a[kMaxModes][2], as[kMaxModes][2], anew[kMaxModes][2], ka[7][kMaxModes][2], S[kMaxModes][2];
    double c[kMaxModes], serr[kMaxModes];
    double pol[kMaxModes][6];
    double eta_re[kMaxModes], eta_im[kMaxModes], eta_t0[kMaxModes], eta_i2s2[kMaxModes], eta_wd[kMaxModes];
    double part[32][2 * kMaxModes + 6];     // per-warp partial sums: overlaps (2N) then <m_s> (3 n_sub)
    double wmax[32];
    double red[2 * kMaxModes + 6];
    double red2[2 * kMaxModes + 6];         // COOP: sums over all blocks
    double t, dt, h, target, err;
    long long steps;
    int clamped, sample_hit, accept, done, status, trace_n, took;
    long long accepted, rejected, rhs_evals, trace_stride, trace_acc0;
    double dt_min, dt_max;
};

// defined in cavmag_batch.cu: instantiates and launches k_batch (the C ABI of the batch, and cav_run's CAV_PATH_BLOCK)
int launch_batch_kernel(BatchArgs& A, bool f32, int n_sub, bool two_per_sm, size_t smem_optin, cudaStream_t stream,
                        cudaError_t* cuda_err);
int launch_coop_kernel(BatchArgs& A, bool f32, int n_sub, cudaStream_t stream, cudaError_t* cuda_err);
int pack_polarisation(int N, const double* pol, const double* quad, double* out /*[N][6]*/);

template <int ROW>
__device__ __forceinline__ void batch_stage_state(BatchShared& sh, const int n, const double two_over_gamma) {
    double re = 0.0, im = 0.0;
#pragma unroll
    for (int j = 0; j < ROW; ++j) { re += kA[ROW][j] * sh.ka[j][n][0]; im += kA[ROW][j] * sh.ka[j][n][1]; }
    const double are = sh.a[n][0] + sh.h * re, aim = sh.a[n][1] + sh.h * im;
    sh.as[n][0] = are; sh.as[n][1] = aim;
    sh.c[n] = two_over_gamma * (sh.Gbre[n] * are - sh.Gbim[n] * aim);
}


// The cavity half of the operator-split loop: classic RK4 over H of da/dt = -(i w + kappa) a + i G S + eta(t)
// with the overlap S_n of the current magnetisation held constant; leaves the new amplitude in anew and the RF weight
// c_n = (2/gamma) Re[G_b a_new] that the LLG half keeps constant ("H_rf = h0 * a.real", Listing 1).
__device__ __forceinline__ void split_cavity_step(BatchShared& sh, const int n, const double t, const double H,
                                                  const bool drive, const double two_over_gamma) {
    const double Sre = sh.S[n][0], Sim = sh.S[n][1], Gre = sh.Gre[n], Gim = sh.Gim[n];
    const double om = sh.omega[n], ka = sh.kappa[n];
    auto f = [&](const double are, const double aim, const double tt, double& kre, double& kim) {
        kre = (-ka * are + om * aim) - (Gre * Sim + Gim * Sre);
        kim = (-ka * aim - om * are) + (Gre * Sre - Gim * Sim);
        if (drive) {
            const double x = tt - sh.eta_t0[n];
            const double env = exp(-(x * x) * sh.eta_i2s2[n]);
            double sn, cs;
            sincos(sh.eta_wd[n] * x, &sn, &cs);
            kre += env * (sh.eta_re[n] * cs + sh.eta_im[n] * sn);
            kim += env * (sh.eta_im[n] * cs - sh.eta_re[n] * sn);
        }
    };
    const double ar = sh.a[n][0], ai = sh.a[n][1];
    double k1r, k1i, k2r, k2i, k3r, k3i, k4r, k4i;
    f(ar, ai, t, k1r, k1i);
    f(ar + 0.5 * H * k1r, ai + 0.5 * H * k1i, t + 0.5 * H, k2r, k2i);
    f(ar + 0.5 * H * k2r, ai + 0.5 * H * k2i, t + 0.5 * H, k3r, k3i);
    f(ar + H * k3r, ai + H * k3i, t + H, k4r, k4i);
    const double nr = ar + (H / 6.0) * (k1r + 2.0 * k2r + 2.0 * k3r + k4r);
    const double ni = ai + (H / 6.0) * (k1i + 2.0 * k2i + 2.0 * k3i + k4i);
    sh.anew[n][0] = nr; sh.anew[n][1] = ni;
    sh.c[n] = two_over_gamma * (sh.Gbre[n] * nr - sh.Gbim[n] * ni);
}

// MAXT: block-size bucket (128 / 256 / 512 / 1024 threads) - the register budget per thread follows from it.  MINB = 2 (the
// 512-thread ferromagnet bucket, chosen by the host when there are more replicas than SMs) asks for two blocks per SM: 64
// registers and < 100 B of spills make one replica ~10 % slower, but the barrier stalls of one replica hide behind the
// other (+31 % with 1184 replicas of CFG1).
// COOP = true: ONE simulation of up to gridDim.x * blockDim.x cells spread over co-resident blocks (cooperative launch): the
// stage state goes through a double-buffered global array (neighbours are L2 reads), block partial sums and block error
// maxima through global memory, and one grid barrier per evaluation (+ one per step for the error norm) replaces the kernel
// boundary; every block replays the mode algebra and the controller (identical bits), block 0 writes trace and state.
template <typename T, int NSUB, int MAXT, int MINB, bool COOP = false>
__global__ void __launch_bounds__(MAXT, MINB) k_batch(const BatchArgs A) {
    extern __shared__ __align__(16) unsigned char batch_dsm[];
    __shared__ BatchShared sh;
    const int nc = A.nc, N = A.N;
    T* const sm_m = reinterpret_cast<T*>(batch_dsm);                 // [NSUB*3][nc] stage state
    T* const sm_u = sm_m + (size_t)NSUB * 3 * nc;                     // [N][nc] profiles (if u_in_smem)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, nwarp = blockDim.x >> 5;
    const int rep = COOP ? 0 : (int)blockIdx.x;
    const int gcell = COOP ? (int)(blockIdx.x * blockDim.x) + tid : tid;
    const bool active = gcell < nc;
    const int cell = active ? gcell : nc - 1;
    const bool writer = !COOP || blockIdx.x == 0;                    // trace rows, amplitudes and controller state
    const int x = cell % A.nx, yy = (cell / A.nx) % A.ny, z = cell / (A.nx * A.ny);
    unsigned long long epoch = 0;                                    // grid barriers passed (COOP)
    int ev = 0;                                                      // evaluations done (COOP: buffer parity)
    auto grid_barrier = [&]() {
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            atomicAdd(A.bar, 1ull);
            const unsigned long long target = (++epoch) * (unsigned long long)A.nblk;
            unsigned long long seen;
            do { asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(seen) : "l"(A.bar) : "memory"); } while (seen < target);
        }
        __syncthreads();
    };

    // open boundary (G9): an out-of-grid neighbour gets weight 0 and the centre's index
    const T wx = (T)A.ex_wx, wy = (T)A.ex_wy, wz = (T)A.ex_wz;
    const int ixm = x > 0 ? cell - 1 : cell, ixp = x < A.nx - 1 ? cell + 1 : cell;
    const int iym = yy > 0 ? cell - A.nx : cell, iyp = yy < A.ny - 1 ? cell + A.nx : cell;
    const int izm = z > 0 ? cell - A.nx * A.ny : cell, izp = z < A.nz - 1 ? cell + A.nx * A.ny : cell;
    const T wxm = x > 0 ? wx : (T)0, wxp = x < A.nx - 1 ? wx : (T)0;
    const T wym = yy > 0 ? wy : (T)0, wyp = yy < A.ny - 1 ? wy : (T)0;
    const T wzm = z > 0 ? wz : (T)0, wzp = z < A.nz - 1 ? wz : (T)0;

    const T B0x = (T)A.B0[rep * 3 + 0], B0y = (T)A.B0[rep * 3 + 1], B0z = (T)A.B0[rep * 3 + 2];
    const T anp = (T)A.an_pref, axx = (T)A.axis[0], axy = (T)A.axis[1], axz = (T)A.axis[2];
    const T alpha = (T)A.alpha, llg = (T)A.llg, BE = (T)A.B_exch_inter;
    const T* __restrict__ ug = reinterpret_cast<const T*>(A.u);
    T* __restrict__ mg = reinterpret_cast<T*>(A.m) + (size_t)rep * NSUB * 3 * nc;

    // ---- load the replica ----
    T y[NSUB][3];
#pragma unroll
    for (int s = 0; s < NSUB; ++s)
#pragma unroll
        for (int c = 0; c < 3; ++c) y[s][c] = mg[(size_t)(s * 3 + c) * nc + cell];
    if (!COOP && A.u_in_smem)
        for (int i = tid; i < N * nc; i += blockDim.x) sm_u[i] = ug[i];
    if (tid < N) {
        const double* mp = A.modep + (A.modep_per_rep ? (size_t)rep * 7 * N : 0);
        sh.omega[tid] = mp[tid]; sh.kappa[tid] = mp[N + tid]; sh.Gre[tid] = mp[2 * N + tid];
        sh.Gim[tid] = mp[3 * N + tid]; sh.invW[tid] = mp[4 * N + tid];
        sh.Gbre[tid] = mp[5 * N + tid]; sh.Gbim[tid] = mp[6 * N + tid];
        const double are = A.a[((size_t)rep * N + tid) * 2], aim = A.a[((size_t)rep * N + tid) * 2 + 1];
        sh.a[tid][0] = are; sh.a[tid][1] = aim;
        sh.as[tid][0] = are; sh.as[tid][1] = aim;                       // stage 1 evaluates f(m_0, a_0)
        sh.c[tid] = A.two_over_gamma * (sh.Gbre[tid] * are - sh.Gbim[tid] * aim);
        if (A.drive) {
            sh.eta_re[tid] = A.drive[tid]; sh.eta_im[tid] = A.drive[N + tid]; sh.eta_t0[tid] = A.drive[2 * N + tid];
            sh.eta_i2s2[tid] = A.drive[3 * N + tid]; sh.eta_wd[tid] = A.drive[4 * N + tid];
        }
        if (A.pol) {
#pragma unroll
            for (int i = 0; i < 6; ++i) sh.pol[tid][i] = A.pol[6 * tid + i];
        }
    }
    if (tid == 0) {
        const BatchCtl& cl = A.ctl[rep];
        sh.t = cl.t; sh.dt_min = cl.dt_min; sh.dt_max = cl.dt_max; sh.err = cl.last_err;
        sh.accepted = cl.accepted; sh.rejected = cl.rejected; sh.rhs_evals = cl.rhs_evals; sh.trace_acc0 = cl.trace_acc0;
        sh.status = cl.status; sh.trace_n = cl.trace_n; sh.steps = 0; sh.took = 0;
        const bool adaptive = A.tol > 0.0;
        if (adaptive) sh.dt = A.dt_init > 0.0 ? A.dt_init : (cl.dt > 0.0 ? cl.dt : 1e-14);
        else {
            sh.dt = A.fixed_dt;
            const long long st = llround(A.sample_dt / A.fixed_dt);
            sh.trace_stride = st < 1 ? 1 : st;
        }
    }
    __syncthreads();
    const T* __restrict__ up = (!COOP && A.u_in_smem) ? sm_u : ug;
    const bool polar = A.pol != nullptr;
    const bool split = A.split_nllg > 0;

    // ---- one evaluation of the coupled right-hand side at stage s (1..7): slope k of the own cell, and in
    //      thread n the mode slope ka_s and the amplitudes / RF weights of the next stage state ----
    auto eval = [&](auto stage_tag, const T (&ms)[NSUB][3], T (&k)[NSUB][3]) {
        constexpr int s = decltype(stage_tag)::value;
        constexpr int nsum_extra = (s == 7) ? 3 * NSUB : 0;
        T* const fld = COOP ? reinterpret_cast<T*>(A.gms[ev & 1]) : sm_m;      // where neighbours read the stage state
        if (active) {
#pragma unroll
            for (int q = 0; q < NSUB; ++q)
#pragma unroll
                for (int c = 0; c < 3; ++c) fld[(size_t)(q * 3 + c) * nc + cell] = ms[q][c];
        }
        // COOP: [A] publishes c_n of this stage before the mode loop.  One block per simulation: c_n was published by the
        // previous evaluation's [B] (stages 1-2: written since by the step's first stage state - one more barrier), and [A]
        // sits behind the mode loop, where it also publishes the block's partial sums: the mode thread's fp64 chain then
        // runs beside the other warps' stencil instead of after it.
        if constexpr (COOP || s <= 2) __syncthreads();
        T mcx, mcy, mcz;
        if constexpr (NSUB == 1) { mcx = ms[0][0]; mcy = ms[0][1]; mcz = ms[0][2]; }
        else { mcx = (T)0.5 * (ms[0][0] + ms[1][0]); mcy = (T)0.5 * (ms[0][1] + ms[1][1]); mcz = (T)0.5 * (ms[0][2] + ms[1][2]); }
        T brf = (T)0, brfy = (T)0, brfz = (T)0;
        for (int n = 0; n < N; ++n) {
            const T un = up[(size_t)n * nc + cell];
            T ux, uy;                                                // u (m_c.p - i m_c.q): real part, minus imaginary part
            if (!polar) {                                            // p = x^, q = y^
                brf += (T)sh.c[n] * un;
                ux = un * mcx; uy = un * mcy;
            } else {                                                 // reading G32: field along p_n, coupling to m.p_n - i m.q_n
                const double cn = sh.c[n];
                brf += (T)(cn * sh.pol[n][0]) * un; brfy += (T)(cn * sh.pol[n][1]) * un; brfz += (T)(cn * sh.pol[n][2]) * un;
                ux = un * (mcx * (T)sh.pol[n][0] + mcy * (T)sh.pol[n][1] + mcz * (T)sh.pol[n][2]);
                uy = un * (mcx * (T)sh.pol[n][3] + mcy * (T)sh.pol[n][4] + mcz * (T)sh.pol[n][5]);
            }
            double px = active ? (double)ux : 0.0, py = active ? (double)uy : 0.0;
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
                px += __shfl_xor_sync(0xffffffffu, px, o);
                py += __shfl_xor_sync(0xffffffffu, py, o);
            }
            if (lane == 0) { sh.part[warp][2 * n] = px; sh.part[warp][2 * n + 1] = py; }
        }
        if constexpr (s == 7) {                                      // <m_s> of the candidate, for the trace
#pragma unroll
            for (int i = 0; i < 3 * NSUB; ++i) {
                double v = active ? (double)ms[i / 3][i % 3] : 0.0;
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
                if (lane == 0) sh.part[warp][2 * N + i] = v;
            }
        }
        // thread n: S_n, the mode slope ka_s and the amplitudes / RF weights of the next stage state; a second warp: <m_s>
        auto mode_block = [&]() {
        if (tid < N) {
            const int n = tid;
            double sx = 0.0, sy = 0.0;
            if constexpr (COOP) {
                sx = sh.red2[2 * n]; sy = sh.red2[2 * n + 1];
            } else {
                for (int w = 0; w < nwarp; ++w) { sx += sh.part[w][2 * n]; sy += sh.part[w][2 * n + 1]; }
            }
            const double Sre = sx * sh.invW[n], Sim = -sy * sh.invW[n];
            sh.S[n][0] = Sre; sh.S[n][1] = Sim;
            if (split) {                                             // operator-split loop: the amplitudes advance once per cavity step
                if constexpr (s == 7) sh.serr[n] = 0.0;
            } else {
            const double are = sh.as[n][0], aim = sh.as[n][1];
            const double Gre = sh.Gre[n], Gim = sh.Gim[n];
            double kre = (-sh.kappa[n] * are + sh.omega[n] * aim) - (Gre * Sim + Gim * Sre);
            double kim = (-sh.kappa[n] * aim - sh.omega[n] * are) + (Gre * Sre - Gim * Sim);
            if (A.drive) {          // + eta_n(t + c_s h)  (Eq. 1 / Eq. 12; stage 1 runs before h is set: c_1 = 0)
                const double x = (s == 1 ? sh.t : sh.t + kC[s - 1] * sh.h) - sh.eta_t0[n];
                const double env = exp(-(x * x) * sh.eta_i2s2[n]);
                double sn, cs;
                sincos(sh.eta_wd[n] * x, &sn, &cs);
                kre += env * (sh.eta_re[n] * cs + sh.eta_im[n] * sn);
                kim += env * (sh.eta_im[n] * cs - sh.eta_re[n] * sn);
            }
            sh.ka[s - 1][n][0] = kre; sh.ka[s - 1][n][1] = kim;
            if constexpr (s >= 2 && s <= 5) batch_stage_state<s>(sh, n, A.two_over_gamma);
            else if constexpr (s == 6) {
                batch_stage_state<6>(sh, n, A.two_over_gamma);       // row 6 = b: the 5th-order candidate
                sh.anew[n][0] = sh.as[n][0]; sh.anew[n][1] = sh.as[n][1];
            } else if constexpr (s == 7) {
                double ere = 0.0, eim = 0.0;
#pragma unroll
                for (int j = 0; j < 7; ++j) { ere += kD[j] * sh.ka[j][n][0]; eim += kD[j] * sh.ka[j][n][1]; }
                const double e = fabs(sh.h) * sqrt(ere * ere + eim * eim);
                sh.serr[n] = (e < CUDART_INF) ? e : CUDART_INF;
            }
            }
        } else if (s == 7 && tid >= 32 && tid < 32 + 3 * NSUB) {     // a second warp sums <m_s>
            const int i = tid - 32;
            double v = 0.0;
            if constexpr (COOP) {
                v = sh.red2[2 * N + i];
            } else {
                for (int w = 0; w < nwarp; ++w) v += sh.part[w][2 * N + i];
            }
            sh.red[i] = v * A.inv_nc;
        }
        };
        if constexpr (!COOP) {
            __syncthreads();                                         // [A] stage state and partial sums of the block published
            mode_block();
        }
        if constexpr (COOP) {
            __syncthreads();
            if (tid < 2 * N + nsum_extra) {                          // fixed-order block sum -> this block's slot
                double v = 0.0;
                for (int w = 0; w < nwarp; ++w) v += sh.part[w][tid];
                A.cpart[ev & 1][(size_t)tid * A.nblk + blockIdx.x] = v;
            }
            grid_barrier();                                          // stage state, partials and c_n of all blocks published
        }
        auto rd = [&](const T* f, int i) -> T {
            if constexpr (COOP) return __ldcg(f + i);                // written by other SMs: read at L2
            else return f[i];
        };
#pragma unroll
        for (int q = 0; q < NSUB; ++q) {
            T lap[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const T* f = fld + (size_t)(q * 3 + c) * nc;
                const T m0 = ms[q][c];
                T l = (rd(f, ixm) - m0) * wxm;
                l += (rd(f, ixp) - m0) * wxp;
                l += (rd(f, iym) - m0) * wym;
                l += (rd(f, iyp) - m0) * wyp;
                l += (rd(f, izm) - m0) * wzm;
                l += (rd(f, izp) - m0) * wzp;
                lap[c] = l;
            }
            const T mx = ms[q][0], my = ms[q][1], mz = ms[q][2];
            T Bx, By, Bz;
            material_field(mx, my, mz, lap[0], lap[1], lap[2], B0x, B0y, B0z, anp, axx, axy, axz, Bx, By, Bz);
            Bx += brf;
            if (polar) { By += brfy; Bz += brfz; }
            if constexpr (NSUB == 2) { Bx -= BE * ms[1 - q][0]; By -= BE * ms[1 - q][1]; Bz -= BE * ms[1 - q][2]; }
            llg_slope(mx, my, mz, Bx, By, Bz, alpha, llg, k[q][0], k[q][1], k[q][2]);
        }
        if constexpr (COOP)                                          // fixed-order sum over the blocks' slots (every block: same bits)
            reduce_block_partials(A.cpart[ev & 1], A.nblk, 2 * N + nsum_extra, A.nblk, warp, nwarp, lane, sh.red2);
        __syncthreads();                                             // [B] stage-state buffer free again; COOP: partial sums published; else: c_n, a_s of the next stage published
        if constexpr (COOP) mode_block();
        if (tid == 0) sh.rhs_evals++;
        ++ev;
    };


    // ---- k1 of the loaded state ----
    T k1[NSUB][3], k2[NSUB][3], k3[NSUB][3], k4[NSUB][3], k5[NSUB][3], k6[NSUB][3], k7[NSUB][3], ms[NSUB][3], yn[NSUB][3];
    eval(std::integral_constant<int, 1>{}, y, k1);
    const bool adaptive = A.tol > 0.0;

    for (;;) {
        // ---- start of a step (thread 0): anything left to do?  h for this step (prepare_h in stage_kernel.cuh) ----
        if (tid == 0) {
            const bool done = !(sh.t < A.t_end) || (A.max_steps > 0 && sh.steps >= A.max_steps) || sh.status != 0;
            sh.done = done ? 1 : 0;
            double h = sh.dt, target = A.t_end;
            int sample_hit = 0;
            if (adaptive && A.sample_dt > 0.0 && sh.trace_n < A.trace_cap) {
                const double ts = A.trace_t0 + (double)(sh.trace_n + 1) * A.sample_dt;
                if (ts <= target) { target = ts; sample_hit = 1; }
            }
            int clamped = 0;
            if (sh.t + h * (1.0 + 1e-12) >= target) { h = target - sh.t; clamped = 1; }
            sh.h = h; sh.target = target; sh.clamped = clamped; sh.sample_hit = sample_hit;
        }
        __syncthreads();
        if (sh.done) break;
        if (split) {
            // Listing 1: the overlaps S_n of the current m are in sh.S (7th evaluation of the last step,
            // or the evaluation before the loop); every split_nllg sub-steps: cavity RK4 over the whole cavity step, then
            // the slope k1 in the NEW constant RF field (no FSAL across a field jump)
            if (sh.steps % A.split_nllg == 0) {
                if (tid < N) split_cavity_step(sh, tid, sh.t, sh.h * (double)A.split_nllg, A.drive != nullptr, A.two_over_gamma);
                eval(std::integral_constant<int, 1>{}, y, k1);
            }
        } else if (tid < N) batch_stage_state<1>(sh, tid, A.two_over_gamma);      // a_2 = a_0 + h a21 ka_1
        const T h = (T)sh.h;

        // stage states m_s = m_0 + h sum_j a_sj k_j (dp_state<ROW>, stage_kernel.cuh) and their evaluations
        auto stage_state = [&](auto row_tag, auto&&... kj) {
            constexpr int ROW = decltype(row_tag)::value;
#pragma unroll
            for (int q = 0; q < NSUB; ++q)
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const T kv[ROW] = {kj[q][c]...};
                    ms[q][c] = dp_state<ROW>(y[q][c], kv, h);
                }
        };
        stage_state(std::integral_constant<int, 1>{}, k1);
        eval(std::integral_constant<int, 2>{}, ms, k2);
        stage_state(std::integral_constant<int, 2>{}, k1, k2);
        eval(std::integral_constant<int, 3>{}, ms, k3);
        stage_state(std::integral_constant<int, 3>{}, k1, k2, k3);
        eval(std::integral_constant<int, 4>{}, ms, k4);
        stage_state(std::integral_constant<int, 4>{}, k1, k2, k3, k4);
        eval(std::integral_constant<int, 5>{}, ms, k5);
        stage_state(std::integral_constant<int, 5>{}, k1, k2, k3, k4, k5);
        eval(std::integral_constant<int, 6>{}, ms, k6);

        // ---- 5th-order candidate, renormalised per cell (G13), 7th evaluation, error (G12) ----
        T e2max = (T)0;
#pragma unroll
        for (int q = 0; q < NSUB; ++q) {
            T er[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) {
                const T kv[6] = {k1[q][c], (T)0, k3[q][c], k4[q][c], k5[q][c], k6[q][c]};      // b_2 = d_2 = 0
                yn[q][c] = dp_state<6>(y[q][c], kv, h);
                er[c] = dp_error6(kv, h);
            }
            if (A.renormalize) {
                const T inv = rsqrt_t<T>(yn[q][0] * yn[q][0] + yn[q][1] * yn[q][1] + yn[q][2] * yn[q][2]);
                yn[q][0] *= inv; yn[q][1] *= inv; yn[q][2] *= inv;
            }
            k6[q][0] = er[0]; k6[q][1] = er[1]; k6[q][2] = er[2];      // k6 is dead: keep the partial error there
        }
        eval(std::integral_constant<int, 7>{}, yn, k7);
#pragma unroll
        for (int q = 0; q < NSUB; ++q) {
            const T e2 = dp_error7_sq(k6[q][0], k6[q][1], k6[q][2], k7[q][0], k7[q][1], k7[q][2], h);
            if (active) e2max = fmax(e2max, e2);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) e2max = fmax(e2max, __shfl_xor_sync(0xffffffffu, e2max, o));
        if (lane == 0) sh.wmax[warp] = (double)e2max;
        __syncthreads();                                                 // [C]
        if constexpr (COOP) {                                            // max over all blocks (order-independent)
            double* const gmax = A.cmax[(int)(sh.steps & 1)];
            if (tid == 0) {
                double mxb = 0.0;
                for (int w = 0; w < nwarp; ++w) mxb = fmax(mxb, sh.wmax[w]);
                gmax[blockIdx.x] = mxb;
            }
            grid_barrier();
            if (warp == 0) {
                double v = 0.0;
                for (int b = lane; b < A.nblk; b += 32) v = fmax(v, __ldcg(gmax + b));
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_xor_sync(0xffffffffu, v, o));
                if (lane == 0) sh.wmax[0] = v;
            }
            __syncthreads();
        }

        // ---- controller (stage_finish<7> in stage_kernel.cuh, same constants) ----
        if (tid == 0) {
            sh.took = 0;
            double mx = 0.0;
            for (int w = 0; w < (COOP ? 1 : nwarp); ++w) mx = fmax(mx, sh.wmax[w]);
            double err = sqrt(mx);
            for (int n = 0; n < N; ++n) err = fmax(err, sh.serr[n]);
            const bool finite = err < CUDART_INF;
            const double hh = sh.h;
            bool accept;
            if (adaptive) accept = finite && err <= A.tol;
            else { accept = true; if (!finite) { accept = false; sh.status = -5; } }
            double fac;
            if (!finite) fac = 0.5;
            else if (err == 0.0) fac = 2.0;
            else { fac = 0.8 * fifth_root(fmin(fmax(A.tol / err, 1e-2), 1e3)); fac = fmin(fmax(fac, 0.5), 2.0); }
            sh.steps++;
            sh.err = err;
            if (accept) {
                sh.t = sh.clamped ? sh.target : sh.t + hh;
                sh.accepted++;
                sh.dt_min = fmin(sh.dt_min, hh);
                sh.dt_max = fmax(sh.dt_max, hh);
                if (adaptive) { const double prop = hh * fac; sh.dt = sh.clamped ? fmax(prop, sh.dt) : prop; }
                const bool take = A.trace != nullptr && A.sample_dt > 0.0 && sh.trace_n < A.trace_cap &&      // every block counts,
                                  (adaptive ? (sh.clamped && sh.sample_hit)
                                            : ((sh.accepted - sh.trace_acc0) % sh.trace_stride == 0));
                if (take && writer) {                                                                       // block 0 writes
                    double* row = A.trace + ((size_t)rep * A.trace_cap + sh.trace_n) * A.row_len;
                    row[0] = sh.t;
                    for (int n = 0; n < N; ++n) {
                        row[1 + 2 * n] = sh.anew[n][0]; row[2 + 2 * n] = sh.anew[n][1];
                        row[1 + 2 * N + 2 * n] = sh.S[n][0]; row[2 + 2 * N + 2 * n] = sh.S[n][1];
                    }
                    for (int i = 0; i < 3 * NSUB; ++i) row[1 + 4 * N + i] = sh.red[i];
                }
                if (take) sh.trace_n++;
                sh.took = take ? 1 : 0;
            } else if (sh.status == 0) {
                sh.rejected++;
                sh.dt = hh * fac;
                sh.took = 0;
            }
            if (adaptive && !(sh.dt > 1e-20)) sh.status = -6;
            sh.accept = accept ? 1 : 0;
        }
        __syncthreads();                                                 // [D]
        if (A.spec != nullptr && sh.took && sh.accept && writer) {       // Fourier sums of this sample (a_new, S of the new state)
            dft_accumulate(A.spec + (size_t)rep * A.spec_K * 2 * (2 * N + NSUB), A.spec_K, A.spec_w0, A.spec_dw, N, sh.t, sh.anew, sh.S,
                           sh.red, NSUB, tid, (int)blockDim.x);
            if (tid == 0) A.spec_n[rep]++;
        }
        if (sh.accept) {                                                 // y := y_new, FSAL: k1 := k7
#pragma unroll
            for (int q = 0; q < NSUB; ++q)
#pragma unroll
                for (int c = 0; c < 3; ++c) { y[q][c] = yn[q][c]; k1[q][c] = k7[q][c]; }
            if (tid < N) {
                sh.a[tid][0] = sh.anew[tid][0]; sh.a[tid][1] = sh.anew[tid][1];
                sh.ka[0][tid][0] = sh.ka[6][tid][0]; sh.ka[0][tid][1] = sh.ka[6][tid][1];
            }
        }
    }

    // ---- store the replica ----
    if (active) {
#pragma unroll
        for (int q = 0; q < NSUB; ++q)
#pragma unroll
            for (int c = 0; c < 3; ++c) mg[(size_t)(q * 3 + c) * nc + cell] = y[q][c];
    }
    if (writer && tid < N) { A.a[((size_t)rep * N + tid) * 2] = sh.a[tid][0]; A.a[((size_t)rep * N + tid) * 2 + 1] = sh.a[tid][1]; }
    if (writer && tid == 0) {
        BatchCtl& cl = A.ctl[rep];
        cl.t = sh.t; cl.dt = sh.dt; cl.dt_min = sh.dt_min; cl.dt_max = sh.dt_max; cl.last_err = sh.err;
        cl.accepted = sh.accepted; cl.rejected = sh.rejected; cl.rhs_evals = sh.rhs_evals;
        cl.status = sh.status; cl.trace_n = sh.trace_n;
    }
}
}  // namespace cavmag
