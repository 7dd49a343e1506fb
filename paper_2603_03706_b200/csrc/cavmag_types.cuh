// Device-side state shared by the stage kernels and the C-ABI layer (CUDA path only).
// Notation follows arXiv 2603.03706: m, a_n, u_n, S_n, G_n, kappa_n, omega_n.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace cavmag {

constexpr int kMaxModes = 32;          // CAV_MAX_MODES
constexpr int kBlock = 128;            // threads per stage-kernel block
constexpr int kMaxSums = 2 * kMaxModes + 6;   // overlap sums (2N) + <m_s> (3 n_sub)
constexpr int kMaxBlocks = 16384;      // upper bound on stage-kernel grid size (partials capacity)

// Dormand-Prince 5(4) coefficients (Dormand & Prince 1980); the paper names only
// "RK45 adaptive" — DESIGN.md reading G11.
// Row s (0-based) holds a_{s+1,j}; row 6 equals b (FSAL).
#define CAVMAG_DP_A                                                                      \
    {{0, 0, 0, 0, 0, 0, 0},                                                              \
     {1.0 / 5.0, 0, 0, 0, 0, 0, 0},                                                      \
     {3.0 / 40.0, 9.0 / 40.0, 0, 0, 0, 0, 0},                                            \
     {44.0 / 45.0, -56.0 / 15.0, 32.0 / 9.0, 0, 0, 0, 0},                                \
     {19372.0 / 6561.0, -25360.0 / 2187.0, 64448.0 / 6561.0, -212.0 / 729.0, 0, 0, 0},   \
     {9017.0 / 3168.0, -355.0 / 33.0, 46732.0 / 5247.0, 49.0 / 176.0, -5103.0 / 18656.0, 0, 0}, \
     {35.0 / 384.0, 0, 500.0 / 1113.0, 125.0 / 192.0, -2187.0 / 6784.0, 11.0 / 84.0, 0}}
// d = b - bhat (error weights)
#define CAVMAG_DP_D                                                                      \
    {35.0 / 384.0 - 5179.0 / 57600.0, 0.0, 500.0 / 1113.0 - 7571.0 / 16695.0,            \
     125.0 / 192.0 - 393.0 / 640.0, -2187.0 / 6784.0 + 92097.0 / 339200.0,               \
     11.0 / 84.0 - 187.0 / 2100.0, -1.0 / 40.0}

// Controller + mode state.  Two instances in device memory per simulation: the canonical one (StageArgs::ctrl,
// the one the host pulls and pushes) and a step-boundary copy (StageArgs::ctrl0).  Written only by single-block code
// (k_begin, the last-arriving block of a stage kernel, block 0 of a TMA stage kernel's prologue); read by every block.
// A kernel whose block 0 rewrites fields that the other blocks of the SAME kernel still have to read (the step
// controller in the prologue of the TMA stage-2 kernel) reads one instance and writes the other.
struct Ctrl {
    // ---- run control ----
    double t, t_end, dt, h, tol, fixed_dt, target;
    long long max_steps, steps_run;
    int adaptive, done, status, clamped, sample_hit;
    // ---- buffer rotation ----
    int ycur;       // Y[ycur] = m_0, Y[1-ycur] = m_new
    int k1slot;     // K[k1slot] = k1, K[6-k1slot] = k7   (k1slot in {0,6}); k2..k6 = K[1..5]
    int k1_valid;
    // ---- statistics ----
    long long accepted, rejected, rhs_evals;
    double dt_min, dt_max, last_err;
    // ---- cavity modes (always fp64) ----
    int N;
    double gamma, two_over_gamma;   // two_over_gamma = 2/gamma (host-computed: no fp64 division on the critical path)
    double omega[kMaxModes], kappa[kMaxModes], Gre[kMaxModes], Gim[kMaxModes], invW[kMaxModes];
    double Gbre[kMaxModes], Gbim[kMaxModes];   // backward coupling G_b of the feedback field (= G unless cav_set_backaction)
    double a[kMaxModes][2];        // a_0: amplitudes of the current accepted state
    double as[2][kMaxModes][2];    // a_s: amplitudes of the state stage s is evaluated at, in as[s & 1] (double-buffered:
                                   // on the TMA path block 0 of kernel s+1 writes a_{s+1} while the other blocks still read a_s)
    double anew[kMaxModes][2];     // 5th-order candidate
    double ka[7][kMaxModes][2];    // mode slopes ka_1..ka_7
    double S[kMaxModes][2];        // overlaps of the last evaluated stage state
    double c[kMaxModes];           // (2/gamma) Re[G_n a_s,n]: RF-field weights for the next kernel
    double mavg[6];                // <m_s> of the last accepted state
    // ---- external drive eta_n(t) = A_n exp(-(t-t0)^2 i2s2) exp(-i wd (t-t0)) ----
    int drive_on, drive_pad;
    double eta_re[kMaxModes], eta_im[kMaxModes], eta_t0[kMaxModes], eta_i2s2[kMaxModes], eta_wd[kMaxModes];
    // ---- trace ----
    double sample_dt, trace_t0;
    int trace_cap, trace_n;
    long long trace_stride, trace_acc0;
    // ---- on-device spectroscopy: Fourier sums at the trace samples ----
    int spec_K, took;              // bins (0: off); took: the controller just stored a trace sample (transient)
    double spec_w0, spec_dw;       // w_k = spec_w0 + k spec_dw
    long long spec_n;              // samples accumulated
    // ---- last-block-done counter ----
    unsigned int arrive;
    int pend7;      // TMA path: stage 7 of the step in flight is still to be finished (mode ODE, error norm, controller) by
                    // the prologue of the next stage-2 kernel
};

// Arguments of every stage kernel (by value; fixed for the lifetime of a CUDA graph).
struct StageArgs {
    Ctrl* ctrl;          // canonical instance
    Ctrl* ctrl0;         // step-boundary copy: written by block 0 of the TMA stage-7 kernel (and k_begin / stage 1), read by
                         // every block of the TMA stage-2 kernel, whose block 0 writes the new state to `ctrl`
    void* Y[2];          // state ping-pong
    void* MS[2];         // materialised stage states (MS[0] doubles as the partial-error field)
    void* K[7];          // slope fields
    const void* u;       // [N][nc]
    double* partial;     // [2][kMaxSums][pstride] block partial sums, double-buffered by stage parity (stage_partials())
    double* partial_max; // [pstride] block max of |e|^2
    const void* bdem;    // [3][nc] dipolar field of the state this stage is evaluated at (generic kernels only), or nullptr
    const double* pol;   // [N][6] polarisation p_n and quadrature axis q_n per mode (generic polarisation kernels only), or nullptr
    double* spec;        // [spec_K][2N][2] Fourier sums X_k += x(t_j) exp(+i w_k t_j), x = a_1..a_N, S_1..S_N, or nullptr
    unsigned long long cond_handle;   // cudaGraphConditionalHandle (0: none)
    int pstride;
    int nx, ny, nz;
    int iters;           // block-iterations per block (kBlock*VEC cells each)
    int serpentine;      // 1: odd stages sweep the grid backwards (L2 reuse across kernels)
    long long nc;        // cells
    // Memory layout of every cell field and of u: rows of `pitch` elements (pitch >= nx; pitch == nx unless the grid is
    // large, nx * sizeof(T) is not a multiple of 16 bytes and the TMA path needs 16-byte row strides), `ncp` = pitch * ny * nz
    // elements per component.  Only the TMA kernels understand pitch > nx; the C ABI always takes and returns dense arrays.
    int pitch;
    long long ncp;
    double inv_nc;       // 1/nc
    long long nvec;      // nc / VEC
    double B0[3];
    double ex_wx, ex_wy, ex_wz;   // (2A/Ms)/D_d^2, tesla
    double an_pref;               // 2Ku/Ms, tesla
    double axis[3];
    double alpha, llg;            // llg = -gamma/(1+alpha^2)
    double B_exch_inter;
    int renormalize;
#ifdef CAVMAG_PROBE
    unsigned long long* probe;   // [8 stages][gridDim.x][32] timestamps (profiling builds only)
#endif
};

}  // namespace cavmag
