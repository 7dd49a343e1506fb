/* =====================================================================================
 * cavmag.h — C ABI of the B200-native (sm_100a) cavity-magnonics hot path.
 *
 * What it computes (arXiv 2603.03706, tier 1; citations are /root/reference/PAPER.md lines):
 * the Landau-Lifshitz-Gilbert equation on a finite-difference grid, integrated TOGETHER
 * with N cavity-mode ODEs in one adaptive Dormand-Prince RK5(4) step, entirely on the
 * device with no per-step host synchronisation.
 *
 *   S_n      = (1/W_n) sum_r u_n(r) (m_c,x - i m_c,y)(r)          PAPER.md:156 Eq. 18, :45 Eq. 2
 *   da_n/dt  = -(i w_n + kappa_n) a_n + i G_n S_n,  G_n = g_n + Gamma_n e^{i Phi_n}
 *                                                                PAPER.md:119 Eq. 12, :317 Eq. 19
 *   B_rf(r)  = x^ (2/gamma) sum_n u_n(r) Re[G_n a_n]              PAPER.md:54 Eq. 3, :65 Eq. 5, :121 Eq. 13, :159
 *   B_s(r)   = B0 + (2A/Ms) sum_{6 nb in grid} (m_nb - m)/D^2 + (2Ku/Ms)(m.k^)k^ + B_rf
 *              - B_exch_inter m_other(r)   [two-sublattice antiferromagnet, PAPER.md:132-144]
 *   dm_s/dt  = -gamma/(1+alpha^2) [ m x B + alpha m x (m x B) ]
 *   m_c      = m_1  or (m_1 + m_2)/2
 *
 * The readings of everything the paper leaves open (signs, normalisation, tableau, step
 * controller, boundary condition) are listed in DESIGN.md ("Readings").
 *
 * Conventions
 *   - SI units: metres, tesla, A/m, J/m, J/m^3; every rate in rad/s.
 *   - Cell fields are SoA, component-major, x fastest:
 *       m : [n_sub][3][nz][ny][nx]      u : [N][nz][ny][nx]
 *     in the precision chosen at cav_create (CAV_F32 -> float, CAV_F64 -> double).
 *   - Mode amplitudes are always double: a : [N][2] = (Re, Im).
 *   - "host or device" pointers carry an explicit is_device flag. Device pointers must be
 *     on the current CUDA device and are read/written on the simulation's stream.
 *   - Ownership: every input array is copied during the call; outputs are written into
 *     caller memory. The library owns all of its device buffers (freed by cav_destroy).
 *   - cav_run* only enqueue work on the stream (asynchronous). cav_get_*, cav_sync and
 *     cav_destroy synchronise the stream. Errors raised on the device (non-finite error
 *     norm, step-size underflow) surface as the return value of the next synchronising call.
 *   - Every function returns CAV_OK (0) or a negative cav_status. No exceptions cross the
 *     boundary. A handle is not thread-safe; distinct handles are independent.
 * ===================================================================================== */
#ifndef CAVMAG_H_
#define CAVMAG_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct cav_sim cav_sim; /* opaque */

typedef enum {
    CAV_OK = 0,
    CAV_E_ARG = -1,           /* invalid argument (NULL, non-positive size, N > CAV_MAX_MODES ...) */
    CAV_E_STATE = -2,         /* call order: e.g. cav_run before cav_set_m */
    CAV_E_CUDA = -3,          /* a CUDA runtime call failed; see cav_last_cuda_error */
    CAV_E_NOMEM = -4,         /* device or host allocation failed */
    CAV_E_NONFINITE = -5,     /* error norm became NaN/Inf in fixed-step mode */
    CAV_E_DT_UNDERFLOW = -6,  /* adaptive step proposal fell below 1e-20 s */
    CAV_E_SINGULAR_NORM = -7, /* CAV_NORM_SUM_U with |sum_r u_n| < 1e-6 N_cells */
    CAV_E_UNSUPPORTED = -8    /* no CUDA device / device is not sm_100 / requested kernel path not eligible for this problem */
} cav_status;

enum { CAV_F32 = 0, CAV_F64 = 1 };
enum { CAV_NORM_NCELLS = 0, CAV_NORM_SUM_U = 1 };
enum { CAV_LAUNCH_GRAPH = 0, CAV_LAUNCH_STREAM = 1 };
enum { CAV_PATH_AUTO = 0, CAV_PATH_GENERIC = 1, CAV_PATH_TMA = 2, CAV_PATH_BLOCK = 3, CAV_PATH_COOP = 4 };
#define CAV_MAX_MODES 32

/* Finite-difference grid: nx*ny*nz cells of size dx*dy*dz (metres). */
typedef struct {
    int nx, ny, nz;
    double dx, dy, dz;
} cav_grid;

/* Material and model parameters ("the paper's statement of the problem"). */
typedef struct {
    double Ms;           /* saturation magnetisation, A/m */
    double Aex;          /* exchange stiffness, J/m (6-neighbour stencil, open boundaries) */
    double Ku;           /* uniaxial anisotropy, J/m^3 */
    double ku_axis[3];   /* anisotropy axis (normalised internally; ignored if Ku == 0) */
    double alpha;        /* Gilbert damping */
    double gamma;        /* gyromagnetic ratio, rad/(s T); PAPER.md:56 uses 1.76e11 */
    double B0[3];        /* static field, tesla */
    int n_sub;           /* 1 ferromagnet, 2 two-sublattice antiferromagnet */
    double B_exch_inter; /* tesla; n_sub == 2: B_s += -B_exch_inter * m_other(r) */
    int precision;       /* CAV_F32 | CAV_F64 for the cell fields */
    int renormalize;     /* 1: m_new = y5/|y5| per cell before the 7th evaluation (default 1) */
    int overlap_norm;    /* CAV_NORM_NCELLS (Eq. 18, default) | CAV_NORM_SUM_U */
} cav_params;

typedef struct {
    long long accepted;  /* accepted RK45 steps since creation */
    long long rejected;  /* rejected RK45 steps */
    long long rhs_evals; /* evaluations of the coupled right-hand side (= stage-kernel launches) */
    double dt_min;       /* smallest / largest accepted step */
    double dt_max;
    double dt_next;      /* current step proposal */
    double t;            /* simulated time, s */
    double last_err;     /* error norm of the last attempted step */
} cav_stats;

/* Create a simulation on the current CUDA device. Allocates all device buffers
 * (11 cell fields of n_sub*3*nx*ny*nz elements, reduction scratch, controller state). */
int cav_create(const cav_grid* grid, const cav_params* params, cav_sim** out);
int cav_destroy(cav_sim* sim);

/* Use an existing CUDA stream (a cudaStream_t, e.g. torch's current stream) for all work.
 * Default: a stream the library creates. Synchronises the old stream first. */
int cav_set_stream(cav_sim* sim, void* cuda_stream);

/* CAV_LAUNCH_GRAPH (default): cav_run is one CUDA-graph launch whose body is a conditional
 * WHILE node looping on the device.  CAV_LAUNCH_STREAM: the host enqueues the stage kernels
 * in chunks and polls the device 'done' flag once per chunk (debug / profiling aid). */
int cav_set_launch_mode(cav_sim* sim, int mode);

/* Cavity modes (PAPER.md:119 Eq. 12, :154 profiles, :317 Eq. 19).
 *   u      [N][nz][ny][nx] in the simulation's precision, host or device
 *   omega, kappa, g, Gamma, Phi : host arrays [N] (rad/s, rad); Gamma and Phi may be NULL (= 0)
 * N may be 0 (plain LLG; u ignored). Replaces any previous mode set and zeroes a. */
int cav_set_modes(cav_sim* sim, int N, const void* u, int u_is_device, const double* omega,
                  const double* kappa, const double* g, const double* Gamma, const double* Phi);

/* Non-reciprocal coupling: a backward (cavity-to-magnon) coupling G_b,n = g_b,n + Gamma_b,n e^{i Phi_b,n}
 * for the feedback field, B_rf,x = (2/gamma) sum_n u_n Re[G_b,n a_n] (h0 = 2 g_b/gamma), while the mode ODE keeps the forward
 * coefficient i G_n of cav_set_modes.  Host arrays [N] (rad/s, rad); Gamma_b, Phi_b may be NULL (= 0); g_b == NULL restores
 * reciprocal coupling (G_b = G).  Call after cav_set_modes (a new mode set is reciprocal again). */
int cav_set_backaction(cav_sim* sim, const double* g_b, const double* Gamma_b, const double* Phi_b);

/* External microwave drive eta_n(t) of Eq. 1 / Eq. 12, as the Gaussian pulse of the paper's
 * spectroscopy protocol (sigma = 20 ps, t0 = 0.1 ns) with an optional carrier (reading G27):
 *     eta_n(t) = A_n exp(-(t - t0_n)^2 / (2 sigma_n^2)) exp(-i omega_d,n (t - t0_n)),
 * added to da_n/dt at the stage times t + c_s h of the RK45 step.
 *   amp_re_im [N][2] complex amplitude A_n (units of a per second); NULL switches the drive off
 *   t0, sigma [N] seconds (sigma > 0, else CAV_E_ARG); omega_d [N] rad/s or NULL (= 0: baseband pulse)
 * Host arrays, copied.  Call after cav_set_modes (a new mode set clears the drive). */
int cav_set_drive(cav_sim* sim, const double* amp_re_im, const double* t0, const double* sigma, const double* omega_d);

/* Magnetisation [n_sub][3][nz][ny][nx] in the simulation's precision. Normalised per cell on entry. */
int cav_set_m(cav_sim* sim, const void* m, int is_device);
int cav_get_m(cav_sim* sim, void* m_out, int is_device);

/* Mode amplitudes, host arrays [N][2] doubles. */
int cav_set_a(cav_sim* sim, const double* a_re_im);
int cav_get_a(cav_sim* sim, double* a_out);

/* Slopes of the current state: dm/dt [n_sub][3][nz][ny][nx] (simulation precision, host or device)
 * and da/dt [N][2] (host). Evaluates the coupled right-hand side once if it is not cached. */
int cav_get_dmdt(cav_sim* sim, void* out, int is_device);
int cav_get_dadt(cav_sim* sim, double* out);

/* Overlaps S_n of the current state (from the last evaluation of the right-hand side), [N][2]. */
int cav_get_overlaps(cav_sim* sim, double* S_out);

/* Advance to t_end.  Exactly one of tol > 0 (adaptive DP5(4), absolute max-norm tolerance)
 * or fixed_dt > 0 (fixed step).  dt_init <= 0: keep the current proposal (1e-14 s initially). */
int cav_run(cav_sim* sim, double t_end, double tol, double fixed_dt, double dt_init);

/* As cav_run, but stop after max_steps attempted steps (accepted + rejected) if max_steps > 0.
 * t_end may be +inf when max_steps > 0. */
int cav_run_steps(cav_sim* sim, double t_end, double tol, double fixed_dt, double dt_init,
                  long long max_steps);

/* Wait for all enqueued work; returns the device status (CAV_OK, CAV_E_NONFINITE, ...). */
int cav_sync(cav_sim* sim);

int cav_get_time(cav_sim* sim, double* t, double* dt_next);
int cav_set_time(cav_sim* sim, double t);
int cav_get_stats(cav_sim* sim, cav_stats* out);

/* Device-side trace: one row per sample,
 *   [t, a(re,im) x N, S(re,im) x N, <m_s>(x,y,z) x n_sub]     (1 + 4N + 3 n_sub doubles)
 * adaptive runs clamp steps onto t_set + k*sample_dt; fixed-step runs sample every
 * round(sample_dt/fixed_dt) accepted steps.  capacity rows are kept on the device; sampling
 * stops when full.  sample_dt <= 0 disables.  Resets the trace. */
int cav_set_trace(cav_sim* sim, double sample_dt, int capacity);
int cav_trace_row_len(cav_sim* sim, int* row_len);
int cav_get_trace(cav_sim* sim, double* out /* [capacity][row_len] host */, int* n_samples);

/* Tuning knob (optional): cells per thread block of the stage kernel; 0 = automatic. */
int cav_set_block_cells(cav_sim* sim, int cells_per_block);

/* Tuning knob (optional): 1 (default) = odd stages sweep the grid in reverse block order so that
 * the tail of one stage's data is still in L2 when the next stage starts; 0 = always forward. */
int cav_set_sweep_order(cav_sim* sim, int serpentine);

/* Which implementation of the fused stage kernel runs (same arithmetic, PAPER.md:150-159 / DESIGN.md "Kernels"):
 *   CAV_PATH_TMA      persistent TMA/mbarrier-pipelined kernel; needs 16-byte row strides and a mode count whose streams fit
 *                     the shared-memory rings, else cav_set_kernel_path returns CAV_E_UNSUPPORTED.  Grids of more than
 *                     512 x (number of SMs) cells whose nx*sizeof(T) is not a multiple of 16 are stored with padded rows
 *                     inside the library (the ABI arrays stay dense) and run on this path only: GENERIC / BLOCK / COOP
 *                     then return CAV_E_UNSUPPORTED; smaller grids with such an nx are not eligible;
 *   CAV_PATH_GENERIC  register/LDG kernel for any shape;
 *   CAV_PATH_BLOCK    grids of at most 1024 cells: the whole run in ONE thread block (the batched small-grid kernel with a
 *                     single replica: stage state in shared memory, slopes in registers, no launch per stage); the
 *                     slope of the final state is not cached (the next run re-evaluates k1: rhs_evals counts it);
 *                     CAV_E_UNSUPPORTED for larger grids;
 *   CAV_PATH_COOP     grids of 1025 .. 512 x (number of SMs) cells: the whole run in ONE cooperative launch of
 *                     ceil(cells/512) co-resident blocks, a grid barrier per evaluation instead of a kernel boundary (the
 *                     same kernel as BLOCK, stage state and block partials through global memory); like BLOCK it does not
 *                     cache the final slope.  Cooperative grids do not overlap with each other: for many concurrent
 *                     simulations on several streams (a sweep) choose GENERIC.  CAV_E_UNSUPPORTED outside that range;
 *   CAV_PATH_AUTO     (default) BLOCK up to 1024 cells; COOP up to 512 x (number of SMs) cells; above that TMA when
 *                     eligible, else GENERIC.
 * cav_get_kernel_path reports what the next run will use (CAV_PATH_GENERIC, _TMA, _BLOCK or _COOP). */
int cav_set_kernel_path(cav_sim* sim, int path);
int cav_get_kernel_path(cav_sim* sim, int* path);

/* Tuning knob (optional): 1 (default) = inside the device-side step loop, consecutive stage kernels of the TMA path
 * are joined by programmatic dependencies (the next kernel's blocks become resident and run their data-independent
 * prologue while the previous kernel drains; results are unchanged); 0 = full kernel-to-kernel dependencies.
 * cav_get_stage_overlap reports whether the graph of the last run was built with them (0 before any run, on the
 * generic path, in CAV_LAUNCH_STREAM mode, or when the driver refused the edges and the library fell back). */
int cav_set_stage_overlap(cav_sim* sim, int on);
int cav_get_stage_overlap(cav_sim* sim, int* active);

/* ---------------------------------------------------------------------------------------------------------
 * Variants.
 * --------------------------------------------------------------------------------------------------------- */

/* Per-mode polarisation.  The paper applies every mode's RF field along x^ and couples it to
 * m^- = m_x - i m_y (Eqs. 1-2).  With a polarisation p_n and a quadrature axis q_n per mode
 *     S_n = (1/W_n) sum_r u_n(r) (m_c.p_n - i m_c.q_n),      B_rf(r) = sum_n c_n u_n(r) p_n
 * (reading G32; p = x^, q = y^ is the paper's case).  pol: [N][3] host, normalised on entry; quad: [N][3] host,
 * used as given, or NULL for q_n = z^ x p_n (static field along z^).  pol == NULL restores x^.  Call after cav_set_modes
 * (a new mode set restores x^).  Implemented in the small-grid kernel (CAV_PATH_BLOCK / CAV_PATH_COOP), in the TMA stage
 * kernels for up to 8 modes (their own instantiation) and in the generic stage kernels, which a run with more modes uses
 * whatever cav_set_kernel_path says; CAV_E_UNSUPPORTED together with cav_set_demag, in a joint sweep, or with more than
 * 8 modes on a grid stored with padded rows. */
int cav_set_polarisation(cav_sim* sim, const double* pol, const double* quad);

/* Integrator.  CAV_INTEGRATOR_UNIFIED (default): LLG and mode ODEs in ONE Dormand-Prince step (tier 1).
 * CAV_INTEGRATOR_SPLIT: the paper's tier-2 co-simulation loop (PAPER.md:169-193 Listing 1, :199), kept as a comparison
 * scheme: per step dt, (i) read the overlaps S_n of the current m, (ii) advance a_n over dt by classic RK4 with S_n held
 * constant, (iii) set the RF field from the new a_n and hold it constant, (iv) advance the LLG equation over dt by n_llg
 * Dormand-Prince steps of dt/n_llg (reading G33).  Fixed step only: cav_run* must be called with
 * fixed_dt = dt (CAV_E_ARG otherwise); max_steps counts co-simulation steps; the statistics count LLG sub-steps
 * (accepted = steps x n_llg, 6 n_llg + 1 evaluations per step); choose a trace sample_dt that is a multiple of dt.
 * Small-grid kernel only: CAV_E_UNSUPPORTED for grids of more than 512 x (number of SMs) cells; the run uses
 * CAV_PATH_BLOCK / CAV_PATH_COOP whatever cav_set_kernel_path says. */
enum { CAV_INTEGRATOR_UNIFIED = 0, CAV_INTEGRATOR_SPLIT = 1 };
int cav_set_integrator(cav_sim* sim, int integrator, int n_llg);

/* Dipolar (demagnetising) field.  The paper switches it off ("Dipolar interactions are
 * disabled"), so it is off by default; on = 1 adds
 *     B_d(r_i) = -mu0 Ms sum_j N(r_i - r_j) . m_tot(r_j)       (open boundary; N: Newell's cell-averaged tensor; m_tot: sum
 * over the sublattices) to the effective field of every evaluation, as a zero-padded FFT convolution (cuFFT, loaded on
 * demand: CAV_E_UNSUPPORTED if it cannot be, for the transforms along x; the y and z transforms of the occupied rows and
 * planes and the tensor product are kernels of this library) in front of each stage kernel.  A different roofline from
 * the fused stencil: runs use the generic stage kernels whatever cav_set_kernel_path says.  In CAV_LAUNCH_GRAPH mode cuFFT's launches are recorded by stream capture into the body of
 * the run graph's WHILE node, so cav_run stays one asynchronous graph launch with no host round trip (if that capture
 * is refused the run is enqueued from the host, as in CAV_LAUNCH_STREAM).  Not available with cav_set_polarisation / the split integrator,
 * nor for grids stored with padded rows (CAV_E_UNSUPPORTED).  DESIGN.md reading G34. */
int cav_set_demag(cav_sim* sim, int on);

/* On-device spectroscopy: the Fourier sums behind the paper's spectra |FFT(m^-)|^2 + |FFT(a)|^2,
 * accumulated inside the step controller at every trace sample (cav_set_trace decides when) instead of copying the
 * trace to the host:   X[k][sig] += x_sig(t_j) exp(+i w_k t_j),   w_k = omega_lo + k (omega_hi - omega_lo)/(n_bins - 1),
 * for the 2N + n_sub signals x = a_1..a_N, S_1..S_N, mu_1..mu_nsub with mu_s = <m_s,x> - i <m_s,y> the plain average of
 * sublattice s (the paper's m^-; (mu_1 - mu_2)/2 is the Neel vector's transverse part, PAPER.md:335 - the sums are linear)
 * (a component ~ exp(-i w0 t), peaks at w_k = w0; a frequency grid finer than 1/T is the paper's zero
 * padding).  Any path, any grid, N = 0 included.  n_bins = 0 switches it off; the call zeroes the sums; a new mode set
 * drops them.  cav_get_spectrum copies [n_bins][2N + n_sub][2] doubles to the host and reports the number of samples
 * accumulated. */
int cav_set_spectrum(cav_sim* sim, int n_bins, double omega_lo, double omega_hi);
int cav_get_spectrum(cav_sim* sim, double* out /* [n_bins][2N + n_sub][2] host */, long long* n_samples);

/* Number of kernels this library has launched for this handle (stage kernels + setup). */
int cav_get_launch_count(cav_sim* sim, long long* n);

/* ---------------------------------------------------------------------------------------------------------
 * Batched sweeps of small grids.  The paper's own workloads are parameter sweeps of a tiny grid
 * (8 x 8 x 1 cells x 41 / 21 field values): independent simulations that differ in B0
 * and/or the mode parameters.  A batch integrates n_rep such replicas in ONE kernel launch: one thread block per
 * replica, one thread per cell, the whole adaptive RK45 loop of the same coupled system (same tableau, controller,
 * error norm and renormalisation as cav_run) inside the kernel with the stage
 * state in shared memory and the slopes in registers - no kernel launch, no global-memory round trip and no
 * grid-wide reduction per stage.  Limits: nx*ny*nz <= 1024 cells, N <= CAV_MAX_MODES.
 * All arrays are HOST arrays copied at the call; replicas are laid out [n_rep][...] with the single-simulation
 * layouts above.  Not thread-safe per handle.
 * --------------------------------------------------------------------------------------------------------- */
typedef struct cav_batch cav_batch; /* opaque */

/* params->B0 is the default static field of every replica.  CAV_E_ARG if the grid has more than 1024 cells. */
int cav_batch_create(const cav_grid* grid, const cav_params* params, int n_rep, cav_batch** out);
int cav_batch_destroy(cav_batch* b);
int cav_batch_set_stream(cav_batch* b, void* cuda_stream);

/* Static field per replica, [n_rep][3] tesla. */
int cav_batch_set_field(cav_batch* b, const double* B0);

/* Modes: profiles u [N][nz][ny][nx] (batch precision) are common to all replicas; omega, kappa, g, Gamma, Phi are
 * [N] (per_replica == 0) or [n_rep][N] (per_replica != 0); Gamma, Phi may be NULL.  Zeroes the amplitudes. */
int cav_batch_set_modes(cav_batch* b, int N, const void* u, const double* omega, const double* kappa,
                        const double* g, const double* Gamma, const double* Phi, int per_replica);

/* Initial magnetisation [n_sub][3][nz][ny][nx] for all replicas (per_replica == 0) or [n_rep][n_sub][3][nz][ny][nx];
 * normalised per cell on entry.  Amplitudes [N][2] or [n_rep][N][2]. */
int cav_batch_set_m(cav_batch* b, const void* m, int per_replica);
int cav_batch_set_a(cav_batch* b, const double* a_re_im, int per_replica);

/* Backward coupling as cav_set_backaction, common to all replicas ([N] arrays).  Call after cav_batch_set_modes. */
int cav_batch_set_backaction(cav_batch* b, const double* g_b, const double* Gamma_b, const double* Phi_b);

/* Drive as cav_set_drive, common to all replicas ([N] arrays).  Call after cav_batch_set_modes. */
int cav_batch_set_drive(cav_batch* b, const double* amp_re_im, const double* t0, const double* sigma, const double* omega_d);

/* Polarisation, integrator and spectrum as cav_set_polarisation / cav_set_integrator / cav_set_spectrum, common to all
 * replicas; the spectrum is kept per replica: [n_rep][n_bins][2N + n_sub][2], n_samples [n_rep].  Call after cav_batch_set_modes. */
int cav_batch_set_polarisation(cav_batch* b, const double* pol, const double* quad);
int cav_batch_set_integrator(cav_batch* b, int integrator, int n_llg);
int cav_batch_set_spectrum(cav_batch* b, int n_bins, double omega_lo, double omega_hi);
int cav_batch_get_spectrum(cav_batch* b, double* out, long long* n_samples);

/* Trace rows as cav_set_trace, per replica; resets the traces. */
int cav_batch_set_trace(cav_batch* b, double sample_dt, int capacity);
int cav_batch_trace_row_len(cav_batch* b, int* row_len);

/* Advance every replica to t_end (or by max_steps attempted steps if max_steps > 0); arguments as cav_run_steps.
 * Asynchronous on the stream; the cav_batch_get_* calls synchronise. */
int cav_batch_run(cav_batch* b, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps);

/* Results.  cav_batch_get_stats also returns the first non-zero device status of any replica. */
int cav_batch_get_m(cav_batch* b, void* m_out /* [n_rep][n_sub][3][nz][ny][nx] */);
int cav_batch_get_a(cav_batch* b, double* a_out /* [n_rep][N][2] */);
int cav_batch_get_stats(cav_batch* b, cav_stats* out /* [n_rep] */);
int cav_batch_get_trace(cav_batch* b, double* out /* [n_rep][capacity][row_len] */, int* n_samples /* [n_rep] */);

/* ---------------------------------------------------------------------------------------------------------
 * Sweeps of mid-size grids: several simulations in one launch (the paper's 41-point field sweep, PAPER.md:229, :335,
 * on grids that are too large for cav_batch and too small to fill the GPU alone, e.g. 64 x 64 x 16 cells).
 * A sweep is a joint LAUNCHER over ordinary cav_sim handles: create and configure every simulation as usual (same grid,
 * precision, material and cell constants and number of modes; at most 8 modes (2 for the antiferromagnet); B0, mode parameters, profiles
 * and state may differ; all on the same stream), then cav_sweep_run advances all of them in ONE device-side loop: the
 * plane-tiles of all simulations form one work list for the persistent TMA grid, and every simulation keeps its own step
 * size, accept/reject decisions, trace and statistics.  Afterwards every cav_get_* / cav_set_* call works on the single
 * handles as before; results are the same as running each simulation alone up to the summation order of the overlap sums.
 * Do not run a member simulation while a sweep run is in flight; create the sweep after cav_set_modes (it is re-planned
 * automatically when traces / spectra are re-allocated).  CAV_E_UNSUPPORTED when the TMA path is not eligible.
 * --------------------------------------------------------------------------------------------------------- */
typedef struct cav_sweep cav_sweep; /* opaque */
int cav_sweep_create(cav_sim* const* sims, int n, cav_sweep** out);
int cav_sweep_destroy(cav_sweep* sweep);
/* Arguments as cav_run_steps, applied to every simulation.  Asynchronous on the simulations' stream. */
int cav_sweep_run(cav_sweep* sweep, double t_end, double tol, double fixed_dt, double dt_init, long long max_steps);

/* ---------------------------------------------------------------------------------------------------------
 * An entry point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid it): the overlaps of a given state with given mode profiles,
 *     S_n = (1/N_cells) sum_r u_n(r) (m_c,x(r) - i m_c,y(r)),   m_c = the mean over the sublattices
 * (Eq. 18 with the paper's polarisation x^; CAV_NORM_NCELLS), the same two-pass fixed-order reduction
 * as the stage kernels' (block partials in fp64, then one sum in block order: results are bitwise reproducible).
 *   m_dev  [n_sub][3][nz][ny][nx], u_dev [N][nz][ny][nx]: DEVICE buffers in `precision` (CAV_F32 | CAV_F64), read only
 *   S_out_dev [N][2] doubles (Re, Im): DEVICE buffer, written; the caller owns all three
 *   cuda_stream: a cudaStream_t (NULL = the default stream); the call is asynchronous on it
 * No handle, no cudaMalloc / cudaFree / allocating library routine: the block partials live in ONE file-scope __device__
 * array of CAV_NOALLOC_SCRATCH_BYTES (1 MiB + 256 B) that every GPU loading the library holds until exit.  Hence the
 * limits: nx*ny*nz <= CAV_NOALLOC_MAX_CELLS (2^24, the largest configuration of BASELINE.json) and N <= CAV_MAX_MODES;
 * beyond them CAV_E_UNSUPPORTED, with the reason in cav_noalloc_last_error().  Every call on a device shares that array
 * (the call clears the words that must start at zero itself): calls that overlap on the GPU - two streams, or two
 * threads - RACE; serialise them (one stream, or events).  Other errors: CAV_E_ARG, CAV_E_CUDA.
 * --------------------------------------------------------------------------------------------------------- */
#define CAV_NOALLOC_MAX_CELLS (1LL << 24)
#define CAV_NOALLOC_SCRATCH_BYTES (256 + 8 * (CAV_NOALLOC_MAX_CELLS / 8192) * 2 * CAV_MAX_MODES)
int cav_overlaps_noalloc(const void* m_dev, const void* u_dev, int precision, int nx, int ny, int nz, int n_sub, int N,
                         double* S_out_dev, void* cuda_stream);
/* Text of the calling thread's last cav_overlaps_noalloc failure ("" after a success). */
const char* cav_noalloc_last_error(void);

const char* cav_strerror(int status);
const char* cav_last_cuda_error(cav_sim* sim);
const char* cav_version(void);

#ifdef __cplusplus
}
#endif
#endif /* CAVMAG_H_ */
