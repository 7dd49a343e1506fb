// =====================================================================================
//  cavmag_oracle.cpp — TEST INFRASTRUCTURE, NOT THE PRODUCT.
//
//  Plain, slow, obviously-correct fp64 CPU implementation of the hot path of
//  arXiv 2603.03706 tier 1: the Landau-Lifshitz-Gilbert equation
//  on a finite-difference grid integrated together with N cavity-mode ODEs in ONE
//  Dormand-Prince RK5(4) step.  Only tests/, __graft_entry__.smoke() and bench.py's
//  cpu_baseline / --impl reference leg may call this.  It shares no code, header, table
//  or helper with paper_2603_03706_b200/ (the CUDA path) and neither includes the other.
//
//  It is an iteration, so the oracle is the algorithm written out step by step in the
//  paper's notation (readings G1..G30 of SURVEY.md section 8(c), restated in DESIGN.md):
//
//    state   m_s(r) in R^3, |m|=1, s = 1[,2] sublattices;   a_n in C, n = 1..N
//    (1) m_c  = m_1  or (m_1+m_2)/2
//    (2) S_n  = (1/W_n) sum_r u_n(r) (m_c,x - i m_c,y)       PAPER.md:156 Eq.18, :45 Eq.2
//    (3) G_n  = g_n + Gamma_n e^{i Phi_n};
//        da_n/dt = -(i w_n + kappa_n) a_n + i G_n S_n + eta_n(t)   PAPER.md:119 Eq.12, :317 Eq.19
//        eta_n(t) = A_n exp(-(t-t0_n)^2/(2 sigma_n^2)) exp(-i w_d,n (t-t0_n))   Gaussian pulse
//        (evaluated at the stage times t + c_s h; absent unless drive arrays are given - reading G27)
//    (4) c_n  = (2/gamma) Re[G_b,n a_n];  B_rf(r) = x^ sum_n c_n u_n(r)      (G_b = G unless a separate backward
//        coupling is given: non-reciprocal g_f != g_b with h0 = 2 g_b/gamma)
//                                                           PAPER.md:65 Eq.5, :121 Eq.13, :159
//        Per-mode polarisation (the paper fixes x^): with a unit vector p_n and a
//        quadrature axis q_n (default z^ x p_n) the mode couples to  m_c.p_n - i m_c.q_n  in (2) and its field
//        points along p_n in (4).  p = x^, q = y^ is the paper's case (reading G32).
//    (5) B_s  = B0 + (2A/Ms) sum_{d,+-} [m_s(r +- e_d) - m_s(r)]/D_d^2   (open boundary)
//             + (2Ku/Ms)(m_s . k^) k^ + B_rf - B_E m_other
//    (6) dm_s/dt = -gamma/(1+alpha^2) [ m x B + alpha m x (m x B) ]
//
//  Pins (tests/test_oracle_*.py, -m "not gpu"): Kittel line (Eq. 9), polariton branches
//  (Eq. 6/7), Rabi period pi/g, N+1 arrowhead eigenvalues (Eq. 14), level attraction
//  (Eq. 20), discrete spin-wave dispersion + overlap coupling, selection rule (Eq. 10/11),
//  AFMR (Eq. 15/16), |m| conservation, convergence order 5, scipy DOP853 cross-check.
//  PARITY UNPINNED: the step-size controller constants (0.8, 1/5, [0.5,2]), the error-norm
//  composition and the default initial step — the paper names "RK45 adaptive" only
//  (PAPER.md:150); adaptive runs are compared on observables.
//
//  Second integrator, orc_run_split: the paper's TIER-2 operator-split loop (PAPER.md:169-193 Listing 1, :199),
//  kept as a comparison scheme: per step dt, (i) read the overlaps S_n of the current m,
//  (ii) advance a_n over dt by classic RK4 with S_n held constant, (iii) set the RF field from the NEW a_n and hold it
//  constant, (iv) advance the LLG equation over dt.  Reading G33: step (iv) = n_llg Dormand-Prince 5(4) steps of dt/n_llg
//  with the same per-cell renormalisation as the unified step (mumax+ runs its own adaptive solver there, unspecified).
//  Pins: first-order convergence of the Rabi period to pi/g and the printed errors (Fig. 11).
//
//  orc_dft: the plain discrete Fourier sum X(w) = sum_j x_j exp(+i w t_j) of a sampled complex trace at arbitrary
//  frequencies w (signals ~ exp(-i w t)) - the definition behind the paper's zero-padded FFT spectra
//  |FFT(m^-)|^2 + |FFT(a)|^2.  Pinned against numpy.fft on the FFT grid.
//
//  Dipolar (demagnetising) field: the paper switches it off ("Dipolar interactions are
//  disabled", :97 Walker modes "not considered"); real samples need it, so it is an OPTIONAL term here (reading G34):
//      B_d(r_i) = -mu0 Ms sum_j N(r_i - r_j) . m_tot(r_j),   m_tot = sum over sublattices,  open boundary (finite sample)
//  with N the demagnetising tensor between two uniformly magnetised cells averaged over the target cell (Newell,
//  Williams & Dunlop 1993, restated in orc_demag_tensor).  The oracle is the plain definition: a direct O(N_cells^2) sum.
//  Pins: self term of a cube = 1/3, trace 1 at the origin and 0 elsewhere, point-dipole far field, brute-force
//  sub-cell dipole sums, demagnetising factors of a uniformly magnetised cube / slab.
//
//  Build:  g++ -O2 -ffp-contract=off -fopenmp -shared -fPIC  (see oracle/build.py)
// =====================================================================================
#include <cmath>
#include <cstdlib>
#include <cstring>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

extern "C" {

struct orc_problem {
    int nx, ny, nz;
    double dx, dy, dz;
    double Ms, Aex, Ku;
    double axis[3];          // unit anisotropy axis k^
    double alpha, gamma;
    double B0[3];            // tesla
    int n_sub;               // 1 ferromagnet, 2 two-sublattice antiferromagnet
    double B_exch_inter;     // tesla; AFM: B_s += -B_exch_inter * m_other(r)
    int renormalize;         // 1: m_new = y5/|y5| before the 7th evaluation
    int norm_sum_u;          // 0: W_n = N_cells (Eq. 18);  1: W_n = sum_r u_n(r)
    int N;                   // number of cavity modes
    const double* u;         // [N][nz][ny][nx]
    const double* omega;     // [N] rad/s
    const double* kappa;     // [N] rad/s
    const double* g;         // [N] rad/s
    const double* Gamma;     // [N] rad/s
    const double* Phi;       // [N] rad
    // external drive eta_n(t) (PAPER.md:43 Eq. 1, :119 Eq. 12; Gaussian pulse of PAPER.md:229); eta_amp == NULL: none
    const double* eta_amp;   // [N][2] complex amplitude A_n (units of a per second)
    const double* eta_t0;    // [N] pulse centre, s
    const double* eta_sigma; // [N] pulse width, s
    const double* eta_wd;    // [N] carrier, rad/s (NULL: baseband pulse)
    // non-reciprocal coupling: backward (cavity-to-magnon) coupling G_b = g_b + Gamma_b e^{i Phi_b} used in
    // the feedback field h0 = 2 g_b / gamma; g_b == NULL: reciprocal (G_b = G)
    const double* g_b;       // [N] rad/s
    const double* Gamma_b;   // [N] rad/s (NULL: 0)
    const double* Phi_b;     // [N] rad   (NULL: 0)
    // per-mode polarisation (reading G32): pol == NULL: every mode along x^ with quadrature y^
    const double* pol;       // [N][3] unit vectors p_n: direction of the mode's RF field
    const double* quad;      // [N][3] quadrature axes q_n (NULL: q_n = z^ x p_n): the mode couples to m.p_n - i m.q_n
    // dipolar field (reading G34): NULL = off (the paper's setting)
    const double* demag_N;   // [(2nz-1)][(2ny-1)][(2nx-1)][6] tensor N(dx_i, dy_j, dz_k) for offsets -(n-1)..(n-1): xx,yy,zz,xy,xz,yz
};

struct orc_stats {
    long long accepted, rejected, rhs_evals;
    double dt_min, dt_max, dt_next, t;
    int status;              // 0 ok, 1 non-finite, 2 dt underflow
};

void orc_set_threads(int n) {
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
int orc_get_threads(void) {
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

}  // extern "C"

namespace {

inline long long ncell(const orc_problem* P) { return (long long)P->nx * P->ny * P->nz; }

// polarisation p_n and quadrature axis q_n of mode n (reading G32): x^, y^ unless given; q defaults to z^ x p
void mode_axes(const orc_problem* P, int n, double* pv, double* qv) {
    if (!P->pol) { pv[0] = 1.0; pv[1] = 0.0; pv[2] = 0.0; qv[0] = 0.0; qv[1] = 1.0; qv[2] = 0.0; return; }
    for (int i = 0; i < 3; ++i) pv[i] = P->pol[3 * n + i];
    if (P->quad) { for (int i = 0; i < 3; ++i) qv[i] = P->quad[3 * n + i]; }
    else { qv[0] = -pv[1]; qv[1] = pv[0]; qv[2] = 0.0; }      // z^ x p
}

// ---- step (2): S_n = (1/W_n) sum_r u_n(r) (m_c,x(r) - i m_c,y(r)) ---------------------
// Summed plane by plane in fixed z order so the result does not depend on the thread count.
void overlaps(const orc_problem* P, const double* m, double* S /*[N][2]*/) {
    const long long nc = ncell(P), plane = (long long)P->nx * P->ny;
    for (int n = 0; n < P->N; ++n) {
        const double* un = P->u + (long long)n * nc;
        double pv[3], qv[3];
        mode_axes(P, n, pv, qv);
        std::vector<double> pre(P->nz), pim(P->nz), pw(P->nz);
#pragma omp parallel for schedule(static)
        for (int z = 0; z < P->nz; ++z) {
            double sre = 0.0, sim = 0.0, sw = 0.0;
            for (long long i = (long long)z * plane; i < (long long)(z + 1) * plane; ++i) {
                double mcx, mcy, mcz;
                if (P->n_sub == 1) {
                    mcx = m[0 * nc + i];
                    mcy = m[1 * nc + i];
                    mcz = m[2 * nc + i];
                } else {  // step (1): net magnetisation couples
                    mcx = 0.5 * (m[0 * nc + i] + m[3 * nc + 0 * nc + i]);
                    mcy = 0.5 * (m[1 * nc + i] + m[3 * nc + 1 * nc + i]);
                    mcz = 0.5 * (m[2 * nc + i] + m[3 * nc + 2 * nc + i]);
                }
                if (!P->pol) {
                    sre += un[i] * mcx;       // Re[u (mx - i my)] = u mx
                    sim += -(un[i] * mcy);    // Im[u (mx - i my)] = -u my
                } else {                      // u (m.p - i m.q)
                    sre += un[i] * (mcx * pv[0] + mcy * pv[1] + mcz * pv[2]);
                    sim += -(un[i] * (mcx * qv[0] + mcy * qv[1] + mcz * qv[2]));
                }
                sw += un[i];
            }
            pre[z] = sre; pim[z] = sim; pw[z] = sw;
        }
        double sre = 0.0, sim = 0.0, sw = 0.0;
        for (int z = 0; z < P->nz; ++z) { sre += pre[z]; sim += pim[z]; sw += pw[z]; }
        const double W = P->norm_sum_u ? sw : (double)nc;
        S[2 * n + 0] = sre / W;
        S[2 * n + 1] = sim / W;
    }
}

// ---- steps (3), (4): mode slopes da_n/dt from given overlaps S, and the RF weights c_n = (2/gamma) Re[G_b,n a_n] ----
void mode_rhs(const orc_problem* P, double t, const double* a, const double* S, double* da, double* c) {
    for (int n = 0; n < P->N; ++n) {
        const double Gre = P->g[n] + P->Gamma[n] * std::cos(P->Phi[n]);
        const double Gim = P->Gamma[n] * std::sin(P->Phi[n]);
        const double are = a[2 * n], aim = a[2 * n + 1];
        const double Sre = S[2 * n], Sim = S[2 * n + 1];
        // -(i w + kappa) a  =  (-kappa are + w aim) + i (-kappa aim - w are)
        // i G S             =  (-(Gre Sim + Gim Sre)) + i (Gre Sre - Gim Sim)
        if (da) {
            da[2 * n + 0] = (-P->kappa[n] * are + P->omega[n] * aim) - (Gre * Sim + Gim * Sre);
            da[2 * n + 1] = (-P->kappa[n] * aim - P->omega[n] * are) + (Gre * Sre - Gim * Sim);
            if (P->eta_amp) {   // + eta_n(t): Gaussian envelope times carrier e^{-i w_d (t - t0)}
                const double x = t - P->eta_t0[n];
                const double env = std::exp(-(x * x) / (2.0 * P->eta_sigma[n] * P->eta_sigma[n]));
                const double ph = P->eta_wd ? P->eta_wd[n] * x : 0.0;
                const double Are = P->eta_amp[2 * n], Aim = P->eta_amp[2 * n + 1];
                da[2 * n + 0] += env * (Are * std::cos(ph) + Aim * std::sin(ph));
                da[2 * n + 1] += env * (Aim * std::cos(ph) - Are * std::sin(ph));
            }
        }
        if (c) {
            double Gbre = Gre, Gbim = Gim;                        // backward coupling: reciprocal unless given
            if (P->g_b) {
                const double Gm = P->Gamma_b ? P->Gamma_b[n] : 0.0, Ph = P->Phi_b ? P->Phi_b[n] : 0.0;
                Gbre = P->g_b[n] + Gm * std::cos(Ph);
                Gbim = Gm * std::sin(Ph);
            }
            c[n] = (2.0 / P->gamma) * (Gbre * are - Gbim * aim);   // (2/gamma) Re[G_b a]
        }
    }
}

// ---- dipolar field (reading G34): B_d(r_i) = -mu0 Ms sum_j N(r_i - r_j) . m_tot(r_j), direct sum over all pairs ----
void demag_field(const orc_problem* P, const double* m, double* bd /*[3][nc]*/) {
    const int nx = P->nx, ny = P->ny, nz = P->nz;
    const long long nc = ncell(P);
    const int tx = 2 * nx - 1, ty = 2 * ny - 1;
    const double pref = -4e-7 * M_PI * P->Ms;
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < nc; ++i) {
        const int xi = (int)(i % nx), yi = (int)((i / nx) % ny), zi = (int)(i / ((long long)nx * ny));
        double hx = 0.0, hy = 0.0, hz = 0.0;
        for (int zj = 0; zj < nz; ++zj)
            for (int yj = 0; yj < ny; ++yj)
                for (int xj = 0; xj < nx; ++xj) {
                    const long long j = ((long long)zj * ny + yj) * nx + xj;
                    double mx = m[j], my = m[nc + j], mz = m[2 * nc + j];
                    if (P->n_sub == 2) { mx += m[3 * nc + j]; my += m[4 * nc + j]; mz += m[5 * nc + j]; }
                    const double* T = P->demag_N + 6 * (((long long)(zi - zj + nz - 1) * ty + (yi - yj + ny - 1)) * tx + (xi - xj + nx - 1));
                    hx += T[0] * mx + T[3] * my + T[4] * mz;
                    hy += T[3] * mx + T[1] * my + T[5] * mz;
                    hz += T[4] * mx + T[5] * my + T[2] * mz;
                }
        bd[i] = pref * hx; bd[nc + i] = pref * hy; bd[2 * nc + i] = pref * hz;
    }
}

// ---- steps (5), (6): dm/dt of every cell for given RF weights c_n ----
void llg_rhs(const orc_problem* P, const double* m, const double* c, double* dm) {
    const int nx = P->nx, ny = P->ny, nz = P->nz, N = P->N;
    const long long nc = ncell(P);
    const double pref_ex = 2.0 * P->Aex / P->Ms;
    const double pref_an = 2.0 * P->Ku / P->Ms;
    const double wx = 1.0 / (P->dx * P->dx), wy = 1.0 / (P->dy * P->dy), wz = 1.0 / (P->dz * P->dz);
    const double llg = -P->gamma / (1.0 + P->alpha * P->alpha);
    std::vector<double> bdem;                                   // dipolar field of the total magnetisation, [3][nc]
    if (P->demag_N) { bdem.assign(3 * (size_t)nc, 0.0); demag_field(P, m, bdem.data()); }
    std::vector<double> cp(3 * (size_t)(N > 0 ? N : 1));      // c_n p_n (general polarisation only)
    if (P->pol)
        for (int n = 0; n < N; ++n) {
            double pv[3], qv[3];
            mode_axes(P, n, pv, qv);
            for (int i = 0; i < 3; ++i) cp[3 * n + i] = c[n] * pv[i];
        }

    for (int s = 0; s < P->n_sub; ++s) {
        const double* ms = m + (long long)s * 3 * nc;
        const double* mo = (P->n_sub == 2) ? m + (long long)(1 - s) * 3 * nc : nullptr;
        double* ds = dm + (long long)s * 3 * nc;
#pragma omp parallel for schedule(static)
        for (int z = 0; z < nz; ++z)
            for (int y = 0; y < ny; ++y)
                for (int x = 0; x < nx; ++x) {
                    const long long i = ((long long)z * ny + y) * nx + x;
                    const double mx = ms[i], my = ms[nc + i], mz = ms[2 * nc + i];
                    // step (5): effective field
                    double Bx = P->B0[0], By = P->B0[1], Bz = P->B0[2];
                    double lx = 0.0, ly = 0.0, lz = 0.0;   // sum over in-grid neighbours
                    if (x > 0)      { long long j = i - 1;  lx += (ms[j] - mx) * wx; ly += (ms[nc + j] - my) * wx; lz += (ms[2 * nc + j] - mz) * wx; }
                    if (x < nx - 1) { long long j = i + 1;  lx += (ms[j] - mx) * wx; ly += (ms[nc + j] - my) * wx; lz += (ms[2 * nc + j] - mz) * wx; }
                    if (y > 0)      { long long j = i - nx; lx += (ms[j] - mx) * wy; ly += (ms[nc + j] - my) * wy; lz += (ms[2 * nc + j] - mz) * wy; }
                    if (y < ny - 1) { long long j = i + nx; lx += (ms[j] - mx) * wy; ly += (ms[nc + j] - my) * wy; lz += (ms[2 * nc + j] - mz) * wy; }
                    if (z > 0)      { long long j = i - (long long)nx * ny; lx += (ms[j] - mx) * wz; ly += (ms[nc + j] - my) * wz; lz += (ms[2 * nc + j] - mz) * wz; }
                    if (z < nz - 1) { long long j = i + (long long)nx * ny; lx += (ms[j] - mx) * wz; ly += (ms[nc + j] - my) * wz; lz += (ms[2 * nc + j] - mz) * wz; }
                    Bx += pref_ex * lx; By += pref_ex * ly; Bz += pref_ex * lz;
                    const double mk = mx * P->axis[0] + my * P->axis[1] + mz * P->axis[2];
                    Bx += pref_an * mk * P->axis[0]; By += pref_an * mk * P->axis[1]; Bz += pref_an * mk * P->axis[2];
                    if (!P->pol) {
                        double brf = 0.0;
                        for (int n = 0; n < N; ++n) brf += c[n] * P->u[(long long)n * nc + i];
                        Bx += brf;                       // RF field along x^
                    } else {                             // RF field sum_n c_n u_n(r) p_n (reading G32)
                        double bx = 0.0, by = 0.0, bz = 0.0;
                        for (int n = 0; n < N; ++n) {
                            const double un = P->u[(long long)n * nc + i];
                            bx += cp[3 * n] * un; by += cp[3 * n + 1] * un; bz += cp[3 * n + 2] * un;
                        }
                        Bx += bx; By += by; Bz += bz;
                    }
                    if (mo) { Bx -= P->B_exch_inter * mo[i]; By -= P->B_exch_inter * mo[nc + i]; Bz -= P->B_exch_inter * mo[2 * nc + i]; }
                    if (P->demag_N) { Bx += bdem[i]; By += bdem[nc + i]; Bz += bdem[2 * nc + i]; }
                    // step (6): LLG in explicit Landau-Lifshitz form
                    const double tx = my * Bz - mz * By, ty = mz * Bx - mx * Bz, tz = mx * By - my * Bx;   // m x B
                    const double dx_ = my * tz - mz * ty, dy_ = mz * tx - mx * tz, dz_ = mx * ty - my * tx; // m x (m x B)
                    ds[i]          = llg * (tx + P->alpha * dx_);
                    ds[nc + i]     = llg * (ty + P->alpha * dy_);
                    ds[2 * nc + i] = llg * (tz + P->alpha * dz_);
                }
    }
}

// ---- the coupled right-hand side f(t, m, a): every term at the same state (no operator splitting) ----
void rhs(const orc_problem* P, double t, const double* m, const double* a, double* dm, double* da, double* S_out) {
    const int N = P->N;
    std::vector<double> S(2 * (size_t)(N > 0 ? N : 1));
    overlaps(P, m, S.data());
    if (S_out) std::memcpy(S_out, S.data(), sizeof(double) * 2 * N);
    std::vector<double> c((size_t)(N > 0 ? N : 1));
    mode_rhs(P, t, a, S.data(), da, c.data());
    llg_rhs(P, m, c.data(), dm);
}

// Dormand-Prince 5(4) (Dormand & Prince 1980), textbook constants — the paper gives none (G11).
const double A21 = 1.0 / 5.0;
const double A31 = 3.0 / 40.0, A32 = 9.0 / 40.0;
const double A41 = 44.0 / 45.0, A42 = -56.0 / 15.0, A43 = 32.0 / 9.0;
const double A51 = 19372.0 / 6561.0, A52 = -25360.0 / 2187.0, A53 = 64448.0 / 6561.0, A54 = -212.0 / 729.0;
const double A61 = 9017.0 / 3168.0, A62 = -355.0 / 33.0, A63 = 46732.0 / 5247.0, A64 = 49.0 / 176.0, A65 = -5103.0 / 18656.0;
const double B1 = 35.0 / 384.0, B3 = 500.0 / 1113.0, B4 = 125.0 / 192.0, B5 = -2187.0 / 6784.0, B6 = 11.0 / 84.0;
const double BH1 = 5179.0 / 57600.0, BH3 = 7571.0 / 16695.0, BH4 = 393.0 / 640.0, BH5 = -92097.0 / 339200.0,
             BH6 = 187.0 / 2100.0, BH7 = 1.0 / 40.0;

struct Work {
    long long nm; int na;
    std::vector<double> k[7], ka[7], ys, as, ynew, anew;
    void init(long long nm_, int na_) {
        nm = nm_; na = na_;
        for (int j = 0; j < 7; ++j) { k[j].assign(nm, 0.0); ka[j].assign(na > 0 ? na : 1, 0.0); }
        ys.assign(nm, 0.0); ynew.assign(nm, 0.0); as.assign(na > 0 ? na : 1, 0.0); anew.assign(na > 0 ? na : 1, 0.0);
    }
};

// y_s = y + h sum_j coef_j k_j   (for both the cell field and the mode amplitudes)
void combine(Work& W, const double* y, const double* a, double h, const double* coef, int nk, double* yo, double* ao) {
#pragma omp parallel for schedule(static)
    for (long long i = 0; i < W.nm; ++i) {
        double acc = 0.0;
        for (int j = 0; j < nk; ++j) acc += coef[j] * W.k[j][i];
        yo[i] = y[i] + h * acc;
    }
    for (int i = 0; i < W.na; ++i) {
        double acc = 0.0;
        for (int j = 0; j < nk; ++j) acc += coef[j] * W.ka[j][i];
        ao[i] = a[i] + h * acc;
    }
}

// One DP5(4) trial step of size h from (m,a) with k1 already in W.k[0], W.ka[0].
// Leaves the candidate in W.ynew/W.anew, k7 in W.k[6]/W.ka[6], returns the error norm.
double trial_step(const orc_problem* P, Work& W, double t, const double* m, const double* a, double h, double* S7) {
    const long long nc = ncell(P);
    { const double c[] = {A21};                     combine(W, m, a, h, c, 1, W.ys.data(), W.as.data()); rhs(P, t + (1.0 / 5.0) * h, W.ys.data(), W.as.data(), W.k[1].data(), W.ka[1].data(), nullptr); }
    { const double c[] = {A31, A32};                combine(W, m, a, h, c, 2, W.ys.data(), W.as.data()); rhs(P, t + (3.0 / 10.0) * h, W.ys.data(), W.as.data(), W.k[2].data(), W.ka[2].data(), nullptr); }
    { const double c[] = {A41, A42, A43};           combine(W, m, a, h, c, 3, W.ys.data(), W.as.data()); rhs(P, t + (4.0 / 5.0) * h, W.ys.data(), W.as.data(), W.k[3].data(), W.ka[3].data(), nullptr); }
    { const double c[] = {A51, A52, A53, A54};      combine(W, m, a, h, c, 4, W.ys.data(), W.as.data()); rhs(P, t + (8.0 / 9.0) * h, W.ys.data(), W.as.data(), W.k[4].data(), W.ka[4].data(), nullptr); }
    { const double c[] = {A61, A62, A63, A64, A65}; combine(W, m, a, h, c, 5, W.ys.data(), W.as.data()); rhs(P, t + (1.0) * h, W.ys.data(), W.as.data(), W.k[5].data(), W.ka[5].data(), nullptr); }
    { const double c[] = {B1, 0.0, B3, B4, B5, B6}; combine(W, m, a, h, c, 6, W.ynew.data(), W.anew.data()); }
    if (P->renormalize) {   // G13: normalise the 5th-order solution per cell before the 7th evaluation
        for (int s = 0; s < P->n_sub; ++s) {
            double* y = W.ynew.data() + (long long)s * 3 * nc;
#pragma omp parallel for schedule(static)
            for (long long i = 0; i < nc; ++i) {
                const double n2 = y[i] * y[i] + y[nc + i] * y[nc + i] + y[2 * nc + i] * y[2 * nc + i];
                const double inv = 1.0 / std::sqrt(n2);
                y[i] *= inv; y[nc + i] *= inv; y[2 * nc + i] *= inv;
            }
        }
    }
    rhs(P, t + h, W.ynew.data(), W.anew.data(), W.k[6].data(), W.ka[6].data(), S7);   // c_7 = 1
    // e = h sum_j d_j k_j,  d = b - bhat
    const double d[7] = {B1 - BH1, 0.0, B3 - BH3, B4 - BH4, B5 - BH5, B6 - BH6, -BH7};
    double err = 0.0;
    bool bad = false;
    for (int s = 0; s < P->n_sub; ++s) {
        const long long o = (long long)s * 3 * nc;
        double emax = 0.0; int nbad = 0;
#pragma omp parallel for schedule(static) reduction(max : emax) reduction(+ : nbad)
        for (long long i = 0; i < nc; ++i) {
            double e2 = 0.0;
            for (int cidx = 0; cidx < 3; ++cidx) {
                double acc = 0.0;
                for (int j = 0; j < 7; ++j) acc += d[j] * W.k[j][o + cidx * nc + i];
                acc *= h;
                e2 += acc * acc;
            }
            const double e = std::sqrt(e2);
            if (!std::isfinite(e)) nbad++;
            else if (e > emax) emax = e;
        }
        if (nbad) bad = true;
        if (emax > err) err = emax;
    }
    for (int n = 0; n < P->N; ++n) {   // mode amplitudes enter the same max-norm (G12)
        double ere = 0.0, eim = 0.0;
        for (int j = 0; j < 7; ++j) { ere += d[j] * W.ka[j][2 * n]; eim += d[j] * W.ka[j][2 * n + 1]; }
        const double e = std::fabs(h) * std::sqrt(ere * ere + eim * eim);
        if (!std::isfinite(e)) bad = true;
        else if (e > err) err = e;
    }
    return bad ? NAN : err;
}

}  // namespace

extern "C" {

// f(t, m, a): dm [n_sub][3][nc], da [N][2], S [N][2] (may be NULL).
void orc_rhs(const orc_problem* P, double t, const double* m, const double* a, double* dm, double* da, double* S) {
    rhs(P, t, m, a, dm, da, S);
}

// Integrate from *t to t_end (or for max_steps attempted steps if max_steps > 0).
//   tol > 0: adaptive (fixed_dt ignored);  tol <= 0: fixed step fixed_dt.
//   m [n_sub][3][nc] and a [N][2] are updated in place; *dt_io carries the step proposal.
//   Trace: sample_dt > 0 and trace != NULL: rows of (1 + 4N + 3 n_sub) doubles
//          [t, a(re,im)xN, S(re,im)xN, <m_s>(x,y,z) x n_sub], at most trace_cap rows.
//          adaptive: steps are clamped onto t0 + k*sample_dt; fixed: every round(sample_dt/dt) steps.
int orc_run(const orc_problem* P, double* m, double* a, double* t_io, double t_end, double tol, double fixed_dt,
            double* dt_io, long long max_steps, double sample_dt, double* trace, int trace_cap, int* n_trace,
            orc_stats* st) {
    const long long nc = ncell(P), nm = (long long)P->n_sub * 3 * nc;
    const int na = 2 * P->N;
    const bool adaptive = tol > 0.0;
    Work W; W.init(nm, na);
    double t = *t_io;
    double dt = adaptive ? ((dt_io && *dt_io > 0.0) ? *dt_io : 1e-14) : fixed_dt;
    orc_stats s = {0, 0, 0, INFINITY, 0.0, dt, t, 0};
    std::vector<double> S7((size_t)(na > 0 ? na : 1));

    rhs(P, t, m, a, W.k[0].data(), W.ka[0].data(), nullptr);   // k1 = f(t, y), once; afterwards FSAL
    s.rhs_evals++;

    const int rowlen = 1 + 4 * P->N + 3 * P->n_sub;
    int ntr = 0;
    const bool tracing = trace && sample_dt > 0.0 && trace_cap > 0;
    const double t0 = t;
    long long stride = 1;
    if (tracing && !adaptive) { stride = llround(sample_dt / fixed_dt); if (stride < 1) stride = 1; }
    long long steps = 0;

    while (t < t_end && (max_steps <= 0 || steps < max_steps)) {
        double h = dt;
        double target = t_end;
        bool sample_hit = false;
        if (tracing && adaptive && ntr < trace_cap) {
            const double ts = t0 + (double)(ntr + 1) * sample_dt;
            if (ts <= target) { target = ts; sample_hit = true; }
        }
        bool clamped = false;
        if (t + h * (1.0 + 1e-12) >= target) { h = target - t; clamped = true; }
        const double err = trial_step(P, W, t, m, a, h, S7.data());
        s.rhs_evals += 6;
        steps++;
        bool accept;
        if (adaptive) accept = std::isfinite(err) && err <= tol;
        else {
            accept = true;
            if (!std::isfinite(err)) { s.status = 1; break; }
        }
        double fac;
        if (!std::isfinite(err)) fac = 0.5;
        else if (err == 0.0) fac = 2.0;
        else { fac = 0.8 * std::pow(tol / err, 0.2); if (fac < 0.5) fac = 0.5; if (fac > 2.0) fac = 2.0; }
        if (accept) {
            t = clamped ? target : t + h;
            std::memcpy(m, W.ynew.data(), sizeof(double) * nm);
            if (na) std::memcpy(a, W.anew.data(), sizeof(double) * na);
            W.k[0].swap(W.k[6]); W.ka[0].swap(W.ka[6]);       // FSAL: k1 := k7
            s.accepted++;
            if (h < s.dt_min) s.dt_min = h;
            if (h > s.dt_max) s.dt_max = h;
            if (adaptive) { const double prop = h * fac; dt = clamped ? (prop > dt ? prop : dt) : prop; }
            const bool take = tracing && ntr < trace_cap &&
                              (adaptive ? (clamped && sample_hit) : (s.accepted % stride == 0));
            if (take) {
                double* row = trace + (long long)ntr * rowlen;
                row[0] = t;
                for (int i = 0; i < na; ++i) row[1 + i] = a[i];
                for (int i = 0; i < na; ++i) row[1 + na + i] = S7[i];
                for (int sub = 0; sub < P->n_sub; ++sub)
                    for (int cidx = 0; cidx < 3; ++cidx) {
                        const double* f = m + ((long long)sub * 3 + cidx) * nc;
                        double acc = 0.0;
                        for (long long i = 0; i < nc; ++i) acc += f[i];
                        row[1 + 2 * na + 3 * sub + cidx] = acc / (double)nc;
                    }
                ntr++;
            }
        } else {
            s.rejected++;
            dt = h * fac;
        }
        if (adaptive && !(dt > 1e-20)) { s.status = 2; break; }
    }
    *t_io = t;
    if (dt_io) *dt_io = dt;
    if (n_trace) *n_trace = ntr;
    s.dt_next = dt; s.t = t;
    if (st) *st = s;
    return s.status;
}

// ---- the paper's tier-2 operator-split loop as a comparison integrator (PAPER.md:169-193 Listing 1, :199) ----
// n_steps steps of size dt from *t_io.  Per step:
//   (i)   S_n = overlaps of the current m                               ("Read magnetization from GPU")
//   (ii)  a_n <- classic RK4 over dt of da/dt = -(i w + kappa) a + i G S + eta(t) with S held constant
//                                                                        ("Step cavity ODE (CPU, RK4)")
//   (iii) c_n = (2/gamma) Re[G_b a_n] from the NEW amplitudes, held constant   ("H_rf = h0 * a.real", then bias field)
//   (iv)  m <- n_llg Dormand-Prince 5(4) steps of dt/n_llg of the LLG equation in that constant RF field, each followed
//         by the per-cell renormalisation of the unified step                  ("world.timesolver.run(dt)"; reading G33)
// Trace rows as orc_run, one per step (sample_every steps), S = overlaps of the state the row belongs to.
int orc_run_split(const orc_problem* P, double* m, double* a, double* t_io, double dt, long long n_steps, int n_llg,
                  long long sample_every, double* trace, int trace_cap, int* n_trace) {
    const long long nc = ncell(P), nm = (long long)P->n_sub * 3 * nc;
    const int N = P->N, na = 2 * N;
    if (n_llg < 1) n_llg = 1;
    std::vector<double> S((size_t)(na > 0 ? na : 1)), c((size_t)(N > 0 ? N : 1));
    std::vector<double> k1a(na > 0 ? na : 1), k2a(na > 0 ? na : 1), k3a(na > 0 ? na : 1), k4a(na > 0 ? na : 1), tmp(na > 0 ? na : 1);
    std::vector<double> k[6], ys(nm);
    for (auto& v : k) v.assign(nm, 0.0);
    const int rowlen = 1 + 4 * N + 3 * P->n_sub;
    int ntr = 0;
    double t = *t_io;
    for (long long step = 0; step < n_steps; ++step) {
        overlaps(P, m, S.data());                                                     // (i)
        // (ii) classic RK4, S frozen
        mode_rhs(P, t, a, S.data(), k1a.data(), nullptr);
        for (int i = 0; i < na; ++i) tmp[i] = a[i] + 0.5 * dt * k1a[i];
        mode_rhs(P, t + 0.5 * dt, tmp.data(), S.data(), k2a.data(), nullptr);
        for (int i = 0; i < na; ++i) tmp[i] = a[i] + 0.5 * dt * k2a[i];
        mode_rhs(P, t + 0.5 * dt, tmp.data(), S.data(), k3a.data(), nullptr);
        for (int i = 0; i < na; ++i) tmp[i] = a[i] + dt * k3a[i];
        mode_rhs(P, t + dt, tmp.data(), S.data(), k4a.data(), nullptr);
        for (int i = 0; i < na; ++i) a[i] = a[i] + (dt / 6.0) * (k1a[i] + 2.0 * k2a[i] + 2.0 * k3a[i] + k4a[i]);
        mode_rhs(P, t + dt, a, S.data(), nullptr, c.data());                          // (iii)
        // (iv) LLG over dt in the constant field
        const double h = dt / (double)n_llg;
        for (int sub = 0; sub < n_llg; ++sub) {
            const double A[6][5] = {{0, 0, 0, 0, 0}, {A21, 0, 0, 0, 0}, {A31, A32, 0, 0, 0}, {A41, A42, A43, 0, 0},
                                    {A51, A52, A53, A54, 0}, {A61, A62, A63, A64, A65}};
            llg_rhs(P, m, c.data(), k[0].data());
            for (int st = 1; st < 6; ++st) {
#pragma omp parallel for schedule(static)
                for (long long i = 0; i < nm; ++i) {
                    double acc = 0.0;
                    for (int j = 0; j < st; ++j) acc += A[st][j] * k[j][i];
                    ys[i] = m[i] + h * acc;
                }
                llg_rhs(P, ys.data(), c.data(), k[st].data());
            }
            const double b[6] = {B1, 0.0, B3, B4, B5, B6};
#pragma omp parallel for schedule(static)
            for (long long i = 0; i < nm; ++i) {
                double acc = 0.0;
                for (int j = 0; j < 6; ++j) acc += b[j] * k[j][i];
                m[i] = m[i] + h * acc;
            }
            if (P->renormalize) {
                for (int s = 0; s < P->n_sub; ++s) {
                    double* y = m + (long long)s * 3 * nc;
#pragma omp parallel for schedule(static)
                    for (long long i = 0; i < nc; ++i) {
                        const double n2 = y[i] * y[i] + y[nc + i] * y[nc + i] + y[2 * nc + i] * y[2 * nc + i];
                        const double inv = 1.0 / std::sqrt(n2);
                        y[i] *= inv; y[nc + i] *= inv; y[2 * nc + i] *= inv;
                    }
                }
            }
        }
        t = *t_io + (double)(step + 1) * dt;
        if (trace && trace_cap > 0 && sample_every > 0 && (step + 1) % sample_every == 0 && ntr < trace_cap) {
            overlaps(P, m, S.data());
            double* row = trace + (long long)ntr * rowlen;
            row[0] = t;
            for (int i = 0; i < na; ++i) row[1 + i] = a[i];
            for (int i = 0; i < na; ++i) row[1 + na + i] = S[i];
            for (int sub = 0; sub < P->n_sub; ++sub)
                for (int cidx = 0; cidx < 3; ++cidx) {
                    const double* f = m + ((long long)sub * 3 + cidx) * nc;
                    double acc = 0.0;
                    for (long long i = 0; i < nc; ++i) acc += f[i];
                    row[1 + 2 * na + 3 * sub + cidx] = acc / (double)nc;
                }
            ntr++;
        }
    }
    *t_io = t;
    if (n_trace) *n_trace = ntr;
    for (long long i = 0; i < nm; ++i) if (!std::isfinite(m[i])) return 1;
    return 0;
}

// ---- the plain discrete Fourier sum of a sampled complex trace ----
// X[k] = sum_j x[j] exp(+i w[k] t[j]) for n samples (x as [n][2] = Re, Im) and nw angular frequencies w: a component
// x ~ exp(-i w0 t) (the paper's sign convention) peaks at w = w0.  out is [nw][2].
void orc_dft(const double* t, const double* x, int n, const double* w, int nw, double* out) {
    for (int k = 0; k < nw; ++k) {
        double re = 0.0, im = 0.0;
        for (int j = 0; j < n; ++j) {
            const double ph = w[k] * t[j];
            const double cs = std::cos(ph), sn = std::sin(ph);
            re += x[2 * j] * cs - x[2 * j + 1] * sn;
            im += x[2 * j] * sn + x[2 * j + 1] * cs;
        }
        out[2 * k] = re; out[2 * k + 1] = im;
    }
}

// ---- demagnetising tensor between two equal rectangular cells (Newell, Williams & Dunlop, J. Geophys. Res. 98, 9551
//      (1993)), restated: with V = dx dy dz and the second-difference weights w = (1, -2, 1),
//        N_xx(X,Y,Z) = -1/(4 pi V) sum_{i,j,k in {-1,0,1}} w_i w_j w_k f(X + i dx, Y + j dy, Z + k dz)
//        N_xy(X,Y,Z) = -1/(4 pi V) sum_{i,j,k}              w_i w_j w_k g(X + i dx, Y + j dy, Z + k dz)
//      the other components by permuting the axes.  f is even in x, y, z; g is odd in x and y, even in z. ----
static double newell_f(double x, double y, double z) {
    x = std::fabs(x); y = std::fabs(y); z = std::fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = std::sqrt(x2 + y2 + z2);
    double r = (1.0 / 6.0) * (2.0 * x2 - y2 - z2) * R;
    if (y > 0.0 && x2 + z2 > 0.0) r += 0.5 * y * (z2 - x2) * std::asinh(y / std::sqrt(x2 + z2));
    if (z > 0.0 && x2 + y2 > 0.0) r += 0.5 * z * (y2 - x2) * std::asinh(z / std::sqrt(x2 + y2));
    if (x > 0.0 && y > 0.0 && z > 0.0) r -= x * y * z * std::atan(y * z / (x * R));
    return r;
}
static double newell_g(double x, double y, double z) {
    z = std::fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = std::sqrt(x2 + y2 + z2);
    double r = -x * y * R / 3.0;
    if (x2 + y2 > 0.0) r += x * y * z * std::asinh(z / std::sqrt(x2 + y2));
    if (y2 + z2 > 0.0) r += (y / 6.0) * (3.0 * z2 - y2) * std::asinh(x / std::sqrt(y2 + z2));
    if (x2 + z2 > 0.0) r += (x / 6.0) * (3.0 * z2 - x2) * std::asinh(y / std::sqrt(x2 + z2));
    if (z > 0.0) r -= (z * z2 / 6.0) * std::atan(x * y / (z * R));
    if (y != 0.0) r -= (z * y2 / 2.0) * std::atan(x * z / (y * R));
    if (x != 0.0) r -= (z * x2 / 2.0) * std::atan(y * z / (x * R));
    return r;
}
static double newell_sum(double (*fn)(double, double, double), double X, double Y, double Z, double dx, double dy, double dz) {
    const double w[3] = {1.0, -2.0, 1.0};
    double acc = 0.0;
    for (int i = -1; i <= 1; ++i)
        for (int j = -1; j <= 1; ++j)
            for (int k = -1; k <= 1; ++k) acc += w[i + 1] * w[j + 1] * w[k + 1] * fn(X + i * dx, Y + j * dy, Z + k * dz);
    return -acc / (4.0 * M_PI * dx * dy * dz);
}

// out[(2nz-1)][(2ny-1)][(2nx-1)][6] = (N_xx, N_yy, N_zz, N_xy, N_xz, N_yz) at the offsets (i dx, j dy, k dz), |i| < nx etc.
void orc_demag_tensor(int nx, int ny, int nz, double dx, double dy, double dz, double* out) {
    const int tx = 2 * nx - 1, ty = 2 * ny - 1, tz = 2 * nz - 1;
    // work in units of dx so that the formulas see numbers of order one
    const double sy = dy / dx, sz = dz / dx;
#pragma omp parallel for schedule(static)
    for (int k = 0; k < tz; ++k)
        for (int j = 0; j < ty; ++j)
            for (int i = 0; i < tx; ++i) {
                const double X = (double)(i - (nx - 1)), Y = (double)(j - (ny - 1)) * sy, Z = (double)(k - (nz - 1)) * sz;
                double* o = out + 6 * (((long long)k * ty + j) * tx + i);
                o[0] = newell_sum(newell_f, X, Y, Z, 1.0, sy, sz);
                o[1] = newell_sum(newell_f, Y, X, Z, sy, 1.0, sz);
                o[2] = newell_sum(newell_f, Z, Y, X, sz, sy, 1.0);
                o[3] = newell_sum(newell_g, X, Y, Z, 1.0, sy, sz);
                o[4] = newell_sum(newell_g, X, Z, Y, 1.0, sz, sy);
                o[5] = newell_sum(newell_g, Y, Z, X, sy, sz, 1.0);
            }
}

// The tableau, exposed so the tests can check its identities (row sums, sum b = 1, sum d = 0).
void orc_tableau(double* a /*[7][7]*/, double* b /*[7]*/, double* bhat /*[7]*/, double* c /*[7]*/) {
    const double A[7][7] = {{0}, {A21}, {A31, A32}, {A41, A42, A43}, {A51, A52, A53, A54},
                            {A61, A62, A63, A64, A65}, {B1, 0.0, B3, B4, B5, B6}};
    const double Bv[7] = {B1, 0.0, B3, B4, B5, B6, 0.0};
    const double BH[7] = {BH1, 0.0, BH3, BH4, BH5, BH6, BH7};
    const double C[7] = {0.0, 1.0 / 5.0, 3.0 / 10.0, 4.0 / 5.0, 8.0 / 9.0, 1.0, 1.0};
    for (int i = 0; i < 7; ++i) { for (int j = 0; j < 7; ++j) a[7 * i + j] = A[i][j]; b[i] = Bv[i]; bhat[i] = BH[i]; c[i] = C[i]; }
}

}  // extern "C"
