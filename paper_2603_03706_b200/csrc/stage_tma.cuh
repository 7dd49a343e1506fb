// The fused RK45 stage kernel, TMA-pipelined variant (hand-written CUDA for sm_100a).
//
// Same arithmetic as stage_kernel.cuh (one launch = one evaluation of the coupled right-hand
// side at stage s, fused with the overlap partials, the next stage state and the error norm; the mode
// ODEs of stages 2..6 are replayed by every block in the next kernel's prologue (deferred_finish), those of
// stages 1 and 7 and the controller run in the last block), but the data movement is Blackwell-native:
//
//   * persistent grid, one CTA per SM; the flattened list of plane-tiles (x-y tile, z) is split
//     into contiguous, equally long runs, one per CTA, so every SM gets the same number of
//     planes and marches in z (each plane of m_s is fetched once per run, plus one halo plane
//     per run end); odd stages walk their run backwards so that a stage starts on data the previous
//     stage left in L2;
//   * a producer warp (one elected lane) issues cp.async.bulk.tensor (TMA) loads of 4-D boxes
//     [comp][1][TY(+2)][TX(+2 HX)] into three shared-memory rings — the stage state with its
//     x/y halo (ring "ms": planes z-1, z, z+1 live), the mode profiles u_n in chunks of 8
//     (ring "u") and the halo-free cell streams y0, k_j, e6 (ring "aux") — completing on
//     mbarriers (expect_tx / complete_tx);
//   * 8 consumer warps (one tile row each, 8 bytes of x per lane) read shared memory only:
//     x neighbours by warp shuffle, y/z neighbours from the halo box / the neighbouring ring
//     slots, so no global load sits on the dependent path and the bytes in flight are set by
//     the ring depth (~100-180 KB per SM) instead of by registers and occupancy;
//   * results go straight from registers to global memory with coalesced 8-byte stores;
//   * inside the run graph consecutive stage kernels are joined by programmatic dependencies: a block's
//     prologue (barrier init, tensor-map prefetch, control words, TMA loads of the streams the previous
//     kernel does not write) runs before griddepcontrol.wait.
//
// Out-of-grid parts of a box are zero-filled by the TMA unit; the open (Neumann) boundary of
// the exchange stencil (reading G9) is applied by substituting the centre value.
#pragma once
#include "stage_kernel.cuh"

namespace cavmag {

constexpr int kTmaTY = 8;                       // tile rows = consumer warps
constexpr int kTmaConsumers = kTmaTY * 32;      // 256 consumer threads
constexpr int kTmaThreads = kTmaConsumers + 32; // + producer warp
constexpr int kTmaRowBytes = 256;               // bytes of x per tile row (64 floats / 32 doubles)
constexpr int kTmaHaloRowBytes = 288;           // row + 16 bytes of x halo on either side (a TMA box must start 16-byte aligned)
constexpr int kTmaHaloBytes = 16;
constexpr int kTmaMaxDepth = 12;

// tensor-map table (device memory, 128 bytes each); H = box with x/y halo, P = plain box
enum TmaMapIndex {
    MAP_H_Y0 = 0, MAP_H_Y1, MAP_H_MS0, MAP_H_MS1, MAP_H_K0, MAP_H_K6,
    MAP_P_Y0, MAP_P_Y1, MAP_P_MS0, MAP_P_K0, MAP_P_K1, MAP_P_K2, MAP_P_K3, MAP_P_K4, MAP_P_K5, MAP_P_K6,
    MAP_P_U, MAP_COUNT
};

constexpr int kTmaUChunk = 8;                   // mode profiles per slot of the u ring

struct TmaArgs {
    const unsigned char* maps;     // [MAP_COUNT][128]
    int Dm, Da, Du;                // ring depths
    int n_uchunks;                 // ceil(N / kTmaUChunk)
    unsigned u_slot_bytes;         // min(N, kTmaUChunk) * 2048
    int ntx, nty;                  // tiles per row / column of the x-y plane
    long long Q;                   // plane-tiles in total = ntx*nty*nz
    unsigned hbox_bytes;           // bytes of one halo box, rounded up to 128
    unsigned hbox_tx;              // bytes TMA writes for one halo box (expect_tx)
    unsigned aux_slot_bytes;       // bytes of one aux slot = n_aux*C * 2048
    unsigned ms_slot_bytes;        // n_halo_fields * hbox_bytes
    int pre_k;                     // 1: k_2..k_{s-2} may be prefetched before the dependency wait (see plan_tma)
    int pre_ctrl;                  // 1: the producer may read Ctrl (written by the stage-2 kernel of this step) before the wait
    int N;                         // number of modes (layout of the stage-7 partial sums: 2N overlaps, then 3 n_sub <m>)
};

// ---- PTX wrappers ----------------------------------------------------------------------
// All shared-memory traffic of the pipeline goes through 32-bit shared-space addresses and explicit
// ld.shared / mbarrier PTX, so that ptxas emits LDS (not generic LD) with immediate offsets.
__device__ __forceinline__ unsigned smem_u32(const void* p) { return (unsigned)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(unsigned bar, unsigned count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(unsigned bar, unsigned bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(unsigned bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ unsigned mbar_try(unsigned bar, unsigned parity) {
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok;
}
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    while (!mbar_try(bar, parity)) {}
}
__device__ __forceinline__ void tma_load_4d(unsigned dst, const void* map, int c0, int c1, int c2, int c3, unsigned bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}
// 8-byte pack (2 floats / 1 double) and scalar loads from a shared-space address
__device__ __forceinline__ Pack<float, 2> lds_pack(unsigned a, const float*) {
    Pack<float, 2> r;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(r.v[0]), "=f"(r.v[1]) : "r"(a));
    return r;
}
__device__ __forceinline__ Pack<double, 1> lds_pack(unsigned a, const double*) {
    Pack<double, 1> r;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(r.v[0]) : "r"(a));
    return r;
}
__device__ __forceinline__ float lds_one(unsigned a, const float*) {
    float r;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(r) : "r"(a));
    return r;
}
__device__ __forceinline__ double lds_one(unsigned a, const double*) {
    double r;
    asm volatile("ld.shared.f64 %0, [%1];" : "=d"(r) : "r"(a));
    return r;
}

// predicated scalar load from a shared-space address (0 when the predicate is off): the two edge lanes of a row take
// their x neighbour from the halo without a divergent branch
__device__ __forceinline__ float lds_one_if(unsigned a, unsigned pred, const float*) {
    float r = 0.0f;
    asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %2, 0;\n@p ld.shared.f32 %0, [%1];\n}\n" : "+f"(r) : "r"(a), "r"(pred));
    return r;
}
__device__ __forceinline__ double lds_one_if(unsigned a, unsigned pred, const double*) {
    double r = 0.0;
    asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %2, 0;\n@p ld.shared.f64 %0, [%1];\n}\n" : "+d"(r) : "r"(a), "r"(pred));
    return r;
}

// number of halo'd fields / plain cell fields the stage streams
template <int STAGE> struct StageStreams {
    static constexpr int n_halo = (STAGE == 2) ? 2 : 1;
    static constexpr int n_aux = (STAGE <= 2) ? 0 : (STAGE == 7) ? 1 : (STAGE == 6) ? 5 : STAGE;   // y0,k1,.. / e6
};

// Deferred finish of stage PREV = STAGE-1, run by the consumer warps of EVERY block of the stage-STAGE kernel while
// the producer warp is already filling the rings: the fixed-order sum of the previous kernel's block partials, the
// mode ODE ka_PREV (Eq. 12 / Eq. 19) and the amplitudes / RF weights c_n of this stage.  All blocks compute the
// same bits from the same inputs; block 0 alone writes the results back to Ctrl.  This replaces the "last block
// to arrive" tail of stages 2..6 (an atomic ticket, two fences and ~4 dependent L2 round trips with 147 SMs
// idle) by work that overlaps the pipeline fill.  Fields written by block 0 (S, ka[PREV-1], as[(PREV+1)&1], c,
// anew, rhs_evals) are never inputs of another block in the same kernel.
constexpr int kCtrlWordsPerConsumer = (kCtrlWords + kTmaConsumers - 1) / kTmaConsumers;

template <int PREV, int NB>
__device__ __forceinline__ bool deferred_finish(const StageArgs& A, Ctrl* __restrict__ gctrl, const int tidc,
                                                unsigned long long* sc_words, double* sred, const int nblk, const bool owner) {
    // nblk blocks wrote partial sums for this simulation (slots 0..nblk-1); `owner` is the one that writes results back
    // one batch of independent loads: the whole Ctrl (a few words per thread) and all 2*NB x gridDim block partials
    // (rows of modes >= N hold stale values that nothing reads)
    const unsigned long long* gcw = reinterpret_cast<const unsigned long long*>(gctrl);
    unsigned long long cw[kCtrlWordsPerConsumer];
#pragma unroll
    for (int k = 0; k < kCtrlWordsPerConsumer; ++k) {
        const int idx = tidc + k * kTmaConsumers;
        cw[k] = idx < kCtrlWords ? __ldcg(gcw + idx) : 0ull;
    }
    if constexpr (NB > 0)
        reduce_block_partials(stage_partials(A, PREV), A.pstride, 2 * NB, nblk, tidc >> 5, kTmaTY, tidc & 31, sred);
#pragma unroll
    for (int k = 0; k < kCtrlWordsPerConsumer; ++k) {
        const int idx = tidc + k * kTmaConsumers;
        if (idx < kCtrlWords) sc_words[idx] = cw[k];
    }
#ifdef CAVMAG_PROBE
    if (tidc == 0) probe_mark(A, PREV + 1, 9);          // Ctrl + partials have landed (this thread's share)
#endif
    asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
#ifdef CAVMAG_PROBE
    if (tidc == 0) probe_mark(A, PREV + 1, 10);         // all consumers' shares are in shared memory
#endif
    Ctrl* const c = reinterpret_cast<Ctrl*>(sc_words);
    const bool live = c->done == 0;                 // done: launched after the run ended (the rest of the last loop iteration, or
                                                    // host-enqueued mode): nothing to finish
    if (live) {
        if (tidc < c->N) {
            const int n = tidc;
            mode_ode_stage<PREV>(c, n, sred, nullptr);
            if (owner) {
                constexpr int nxt = (PREV + 1) & 1;
                gctrl->S[n][0] = c->S[n][0]; gctrl->S[n][1] = c->S[n][1];
                gctrl->ka[PREV - 1][n][0] = c->ka[PREV - 1][n][0]; gctrl->ka[PREV - 1][n][1] = c->ka[PREV - 1][n][1];
                gctrl->as[nxt][n][0] = c->as[nxt][n][0]; gctrl->as[nxt][n][1] = c->as[nxt][n][1];
                gctrl->c[n] = c->c[n];
                if constexpr (PREV == 6) { gctrl->anew[n][0] = c->anew[n][0]; gctrl->anew[n][1] = c->anew[n][1]; }
            }
        }
        if (tidc == 0) {
            c->rhs_evals++;                             // evaluation PREV is complete
            if (owner) gctrl->rhs_evals = c->rhs_evals;
        }
    }
    if constexpr (PREV == 6) {
        // The stage-7 kernel hands the step over to the next stage-2 kernel through the boundary copy: block 0 stores
        // its whole working copy there (also when the run is over, so that both instances end up equal).  No block of
        // THIS kernel reads ctrl0, and the stage-2 kernel starts after this one has completed.
        if (owner) {
            asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
            unsigned long long* const g0 = reinterpret_cast<unsigned long long*>(A.ctrl0);
            for (int idx = tidc; idx < kCtrlWords; idx += kTmaConsumers) g0[idx] = sc_words[idx];
        }
    }
    return live;
}

// Deferred finish of stage 7 AND the step controller, run by the consumer warps of every block of the stage-2 kernel of
// the next loop iteration (all blocks compute the same bits from the same inputs).  It replaces the "last block to
// arrive" tail of the stage-7 kernel - a ticket, the second reduction pass, the controller and the graph condition
// on ONE block with 147 SMs idle, ~10 us of every step on cfg3 - by a prologue that every block runs at once.
//   reads : the boundary copy ctrl0 (written by block 0 of the stage-7 kernel, by k_begin or by stage 1), the stage-7
//           block partials (2N overlap sums of m_new, 3 n_sub sums for <m>) and the blocks' error maxima
//   does  : ka_7 and the mode error (Eq. 12 at the candidate), err = max(cells, modes), accept / reject, dt, t, buffer
//           rotation, trace row, done, h of the step that starts now, a_2 and its RF weights
//   writes: block 0 stores the whole new state to the canonical instance `ctrl` (never read by a block of this kernel),
//           the trace row, and the WHILE condition of the run graph.  The condition lags by one iteration: the loop
//           body that finds `done` is empty from here on (every later kernel of it returns at once).
// The producer warp learns buffer indices and `done` from the shared copy through named barrier 2 (bar.arrive here,
// bar.sync there).  Returns false when the run is over.
template <int NB, int NSUB>
__device__ __forceinline__ bool deferred_finish7(const StageArgs& A, const TmaArgs& TA, const int tidc,
                                                 unsigned long long* sc_words, double* sred, double* serr, double* trace,
                                                 const int nblk, const bool owner, unsigned int* live_count, int& spec_miss) {
    // live_count != nullptr (joint launch of several simulations): the owner reports "this simulation goes on" there
    // instead of setting the WHILE condition itself
    const unsigned long long* gcw = reinterpret_cast<const unsigned long long*>(A.ctrl0);
    unsigned long long cw[kCtrlWordsPerConsumer];
#pragma unroll
    for (int k = 0; k < kCtrlWordsPerConsumer; ++k) {
        const int idx = tidc + k * kTmaConsumers;
        cw[k] = idx < kCtrlWords ? __ldcg(gcw + idx) : 0ull;
    }
    const int N = TA.N, warp = tidc >> 5, lane = tidc & 31;
    const int nsum = 2 * N + 3 * NSUB;
    // warps 0..6 sum the partials, warp 7 takes the error maxima (stale values when no stage 7 is pending: not used)
    if (warp < kTmaTY - 1) reduce_block_partials(stage_partials(A, 7), A.pstride, nsum, nblk, warp, kTmaTY - 1, lane, sred);
    else {
        const double mx = reduce_block_max(A.partial_max, nblk, lane);
        if (lane == 0) serr[kMaxModes] = mx;
    }
#pragma unroll
    for (int k = 0; k < kCtrlWordsPerConsumer; ++k) {
        const int idx = tidc + k * kTmaConsumers;
        if (idx < kCtrlWords) sc_words[idx] = cw[k];
    }
    asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
    Ctrl* const c = reinterpret_cast<Ctrl*>(sc_words);
    // what the producer warp assumes while this runs (it reads the same words from ctrl0): the pending step is accepted,
    // i.e. the buffer indices flip; every thread keeps the prediction to compare it with the verdict
    const int done_in = c->done;
    const int ycur_pred = c->pend7 ? (c->ycur ^ 1) : c->ycur, k1_pred = c->pend7 ? 6 - c->k1slot : c->k1slot;
    const bool write = owner;
    if (c->done == 0 && c->pend7 != 0) {            // uniform over the block (and over the grid)
        if (tidc < N) mode_ode_stage<7>(c, tidc, sred, serr);
        asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
        if (tidc == 0) {
            const int accept = controller_step(c, serr[kMaxModes], serr, sred, N, NSUB, A.inv_nc, trace, write);
            serr[kMaxModes + 1] = (double)accept;
        }
        asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
        if (write && A.spec != nullptr && c->spec_K > 0 && c->took)       // Fourier sums of this trace sample
            dft_accumulate(A.spec, c->spec_K, c->spec_w0, c->spec_dw, N, c->t, c->anew, c->S, c->mavg, NSUB, tidc, kTmaConsumers);
        if (tidc < N && serr[kMaxModes + 1] != 0.0) {     // y := y_new (modes), FSAL: ka_1 := ka_7
            c->a[tidc][0] = c->anew[tidc][0]; c->a[tidc][1] = c->anew[tidc][1];
            c->ka[0][tidc][0] = c->ka[6][tidc][0]; c->ka[0][tidc][1] = c->ka[6][tidc][1];
        }
        asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
        if (tidc == 0) {                                  // start of the next step
            const bool done = !(c->t < c->t_end) || (c->max_steps > 0 && c->steps_run >= c->max_steps) || c->status != 0;
            c->done = done ? 1 : 0;
            prepare_h(c);
        }
        asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
        if (tidc < N) mode_stage_state<1>(c, tidc);       // a_2 = a_0 + h a21 ka_1
    }
    if (tidc == 0) c->pend7 = c->done ? 0 : 1;            // a step starts now: its stage 7 will be pending
    asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
    spec_miss = (done_in == 0 && (c->done != 0 || c->ycur != ycur_pred || c->k1slot != k1_pred)) ? 1 : 0;
    asm volatile("bar.arrive 2, %0;" ::"n"(kTmaThreads) : "memory");      // the producer warp may read the shared copy
#ifdef CAVMAG_PROBE
    if (tidc == 0) probe_mark(A, 2, 10);                // verdict and the new step's control data are in shared memory
#endif
    const bool live = c->done == 0;
    if (write) {
        unsigned long long* const g1 = reinterpret_cast<unsigned long long*>(A.ctrl);
        for (int idx = tidc; idx < kCtrlWords; idx += kTmaConsumers) g1[idx] = sc_words[idx];
        if (tidc == 0) {
            // A run bounded by max_steps knows its last step when that step STARTS (rejected steps count): the loop can
            // stop after this body, and the stage-2 kernel that follows the WHILE node finishes the step.  A run bounded
            // by t_end only learns it from the controller: the condition then lags one iteration (empty kernels).
            const bool last = c->max_steps > 0 && c->steps_run + 1 >= c->max_steps;
            if (live_count != nullptr) { if (live && !last) atomicAdd(live_count, 1u); }
            else if (A.cond_handle != 0ull)
                cudaGraphSetConditional((cudaGraphConditionalHandle)A.cond_handle, (live && !last) ? 1u : 0u);
        }
    }
    return live;
}

// Joint launch of R independent simulations of the same shape (a field sweep of a mid-size grid): the
// plane-tiles of all of them form ONE list that the persistent grid cuts into equal runs, so a block may work on (at
// most a few) different simulations one after the other - a "sub-run" each, with that simulation's buffers, Ctrl, tensor
// maps and partial-sum slots.  Every simulation keeps its own step size and accept/reject decisions.
struct RepPtrs {
    Ctrl* ctrl; Ctrl* ctrl0;
    void* Y[2]; void* MS[2]; void* K[7];
    const void* u;
    double* partial; double* partial_max; double* spec; double* trace;
    const unsigned char* maps;
    const unsigned char* umap;      // tensor map of the mode profiles: the member's own, or member 0's when all members share
                                    // the same profiles (one copy then serves every member out of L2)
    double B0[3];
};
struct SweepArgs {
    const RepPtrs* reps;            // [R] in device memory
    int R;
    unsigned int* live;             // simulations that go on after this step (stage 2 adds, stage 3 turns it into the WHILE condition)
    unsigned long long cond_handle;
};

// POL: per-mode polarisation (A.pol, reading G32; cav_set_polarisation) - its own instantiation, up to 8 modes: the RF field
// of mode n points along p_n, and the overlap is taken with m.p_n - i m.q_n.  The consumers accumulate the three raw sums
// sum u_n m_c per mode and project them on p_n, q_n once, before the block reduction (the projection is linear).
template <typename T, int STAGE, int NSUB, int NB, bool SWEEP, bool POL = false>
__device__ __forceinline__ void stage_tma_body(const StageArgs& A, const TmaArgs& TA, double* __restrict__ trace0, const SweepArgs& SW) {
    static_assert(!(SWEEP && STAGE == 1), "stage 1 of a joint launch runs as one ordinary launch per simulation");
    static_assert(!POL || (!SWEEP && NB >= 1 && NB <= 8), "polarisation: single simulations with 1..8 modes");
    constexpr int VEC = 8 / (int)sizeof(T);              // cells per lane: 2 floats / 1 double
    constexpr int TX = kTmaRowBytes / (int)sizeof(T);    // cells per tile row
    constexpr int HX = kTmaHaloBytes / (int)sizeof(T);   // x halo in cells (16 bytes: 4 floats / 2 doubles)
    constexpr int C = 3 * NSUB;
    constexpr int NH = StageStreams<STAGE>::n_halo;
    constexpr int NAUX = StageStreams<STAGE>::n_aux;
    constexpr int NCH = (NB + kTmaUChunk - 1) / kTmaUChunk;          // u chunks per plane
    constexpr int UCB = NB < kTmaUChunk ? NB : kTmaUChunk;           // modes per chunk (box depth)
    constexpr int HPLANE = kTmaHaloRowBytes * (kTmaTY + 2);          // one comp of a halo box
    constexpr int APLANE = kTmaRowBytes * kTmaTY;                    // one comp of a plain box
    using P = Pack<T, VEC>;
    const T* const tag = nullptr;

    if (threadIdx.x == 0) CAVMAG_MARK(0);
    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bars[6 * kTmaMaxDepth];
    __shared__ T s_cn[NB > 0 ? NB : 1];
    __shared__ T s_pq[POL ? 6 * NB : 1];         // p_n, q_n (constant during a run: loaded before the dependency wait)

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int nx = A.nx, ny = A.ny, nz = A.nz;
    const long long nc = A.ncp;                 // component stride in memory (rows padded to 16 bytes: cavmag_types.cuh)
    const int Dm = TA.Dm, Da = TA.Da, Du = TA.Du;

    const unsigned ms_ring = (smem_u32(smem_raw) + 127u) & ~127u;
    const unsigned aux_ring = ms_ring + (unsigned)Dm * TA.ms_slot_bytes;
    const unsigned u_ring = aux_ring + (unsigned)Da * TA.aux_slot_bytes;
    const unsigned full_ms = smem_u32(&bars[0]), empty_ms = smem_u32(&bars[kTmaMaxDepth]);
    const unsigned full_aux = smem_u32(&bars[2 * kTmaMaxDepth]), empty_aux = smem_u32(&bars[3 * kTmaMaxDepth]);
    const unsigned full_u = smem_u32(&bars[4 * kTmaMaxDepth]), empty_u = smem_u32(&bars[5 * kTmaMaxDepth]);

    // ---- prologue that does not depend on the previous stage kernel (overlaps its tail under a
    //      programmatic graph edge): barrier init, tensor-map prefetch ----
    if (tid == 0) {
        for (int i = 0; i < Dm; ++i) { mbar_init(full_ms + 8 * i, 1); mbar_init(empty_ms + 8 * i, kTmaTY); }
        for (int i = 0; i < Da; ++i) { mbar_init(full_aux + 8 * i, 1); mbar_init(empty_aux + 8 * i, kTmaTY); }
        for (int i = 0; i < Du; ++i) { mbar_init(full_u + 8 * i, 1); mbar_init(empty_u + 8 * i, kTmaTY); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (warp == kTmaTY && lane < MAP_COUNT)
        asm volatile("prefetch.tensormap [%0];" ::"l"(TA.maps + 128 * lane) : "memory");
    __syncthreads();                            // the barriers are initialised before the producer arms them
    // Let the next stage kernel be scheduled as SMs drain.  Every thread executes griddepcontrol.wait (the previous
    // kernel has completed and flushed) before it touches anything that kernel wrote - the consumers at once, the
    // producer lane after it has prefetched what the previous kernel does NOT write (kPre below).  Both
    // instructions are no-ops without a programmatic dependency.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    // What the producer lane may issue BEFORE the dependency wait (DRAM is under-used while the previous kernel's
    // slowest blocks finish, and this fill is ~10 % of a stage):
    //   * the mode profiles u: never written, always safe, in every stage >= 2;
    //   * the aux streams y0, k1 (written before this loop iteration started) - but WHICH buffers they are (ycur,
    //     k1slot) and whether the run is over is decided by the controller in the prologue of this step's stage-2
    //     kernel, so the producer must first read Ctrl; and k_2..k_{s-2}, written by kernel s-2.
    // Programmatic edges are NOT transitive: kernel s may be launched while kernel s-2 is still running, unless a block
    // of kernel s can only become resident on an SM that a block of kernel s-1 has left (which has passed its own
    // wait, so kernel s-2 has completed).  The host sets TA.pre_ctrl (stages >= 4: Ctrl as written by this step's
    // stage-2 kernel) and TA.pre_k only when that holds: one CTA per SM (every stage's shared memory exceeds half an
    // SM) and a grid of exactly n_sm blocks.  Otherwise only u is fetched early and everything else follows the wait.
    constexpr bool kPre = STAGE >= 2;

    constexpr bool kDeferred = STAGE >= 2;      // this kernel first finishes the previous stage (deferred_finish / deferred_finish7)
    constexpr int NRED = STAGE == 2 ? 2 * NB + 3 * NSUB : (NB > 0 ? 2 * NB : 1);
    __shared__ __align__(16) unsigned long long s_ctrl[kDeferred ? kCtrlWords : 1];
    __shared__ double s_red[kDeferred ? NRED : 1];
    __shared__ double s_err[STAGE == 2 ? kMaxModes + 2 : 1];      // stage 2: mode errors, max |e|^2, accept flag

    // this CTA's run of plane-tiles; tile coordinates are advanced incrementally (no divisions in the loops)
    const long long Qtot = SWEEP ? TA.Q * (long long)SW.R : TA.Q;
    const long long cq0 = (Qtot * (long long)blockIdx.x) / gridDim.x;
    const long long cq1 = (Qtot * (long long)(blockIdx.x + 1)) / gridDim.x;
    // Sweep direction: odd stages walk their run backwards (cav_set_sweep_order), so a block starts stage s+1 on the
    // plane-tiles it finished stage s with - their stage state, slopes, y0 and profiles are still in the 126 MB L2.
    const int dir = (A.serpentine && (STAGE & 1)) ? -1 : 1;
    const int zfirst = dir > 0 ? 0 : nz - 1, zlast = dir > 0 ? nz - 1 : 0;
    // sub-runs: one per simulation this block's run touches (exactly one without SWEEP)
    const int r_lo = SWEEP ? (int)(cq0 / TA.Q) : 0;
    const int r_hi = SWEEP ? (cq1 > cq0 ? (int)((cq1 - 1) / TA.Q) : r_lo - 1) : 0;
    const int nsr = SWEEP ? r_hi - r_lo + 1 : 1;
    StageArgs Arep;                                  // SWEEP: the arguments of the current simulation
    double* trace = trace0;
    const unsigned char* rep_maps = TA.maps;
    const unsigned char* rep_umap = TA.maps + 128 * MAP_P_U;
    long long ql0 = cq0, ql1 = cq1;                  // the sub-run, in plane-tiles of its own simulation
    int slot = (int)blockIdx.x, nblk_r = (int)gridDim.x;       // this block's partial-sum slot / blocks working on the simulation
    int nplanes = 0, z0 = 0, tx0 = 0, ty0 = 0;                 // the sub-run: length and first plane-tile in sweep order
    auto set_geometry = [&]() {                                // (64-bit divisions: once per block, not once per role)
        nplanes = (int)(ql1 - ql0);
        const long long qs = dir > 0 ? ql0 : ql1 - 1;
        const long long t0 = qs / nz;
        z0 = (int)(qs - t0 * nz);
        tx0 = (int)(t0 % TA.ntx); ty0 = (int)(t0 / TA.ntx);
    };
    if constexpr (!SWEEP) set_geometry();
    auto enter_subrun = [&](const int sr) {
        if constexpr (SWEEP) {
            const int r = dir > 0 ? r_lo + sr : r_hi - sr;
            const long long base = (long long)r * TA.Q, G = gridDim.x;
            ql0 = (cq0 > base ? cq0 : base) - base;
            ql1 = (cq1 < base + TA.Q ? cq1 : base + TA.Q) - base;
            long long bf = (base * G) / Qtot;                        // first block whose run reaches into simulation r
            while ((Qtot * (bf + 1)) / G <= base) ++bf;
            long long bl = ((base + TA.Q) * G - 1) / Qtot;           // last block whose run starts before its end
            if (bl > G - 1) bl = G - 1;
            while ((Qtot * bl) / G >= base + TA.Q) --bl;
            slot = (int)((long long)blockIdx.x - bf);
            nblk_r = (int)(bl - bf + 1);
            const RepPtrs& rp = SW.reps[r];
            Arep = A;
            Arep.ctrl = rp.ctrl; Arep.ctrl0 = rp.ctrl0;
            Arep.Y[0] = rp.Y[0]; Arep.Y[1] = rp.Y[1]; Arep.MS[0] = rp.MS[0]; Arep.MS[1] = rp.MS[1];
#pragma unroll
            for (int i = 0; i < 7; ++i) Arep.K[i] = rp.K[i];
            Arep.u = rp.u; Arep.partial = rp.partial; Arep.partial_max = rp.partial_max; Arep.spec = rp.spec;
            Arep.B0[0] = rp.B0[0]; Arep.B0[1] = rp.B0[1]; Arep.B0[2] = rp.B0[2];
            Arep.cond_handle = 0ull;
            trace = rp.trace;
            rep_maps = rp.maps;
            rep_umap = rp.umap;
            set_geometry();
        }
    };
    const StageArgs& Aouter = A;
    // next plane-tile of the run in sweep order; returns true when the tile column changes
    auto advance = [&](int& z, int& tx, int& ty) -> bool {
        z += dir;
        if (z == nz) { z = 0; if (++tx == TA.ntx) { tx = 0; ++ty; } return true; }
        if (z < 0) { z = nz - 1; if (--tx < 0) { tx = TA.ntx - 1; --ty; } return true; }
        return false;
    };

    // Each role fetches what it needs from Ctrl with ONE batch of independent loads (one L2 round trip after the
    // dependency wait): the producer four words, the consumers the whole struct or, in stages 1-2, a few fields.
    int N, ycur, k1slot;

    if (warp == kTmaTY) {
        // =============================== TMA producer ===============================
        int hm = 0, ha = 0, hu = 0;                 // ring heads, carried over the sub-runs
        unsigned pm = 1, pa = 1, pu = 1;            // parity to wait on for "empty" (first pass: passes immediately)
        for (int sr = 0; sr < nsr; ++sr) {
            enter_subrun(sr);
            const StageArgs& A = SWEEP ? Arep : Aouter;
            Ctrl* const ctrl = A.ctrl;
        int done = 0;
        bool have_ctrl = false;
        if constexpr (STAGE == 1) {
            asm volatile("griddepcontrol.wait;" ::: "memory");
            done = ctrl->k1_valid; N = ctrl->N; ycur = ctrl->ycur; k1slot = ctrl->k1slot;
            have_ctrl = true;
        } else if constexpr (STAGE >= 3) {
            if (TA.pre_ctrl) {
                done = ctrl->done; N = ctrl->N; ycur = ctrl->ycur; k1slot = ctrl->k1slot;
                have_ctrl = true;
            }
        }
        if (have_ctrl && done) return;             // (never in a joint launch: pre_ctrl is off there)
        const bool issuer = lane == 0 && nplanes > 0;
        const unsigned char* maps = rep_maps;
        auto mp = [&](int i) { return (const void*)(maps + 128 * i); };
        const void* hmap0 = nullptr;
        const void* hmap1 = nullptr;                    // STAGE 2 only
        const void* amap[5] = {nullptr, nullptr, nullptr, nullptr, nullptr};
        auto setup_maps = [&]() {                       // needs ycur, k1slot
            hmap0 = STAGE == 1 ? mp(MAP_H_Y0 + ycur) : STAGE == 2 ? mp(MAP_H_Y0 + ycur)
                    : STAGE == 7 ? mp(MAP_H_Y0 + (1 - ycur))
                    : (STAGE == 3 || STAGE == 5) ? mp(MAP_H_MS0) : mp(MAP_H_MS1);
            hmap1 = mp(k1slot == 0 ? MAP_H_K0 : MAP_H_K6);
            if constexpr (STAGE >= 3 && STAGE <= 6) {
                amap[0] = mp(MAP_P_Y0 + ycur);
                amap[1] = mp(k1slot == 0 ? MAP_P_K0 : MAP_P_K6);
                if constexpr (STAGE == 6) { amap[2] = mp(MAP_P_K2); amap[3] = mp(MAP_P_K3); amap[4] = mp(MAP_P_K4); }
                else {
#pragma unroll
                    for (int j = 1; j < STAGE - 1; ++j) amap[1 + j] = mp(MAP_P_K0 + j);
                }
            } else if constexpr (STAGE == 7) {
                amap[0] = mp(MAP_P_MS0);      // e6
            }
        };
        if (have_ctrl) setup_maps();
        const void* umap = (const void*)rep_umap;
        constexpr unsigned aux_tx = (unsigned)(NAUX * C) * (unsigned)APLANE;
        constexpr unsigned u_tx = (unsigned)UCB * (unsigned)APLANE;   // the full box is always counted (OOB modes zero-filled)
        int pre_a = 0, pre_u = 0;                   // aux slots armed / u slots filled before the dependency wait
        int spec_slots = 0;                         // stage 2: ms slots filled speculatively before the controller's verdict
        const int npre = (NAUX > 1) ? (TA.pre_k ? NAUX - 1 : (NAUX - 1 < 2 ? NAUX - 1 : 2)) : 0;   // aux fields fetched before the wait
        if constexpr (kPre) {
            if (!SWEEP && issuer) {                 // (a joint launch fetches nothing before the wait)
                int zz = z0, txx = tx0, tyy = ty0;
                for (int p = 0; p < nplanes; ++p) {
                    const bool do_u = NB > 0 && pre_u + NCH <= Du;
                    const bool do_a = NAUX > 1 && have_ctrl && pre_a < Da;
                    if (!do_u && !do_a) break;
                    const int x0 = txx * TX, y0 = tyy * kTmaTY;
                    if constexpr (NB > 0) {
                        if (do_u) {
#pragma unroll 1
                            for (int ch = 0; ch < NCH; ++ch) {
                                const unsigned bar = full_u + 8 * pre_u;
                                mbar_expect_tx(bar, u_tx);
                                tma_load_4d(u_ring + (unsigned)pre_u * u_tx, umap, x0, y0, zz, ch * kTmaUChunk, bar);
                                ++pre_u;
                            }
                        }
                    }
                    if constexpr (NAUX > 1) {
                        if (do_a) {
                            const unsigned bar = full_aux + 8 * pre_a;
                            mbar_expect_tx(bar, aux_tx);            // the whole slot; the other fields follow after the wait
                            unsigned dst = aux_ring + (unsigned)pre_a * aux_tx;
#pragma unroll
                            for (int f = 0; f < NAUX - 1; ++f) {
                                if (f < npre) tma_load_4d(dst, amap[f], x0, y0, zz, 0, bar);
                                dst += C * APLANE;
                            }
                            ++pre_a;
                        }
                    }
                    advance(zz, txx, tyy);
                }
            }
            __syncwarp();
            if (!SWEEP || sr == 0) asm volatile("griddepcontrol.wait;" ::: "memory");
            CAVMAG_MARK(13);
            if constexpr (STAGE == 2) {
                // The consumers are finishing the previous step (deferred_finish7: ~5 us for loads, mode algebra and the
                // controller).  The buffer indices of THIS step depend on its verdict, but a step is almost always
                // accepted: issue the first stage-state tiles now for "accept" (indices flipped) and check afterwards.
                bool spec = false;
                if constexpr (!SWEEP) {
                    const Ctrl* const c0 = A.ctrl0;             // complete: written by the stage-7 kernel / k_begin / stage 1
                    const int d0 = c0->done, p7 = c0->pend7, y0c = c0->ycur, k0c = c0->k1slot;
                    if (!d0) { ycur = p7 ? (y0c ^ 1) : y0c; k1slot = p7 ? 6 - k0c : k0c; spec = true; }
                    if (spec && issuer) {
                        setup_maps();
                        int zz = z0, txx = tx0, tyy = ty0;
                        for (int p = 0; p < nplanes; ++p) {         // the slots the main loop will ask for, in its order
                            const int need = (p == 0 || zz == zfirst) ? 3 : 1;
                            if (spec_slots + need > Dm) break;
                            const int x0 = txx * TX, y0 = tyy * kTmaTY;
                            for (int i = 0; i < need; ++i) {
                                const int zq = need == 3 ? zz - dir + i * dir : zz + dir;
                                const unsigned bar = full_ms + 8 * spec_slots;
                                mbar_expect_tx(bar, NH * TA.hbox_tx);
                                const unsigned dst = ms_ring + (unsigned)spec_slots * TA.ms_slot_bytes;
                                tma_load_4d(dst, hmap0, x0 - HX, y0 - 1, zq, 0, bar);
                                if constexpr (NH == 2) tma_load_4d(dst + TA.hbox_bytes, hmap1, x0 - HX, y0 - 1, zq, 0, bar);
                                ++spec_slots;
                            }
                            advance(zz, txx, tyy);
                        }
                    }
                    __syncwarp();
                }
                // verdict and buffer indices in s_ctrl
                asm volatile("bar.sync 2, %0;" ::"n"(kTmaThreads) : "memory");
                const Ctrl* const sc = reinterpret_cast<const Ctrl*>(s_ctrl);
                const int ys = ycur, ks = k1slot;
                done = sc->done; N = sc->N; ycur = sc->ycur; k1slot = sc->k1slot;
                if (spec && (done || ycur != ys || k1slot != ks)) {
                    // rejected step (or the run is over): the tiles fetched are the wrong buffers.  Let them land, burn the
                    // phase of the untouched slots as well, and start over - the consumers know (spec_miss) that every
                    // "full" barrier of the ms ring is one phase ahead.
                    if (issuer) {
                        for (int i = 0; i < spec_slots; ++i) mbar_wait(full_ms + 8 * i, 0u);
                        for (int i = spec_slots; i < Dm; ++i) mbar_expect_tx(full_ms + 8 * i, 0u);
                    }
                    spec_slots = 0;
                }
                setup_maps();
            } else if (!have_ctrl) {
                done = ctrl->done; N = ctrl->N; ycur = ctrl->ycur; k1slot = ctrl->k1slot;
                setup_maps();
            }
            if (done) {                             // the run is over: let the early profile loads land, then leave
                if (issuer)
                    for (int i = 0; i < pre_u; ++i) mbar_wait(full_u + 8 * i, 0u);
                if constexpr (SWEEP) continue; else return;
            }
        }
        if (issuer) {
            int z = z0, tx = tx0, ty = ty0;
            auto issue_ms = [&](int x0, int y0, int zz) {
                if (spec_slots > 0) {                   // filled before the verdict, same order
                    --spec_slots;
                    if (++hm == Dm) { hm = 0; pm ^= 1u; }
                    return;
                }
                mbar_wait(empty_ms + 8 * hm, pm);
                const unsigned bar = full_ms + 8 * hm;
                mbar_expect_tx(bar, NH * TA.hbox_tx);
                const unsigned dst = ms_ring + (unsigned)hm * TA.ms_slot_bytes;
                tma_load_4d(dst, hmap0, x0 - HX, y0 - 1, zz, 0, bar);
                if constexpr (NH == 2) tma_load_4d(dst + TA.hbox_bytes, hmap1, x0 - HX, y0 - 1, zz, 0, bar);
                if (++hm == Dm) { hm = 0; pm ^= 1u; }
            };
            for (int p = 0; p < nplanes; ++p) {
                const int x0 = tx * TX, y0 = ty * kTmaTY;
                if (p == 0 || z == zfirst) { issue_ms(x0, y0, z - dir); issue_ms(x0, y0, z); }
                issue_ms(x0, y0, z + dir);
                if constexpr (NB > 0) {
#pragma unroll 1
                    for (int ch = 0; ch < NCH; ++ch) {       // mode profiles, UCB per slot (out-of-range modes zero-filled)
                        if (pre_u > 0) { --pre_u; }          // filled before the dependency wait
                        else {
                            mbar_wait(empty_u + 8 * hu, pu);
                            const unsigned bar = full_u + 8 * hu;
                            mbar_expect_tx(bar, u_tx);
                            tma_load_4d(u_ring + (unsigned)hu * u_tx, umap, x0, y0, z, ch * kTmaUChunk, bar);
                        }
                        if (++hu == Du) { hu = 0; pu ^= 1u; }
                    }
                }
                if constexpr (NAUX > 0) {
                    const unsigned bar = full_aux + 8 * ha;
                    unsigned dst = aux_ring + (unsigned)ha * aux_tx;
                    if (pre_a > 0) {                          // armed before the dependency wait: k_{s-1} (and what npre left out) is missing
                        --pre_a;
#pragma unroll
                        for (int f = 0; f < NAUX; ++f)
                            if (f >= npre) tma_load_4d(dst + (unsigned)(f * C * APLANE), amap[f], x0, y0, z, 0, bar);
                    } else {
                        mbar_wait(empty_aux + 8 * ha, pa);
                        mbar_expect_tx(bar, aux_tx);
#pragma unroll
                        for (int f = 0; f < NAUX; ++f) {
                            tma_load_4d(dst, amap[f], x0, y0, z, 0, bar);
                            dst += C * APLANE;
                        }
                    }
                    if (++ha == Da) { ha = 0; pa ^= 1u; }
                }
                advance(z, tx, ty);
            }
            CAVMAG_MARK(6);
        }
        }   // sub-runs
    } else {
        // ================================ consumers =================================
        int hm = 0, ha = 0, hu = 0, tm = 0;          // ring heads (next slot to acquire) and the ms tail (next to release), carried over the sub-runs
        unsigned pm = 0, pa = 0, pu = 0;             // parity to wait on for "full"
        for (int sr = 0; sr < nsr; ++sr) {
            enter_subrun(sr);
            const StageArgs& A = SWEEP ? Arep : Aouter;
            Ctrl* const ctrl = A.ctrl;
        if constexpr (POL) {
            if (tid < 6 * NB) s_pq[tid] = (tid / 6 < TA.N) ? (T)A.pol[tid] : (T)0;      // (visible after the consumers' barrier below)
        }
        if (!SWEEP || sr == 0) {
            asm volatile("griddepcontrol.wait;" ::: "memory");
            if constexpr (SWEEP && STAGE == 3) {
                // the stage-2 kernel has completed: its owners have counted the simulations that go on
                if (blockIdx.x == 0 && tid == 0) {
                    const unsigned int v = atomicExch(SW.live, 0u);
                    if (SW.cond_handle != 0ull) cudaGraphSetConditional((cudaGraphConditionalHandle)SW.cond_handle, v > 0u ? 1u : 0u);
                }
            }
        }
        if (tid == 0) CAVMAG_MARK(15);
        double hd;
        if constexpr (STAGE == 2) {
            // finish stage 7 of the previous step, run the controller, start this step (all blocks, same bits)
            int spec_miss = 0;
            if (!deferred_finish7<NB, NSUB>(A, TA, tid, s_ctrl, s_red, s_err, trace, nblk_r, slot == 0, SWEEP ? SW.live : nullptr, spec_miss)) {
                if constexpr (SWEEP) continue; else return;
            }
            if constexpr (!SWEEP) { if (spec_miss) pm = 1u; }      // the producer re-issued its speculative tiles: ms "full" barriers are one phase ahead
            const Ctrl* const sc = reinterpret_cast<const Ctrl*>(s_ctrl);
            N = sc->N; ycur = sc->ycur; k1slot = sc->k1slot; hd = sc->h;
            if (NB > 0 && tid < NB) s_cn[tid] = (tid < N) ? (T)sc->c[tid] : (T)0;
        } else if constexpr (kDeferred) {
            if (!deferred_finish<STAGE - 1, NB>(A, ctrl, tid, s_ctrl, s_red, nblk_r, slot == 0)) {
                if constexpr (SWEEP) continue; else return;
            }
            const Ctrl* const sc = reinterpret_cast<const Ctrl*>(s_ctrl);
            N = sc->N; ycur = sc->ycur; k1slot = sc->k1slot; hd = sc->h;
            if (NB > 0 && tid < NB) s_cn[tid] = (tid < N) ? (T)sc->c[tid] : (T)0;
        } else {
            const int done = ctrl->k1_valid;            // stage 1: k1 of a fresh state
            N = ctrl->N; ycur = ctrl->ycur; k1slot = ctrl->k1slot; hd = ctrl->h;
            double cv = 0.0;
            if (NB > 0 && tid < NB) cv = ctrl->c[tid];
            if (done) return;
            if (NB > 0 && tid < NB) s_cn[tid] = (tid < N) ? (T)cv : (T)0;
        }
        asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
        if (tid == 0) CAVMAG_MARK(1);
        const T h = (T)hd;
        const T ha21 = h * (T)kA[1][0];
        T cn_reg[(NB > 0 && NB <= 8) ? NB : 1];
        if constexpr (NB > 0 && NB <= 8) {
#pragma unroll
            for (int n = 0; n < NB; ++n) cn_reg[n] = s_cn[n];
        }
        T cp_reg[POL ? 3 * NB : 1];                 // c_n p_n: the RF field of mode n per unit of u_n
        if constexpr (POL) {
#pragma unroll
            for (int n = 0; n < NB; ++n)
#pragma unroll
                for (int k = 0; k < 3; ++k) cp_reg[3 * n + k] = s_cn[n] * s_pq[6 * n + k];
        }
        const T B0x = (T)A.B0[0], B0y = (T)A.B0[1], B0z = (T)A.B0[2];
        const T wx = (T)A.ex_wx, wy = (T)A.ex_wy, wz = (T)A.ex_wz;
        const T anp = (T)A.an_pref, axx = (T)A.axis[0], axy = (T)A.axis[1], axz = (T)A.axis[2];
        const T alpha = (T)A.alpha, llg = (T)A.llg, BE = (T)A.B_exch_inter;
        const bool renorm = A.renormalize != 0;

        T* __restrict__ ynew = (T*)(ycur ? A.Y[0] : A.Y[1]);
        T* __restrict__ kout = STAGE == 1 ? (T*)(k1slot ? A.K[6] : A.K[0]) : STAGE == 7 ? (T*)(k1slot ? A.K[0] : A.K[6]) : (T*)A.K[STAGE - 1];
        T* __restrict__ mnext = STAGE == 6 ? ynew : (STAGE == 2 || STAGE == 4) ? (T*)A.MS[0] : (T*)A.MS[1];
        T* __restrict__ e6g = (T*)A.MS[0];

        T ox[NB > 0 ? NB : 1], oy[NB > 0 ? NB : 1], oz[POL ? NB : 1];
#pragma unroll
        for (int n = 0; n < NB; ++n) { ox[n] = (T)0; oy[n] = (T)0; if constexpr (POL) oz[n] = (T)0; }
        T sm[NSUB * 3];
#pragma unroll
        for (int i = 0; i < NSUB * 3; ++i) sm[i] = (T)0;
        T emax2 = (T)0;

        const long long plane = (long long)A.pitch * ny;     // plane stride in memory
        const unsigned crow = (unsigned)((warp + 1) * kTmaHaloRowBytes + kTmaHaloBytes + lane * 8);   // centre, within a comp plane
        const unsigned arow = (unsigned)(warp * kTmaRowBytes + lane * 8);

        int z = z0, tx = tx0, ty = ty0;
        unsigned sm_zm = 0, sm_zc = 0, sm_zp = 0;    // shared addresses of the live stage-state planes
        auto acquire_ms = [&]() -> unsigned {
            mbar_wait(full_ms + 8 * hm, pm);
            const unsigned a = ms_ring + (unsigned)hm * TA.ms_slot_bytes;
            if (++hm == Dm) { hm = 0; pm ^= 1u; }
            return a;
        };
        auto release_ms = [&]() {
            mbar_arrive(empty_ms + 8 * tm);
            if (++tm == Dm) tm = 0;
        };

        // per-tile quantities (refreshed when the tile changes)
        bool active = false;
        long long cell = 0;                          // global cell index of this lane's first cell in plane z
        T wxl = (T)0, wxr = (T)0, wxi = (T)0, wym = (T)0, wyp = (T)0;
        bool new_tile = true;

        // stage state from a halo box (STAGE 2: formed on the fly from y0 and k1)
        auto ldm = [&](unsigned slot, int comp, unsigned off) -> P {
            const unsigned p = slot + (unsigned)(comp * HPLANE) + off;
            P a = lds_pack(p, tag);
            if constexpr (STAGE == 2) {
                const P b = lds_pack(p + TA.hbox_bytes, tag);
#pragma unroll
                for (int v = 0; v < VEC; ++v) a.v[v] = a.v[v] + ha21 * b.v[v];
            }
            return a;
        };
        auto ldm1_if = [&](unsigned slot, int comp, unsigned off, unsigned pred) -> T {
            const unsigned p = slot + (unsigned)(comp * HPLANE) + off;
            T a = lds_one_if(p, pred, tag);
            if constexpr (STAGE == 2) a = a + ha21 * lds_one_if(p + TA.hbox_bytes, pred, tag);
            return a;
        };
        const unsigned is_lane0 = lane == 0 ? 1u : 0u, is_lane31 = lane == 31 ? 1u : 0u;

#pragma unroll 1
        for (int pl = 0; pl < nplanes; ++pl) {
            if (new_tile) {
                const int gx = tx * TX + lane * VEC, gy = ty * kTmaTY + warp;
                active = gx < nx && gy < ny;
                // open boundary (G9): an out-of-grid neighbour gets weight 0; its TMA-zero-filled value is finite
                wxl = gx > 0 ? wx : (T)0;
                wxr = gx + VEC < nx ? wx : (T)0;
                wxi = gx + 1 < nx ? wx : (T)0;          // neighbour inside the lane's pair (a padded row may end on an odd nx)
                wym = gy > 0 ? wy : (T)0;
                wyp = gy < ny - 1 ? wy : (T)0;
                cell = (long long)z * plane + (long long)gy * A.pitch + gx;
                new_tile = false;
            }
            const bool seg_start = (pl == 0 || z == zfirst);
            const bool seg_end = (pl + 1 == nplanes || z == zlast);
            if (seg_start) { sm_zm = acquire_ms(); sm_zc = acquire_ms(); }
            sm_zp = acquire_ms();
            if (pl == 0 && tid == 0) CAVMAG_MARK(2);
            const T wzm = z > 0 ? wz : (T)0, wzp = z < nz - 1 ? wz : (T)0;

            P mc[NSUB][3];
#pragma unroll
            for (int s = 0; s < NSUB; ++s)
#pragma unroll
                for (int c = 0; c < 3; ++c) mc[s][c] = ldm(sm_zc, s * 3 + c, crow);

            // ---- mode profiles (ring u): RF field and overlap partials of THIS stage state ----
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
                for (int ch = 0; ch < NCH; ++ch) {
                    mbar_wait(full_u + 8 * hu, pu);
                    const unsigned us = u_ring + (unsigned)hu * (unsigned)(UCB * APLANE) + arow;
                    P un[UCB];
#pragma unroll
                    for (int i = 0; i < UCB; ++i) un[i] = lds_pack(us + (unsigned)(i * APLANE), tag);
                    __syncwarp();
                    if (lane == 0) mbar_arrive(empty_u + 8 * hu);
                    if (++hu == Du) { hu = 0; pu ^= 1u; }
#pragma unroll
                    for (int i = 0; i < UCB; ++i) {
                        const int n = ch * kTmaUChunk + i;          // modes >= N: u zero-filled, c_n = 0
                        if constexpr (!POL) {
                            const T cn = (NB <= 8) ? cn_reg[NB <= 8 ? n : 0] : s_cn[n];     // few modes: RF weights live in registers
#pragma unroll
                            for (int v = 0; v < VEC; ++v) {
                                brf[v] += cn * un[i].v[v];
                                ox[n] += un[i].v[v] * mcx[v];
                                oy[n] += un[i].v[v] * mcy[v];
                            }
                        } else {
#pragma unroll
                            for (int v = 0; v < VEC; ++v) {
                                brf[v] += cp_reg[POL ? 3 * n : 0] * un[i].v[v];
                                brfy[v] += cp_reg[POL ? 3 * n + 1 : 0] * un[i].v[v];
                                brfz[v] += cp_reg[POL ? 3 * n + 2 : 0] * un[i].v[v];
                                ox[n] += un[i].v[v] * mcx[v];
                                oy[n] += un[i].v[v] * mcy[v];
                                oz[POL ? n : 0] += un[i].v[v] * mcz[v];
                            }
                        }
                    }
                }
            }
            // ---- halo-free cell streams (ring aux): only the fused tail below reads them ----
            unsigned axf = 0;
            int aslot = 0;
            if constexpr (NAUX > 0) {
                aslot = ha;
                mbar_wait(full_aux + 8 * ha, pa);
                axf = aux_ring + (unsigned)ha * (unsigned)(NAUX * C * APLANE) + arow;
                if (++ha == Da) { ha = 0; pa ^= 1u; }
            }

#pragma unroll
            for (int s = 0; s < NSUB; ++s) {
                // ---- 6-neighbour exchange: sum over in-grid neighbours of (m_nb - m) (2A/Ms)/D^2 ----
                T lap[3][VEC];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const int comp = s * 3 + c;
                    const P nym = ldm(sm_zc, comp, crow - kTmaHaloRowBytes);
                    const P nyp = ldm(sm_zc, comp, crow + kTmaHaloRowBytes);
                    const P nzm = ldm(dir > 0 ? sm_zm : sm_zp, comp, crow);      // sm_zm / sm_zp: previous / next plane of the sweep
                    const P nzp = ldm(dir > 0 ? sm_zp : sm_zm, comp, crow);
                    T xl = __shfl_up_sync(0xffffffffu, mc[s][c].v[VEC - 1], 1);
                    T xr = __shfl_down_sync(0xffffffffu, mc[s][c].v[0], 1);
                    const T xl_h = ldm1_if(sm_zc, comp, crow - (unsigned)sizeof(T), is_lane0);
                    const T xr_h = ldm1_if(sm_zc, comp, crow + 8u, is_lane31);
                    xl = is_lane0 ? xl_h : xl;
                    xr = is_lane31 ? xr_h : xr;
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const T m0 = mc[s][c].v[v];
                        const T left = (v == 0) ? xl : mc[s][c].v[v > 0 ? v - 1 : 0];
                        const T right = (v == VEC - 1) ? xr : mc[s][c].v[v < VEC - 1 ? v + 1 : VEC - 1];
                        T l = (left - m0) * ((v == 0) ? wxl : wx);
                        l += (right - m0) * ((v == VEC - 1) ? wxr : wxi);
                        l += (nym.v[v] - m0) * wym;
                        l += (nyp.v[v] - m0) * wyp;
                        l += (nzm.v[v] - m0) * wzm;
                        l += (nzp.v[v] - m0) * wzp;
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
                    llg_slope(mx, my, mz, Bx, By, Bz, alpha, llg, ks[0].v[v], ks[1].v[v], ks[2].v[v]);
                }

#pragma unroll
                for (int c = 0; c < 3; ++c)
                    if (active) stp<T, VEC>(kout + (long long)(s * 3 + c) * nc + cell, ks[c]);

                if constexpr (STAGE >= 2 && STAGE <= 5) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const int comp = s * 3 + c;
                        P m0v, q[STAGE];               // k_1 .. k_STAGE of this component
                        if constexpr (STAGE == 2) {
                            m0v = lds_pack(sm_zc + (unsigned)(comp * HPLANE) + crow, tag);
                            q[0] = lds_pack(sm_zc + TA.hbox_bytes + (unsigned)(comp * HPLANE) + crow, tag);
                        } else {
                            m0v = lds_pack(axf + (unsigned)(comp * APLANE), tag);
#pragma unroll
                            for (int j = 0; j < STAGE - 1; ++j) q[j] = lds_pack(axf + (unsigned)(((1 + j) * C + comp) * APLANE), tag);
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
                        if (active) stp<T, VEC>(mnext + (long long)comp * nc + cell, out);
                    }
                }
                if constexpr (STAGE == 6) {
                    P y5[3], er[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const int comp = s * 3 + c;
                        const P m0v = lds_pack(axf + (unsigned)(comp * APLANE), tag);
                        const P q1 = lds_pack(axf + (unsigned)((C + comp) * APLANE), tag);
                        const P q3 = lds_pack(axf + (unsigned)((2 * C + comp) * APLANE), tag);
                        const P q4 = lds_pack(axf + (unsigned)((3 * C + comp) * APLANE), tag);
                        const P q5 = lds_pack(axf + (unsigned)((4 * C + comp) * APLANE), tag);
#pragma unroll
                        for (int v = 0; v < VEC; ++v) {
                            const T kv[6] = {q1.v[v], (T)0, q3.v[v], q4.v[v], q5.v[v], ks[c].v[v]};      // b_2 = d_2 = 0: k_2 is not read
                            y5[c].v[v] = dp_state<6>(m0v.v[v], kv, h);
                            er[c].v[v] = dp_error6(kv, h);
                        }
                    }
                    if (renorm) {
#pragma unroll
                        for (int v = 0; v < VEC; ++v) {
                            const T inv = rsqrt_t<T>(y5[0].v[v] * y5[0].v[v] + y5[1].v[v] * y5[1].v[v] + y5[2].v[v] * y5[2].v[v]);
                            y5[0].v[v] *= inv; y5[1].v[v] *= inv; y5[2].v[v] *= inv;
                        }
                    }
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const long long off = (long long)(s * 3 + c) * nc + cell;
                        if (active) { stp<T, VEC>(mnext + off, y5[c]); stp<T, VEC>(e6g + off, er[c]); }
                    }
                }
                if constexpr (STAGE == 7) {
                    P er[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) er[c] = lds_pack(axf + (unsigned)((s * 3 + c) * APLANE), tag);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const T e2 = dp_error7_sq(er[0].v[v], er[1].v[v], er[2].v[v], ks[0].v[v], ks[1].v[v], ks[2].v[v], h);
                        // out-of-grid lanes hold TMA zero fill: e2 = 0 and m = 0, so they need no mask
                        emax2 = fmax(emax2, e2);
                        sm[s * 3 + 0] += mc[s][0].v[v]; sm[s * 3 + 1] += mc[s][1].v[v]; sm[s * 3 + 2] += mc[s][2].v[v];
                    }
                }
            }

            // ---- release the slots this plane no longer needs ----
            __syncwarp();
            if (lane == 0) {
                if constexpr (NAUX > 0) mbar_arrive(empty_aux + 8 * aslot);
                release_ms();                                   // plane z-1
                if (seg_end) { release_ms(); release_ms(); }    // planes z, z+1 (the next segment reloads its own)
            }
            sm_zm = sm_zc; sm_zc = sm_zp;
            cell += dir > 0 ? plane : -plane;
            if (advance(z, tx, ty)) new_tile = true;
        }

        if (tid == 0) CAVMAG_MARK(3);
        // ---- pass 1 of the reductions: warp shuffle tree; lane 0 of each consumer warp deposits ----
        constexpr int NS = 2 * NB + (STAGE == 7 ? 3 * NSUB : 0);
        __shared__ double swarp[kTmaTY][NS > 0 ? NS : 1];
        __shared__ double swmax[kTmaTY];
        {
            T vals[NS > 0 ? NS : 1];
#pragma unroll
            for (int n = 0; n < NB; ++n) {
                if constexpr (!POL) { vals[2 * n] = ox[n]; vals[2 * n + 1] = oy[n]; }
                else {              // sum u (m.p) and sum u (m.q) from the raw sums
                    vals[2 * n] = ox[n] * s_pq[6 * n] + oy[n] * s_pq[6 * n + 1] + oz[POL ? n : 0] * s_pq[6 * n + 2];
                    vals[2 * n + 1] = ox[n] * s_pq[6 * n + 3] + oy[n] * s_pq[6 * n + 4] + oz[POL ? n : 0] * s_pq[6 * n + 5];
                }
            }
            if constexpr (STAGE == 7) {
#pragma unroll
                for (int i = 0; i < 3 * NSUB; ++i) vals[2 * NB + i] = sm[i];
            }
#pragma unroll
            for (int i = 0; i < NS; ++i) {
                T x = vals[i];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
                if (lane == 0) swarp[warp][i] = (double)x;
            }
            if constexpr (STAGE == 7) {
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) emax2 = fmax(emax2, __shfl_xor_sync(0xffffffffu, emax2, o));
                if (lane == 0) swmax[warp] = (double)emax2;
            }
        }
        // consumer-only barrier (the producer warp does not take part)
        asm volatile("bar.sync 1, %0;" ::"n"(kTmaConsumers) : "memory");
        if (tid < NS) {
            const int i = tid;
            const bool used = (i < 2 * NB) ? (i < 2 * N) : true;
            if (used) {
                double acc = 0.0;
#pragma unroll
                for (int w = 0; w < kTmaTY; ++w) acc += swarp[w][i];
                const int comp = (i < 2 * NB) ? i : (2 * N + (i - 2 * NB));
                stage_partials(A, STAGE)[(size_t)comp * A.pstride + slot] = acc;
            }
        }
        if (STAGE == 7 && tid == 0) {
            double mx = 0.0;
#pragma unroll
            for (int w = 0; w < kTmaTY; ++w) mx = fmax(mx, swmax[w]);
            A.partial_max[slot] = mx;
        }
        }   // sub-runs
    }

    // ---- stage 1 (k1 of a fresh state, once per run at most): last-block-done -> second reduction pass, mode ODE,
    //      start of the first step.  Stages 2..7 end here: their finish runs in the prologue of the next stage
    //      kernel (deferred_finish; stage 7 and the step controller: deferred_finish7 in the next stage-2 kernel). ----
    if constexpr (STAGE == 1) {
        // One fence per block: the barrier orders every thread's stores before thread 0's gpu-scope fence
        // (release); the last block's thread 0 fences again after the ticket (acquire) before the barrier that
        // lets its threads read the other blocks' partials.
        __shared__ int s_last;
        Ctrl* const ctrl = A.ctrl;
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            CAVMAG_MARK(4);
            const unsigned int old = atomicAdd(&ctrl->arrive, 1u);
            s_last = (old == gridDim.x - 1) ? 1 : 0;
            if (s_last) __threadfence();
        }
        __syncthreads();
        if (s_last) stage_finish<STAGE>(finish_args(A, STAGE), NSUB, N, trace);
#ifdef CAVMAG_PROBE
        __syncthreads();
        if (tid == 0) { CAVMAG_MARK(5); A.probe[((size_t)STAGE * gridDim.x + blockIdx.x) * 32 + 7] = (unsigned long long)s_last; }
#endif
    } else {
#ifdef CAVMAG_PROBE
        __syncthreads();
        if (tid == 0) { CAVMAG_MARK(4); CAVMAG_MARK(5); }
#endif
    }
}

template <typename T, int STAGE, int NSUB, int NB>
__global__ void __launch_bounds__(kTmaThreads, 1) k_stage_tma(const __grid_constant__ StageArgs A, const __grid_constant__ TmaArgs TA,
                                                              double* __restrict__ trace) {
    stage_tma_body<T, STAGE, NSUB, NB, false>(A, TA, trace, SweepArgs{nullptr, 1, nullptr, 0ull});
}

template <typename T, int STAGE, int NSUB, int NB>
__global__ void __launch_bounds__(kTmaThreads, 1) k_stage_tma_pol(const __grid_constant__ StageArgs A, const __grid_constant__ TmaArgs TA,
                                                                  double* __restrict__ trace) {
    stage_tma_body<T, STAGE, NSUB, NB, false, true>(A, TA, trace, SweepArgs{nullptr, 1, nullptr, 0ull});
}

// Joint launch over SW.R simulations of the same shape: A carries the shared grid / material constants (and simulation
// 0's pointers, unused), SW.reps the per-simulation pointers.
template <typename T, int STAGE, int NSUB, int NB>
__global__ void __launch_bounds__(kTmaThreads, 1) k_stage_tma_sweep(const __grid_constant__ StageArgs A, const __grid_constant__ TmaArgs TA,
                                                                    const __grid_constant__ SweepArgs SW) {
    stage_tma_body<T, STAGE, NSUB, NB, true>(A, TA, nullptr, SW);
}

const void* stage_tma_sweep_kernel_f32(int n_sub, int stage, int nb);
const void* stage_tma_sweep_kernel_f64(int n_sub, int stage, int nb);

#define CAVMAG_TMA_SWEEP_CASES(T, NSUB, NB)                                        \
    switch (stage) {                                                               \
        case 2: return (const void*)k_stage_tma_sweep<T, 2, NSUB, NB>;             \
        case 3: return (const void*)k_stage_tma_sweep<T, 3, NSUB, NB>;             \
        case 4: return (const void*)k_stage_tma_sweep<T, 4, NSUB, NB>;             \
        case 5: return (const void*)k_stage_tma_sweep<T, 5, NSUB, NB>;             \
        case 6: return (const void*)k_stage_tma_sweep<T, 6, NSUB, NB>;             \
        case 7: return (const void*)k_stage_tma_sweep<T, 7, NSUB, NB>;             \
        default: return nullptr;                                                   \
    }
// the sweeps of the paper have 1-3 modes: mode buckets 0, 1, 2 and 8 for the ferromagnet,
// 0, 1 and 2 for the two-sublattice antiferromagnet
#define CAVMAG_DEFINE_TMA_SWEEP_LOOKUP(NAME, T)                                    \
    const void* NAME(int n_sub, int stage, int nb) {                               \
        if (n_sub == 1) {                                                          \
            if (nb == 0) { CAVMAG_TMA_SWEEP_CASES(T, 1, 0) }                       \
            if (nb == 1) { CAVMAG_TMA_SWEEP_CASES(T, 1, 1) }                       \
            if (nb == 2) { CAVMAG_TMA_SWEEP_CASES(T, 1, 2) }                       \
            if (nb == 8) { CAVMAG_TMA_SWEEP_CASES(T, 1, 8) }                       \
        } else {                                                                   \
            if (nb == 0) { CAVMAG_TMA_SWEEP_CASES(T, 2, 0) }                       \
            if (nb == 1) { CAVMAG_TMA_SWEEP_CASES(T, 2, 1) }                       \
            if (nb == 2) { CAVMAG_TMA_SWEEP_CASES(T, 2, 2) }                       \
        }                                                                          \
        return nullptr;                                                            \
    }

const void* stage_tma_kernel_f32_fm(int stage, int nb);
const void* stage_tma_kernel_f32_afm(int stage, int nb);
const void* stage_tma_kernel_f64_fm(int stage, int nb);
const void* stage_tma_kernel_f64_afm(int stage, int nb);

#define CAVMAG_TMA_STAGE_CASES(T, NSUB, NB)                                        \
    switch (stage) {                                                               \
        case 1: return (const void*)k_stage_tma<T, 1, NSUB, NB>;                   \
        case 2: return (const void*)k_stage_tma<T, 2, NSUB, NB>;                   \
        case 3: return (const void*)k_stage_tma<T, 3, NSUB, NB>;                   \
        case 4: return (const void*)k_stage_tma<T, 4, NSUB, NB>;                   \
        case 5: return (const void*)k_stage_tma<T, 5, NSUB, NB>;                   \
        case 6: return (const void*)k_stage_tma<T, 6, NSUB, NB>;                   \
        case 7: return (const void*)k_stage_tma<T, 7, NSUB, NB>;                   \
        default: return nullptr;                                                   \
    }

// per-mode polarisation (k_stage_tma_pol): mode buckets 1, 2, 8
const void* stage_tma_pol_kernel_f32_fm(int stage, int nb);
const void* stage_tma_pol_kernel_f32_afm(int stage, int nb);
const void* stage_tma_pol_kernel_f64_fm(int stage, int nb);
const void* stage_tma_pol_kernel_f64_afm(int stage, int nb);

#define CAVMAG_TMA_POL_STAGE_CASES(T, NSUB, NB)                                    \
    switch (stage) {                                                               \
        case 1: return (const void*)k_stage_tma_pol<T, 1, NSUB, NB>;               \
        case 2: return (const void*)k_stage_tma_pol<T, 2, NSUB, NB>;               \
        case 3: return (const void*)k_stage_tma_pol<T, 3, NSUB, NB>;               \
        case 4: return (const void*)k_stage_tma_pol<T, 4, NSUB, NB>;               \
        case 5: return (const void*)k_stage_tma_pol<T, 5, NSUB, NB>;               \
        case 6: return (const void*)k_stage_tma_pol<T, 6, NSUB, NB>;               \
        case 7: return (const void*)k_stage_tma_pol<T, 7, NSUB, NB>;               \
        default: return nullptr;                                                   \
    }

#define CAVMAG_DEFINE_TMA_POL_LOOKUP(NAME, T, NSUB)                                \
    const void* NAME(int stage, int nb) {                                          \
        if (nb == 1) { CAVMAG_TMA_POL_STAGE_CASES(T, NSUB, 1) }                    \
        if (nb == 2) { CAVMAG_TMA_POL_STAGE_CASES(T, NSUB, 2) }                    \
        if (nb == 8) { CAVMAG_TMA_POL_STAGE_CASES(T, NSUB, 8) }                    \
        return nullptr;                                                            \
    }

#define CAVMAG_DEFINE_TMA_LOOKUP(NAME, T, NSUB)                                    \
    const void* NAME(int stage, int nb) {                                          \
        if (nb == 0) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 0) }                        \
        if (nb == 1) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 1) }                        \
        if (nb == 2) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 2) }                        \
        if (nb == 8) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 8) }                        \
        if (nb == 32) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 32) }                      \
        return nullptr;                                                            \
    }

}  // namespace cavmag
