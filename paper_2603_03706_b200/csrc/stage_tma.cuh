// The fused RK45 stage kernel, TMA-pipelined variant (hand-written CUDA for sm_100a).
//
// Same arithmetic as stage_kernel.cuh (one launch = one evaluation of the coupled right-hand
// side at stage s, fused with the overlap partials, the next stage state, the error norm and,
// in the last block, the mode ODEs + controller), but the data movement is Blackwell-native:
//
//   * persistent grid, one CTA per SM; the flattened list of plane-tiles (x-y tile, z) is split
//     into contiguous, equally long runs, one per CTA, so every SM gets the same number of
//     planes and marches in z (each plane of m_s is fetched once per run, plus one halo plane
//     per run end);
//   * a producer warp (one elected lane) issues cp.async.bulk.tensor (TMA) loads of 4-D boxes
//     [comp][1][TY(+2)][TX(+2 HX)] into three shared-memory rings — the stage state with its
//     x/y halo (ring "ms": planes z-1, z, z+1 live), the mode profiles u_n in chunks of 8
//     (ring "u") and the halo-free cell streams y0, k_j, e6 (ring "aux") — completing on
//     mbarriers (expect_tx / complete_tx);
//   * 8 consumer warps (one tile row each, 8 bytes of x per lane) read shared memory only:
//     x neighbours by warp shuffle, y/z neighbours from the halo box / the neighbouring ring
//     slots, so no global load sits on the dependent path and the bytes in flight are set by
//     the ring depth (~100-180 KB per SM) instead of by registers and occupancy;
//   * results go straight from registers to global memory with coalesced 8-byte stores.
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
};

// ---- PTX wrappers ----------------------------------------------------------------------
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
__device__ __forceinline__ void mbar_wait(unsigned bar, unsigned parity) {
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tma_load_4d(unsigned dst, const void* map, int c0, int c1, int c2, int c3, unsigned bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];"
        ::"r"(dst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(c3), "r"(bar) : "memory");
}

// number of halo'd fields / plain cell fields the stage streams
template <int STAGE> struct StageStreams {
    static constexpr int n_halo = (STAGE == 2) ? 2 : 1;
    static constexpr int n_aux = (STAGE <= 2) ? 0 : (STAGE == 7) ? 1 : (STAGE == 6) ? 5 : STAGE;   // y0,k1,.. / e6
};

template <typename T, int STAGE, int NSUB, int NB>
__global__ void __launch_bounds__(kTmaThreads, 1) k_stage_tma(const StageArgs A, const TmaArgs TA, double* __restrict__ trace) {
    constexpr int VEC = 8 / (int)sizeof(T);              // cells per lane: 2 floats / 1 double
    constexpr int TX = kTmaRowBytes / (int)sizeof(T);    // cells per tile row
    constexpr int HX = kTmaHaloBytes / (int)sizeof(T);   // x halo in cells (16 bytes: 4 floats / 2 doubles)
    constexpr int C = 3 * NSUB;
    constexpr int NH = StageStreams<STAGE>::n_halo;
    constexpr int NAUX = StageStreams<STAGE>::n_aux;
    using P = Pack<T, VEC>;

    Ctrl* ctrl = A.ctrl;
    if (STAGE == 1) { if (ctrl->k1_valid) return; }
    else if (ctrl->done) return;

    extern __shared__ __align__(128) unsigned char smem_raw[];
    __shared__ __align__(8) unsigned long long bars[6 * kTmaMaxDepth];
    __shared__ T s_cn[NB > 0 ? NB : 1];

    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int N = ctrl->N;
    const int nx = A.nx, ny = A.ny, nz = A.nz;
    const long long nc = A.nc;
    const int Dm = TA.Dm, Da = TA.Da, Du = TA.Du;

    unsigned char* smem = (unsigned char*)(((uintptr_t)smem_raw + 127) & ~(uintptr_t)127);
    unsigned char* ms_ring = smem;
    unsigned char* aux_ring = smem + (size_t)Dm * TA.ms_slot_bytes;
    unsigned char* u_ring = aux_ring + (size_t)Da * TA.aux_slot_bytes;
    const unsigned full_ms = smem_u32(&bars[0]), empty_ms = smem_u32(&bars[kTmaMaxDepth]);
    const unsigned full_aux = smem_u32(&bars[2 * kTmaMaxDepth]), empty_aux = smem_u32(&bars[3 * kTmaMaxDepth]);
    const unsigned full_u = smem_u32(&bars[4 * kTmaMaxDepth]), empty_u = smem_u32(&bars[5 * kTmaMaxDepth]);

    if (tid == 0) {
        for (int i = 0; i < Dm; ++i) { mbar_init(full_ms + 8 * i, 1); mbar_init(empty_ms + 8 * i, kTmaTY); }
        for (int i = 0; i < Da; ++i) { mbar_init(full_aux + 8 * i, 1); mbar_init(empty_aux + 8 * i, kTmaTY); }
        for (int i = 0; i < Du; ++i) { mbar_init(full_u + 8 * i, 1); mbar_init(empty_u + 8 * i, kTmaTY); }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    if (NB > 0 && tid < NB) s_cn[tid] = (tid < N) ? (T)ctrl->c[tid] : (T)0;
    __syncthreads();

    // this CTA's run of plane-tiles
    const long long q0 = (TA.Q * (long long)blockIdx.x) / gridDim.x;
    const long long q1 = (TA.Q * (long long)(blockIdx.x + 1)) / gridDim.x;
    const int ycur = ctrl->ycur, k1slot = ctrl->k1slot;

    if (warp == kTmaTY) {
        // =============================== TMA producer ===============================
        if (lane == 0 && q0 < q1) {
            const unsigned char* maps = TA.maps;
            auto mp = [&](int i) { return (const void*)(maps + 128 * i); };
            // halo'd stage-state field(s)
            const void* hmap0 = STAGE == 1 ? mp(MAP_H_Y0 + ycur) : STAGE == 2 ? mp(MAP_H_Y0 + ycur)
                               : STAGE == 7 ? mp(MAP_H_Y0 + (1 - ycur))
                               : (STAGE == 3 || STAGE == 5) ? mp(MAP_H_MS0) : mp(MAP_H_MS1);
            const void* hmap1 = mp(k1slot == 0 ? MAP_H_K0 : MAP_H_K6);     // STAGE 2 only
            const void* amap[5];
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
            const void* umap = mp(MAP_P_U);
            const unsigned aux_tx = (unsigned)(NAUX * C) * (unsigned)(kTmaRowBytes * kTmaTY);
            const int nch = (NB > 0) ? TA.n_uchunks : 0;

            long long t = q0 / nz;
            int z = (int)(q0 - t * nz);
            unsigned jm = 0, ja = 0, ju = 0;
            auto issue_ms = [&](int x0, int y0, int zz) {
                const unsigned slot = jm % (unsigned)Dm, par = (jm / (unsigned)Dm) & 1u;
                mbar_wait(empty_ms + 8 * slot, par ^ 1u);
                const unsigned bar = full_ms + 8 * slot;
                mbar_expect_tx(bar, NH * TA.hbox_tx);
                const unsigned dst = smem_u32(ms_ring + (size_t)slot * TA.ms_slot_bytes);
                tma_load_4d(dst, hmap0, x0 - HX, y0 - 1, zz, 0, bar);
                if constexpr (NH == 2) tma_load_4d(dst + TA.hbox_bytes, hmap1, x0 - HX, y0 - 1, zz, 0, bar);
                ++jm;
            };
            for (long long q = q0; q < q1; ++q) {
                const int x0 = (int)(t % TA.ntx) * TX, y0 = (int)(t / TA.ntx) * kTmaTY;
                if (q == q0 || z == 0) { issue_ms(x0, y0, z - 1); issue_ms(x0, y0, z); }
                issue_ms(x0, y0, z + 1);
                for (int ch = 0; ch < nch; ++ch) {       // mode profiles, 8 per slot (out-of-range modes zero-filled)
                    const unsigned slot = ju % (unsigned)Du, par = (ju / (unsigned)Du) & 1u;
                    mbar_wait(empty_u + 8 * slot, par ^ 1u);
                    const unsigned bar = full_u + 8 * slot;
                    mbar_expect_tx(bar, TA.u_slot_bytes);
                    tma_load_4d(smem_u32(u_ring + (size_t)slot * TA.u_slot_bytes), umap, x0, y0, z, ch * kTmaUChunk, bar);
                    ++ju;
                }
                if constexpr (NAUX > 0) {
                    const unsigned slot = ja % (unsigned)Da, par = (ja / (unsigned)Da) & 1u;
                    mbar_wait(empty_aux + 8 * slot, par ^ 1u);
                    const unsigned bar = full_aux + 8 * slot;
                    mbar_expect_tx(bar, aux_tx);
                    unsigned dst = smem_u32(aux_ring + (size_t)slot * TA.aux_slot_bytes);
#pragma unroll
                    for (int f = 0; f < NAUX; ++f) {
                        tma_load_4d(dst, amap[f], x0, y0, z, 0, bar);
                        dst += C * (kTmaRowBytes * kTmaTY);
                    }
                    ++ja;
                }
                if (++z == nz) { z = 0; ++t; }
            }
        }
    } else {
        // ================================ consumers =================================
        const T h = (T)ctrl->h;
        const T ha21 = h * (T)kA[1][0];
        const T B0x = (T)A.B0[0], B0y = (T)A.B0[1], B0z = (T)A.B0[2];
        const T wx = (T)A.ex_wx, wy = (T)A.ex_wy, wz = (T)A.ex_wz;
        const T anp = (T)A.an_pref, axx = (T)A.axis[0], axy = (T)A.axis[1], axz = (T)A.axis[2];
        const T alpha = (T)A.alpha, llg = (T)A.llg, BE = (T)A.B_exch_inter;

        const T* __restrict__ y0g = (const T*)(ycur ? A.Y[1] : A.Y[0]);
        T* __restrict__ ynew = (T*)(ycur ? A.Y[0] : A.Y[1]);
        T* __restrict__ kout = STAGE == 1 ? (T*)(k1slot ? A.K[6] : A.K[0]) : STAGE == 7 ? (T*)(k1slot ? A.K[0] : A.K[6]) : (T*)A.K[STAGE - 1];
        T* __restrict__ mnext = STAGE == 6 ? ynew : (STAGE == 2 || STAGE == 4) ? (T*)A.MS[0] : (T*)A.MS[1];
        T* __restrict__ e6g = (T*)A.MS[0];
        (void)y0g;

        T ox[NB > 0 ? NB : 1], oy[NB > 0 ? NB : 1];
#pragma unroll
        for (int n = 0; n < NB; ++n) { ox[n] = (T)0; oy[n] = (T)0; }
        T sm[NSUB * 3];
#pragma unroll
        for (int i = 0; i < NSUB * 3; ++i) sm[i] = (T)0;
        T emax2 = (T)0;

        long long t = q0 / nz;
        int z = (int)(q0 - t * nz);
        unsigned jm = 0, ja = 0, ju = 0, jzm = 0, jzc = 0, jzp = 0;
        const int nch = (NB > 0) ? TA.n_uchunks : 0;
        const int crow = (warp + 1) * kTmaHaloRowBytes + kTmaHaloBytes + lane * 8;   // centre, within a comp plane
        constexpr int HPLANE = kTmaHaloRowBytes * (kTmaTY + 2);                            // one comp of a halo box
        constexpr int APLANE = kTmaRowBytes * kTmaTY;                                       // one comp of a plain box
        const int arow = warp * kTmaRowBytes + lane * 8;

        for (long long q = q0; q < q1; ++q) {
            const int x0 = (int)(t % TA.ntx) * TX, y0 = (int)(t / TA.ntx) * kTmaTY;
            const int gx = x0 + lane * VEC, gy = y0 + warp;
            const bool active = gx < nx && gy < ny;
            const bool seg_start = (q == q0 || z == 0);
            const bool seg_end = (q + 1 == q1 || z == nz - 1);
            if (seg_start) {
                jzm = jm++; jzc = jm++;
                mbar_wait(full_ms + 8 * (jzm % (unsigned)Dm), (jzm / (unsigned)Dm) & 1u);
                mbar_wait(full_ms + 8 * (jzc % (unsigned)Dm), (jzc / (unsigned)Dm) & 1u);
            }
            jzp = jm++;
            mbar_wait(full_ms + 8 * (jzp % (unsigned)Dm), (jzp / (unsigned)Dm) & 1u);
            const unsigned char* sm_zm = ms_ring + (size_t)(jzm % (unsigned)Dm) * TA.ms_slot_bytes;
            const unsigned char* sm_zc = ms_ring + (size_t)(jzc % (unsigned)Dm) * TA.ms_slot_bytes;
            const unsigned char* sm_zp = ms_ring + (size_t)(jzp % (unsigned)Dm) * TA.ms_slot_bytes;
            const bool has_l = gx > 0, has_r = gx + VEC < nx;
            const bool has_ym = gy > 0, has_yp = gy < ny - 1, has_zm = z > 0, has_zp = z < nz - 1;

            // stage state from a halo box (STAGE 2: formed on the fly from y0 and k1)
            auto ldm = [&](const unsigned char* slot, int comp, int off) -> P {
                const unsigned char* p = slot + comp * HPLANE + off;
                P a = *reinterpret_cast<const P*>(p);
                if constexpr (STAGE == 2) {
                    const P b = *reinterpret_cast<const P*>(p + TA.hbox_bytes);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) a.v[v] = a.v[v] + ha21 * b.v[v];
                }
                return a;
            };
            auto ldm1 = [&](const unsigned char* slot, int comp, int off) -> T {
                const unsigned char* p = slot + comp * HPLANE + off;
                T a = *reinterpret_cast<const T*>(p);
                if constexpr (STAGE == 2) a = a + ha21 * *reinterpret_cast<const T*>(p + TA.hbox_bytes);
                return a;
            };

            P mc[NSUB][3];
#pragma unroll
            for (int s = 0; s < NSUB; ++s)
#pragma unroll
                for (int c = 0; c < 3; ++c) mc[s][c] = ldm(sm_zc, s * 3 + c, crow);

            // ---- mode profiles (ring u): RF field and overlap partials of THIS stage state ----
            T brf[VEC];
#pragma unroll
            for (int v = 0; v < VEC; ++v) brf[v] = (T)0;
            if constexpr (NB > 0) {
                T mcx[VEC], mcy[VEC];
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    if constexpr (NSUB == 1) { mcx[v] = mc[0][0].v[v]; mcy[v] = mc[0][1].v[v]; }
                    else { mcx[v] = (T)0.5 * (mc[0][0].v[v] + mc[1][0].v[v]); mcy[v] = (T)0.5 * (mc[0][1].v[v] + mc[1][1].v[v]); }
                }
                constexpr int NCH = (NB + kTmaUChunk - 1) / kTmaUChunk;
                constexpr int UCB = NB < kTmaUChunk ? NB : kTmaUChunk;
#pragma unroll
                for (int ch = 0; ch < NCH; ++ch) {
                    if (ch < nch) {
                        const unsigned uslot = ju % (unsigned)Du;
                        mbar_wait(full_u + 8 * uslot, (ju / (unsigned)Du) & 1u);
                        const unsigned char* us = u_ring + (size_t)uslot * TA.u_slot_bytes;
                        ++ju;
#pragma unroll
                        for (int i = 0; i < UCB; ++i) {
                            const int n = ch * kTmaUChunk + i;
                            if (n < N) {
                                const P un = *reinterpret_cast<const P*>(us + i * APLANE + arow);
                                const T cn = s_cn[n];
                                T sx = (T)0, sy = (T)0;
#pragma unroll
                                for (int v = 0; v < VEC; ++v) {
                                    brf[v] += cn * un.v[v];
                                    sx += un.v[v] * mcx[v];
                                    sy += un.v[v] * mcy[v];
                                }
                                if (active) { ox[n] += sx; oy[n] += sy; }
                            }
                        }
                        __syncwarp();
                        if (lane == 0) mbar_arrive(empty_u + 8 * uslot);
                    }
                }
            }
            // ---- halo-free cell streams (ring aux): only the tail below reads them ----
            const unsigned char* axf = nullptr;
            unsigned aslot = 0;
            if constexpr (NAUX > 0) {
                aslot = ja % (unsigned)Da;
                mbar_wait(full_aux + 8 * aslot, (ja / (unsigned)Da) & 1u);
                axf = aux_ring + (size_t)aslot * TA.aux_slot_bytes;
                ++ja;
            }

#pragma unroll
            for (int s = 0; s < NSUB; ++s) {
                T lap[3][VEC];
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    const int comp = s * 3 + c;
                    const P nym = ldm(sm_zc, comp, crow - kTmaHaloRowBytes);
                    const P nyp = ldm(sm_zc, comp, crow + kTmaHaloRowBytes);
                    const P nzm = ldm(sm_zm, comp, crow);
                    const P nzp = ldm(sm_zp, comp, crow);
                    T xl = __shfl_up_sync(0xffffffffu, mc[s][c].v[VEC - 1], 1);
                    T xr = __shfl_down_sync(0xffffffffu, mc[s][c].v[0], 1);
                    if (lane == 0) xl = ldm1(sm_zc, comp, crow - (int)sizeof(T));
                    if (lane == 31) xr = ldm1(sm_zc, comp, crow + 8);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const T m0 = mc[s][c].v[v];
                        T left = (v == 0) ? xl : mc[s][c].v[v > 0 ? v - 1 : 0];
                        T right = (v == VEC - 1) ? xr : mc[s][c].v[v < VEC - 1 ? v + 1 : VEC - 1];
                        if (v == 0 && !has_l) left = m0;
                        if (v == VEC - 1 && !has_r) right = m0;
                        const T ym = has_ym ? nym.v[v] : m0, yp = has_yp ? nyp.v[v] : m0;
                        const T zm = has_zm ? nzm.v[v] : m0, zp = has_zp ? nzp.v[v] : m0;
                        T l = (left - m0) * wx;
                        l += (right - m0) * wx;
                        l += (ym - m0) * wy;
                        l += (yp - m0) * wy;
                        l += (zm - m0) * wz;
                        l += (zp - m0) * wz;
                        lap[c][v] = l;
                    }
                }

                P ks[3];
#pragma unroll
                for (int v = 0; v < VEC; ++v) {
                    const T mx = mc[s][0].v[v], my = mc[s][1].v[v], mz = mc[s][2].v[v];
                    const T mk = mx * axx + my * axy + mz * axz;
                    T Bx = B0x + lap[0][v] + anp * mk * axx + brf[v];
                    T By = B0y + lap[1][v] + anp * mk * axy;
                    T Bz = B0z + lap[2][v] + anp * mk * axz;
                    if constexpr (NSUB == 2) {
                        Bx -= BE * mc[1 - s][0].v[v]; By -= BE * mc[1 - s][1].v[v]; Bz -= BE * mc[1 - s][2].v[v];
                    }
                    const T tx = my * Bz - mz * By, ty = mz * Bx - mx * Bz, tz = mx * By - my * Bx;
                    const T dx = my * tz - mz * ty, dy = mz * tx - mx * tz, dz = mx * ty - my * tx;
                    ks[0].v[v] = llg * (tx + alpha * dx);
                    ks[1].v[v] = llg * (ty + alpha * dy);
                    ks[2].v[v] = llg * (tz + alpha * dz);
                }

                const long long cell = ((long long)z * ny + gy) * nx + gx;
#pragma unroll
                for (int c = 0; c < 3; ++c)
                    if (active) stp<T, VEC>(kout + (long long)(s * 3 + c) * nc + cell, ks[c]);

                if constexpr (STAGE >= 2 && STAGE <= 5) {
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const int comp = s * 3 + c;
                        P acc, m0v;
                        if constexpr (STAGE == 2) {
                            m0v = *reinterpret_cast<const P*>(sm_zc + comp * HPLANE + crow);
                            const P q1 = *reinterpret_cast<const P*>(sm_zc + TA.hbox_bytes + comp * HPLANE + crow);
#pragma unroll
                            for (int v = 0; v < VEC; ++v) acc.v[v] = (T)kA[2][0] * q1.v[v];
                        } else {
                            m0v = *reinterpret_cast<const P*>(axf + comp * APLANE + arow);
                            const P q1 = *reinterpret_cast<const P*>(axf + (C + comp) * APLANE + arow);
#pragma unroll
                            for (int v = 0; v < VEC; ++v) acc.v[v] = (T)kA[STAGE][0] * q1.v[v];
#pragma unroll
                            for (int j = 1; j < STAGE - 1; ++j) {
                                const P qj = *reinterpret_cast<const P*>(axf + ((1 + j) * C + comp) * APLANE + arow);
#pragma unroll
                                for (int v = 0; v < VEC; ++v) acc.v[v] += (T)kA[STAGE][j] * qj.v[v];
                            }
                        }
                        P out;
#pragma unroll
                        for (int v = 0; v < VEC; ++v) {
                            acc.v[v] += (T)kA[STAGE][STAGE - 1] * ks[c].v[v];
                            out.v[v] = m0v.v[v] + h * acc.v[v];
                        }
                        if (active) stp<T, VEC>(mnext + (long long)comp * nc + cell, out);
                    }
                }
                if constexpr (STAGE == 6) {
                    P y5[3], er[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) {
                        const int comp = s * 3 + c;
                        const P m0v = *reinterpret_cast<const P*>(axf + comp * APLANE + arow);
                        const P q1 = *reinterpret_cast<const P*>(axf + (C + comp) * APLANE + arow);
                        const P q3 = *reinterpret_cast<const P*>(axf + (2 * C + comp) * APLANE + arow);
                        const P q4 = *reinterpret_cast<const P*>(axf + (3 * C + comp) * APLANE + arow);
                        const P q5 = *reinterpret_cast<const P*>(axf + (4 * C + comp) * APLANE + arow);
#pragma unroll
                        for (int v = 0; v < VEC; ++v) {
                            T acc = (T)kA[6][0] * q1.v[v];
                            acc += (T)kA[6][2] * q3.v[v];
                            acc += (T)kA[6][3] * q4.v[v];
                            acc += (T)kA[6][4] * q5.v[v];
                            acc += (T)kA[6][5] * ks[c].v[v];
                            y5[c].v[v] = m0v.v[v] + h * acc;
                            T e = (T)kD[0] * q1.v[v];
                            e += (T)kD[2] * q3.v[v];
                            e += (T)kD[3] * q4.v[v];
                            e += (T)kD[4] * q5.v[v];
                            e += (T)kD[5] * ks[c].v[v];
                            er[c].v[v] = h * e;
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
                        if (active) { stp<T, VEC>(mnext + off, y5[c]); stp<T, VEC>(e6g + off, er[c]); }
                    }
                }
                if constexpr (STAGE == 7) {
                    P er[3];
#pragma unroll
                    for (int c = 0; c < 3; ++c) er[c] = *reinterpret_cast<const P*>(axf + (s * 3 + c) * APLANE + arow);
#pragma unroll
                    for (int v = 0; v < VEC; ++v) {
                        const T hd7 = h * (T)kD[6];
                        const T ex = er[0].v[v] + hd7 * ks[0].v[v];
                        const T ey = er[1].v[v] + hd7 * ks[1].v[v];
                        const T ez = er[2].v[v] + hd7 * ks[2].v[v];
                        T e2 = ex * ex + ey * ey + ez * ez;
                        e2 = (e2 < (T)CUDART_INF) ? e2 : (T)CUDART_INF;
                        if (active) {
                            emax2 = fmax(emax2, e2);
                            sm[s * 3 + 0] += mc[s][0].v[v]; sm[s * 3 + 1] += mc[s][1].v[v]; sm[s * 3 + 2] += mc[s][2].v[v];
                        }
                    }
                }
            }

            // ---- release the slots this plane no longer needs ----
            __syncwarp();
            if (lane == 0) {
                if constexpr (NAUX > 0) mbar_arrive(empty_aux + 8 * aslot);
                mbar_arrive(empty_ms + 8 * (jzm % (unsigned)Dm));
                if (seg_end) {
                    mbar_arrive(empty_ms + 8 * (jzc % (unsigned)Dm));
                    mbar_arrive(empty_ms + 8 * (jzp % (unsigned)Dm));
                }
            }
            jzm = jzc; jzc = jzp;
            if (++z == nz) { z = 0; ++t; }
        }

        // ---- pass 1 of the reductions: warp shuffle tree; lane 0 of each consumer warp deposits ----
        constexpr int NS = 2 * NB + (STAGE == 7 ? 3 * NSUB : 0);
        __shared__ double swarp[kTmaTY][NS > 0 ? NS : 1];
        __shared__ double swmax[kTmaTY];
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
                A.partial[(size_t)comp * A.pstride + blockIdx.x] = acc;
            }
        }
        if (STAGE == 7 && tid == 0) {
            double mx = 0.0;
#pragma unroll
            for (int w = 0; w < kTmaTY; ++w) mx = fmax(mx, swmax[w]);
            A.partial_max[blockIdx.x] = mx;
        }
    }

    // ---- last-block-done: second reduction pass, mode ODEs, controller ----
    __shared__ int s_last;
    __threadfence();
    __syncthreads();
    if (tid == 0) {
        const unsigned int old = atomicAdd(&ctrl->arrive, 1u);
        s_last = (old == gridDim.x - 1) ? 1 : 0;
    }
    __syncthreads();
    if (s_last) stage_finish(A, STAGE, NSUB, trace);
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

#define CAVMAG_DEFINE_TMA_LOOKUP(NAME, T, NSUB)                                    \
    const void* NAME(int stage, int nb) {                                          \
        if (nb == 0) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 0) }                        \
        if (nb == 2) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 2) }                        \
        if (nb == 8) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 8) }                        \
        if (nb == 32) { CAVMAG_TMA_STAGE_CASES(T, NSUB, 32) }                      \
        return nullptr;                                                            \
    }

}  // namespace cavmag
