// Dipolar field by FFT convolution (see demag.cuh).
//
// Layout of one evaluation (nz <= 64 and ny <= 512 - 256 in fp64 -, the usual case: films and slabs):
//   gather   stage state, summed over the sublattices -> [3][nz][ny][Px] real, zero-padded in x only
//   cuFFT    batched 1-D R2C along x over the 3 nz ny occupied rows: rows and planes that would only hold zeros are
//            never stored or transformed
//   k_demag_ycol    per (component, z, kx) column and in shared memory: zero-pad the ny rows to Py = 2^qy, FFT along y,
//            frequency index left in bit-reversed order
//   k_demag_zconv   per (ky, kx) column and in shared memory: zero-pad to Pz, FFT along z, product with the tensor's
//            transform, inverse FFT along z, keep z < nz - the full [Pz][Py][Px/2+1] spectrum never exists in memory.
//            The tensor's transform is real and even/odd in every index: one octant of it is stored, as reals.
//   k_demag_ycol    inverse along y, keep the ny rows
//   cuFFT    batched 1-D C2R along x, then the scatter of the first nx cells of a row into the dense field.
// Fallbacks: 2-D cuFFT over all Py rows (ny beyond that, or nx = 1), padded 3-D cuFFT with a separate product kernel (nz > 64,
// where the columns of a block do not fit shared memory).  cuFFT does the x transforms (a library primitive); the tensor,
// the gather, the y and z transforms, the product and the scatter are kernels of this file.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <dlfcn.h>
#include <new>
#include <type_traits>

#include <cufft.h>     // types and enums only: the entry points are resolved with dlsym

#include "../../include/cavmag.h"
#include "demag.cuh"
#include "stage_kernel.cuh"

namespace cavmag {

namespace {

struct FftApi {
    cufftResult (*PlanMany)(cufftHandle*, int, int*, int*, int, int, int*, int, int, cufftType, int) = nullptr;
    cufftResult (*ExecR2C)(cufftHandle, cufftReal*, cufftComplex*) = nullptr;
    cufftResult (*ExecC2R)(cufftHandle, cufftComplex*, cufftReal*) = nullptr;
    cufftResult (*ExecD2Z)(cufftHandle, cufftDoubleReal*, cufftDoubleComplex*) = nullptr;
    cufftResult (*ExecZ2D)(cufftHandle, cufftDoubleComplex*, cufftDoubleReal*) = nullptr;
    cufftResult (*SetStream)(cufftHandle, cudaStream_t) = nullptr;
    cufftResult (*Destroy)(cufftHandle) = nullptr;
    bool ok = false;
};

FftApi& fft_api() {
    static FftApi api;
    static bool tried = false;
    if (tried) return api;
    tried = true;
    const char* names[] = {"libcufft.so.11", "/usr/local/cuda/lib64/libcufft.so.11", "libcufft.so", "/usr/local/cuda/lib64/libcufft.so"};
    void* h = nullptr;
    for (const char* n : names) { h = dlopen(n, RTLD_NOW | RTLD_LOCAL); if (h) break; }
    if (!h) return api;
    api.PlanMany = (decltype(api.PlanMany))dlsym(h, "cufftPlanMany");
    api.ExecR2C = (decltype(api.ExecR2C))dlsym(h, "cufftExecR2C");
    api.ExecC2R = (decltype(api.ExecC2R))dlsym(h, "cufftExecC2R");
    api.ExecD2Z = (decltype(api.ExecD2Z))dlsym(h, "cufftExecD2Z");
    api.ExecZ2D = (decltype(api.ExecZ2D))dlsym(h, "cufftExecZ2D");
    api.SetStream = (decltype(api.SetStream))dlsym(h, "cufftSetStream");
    api.Destroy = (decltype(api.Destroy))dlsym(h, "cufftDestroy");
    api.ok = api.PlanMany && api.ExecR2C && api.ExecC2R && api.ExecD2Z && api.ExecZ2D && api.SetStream && api.Destroy;
    return api;
}

// ---- Newell, Williams & Dunlop (1993): demagnetising tensor between two equal rectangular cells ----
// N_xx(X,Y,Z) = -1/(4 pi V) sum_{i,j,k in {-1,0,1}} w_i w_j w_k f(X + i dx, Y + j dy, Z + k dz),  w = (1,-2,1);  N_xy with g.
__device__ double nw_f(double x, double y, double z) {
    x = fabs(x); y = fabs(y); z = fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = sqrt(x2 + y2 + z2);
    double r = (2.0 * x2 - y2 - z2) * R * (1.0 / 6.0);
    if (y > 0.0 && x2 + z2 > 0.0) r += 0.5 * y * (z2 - x2) * asinh(y / sqrt(x2 + z2));
    if (z > 0.0 && x2 + y2 > 0.0) r += 0.5 * z * (y2 - x2) * asinh(z / sqrt(x2 + y2));
    if (x > 0.0 && y > 0.0 && z > 0.0) r -= x * y * z * atan(y * z / (x * R));
    return r;
}
__device__ double nw_g(double x, double y, double z) {
    z = fabs(z);
    const double x2 = x * x, y2 = y * y, z2 = z * z, R = sqrt(x2 + y2 + z2);
    double r = -x * y * R * (1.0 / 3.0);
    if (x2 + y2 > 0.0) r += x * y * z * asinh(z / sqrt(x2 + y2));
    if (y2 + z2 > 0.0) r += (y * (1.0 / 6.0)) * (3.0 * z2 - y2) * asinh(x / sqrt(y2 + z2));
    if (x2 + z2 > 0.0) r += (x * (1.0 / 6.0)) * (3.0 * z2 - x2) * asinh(y / sqrt(x2 + z2));
    if (z > 0.0) r -= (z * z2 * (1.0 / 6.0)) * atan(x * y / (z * R));
    if (y != 0.0) r -= (0.5 * z * y2) * atan(x * z / (y * R));
    if (x != 0.0) r -= (0.5 * z * x2) * atan(y * z / (x * R));
    return r;
}
template <bool G>
__device__ double nw_sum(double X, double Y, double Z, double dx, double dy, double dz) {
    double acc = 0.0;
    for (int i = -1; i <= 1; ++i)
        for (int j = -1; j <= 1; ++j)
            for (int k = -1; k <= 1; ++k) {
                const double w = (i == 0 ? -2.0 : 1.0) * (j == 0 ? -2.0 : 1.0) * (k == 0 ? -2.0 : 1.0);
                acc += w * (G ? nw_g(X + i * dx, Y + j * dy, Z + k * dz) : nw_f(X + i * dx, Y + j * dy, Z + k * dz));
            }
    return -acc / (4.0 * CUDART_PI * dx * dy * dz);
}

// One component (0..5 = xx, yy, zz, xy, xz, yz) of the tensor on the padded, wrapped grid [Pz][Py][Px] (lengths in units of dx).
__global__ void k_demag_tensor(double* out, int comp, int nx, int ny, int nz, int Px, int Py, int Pz, double sy, double sz) {
    const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long tot = (long long)Px * Py * Pz;
    if (idx >= tot) return;
    const int i = (int)(idx % Px), j = (int)((idx / Px) % Py), k = (int)(idx / ((long long)Px * Py));
    auto off = [](int a, int n, int P, bool& ok) { if (a < n) return a; if (a > P - n) return a - P; ok = false; return 0; };
    bool ok = true;
    const double X = (double)off(i, nx, Px, ok), Y = (double)off(j, ny, Py, ok) * sy, Z = (double)off(k, nz, Pz, ok) * sz;
    double v = 0.0;
    if (ok) {
        switch (comp) {
            case 0: v = nw_sum<false>(X, Y, Z, 1.0, sy, sz); break;
            case 1: v = nw_sum<false>(Y, X, Z, sy, 1.0, sz); break;
            case 2: v = nw_sum<false>(Z, Y, X, sz, sy, 1.0); break;
            case 3: v = nw_sum<true>(X, Y, Z, 1.0, sy, sz); break;
            case 4: v = nw_sum<true>(X, Z, Y, 1.0, sz, sy); break;
            default: v = nw_sum<true>(Y, Z, X, sy, sz, 1.0); break;
        }
    }
    out[idx] = v;
}

// transform of one tensor component -> the plan's table, scaled by -mu0 Ms / (Px Py Pz)
template <typename C>
__global__ void k_store_khat(const cufftDoubleComplex* src, C* dst, long long n, double scale) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    dst[i].x = (decltype(dst[i].x))(src[i].x * scale);
    dst[i].y = (decltype(dst[i].y))(src[i].y * scale);
}

// real part of one tensor component's transform on the octant kz <= Pz/2, ky <= Py/2, kx <= Px/2, scaled.  (The tensor
// is real and, per index, even or odd with a zero at the origin and at the unused offset n: its transform is real, and
// +-1 times itself under k -> P - k.  The imaginary parts left by rounding are dropped.)
template <typename T>
__global__ void k_store_khat_real(const cufftDoubleComplex* src, T* dst, int NZH, int NYH, int NXH, int Py, double scale) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= (long long)NZH * NYH * NXH) return;
    const int kx = (int)(i % NXH), ky = (int)((i / NXH) % NYH), kz = (int)(i / ((long long)NXH * NYH));
    dst[i] = (T)(src[((long long)kz * Py + ky) * NXH + kx].x * scale);
}

// columns (ky, kx) per block of the z convolution: a warp per worker row in fp32 (positions and twiddles are warp-uniform)
template <typename T> struct ZTile { static constexpr int value = sizeof(T) == 4 ? 32 : 16; };

// ---- complex arithmetic and the radix-2 levels of a pass, on values held in registers ----
template <typename C> __device__ __forceinline__ C c_add(const C& a, const C& b) { C r; r.x = a.x + b.x; r.y = a.y + b.y; return r; }
template <typename C> __device__ __forceinline__ C c_sub(const C& a, const C& b) { C r; r.x = a.x - b.x; r.y = a.y - b.y; return r; }
// fp32: a complex number is one 64-bit register pair, and sm_100 adds / multiplies both halves in one instruction
// (FADD2 / FFMA2): half the issue slots of the butterflies' additions
template <> __device__ __forceinline__ float2 c_add<float2>(const float2& a, const float2& b) { return __fadd2_rn(a, b); }
template <> __device__ __forceinline__ float2 c_sub<float2>(const float2& a, const float2& b) { return __ffma2_rn(b, make_float2(-1.0f, -1.0f), a); }
template <typename C> __device__ __forceinline__ C c_mul(const C& a, const C& b) { C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r; }
template <typename C> __device__ __forceinline__ C c_mulc(const C& a, const C& b) { C r; r.x = a.x * b.x + a.y * b.y; r.y = a.y * b.x - a.x * b.y; return r; }   // a conj(b)

// A transform of length P = 2^q runs in passes of up to three radix-2 levels on 2^L values held in registers, with a
// shared-memory exchange between passes.  Forward: decimation in frequency (natural order in, bit-reversed out), spans
// P/2, P/4, .. 1; inverse: decimation in time with conjugate twiddles (bit-reversed in, natural out), the same passes
// mirrored.  Levels per pass, in forward order: threes, a four is two twos (q = 9: 3 3 3, q = 6: 3 3, q = 7: 3 2 2).
__host__ __device__ constexpr int fft_pass_count(int q) { int n = 0; while (q > 0) { q -= (q >= 3 && q != 4) ? 3 : (q >= 2 ? 2 : 1); ++n; } return n; }
__host__ __device__ constexpr int fft_pass_levels(int q, int i) {
    int L = 0;
    for (int k = 0; k <= i; ++k) { L = (q >= 3 && q != 4) ? 3 : (q >= 2 ? 2 : 1); q -= L; }
    return L;
}
__host__ __device__ constexpr int fft_pass_done(int q, int i) { int d = 0; for (int k = 0; k < i; ++k) d += fft_pass_levels(q, k); return d; }   // levels before pass i
__host__ __device__ constexpr int fft_rows(int q) { return (1 << q) / 8 < 1 ? 1 : ((1 << q) / 8 > 32 ? 32 : (1 << q) / 8); }   // blockDim.y: groups of a pass in flight

// The L levels of one pass on v[c][e], e < 2^L: the values of a group sit HQ positions apart (positions p0 + e HQ,
// p0 = (w / HQ) (HQ 2^L) + r, r = w % HQ for group w), level l pairs values d apart (forward d = 2^(L-1-l), inverse 2^l)
// inside a span of HQ d positions; tw[t] = exp(-2 pi i t / P).
template <typename C, int P, int NC, int L, int HQ, bool INV>
__device__ __forceinline__ void fft_levels(C (&v)[NC][1 << L], const C* __restrict__ tw, const int r) {
    constexpr int n = 1 << L;
#pragma unroll
    for (int l = 0; l < L; ++l) {
        const int d = INV ? (1 << l) : (1 << (L - 1 - l));
#pragma unroll
        for (int e = 0; e < n; ++e) {
            if (e & d) continue;
            const C t = tw[(r + (e % d) * HQ) * (P / (2 * HQ * d))];
#pragma unroll
            for (int c = 0; c < NC; ++c) {
                if constexpr (!INV) {
                    const C lo = v[c][e], hi = v[c][e + d];
                    v[c][e] = c_add(lo, hi);
                    v[c][e + d] = c_mul(c_sub(lo, hi), t);
                } else {
                    const C x = c_mulc(v[c][e + d], t), lo = v[c][e];
                    v[c][e] = c_add(lo, x);
                    v[c][e + d] = c_sub(lo, x);
                }
            }
        }
    }
}

// One block: TK consecutive columns (ky, kx) of the half-spectrum, the three field components, the whole z column.
//   F [3][nz][Py][NXH] complex (in place), K [6][Pz/2+1][Py/2+1][NXH] real, Pz = 2^q >= 2 nz - 1 (q = 0: no z transform)
// The first forward pass reads global memory (zero beyond nz); the last forward pass leaves the bit-reversed spectrum of
// its 2^L positions in registers, where it is multiplied by the tensor's transform (pointwise, so at the bit-reversed
// positions) and taken through the first inverse pass - the same positions - at once; the last inverse pass writes the
// planes below nz to global memory.  q = 6: three passes with two shared-memory exchanges.  The inverse is unnormalised
// (1/(Px Py Pz) is folded into K).
__host__ __device__ constexpr int zconv_rows(int q) { return fft_rows(q); }   // blockDim.y

template <typename T, typename C, int q>
__global__ void __launch_bounds__(zconv_rows(q) * ZTile<T>::value)
k_demag_zconv(C* __restrict__ F, const T* __restrict__ K, int nz, int Py, int NXH, int qy_rev) {
    constexpr int Pz = 1 << q;
    constexpr int NJ = zconv_rows(q);
    constexpr int kZTile = ZTile<T>::value;
    constexpr int NP = fft_pass_count(q);
    extern __shared__ __align__(16) unsigned char zsm[];
    C* const sm = reinterpret_cast<C*>(zsm);                    // [3][Pz][kZTile]
    C* const tw = sm + 3 * Pz * kZTile;                         // exp(-2 pi i j / Pz), j < Pz/2
    T* const ks = reinterpret_cast<T*>(tw + (Pz / 2 > 0 ? Pz / 2 : 1));       // the tensor's transform for this block: [6][Pz/2+1][kZTile]
    const int k = threadIdx.x, j = threadIdx.y;
    const long long zs = (long long)Py * NXH;                   // z stride = columns per plane
    const long long col = (long long)blockIdx.x * kZTile + k;
    const bool live = col < zs;
    const int ky_row = live ? (int)(col / NXH) : 0, kx = live ? (int)(col % NXH) : 0;
    // (rows written by k_demag_ycol hold the y frequencies in bit-reversed order: qy_rev = log2 Py there, 0 otherwise)
    const int ky = qy_rev > 0 ? (int)(__brev((unsigned)ky_row) >> (32 - qy_rev)) : ky_row;
    C* const Fc = F + col;                                      // this thread's column: Fc[(c nz + z) zs]
    for (int t = j * kZTile + k; t < Pz / 2; t += NJ * kZTile) {
        double sn, cs;
        sincospi(-2.0 * (double)t / (double)Pz, &sn, &cs);
        tw[t].x = (T)cs; tw[t].y = (T)sn;
    }
    const int kys = ky <= Py / 2 ? ky : Py - ky;
    const T sy = ky <= Py / 2 ? (T)1 : (T)-1;
    constexpr int NZH = Pz / 2 + 1;
    const int NYH = Py / 2 + 1;
    const long long cst = (long long)NZH * NYH * NXH;
    // the block's slice of the tensor's transform goes to shared memory asynchronously: it is needed after the forward passes
    if (live) {
        const T* const Kc = K + (long long)kys * NXH + kx;
        for (int t = j; t < 6 * NZH; t += NJ) {
            const int comp = t / NZH, kzs = t % NZH;
            const unsigned dst = (unsigned)__cvta_generic_to_shared(ks + t * kZTile + k);
            const T* src = Kc + comp * cst + (long long)kzs * NYH * NXH;
            if constexpr (sizeof(T) == 4) asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
            else asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
        }
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
    // G = Khat F at position pos of the (bit-reversed) spectrum, for the three components
    auto product = [&](int pos, C& fx, C& fy, C& fz) {
        const int kz = q > 0 ? (int)(__brev((unsigned)pos) >> ((32 - q) & 31)) : 0;
        const int kzs = kz <= Pz / 2 ? kz : Pz - kz;
        const T sz = kz <= Pz / 2 ? (T)1 : (T)-1;
        const T* const kk = ks + kzs * kZTile + k;
        constexpr int cs6 = NZH * kZTile;
        const T kxx = kk[0], kyy = kk[cs6], kzz = kk[2 * cs6];
        const T kxy = sy * kk[3 * cs6], kxz = sz * kk[4 * cs6], kyz = sy * sz * kk[5 * cs6];
        C gx, gy, gz;
        gx.x = kxx * fx.x + kxy * fy.x + kxz * fz.x; gx.y = kxx * fx.y + kxy * fy.y + kxz * fz.y;
        gy.x = kxy * fx.x + kyy * fy.x + kyz * fz.x; gy.y = kxy * fx.y + kyy * fy.y + kyz * fz.y;
        gz.x = kxz * fx.x + kyz * fy.x + kzz * fz.x; gz.y = kxz * fx.y + kyz * fy.y + kzz * fz.y;
        fx = gx; fy = gy; fz = gz;
    };
    C zero; zero.x = (T)0; zero.y = (T)0;
    if constexpr (q == 0) {                                     // a film: one plane, no z transform
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        if (live && j == 0) {
            C fx = Fc[0], fy = Fc[zs], fz = Fc[2 * zs];          // (nz = 1)
            product(0, fx, fy, fz);
            Fc[0] = fx; Fc[zs] = fy; Fc[2 * zs] = fz;
        }
    } else {
    if constexpr (NP == 1) asm volatile("cp.async.wait_group 0;" ::: "memory");       // one pass: the product is in it
    __syncthreads();                                            // twiddles
    const long long cz = (long long)nz * zs;                    // component stride
    // Step i of 2 NP - 1: forward passes 0 .. NP-2, the middle step (forward pass NP-1, product, inverse pass 0), inverse
    // passes 1 .. NP-1 (inverse pass k mirrors forward pass NP-1-k: the same groups and positions)
    auto step = [&](auto I) {
        constexpr int i = decltype(I)::value;
        constexpr bool mid = i == NP - 1, inv = i > NP - 1;
        constexpr int fi = inv ? 2 * (NP - 1) - i : i;           // the forward pass whose groups this step works on
        constexpr int L = fft_pass_levels(q, fi), n = 1 << L;
        constexpr int HQ = ((Pz / 2) >> fft_pass_done(q, fi)) >> (L - 1);
        constexpr bool first = i == 0, last = i == 2 * NP - 2;
#pragma unroll
        for (int w0 = 0; w0 < Pz / n; w0 += NJ) {
            const int w = w0 + j;
            if (Pz / n < NJ && w >= Pz / n) break;
            const int r = w % HQ, p0 = (w / HQ) * (HQ * n) + r;
            C v[3][n];
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int e = 0; e < n; ++e) {
                    const int pos = p0 + e * HQ;
                    if constexpr (first) v[c][e] = (live && pos < nz) ? Fc[c * cz + pos * zs] : zero;      // zero padding beyond nz
                    else v[c][e] = sm[(c * Pz + pos) * kZTile + k];
                }
            if constexpr (!inv) fft_levels<C, Pz, 3, L, HQ, false>(v, tw, r);
            if constexpr (mid) {
                if (live) {
#pragma unroll
                    for (int e = 0; e < n; ++e) product(p0 + e * HQ, v[0][e], v[1][e], v[2][e]);
                }
            }
            if constexpr (mid || inv) fft_levels<C, Pz, 3, L, HQ, true>(v, tw, r);
#pragma unroll
            for (int c = 0; c < 3; ++c)
#pragma unroll
                for (int e = 0; e < n; ++e) {
                    const int pos = p0 + e * HQ;
                    if constexpr (last) { if (live && pos < nz) Fc[c * cz + pos * zs] = v[c][e]; }         // keep the planes below nz
                    else sm[(c * Pz + pos) * kZTile + k] = v[c][e];
                }
        }
        if constexpr (i == NP - 2) asm volatile("cp.async.wait_group 0;" ::: "memory");    // the next step multiplies
        if constexpr (!last) __syncthreads();
    };
    using std::integral_constant;
    step(integral_constant<int, 0>{});
    if constexpr (2 * NP - 1 > 1) step(integral_constant<int, 1>{});
    if constexpr (2 * NP - 1 > 2) step(integral_constant<int, 2>{});
    if constexpr (2 * NP - 1 > 3) step(integral_constant<int, 3>{});
    if constexpr (2 * NP - 1 > 4) step(integral_constant<int, 4>{});
    }
}

template <typename T, typename C>
const void* zconv_fn(int q) {
    switch (q) {
        case 0: return (const void*)k_demag_zconv<T, C, 0>;
        case 1: return (const void*)k_demag_zconv<T, C, 1>;
        case 2: return (const void*)k_demag_zconv<T, C, 2>;
        case 3: return (const void*)k_demag_zconv<T, C, 3>;
        case 4: return (const void*)k_demag_zconv<T, C, 4>;
        case 5: return (const void*)k_demag_zconv<T, C, 5>;
        case 6: return (const void*)k_demag_zconv<T, C, 6>;
        default: return (const void*)k_demag_zconv<T, C, 7>;
    }
}

// ---- y transform of the occupied rows only ("yfused" layout, Py = 2^q) ----
// After the x transform only ny of the Py rows of a plane are non-zero, and only ny rows of the result are wanted:
//   forward (INV = false): in [planes][ny][NXH]  -> zero-pad to Py, transform along y -> out [planes][Py][NXH], frequency
//                          index in bit-reversed order (the z convolution works column by column and only needs to know
//                          which frequency a row holds);
//   inverse (INV = true):  in [planes][Py][NXH] (bit-reversed) -> transform back -> rows y < ny -> out [planes][ny][NXH].
// Up to three radix-2 levels per pass on eight values in registers (Py = 512: three passes, two shared-memory exchanges);
// the first pass reads global memory, the last one writes it; one component per column.
constexpr int kYTile = 16;           // columns (plane, kx) per block
__host__ __device__ constexpr int ycol_rows(int q) { return fft_rows(q); }   // blockDim.y

template <typename T, typename C, int q, bool INV>
__global__ void __launch_bounds__(ycol_rows(q) * kYTile)
k_demag_ycol(const C* __restrict__ in, C* __restrict__ out, int n_valid, int NXH, long long ncols) {
    constexpr int P = 1 << q, NJ = ycol_rows(q), TK = kYTile;
    constexpr int NP = fft_pass_count(q);
    extern __shared__ __align__(16) unsigned char ysm[];
    C* const sm = reinterpret_cast<C*>(ysm);                    // [P][TK]
    C* const tw = sm + P * TK;                                  // exp(-2 pi i j / P), j < P/2
    const int k = threadIdx.x, j = threadIdx.y;
    const long long col = (long long)blockIdx.x * TK + k;
    const bool live = col < ncols;
    const long long plane = live ? col / NXH : 0;
    const int kx = live ? (int)(col % NXH) : 0;
    const C* const ci = in + plane * (long long)(INV ? P : n_valid) * NXH + kx;      // element stride NXH
    C* const co = out + plane * (long long)(INV ? n_valid : P) * NXH + kx;
    for (int t = j * TK + k; t < P / 2; t += NJ * TK) {
        double sn, cs;
        sincospi(-2.0 * (double)t / (double)P, &sn, &cs);
        tw[t].x = (T)cs; tw[t].y = (T)sn;
    }
    __syncthreads();
    C zero; zero.x = (T)0; zero.y = (T)0;
    auto pass = [&](auto I) {
        constexpr int i = decltype(I)::value;                    // pass index in execution order
        constexpr int fi = INV ? NP - 1 - i : i;                 // the forward pass it mirrors
        constexpr int L = fft_pass_levels(q, fi), n = 1 << L;
        constexpr int HQ = ((P / 2) >> fft_pass_done(q, fi)) >> (L - 1);
        constexpr bool first = i == 0, last = i == NP - 1;
#pragma unroll
        for (int w0 = 0; w0 < P / n; w0 += NJ) {
            const int w = w0 + j;
            if (P / n < NJ && w >= P / n) break;
            const int r = w % HQ, p0 = (w / HQ) * (HQ * n) + r;
            C v[1][n];
#pragma unroll
            for (int e = 0; e < n; ++e) {
                const int pos = p0 + e * HQ;
                if constexpr (first) v[0][e] = (live && (INV || pos < n_valid)) ? ci[(long long)pos * NXH] : zero;    // forward: zero padding beyond n_valid
                else v[0][e] = sm[pos * TK + k];
            }
            fft_levels<C, P, 1, L, HQ, INV>(v, tw, r);
#pragma unroll
            for (int e = 0; e < n; ++e) {
                const int pos = p0 + e * HQ;
                if constexpr (last) { if (live && (!INV || pos < n_valid)) co[(long long)pos * NXH] = v[0][e]; }      // inverse: keep the rows below n_valid
                else sm[pos * TK + k] = v[0][e];
            }
        }
        if constexpr (!last) __syncthreads();
    };
    using std::integral_constant;
    pass(integral_constant<int, 0>{});
    if constexpr (NP > 1) pass(integral_constant<int, 1>{});
    if constexpr (NP > 2) pass(integral_constant<int, 2>{});
    if constexpr (NP > 3) pass(integral_constant<int, 3>{});
}

constexpr int kYColMaxQ = 10;        // fp32: Py <= 1024 ([Py][16] complex columns = 128 KB of shared memory); fp64: Py <= 512

template <typename T, typename C, bool INV>
const void* ycol_fn(int q) {
    switch (q) {
        case 1: return (const void*)k_demag_ycol<T, C, 1, INV>;
        case 2: return (const void*)k_demag_ycol<T, C, 2, INV>;
        case 3: return (const void*)k_demag_ycol<T, C, 3, INV>;
        case 4: return (const void*)k_demag_ycol<T, C, 4, INV>;
        case 5: return (const void*)k_demag_ycol<T, C, 5, INV>;
        case 6: return (const void*)k_demag_ycol<T, C, 6, INV>;
        case 7: return (const void*)k_demag_ycol<T, C, 7, INV>;
        case 8: return (const void*)k_demag_ycol<T, C, 8, INV>;
        case 9: return (const void*)k_demag_ycol<T, C, 9, INV>;
        case 10: return (const void*)k_demag_ycol<T, C, 10, INV>;
        default: return nullptr;
    }
}

// The state stage `stage` is evaluated at, summed over the sublattices, into the zero-padded array [3][Pz][Py][Px]
// (the pad region is zeroed once and never written).  Buffer indices and h as the stage kernel reads them.
constexpr int kGatherRows = 4;       // rows per thread of the gather / scatter kernels (independent loads in flight)

template <typename T, int NSUB>
__global__ void k_demag_gather(const StageArgs A, int stage, T* __restrict__ pad, int Px, int Py, int Pz) {
    const Ctrl* c = A.ctrl;
    if (stage == 1 ? c->k1_valid : c->done) return;
    const int x = blockIdx.x * blockDim.x + threadIdx.x, yb = blockIdx.y * kGatherRows, z = blockIdx.z;   // grid: (ceil(nx / block), ceil(ny / 4), nz)
    if (x >= A.nx) return;
    const long long nc = A.nc;
    const int ycur = c->ycur, k1slot = c->k1slot;
    const T* __restrict__ y0 = (const T*)(ycur ? A.Y[1] : A.Y[0]);
    const T* __restrict__ ynew = (const T*)(ycur ? A.Y[0] : A.Y[1]);
    const T* __restrict__ k1 = (const T*)(k1slot ? A.K[6] : A.K[0]);
    const T* __restrict__ ms = stage == 1 ? y0 : stage == 7 ? ynew : (stage == 3 || stage == 5) ? (const T*)A.MS[0] : (const T*)A.MS[1];
    const T ha21 = (T)c->h * (T)kA[1][0];
    const long long pvol = (long long)Px * Py * Pz;
    T v[kGatherRows][3];
#pragma unroll
    for (int r = 0; r < kGatherRows; ++r) {
        const int y = yb + r;
        const long long i = ((long long)z * A.ny + (y < A.ny ? y : A.ny - 1)) * A.nx + x;
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) {
            T acc = (T)0;
#pragma unroll
            for (int s = 0; s < NSUB; ++s) {             // (compile-time count: every load of the thread is independent)
                const long long off = (long long)(s * 3 + comp) * nc + i;
                acc += stage == 2 ? y0[off] + ha21 * k1[off] : ms[off];
            }
            v[r][comp] = acc;
        }
    }
#pragma unroll
    for (int r = 0; r < kGatherRows; ++r) {
        const int y = yb + r;
        if (y >= A.ny) break;
        const long long o = ((long long)z * Py + y) * Px + x;
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) pad[comp * pvol + o] = v[r][comp];
    }
}

// G_i = sum_j Khat_ij F_j at every frequency point, in place (six symmetric components: xx, yy, zz, xy, xz, yz)
template <typename C>
__global__ void k_demag_product(C* F, const C* K, long long nf) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nf) return;
    const C fx = F[i], fy = F[nf + i], fz = F[2 * nf + i];
    const C kxx = K[i], kyy = K[nf + i], kzz = K[2 * nf + i], kxy = K[3 * nf + i], kxz = K[4 * nf + i], kyz = K[5 * nf + i];
    auto mul = [](const C& a, const C& b) { C r; r.x = a.x * b.x - a.y * b.y; r.y = a.x * b.y + a.y * b.x; return r; };
    auto add3 = [](const C& a, const C& b, const C& c) { C r; r.x = a.x + b.x + c.x; r.y = a.y + b.y + c.y; return r; };
    F[i] = add3(mul(kxx, fx), mul(kxy, fy), mul(kxz, fz));
    F[nf + i] = add3(mul(kxy, fx), mul(kyy, fy), mul(kyz, fz));
    F[2 * nf + i] = add3(mul(kxz, fx), mul(kyz, fy), mul(kzz, fz));
}

template <typename T>
__global__ void k_demag_scatter(const T* __restrict__ conv, T* __restrict__ bdem, int nx, int ny, long long nc, int Px, int Py, int Pz) {
    const int x = blockIdx.x * blockDim.x + threadIdx.x, yb = blockIdx.y * kGatherRows, z = blockIdx.z;   // grid: (ceil(nx / block), ceil(ny / 4), nz)
    if (x >= nx) return;
    const long long pvol = (long long)Px * Py * Pz;
    T v[kGatherRows][3];
#pragma unroll
    for (int r = 0; r < kGatherRows; ++r) {
        const int y = yb + r < ny ? yb + r : ny - 1;
        const long long o = ((long long)z * Py + y) * Px + x;
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) v[r][comp] = conv[comp * pvol + o];
    }
#pragma unroll
    for (int r = 0; r < kGatherRows; ++r) {
        const int y = yb + r;
        if (y >= ny) break;
        const long long i = ((long long)z * ny + y) * nx + x;
#pragma unroll
        for (int comp = 0; comp < 3; ++comp) bdem[comp * nc + i] = v[r][comp];
    }
}

}  // namespace

struct DemagPlan {
    int nx = 0, ny = 0, nz = 0, Px = 0, Py = 0, Pz = 0, n_sub = 1;
    int q = 0;                           // zfused: Pz = 2^q
    bool f32 = true;
    bool zfused = true;                  // z transform + product + inverse z transform in one kernel (nz <= kZFusedMax)
    int zplanes = 0;                     // planes of the work arrays: nz (zfused) or Pz
    long long pvol = 0, nf = 0;          // real points, complex points per component of the work arrays
    void* pad = nullptr;                 // [3][zplanes][Py][Px] real: gathered state (pad region stays zero)
    void* freq = nullptr;                // [3][zplanes][Py][Px/2+1] complex
    void* conv = nullptr;                // [3][zplanes][Py][Px] real: unnormalised convolution (scale folded into khat)
    void* khat = nullptr;                // zfused: [6][Pz/2+1][Py/2+1][Px/2+1] real; else [6][nf] complex
    size_t zsmem = 0;
    const void* zfn = nullptr;           // k_demag_zconv<T, C, q>
    // yfused (zfused, nx > 1, Py = 2^qy <= 1024): cuFFT transforms the ny occupied rows along x only, k_demag_ycol does y
    bool yfused = false;
    int qy = 0;
    void* xf = nullptr;                  // [3][nz][ny][Px/2+1] complex: x-transformed occupied rows (qy > 0)
    size_t ysmem = 0;
    const void* yfwd = nullptr;
    const void* yinv = nullptr;
    int prows = 0;                       // rows per plane of pad / conv: ny (yfused) or Py
    cufftHandle fwd = 0, inv = 0;
    bool have_fwd = false, have_inv = false;
};

constexpr int kZFusedMax = 64;           // largest nz whose z columns (Pz <= 128, three components) and tensor slice fit shared memory

void demag_destroy(DemagPlan* p) {
    if (!p) return;
    FftApi& f = fft_api();
    if (p->have_fwd) f.Destroy(p->fwd);
    if (p->have_inv) f.Destroy(p->inv);
    cudaFree(p->pad); cudaFree(p->freq); cudaFree(p->conv); cudaFree(p->khat); cudaFree(p->xf);
    cudaGetLastError();
    delete p;
}

int demag_create(DemagPlan** out, int nx, int ny, int nz, double dx, double dy, double dz, double Ms, int n_sub, bool f32,
                 cudaStream_t stream, char* err, int err_len) {
    *out = nullptr;
    FftApi& f = fft_api();
    if (!f.ok) { snprintf(err, err_len, "cuFFT (libcufft.so.11) could not be loaded"); return CAV_E_UNSUPPORTED; }
    DemagPlan* p = new (std::nothrow) DemagPlan();
    if (!p) return CAV_E_NOMEM;
    auto fail = [&](int code, const char* what) { snprintf(err, err_len, "demag: %s", what); demag_destroy(p); cudaGetLastError(); return code; };
    p->nx = nx; p->ny = ny; p->nz = nz; p->n_sub = n_sub; p->f32 = f32;
    p->zfused = nz <= kZFusedMax;
    p->Px = nx > 1 ? 2 * nx : 1; p->Py = ny > 1 ? 2 * ny : 1;
    if (p->zfused) { p->Pz = 1; p->q = 0; while (p->Pz < 2 * nz - 1) { p->Pz *= 2; p->q++; } }
    else p->Pz = 2 * nz;
    if (p->zfused && nx > 1) {           // y by k_demag_ycol: Py a power of two >= 2 ny - 1
        int Py2 = 1, qy = 0;
        while (Py2 < 2 * ny - 1) { Py2 *= 2; qy++; }
        if (qy <= (f32 ? kYColMaxQ : kYColMaxQ - 1)) { p->yfused = true; p->Py = Py2; p->qy = qy; }
    }
    p->zplanes = p->zfused ? nz : p->Pz;
    p->prows = p->yfused ? ny : p->Py;
    const int NXH = p->Px / 2 + 1, NYH = p->Py / 2 + 1, NZH = p->Pz / 2 + 1;
    p->pvol = (long long)p->Px * p->prows * p->zplanes;
    p->nf = (long long)p->zplanes * p->Py * NXH;
    const size_t rs = f32 ? 4 : 8, cs = 2 * rs;
    const size_t kbytes = p->zfused ? (size_t)6 * NZH * NYH * NXH * rs : (size_t)6 * p->nf * cs;
    if (cudaMalloc(&p->pad, 3 * p->pvol * rs) != cudaSuccess || cudaMalloc(&p->conv, 3 * p->pvol * rs) != cudaSuccess ||
        cudaMalloc(&p->freq, 3 * p->nf * cs) != cudaSuccess || cudaMalloc(&p->khat, kbytes) != cudaSuccess)
        return fail(CAV_E_NOMEM, "device allocation");
    if (p->yfused && p->qy > 0 && cudaMalloc(&p->xf, (size_t)3 * nz * ny * NXH * cs) != cudaSuccess) return fail(CAV_E_NOMEM, "device allocation");
    if (cudaMemsetAsync(p->pad, 0, 3 * p->pvol * rs, stream) != cudaSuccess) return fail(CAV_E_CUDA, "memset");
    int n3[3] = {p->Pz, p->Py, p->Px};
    int n2[2] = {p->Py, p->Px};
    int n1[1] = {p->Px};
    const int rank = p->yfused ? 1 : (p->zfused ? 2 : 3), batch = p->yfused ? 3 * nz * ny : (p->zfused ? 3 * nz : 3);
    int* const nn = p->yfused ? n1 : (p->zfused ? n2 : n3);
    if (p->yfused && p->qy > 0) {
        p->ysmem = ((size_t)p->Py * kYTile + (size_t)p->Py / 2) * cs;
        p->yfwd = f32 ? ycol_fn<float, cufftComplex, false>(p->qy) : ycol_fn<double, cufftDoubleComplex, false>(p->qy);
        p->yinv = f32 ? ycol_fn<float, cufftComplex, true>(p->qy) : ycol_fn<double, cufftDoubleComplex, true>(p->qy);
        if (cudaFuncSetAttribute(p->yfwd, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->ysmem) != cudaSuccess ||
            cudaFuncSetAttribute(p->yinv, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->ysmem) != cudaSuccess)
            return fail(CAV_E_CUDA, "shared memory for the y transform");
    }
    if (f.PlanMany(&p->fwd, rank, nn, nullptr, 1, 0, nullptr, 1, 0, f32 ? CUFFT_R2C : CUFFT_D2Z, batch) != CUFFT_SUCCESS) return fail(CAV_E_CUDA, "cufftPlanMany (forward)");
    p->have_fwd = true;
    if (f.PlanMany(&p->inv, rank, nn, nullptr, 1, 0, nullptr, 1, 0, f32 ? CUFFT_C2R : CUFFT_Z2D, batch) != CUFFT_SUCCESS) return fail(CAV_E_CUDA, "cufftPlanMany (inverse)");
    p->have_inv = true;
    if (p->zfused) {
        const size_t tk = f32 ? ZTile<float>::value : ZTile<double>::value;
        p->zsmem = ((size_t)3 * p->Pz * tk + (size_t)(p->Pz / 2 > 0 ? p->Pz / 2 : 1)) * cs + (size_t)6 * NZH * tk * rs;
        p->zfn = f32 ? zconv_fn<float, cufftComplex>(p->q) : zconv_fn<double, cufftDoubleComplex>(p->q);
        const cudaError_t e = cudaFuncSetAttribute(p->zfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)p->zsmem);
        if (e != cudaSuccess) return fail(CAV_E_CUDA, "shared memory for the z convolution");
    }
    // tensor table: fp64 on the device, one component at a time through a temporary 3-D D2Z plan on [Pz][Py][Px]
    const long long tvol = (long long)p->Px * p->Py * p->Pz, tnf = (long long)p->Pz * p->Py * NXH;
    double* tn = nullptr;
    cufftDoubleComplex* tk = nullptr;
    cufftHandle tp = 0;
    if (cudaMalloc(&tn, tvol * sizeof(double)) != cudaSuccess || cudaMalloc(&tk, tnf * sizeof(cufftDoubleComplex)) != cudaSuccess) {
        cudaFree(tn); cudaFree(tk);
        return fail(CAV_E_NOMEM, "tensor scratch");
    }
    if (f.PlanMany(&tp, 3, n3, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, 1) != CUFFT_SUCCESS) { cudaFree(tn); cudaFree(tk); return fail(CAV_E_CUDA, "cufftPlanMany (tensor)"); }
    f.SetStream(tp, stream);
    const double scale = -4e-7 * CUDART_PI * Ms / (double)tvol;
    const int tb = 256;
    bool ok = true;
    for (int comp = 0; comp < 6 && ok; ++comp) {
        k_demag_tensor<<<(unsigned)((tvol + tb - 1) / tb), tb, 0, stream>>>(tn, comp, nx, ny, nz, p->Px, p->Py, p->Pz, dy / dx, dz / dx);
        ok = ok && f.ExecD2Z(tp, tn, tk) == CUFFT_SUCCESS;
        if (p->zfused) {
            const long long oct = (long long)NZH * NYH * NXH;
            const unsigned g = (unsigned)((oct + tb - 1) / tb);
            if (f32) k_store_khat_real<float><<<g, tb, 0, stream>>>(tk, (float*)p->khat + comp * oct, NZH, NYH, NXH, p->Py, scale);
            else k_store_khat_real<double><<<g, tb, 0, stream>>>(tk, (double*)p->khat + comp * oct, NZH, NYH, NXH, p->Py, scale);
        } else if (f32) k_store_khat<cufftComplex><<<(unsigned)((p->nf + tb - 1) / tb), tb, 0, stream>>>(tk, (cufftComplex*)p->khat + comp * p->nf, p->nf, scale);
        else k_store_khat<cufftDoubleComplex><<<(unsigned)((p->nf + tb - 1) / tb), tb, 0, stream>>>(tk, (cufftDoubleComplex*)p->khat + comp * p->nf, p->nf, scale);
    }
    ok = ok && cudaStreamSynchronize(stream) == cudaSuccess && cudaGetLastError() == cudaSuccess;
    f.Destroy(tp);
    cudaFree(tn); cudaFree(tk);
    if (!ok) return fail(CAV_E_CUDA, "tensor table");
    *out = p;
    return CAV_OK;
}

int demag_apply(DemagPlan* p, const StageArgs& A, int stage, void* bdem, cudaStream_t stream) {
    FftApi& f = fft_api();
    const int tb = 256;
    const unsigned gf = (unsigned)((p->nf + tb - 1) / tb);
    const int gtb = A.nx >= 256 ? 256 : (A.nx >= 128 ? 128 : (A.nx >= 64 ? 64 : 32));
    const dim3 gc((unsigned)((A.nx + gtb - 1) / gtb), (unsigned)((A.ny + kGatherRows - 1) / kGatherRows), (unsigned)p->nz);
    const int NXH = p->Px / 2 + 1;
    const int tk = p->f32 ? ZTile<float>::value : ZTile<double>::value;
    const dim3 zgrid((unsigned)(((long long)p->Py * NXH + tk - 1) / tk));
    const dim3 zblock((unsigned)tk, (unsigned)zconv_rows(p->q));
    int nzv = p->nz, pyv = p->Py, nxhv = NXH, qyrev = (p->yfused ? p->qy : 0);
    void* zargs[] = {&p->freq, &p->khat, &nzv, &pyv, &nxhv, &qyrev};
    // y transform of the occupied rows (yfused): columns (component, z, kx)
    const bool ycol = p->yfused && p->qy > 0;
    void* const xspec = ycol ? p->xf : p->freq;              // what the x transforms write / read
    long long ncols = (long long)3 * p->nz * NXH;
    int nyv = p->ny;
    const dim3 ygrid((unsigned)((ncols + kYTile - 1) / kYTile));
    const dim3 yblock((unsigned)kYTile, (unsigned)ycol_rows(p->qy));
    void* yfargs[] = {&p->xf, &p->freq, &nyv, &nxhv, &ncols};
    void* yiargs[] = {&p->freq, &p->xf, &nyv, &nxhv, &ncols};
    f.SetStream(p->fwd, stream);
    f.SetStream(p->inv, stream);
    auto run = [&](auto tag_real, auto tag_cplx) -> int {
        using R = decltype(tag_real);
        using Cx = decltype(tag_cplx);
        if (p->n_sub == 1) k_demag_gather<R, 1><<<gc, gtb, 0, stream>>>(A, stage, (R*)p->pad, p->Px, p->prows, p->zplanes);
        else k_demag_gather<R, 2><<<gc, gtb, 0, stream>>>(A, stage, (R*)p->pad, p->Px, p->prows, p->zplanes);
        if constexpr (sizeof(R) == 4) { if (f.ExecR2C(p->fwd, (cufftReal*)p->pad, (cufftComplex*)xspec) != CUFFT_SUCCESS) return CAV_E_CUDA; }
        else { if (f.ExecD2Z(p->fwd, (cufftDoubleReal*)p->pad, (cufftDoubleComplex*)xspec) != CUFFT_SUCCESS) return CAV_E_CUDA; }
        if (ycol && cudaLaunchKernel(p->yfwd, ygrid, yblock, yfargs, p->ysmem, stream) != cudaSuccess) return CAV_E_CUDA;
        if (p->zfused) { if (cudaLaunchKernel(p->zfn, zgrid, zblock, zargs, p->zsmem, stream) != cudaSuccess) return CAV_E_CUDA; }
        else k_demag_product<Cx><<<gf, tb, 0, stream>>>((Cx*)p->freq, (const Cx*)p->khat, p->nf);
        if (ycol && cudaLaunchKernel(p->yinv, ygrid, yblock, yiargs, p->ysmem, stream) != cudaSuccess) return CAV_E_CUDA;
        if constexpr (sizeof(R) == 4) { if (f.ExecC2R(p->inv, (cufftComplex*)xspec, (cufftReal*)p->conv) != CUFFT_SUCCESS) return CAV_E_CUDA; }
        else { if (f.ExecZ2D(p->inv, (cufftDoubleComplex*)xspec, (cufftDoubleReal*)p->conv) != CUFFT_SUCCESS) return CAV_E_CUDA; }
        k_demag_scatter<R><<<gc, gtb, 0, stream>>>((const R*)p->conv, (R*)bdem, A.nx, A.ny, A.nc, p->Px, p->prows, p->zplanes);
        return CAV_OK;
    };
    const int rc = p->f32 ? run(float{}, cufftComplex{}) : run(double{}, cufftDoubleComplex{});
    if (rc) return rc;
    return cudaGetLastError() == cudaSuccess ? CAV_OK : CAV_E_CUDA;
}

}  // namespace cavmag
