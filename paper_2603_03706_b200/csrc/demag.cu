// Dipolar field by FFT convolution (see demag.cuh).  cuFFT does the transforms (a library primitive); the tensor, the
// gather of the stage state, the tensor product and the scatter are kernels of this file.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <dlfcn.h>
#include <new>

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

// The state stage `stage` is evaluated at, summed over the sublattices, into the zero-padded array [3][Pz][Py][Px]
// (the pad region is zeroed once and never written).  Buffer indices and h as the stage kernel reads them.
template <typename T>
__global__ void k_demag_gather(const StageArgs A, int stage, int n_sub, T* pad, int Px, int Py, int Pz) {
    const Ctrl* c = A.ctrl;
    if (stage == 1 ? c->k1_valid : c->done) return;
    const long long nc = A.nc;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nc) return;
    const int ycur = c->ycur, k1slot = c->k1slot;
    const T* y0 = (const T*)(ycur ? A.Y[1] : A.Y[0]);
    const T* ynew = (const T*)(ycur ? A.Y[0] : A.Y[1]);
    const T* k1 = (const T*)(k1slot ? A.K[6] : A.K[0]);
    const T* ms = stage == 1 ? y0 : stage == 7 ? ynew : (stage == 3 || stage == 5) ? (const T*)A.MS[0] : (const T*)A.MS[1];
    const T ha21 = (T)c->h * (T)kA[1][0];
    const int x = (int)(i % A.nx), y = (int)((i / A.nx) % A.ny), z = (int)(i / ((long long)A.nx * A.ny));
    const long long o = ((long long)z * Py + y) * Px + x, pvol = (long long)Px * Py * Pz;
    for (int comp = 0; comp < 3; ++comp) {
        T v = (T)0;
        for (int s = 0; s < n_sub; ++s) {
            const long long off = (long long)(s * 3 + comp) * nc + i;
            v += stage == 2 ? y0[off] + ha21 * k1[off] : ms[off];
        }
        pad[comp * pvol + o] = v;
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
__global__ void k_demag_scatter(const T* conv, T* bdem, int nx, int ny, long long nc, int Px, int Py, int Pz) {
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= nc) return;
    const int x = (int)(i % nx), y = (int)((i / nx) % ny), z = (int)(i / ((long long)nx * ny));
    const long long o = ((long long)z * Py + y) * Px + x, pvol = (long long)Px * Py * Pz;
    for (int comp = 0; comp < 3; ++comp) bdem[comp * nc + i] = conv[comp * pvol + o];
}

}  // namespace

struct DemagPlan {
    int nx = 0, ny = 0, nz = 0, Px = 0, Py = 0, Pz = 0, n_sub = 1;
    bool f32 = true;
    long long pvol = 0, nf = 0;          // padded real points, complex points per component
    void* pad = nullptr;                 // [3][pvol] real: gathered state (pad region stays zero)
    void* freq = nullptr;                // [3][nf] complex
    void* conv = nullptr;                // [3][pvol] real: unnormalised convolution (scale folded into khat)
    void* khat = nullptr;                // [6][nf] complex
    cufftHandle fwd = 0, inv = 0;
    bool have_fwd = false, have_inv = false;
};

void demag_destroy(DemagPlan* p) {
    if (!p) return;
    FftApi& f = fft_api();
    if (p->have_fwd) f.Destroy(p->fwd);
    if (p->have_inv) f.Destroy(p->inv);
    cudaFree(p->pad); cudaFree(p->freq); cudaFree(p->conv); cudaFree(p->khat);
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
    p->Px = nx > 1 ? 2 * nx : 1; p->Py = ny > 1 ? 2 * ny : 1; p->Pz = nz > 1 ? 2 * nz : 1;
    p->pvol = (long long)p->Px * p->Py * p->Pz;
    p->nf = (long long)p->Pz * p->Py * (p->Px / 2 + 1);
    const size_t rs = f32 ? 4 : 8, cs = 2 * rs;
    if (cudaMalloc(&p->pad, 3 * p->pvol * rs) != cudaSuccess || cudaMalloc(&p->conv, 3 * p->pvol * rs) != cudaSuccess ||
        cudaMalloc(&p->freq, 3 * p->nf * cs) != cudaSuccess || cudaMalloc(&p->khat, 6 * p->nf * cs) != cudaSuccess)
        return fail(CAV_E_NOMEM, "device allocation");
    if (cudaMemsetAsync(p->pad, 0, 3 * p->pvol * rs, stream) != cudaSuccess) return fail(CAV_E_CUDA, "memset");
    int n[3] = {p->Pz, p->Py, p->Px};
    if (f.PlanMany(&p->fwd, 3, n, nullptr, 1, 0, nullptr, 1, 0, f32 ? CUFFT_R2C : CUFFT_D2Z, 3) != CUFFT_SUCCESS) return fail(CAV_E_CUDA, "cufftPlanMany (forward)");
    p->have_fwd = true;
    if (f.PlanMany(&p->inv, 3, n, nullptr, 1, 0, nullptr, 1, 0, f32 ? CUFFT_C2R : CUFFT_Z2D, 3) != CUFFT_SUCCESS) return fail(CAV_E_CUDA, "cufftPlanMany (inverse)");
    p->have_inv = true;
    // tensor table: fp64 on the device, one component at a time through a temporary D2Z plan
    double* tn = nullptr;
    cufftDoubleComplex* tk = nullptr;
    cufftHandle tp = 0;
    if (cudaMalloc(&tn, p->pvol * sizeof(double)) != cudaSuccess || cudaMalloc(&tk, p->nf * sizeof(cufftDoubleComplex)) != cudaSuccess) {
        cudaFree(tn); cudaFree(tk);
        return fail(CAV_E_NOMEM, "tensor scratch");
    }
    if (f.PlanMany(&tp, 3, n, nullptr, 1, 0, nullptr, 1, 0, CUFFT_D2Z, 1) != CUFFT_SUCCESS) { cudaFree(tn); cudaFree(tk); return fail(CAV_E_CUDA, "cufftPlanMany (tensor)"); }
    f.SetStream(tp, stream);
    const double scale = -4e-7 * CUDART_PI * Ms / (double)p->pvol;
    const int tb = 256;
    bool ok = true;
    for (int comp = 0; comp < 6 && ok; ++comp) {
        k_demag_tensor<<<(unsigned)((p->pvol + tb - 1) / tb), tb, 0, stream>>>(tn, comp, nx, ny, nz, p->Px, p->Py, p->Pz, dy / dx, dz / dx);
        ok = ok && f.ExecD2Z(tp, tn, tk) == CUFFT_SUCCESS;
        if (f32) k_store_khat<cufftComplex><<<(unsigned)((p->nf + tb - 1) / tb), tb, 0, stream>>>(tk, (cufftComplex*)p->khat + comp * p->nf, p->nf, scale);
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
    const unsigned gc = (unsigned)((A.nc + tb - 1) / tb), gf = (unsigned)((p->nf + tb - 1) / tb);
    f.SetStream(p->fwd, stream);
    f.SetStream(p->inv, stream);
    if (p->f32) {
        k_demag_gather<float><<<gc, tb, 0, stream>>>(A, stage, p->n_sub, (float*)p->pad, p->Px, p->Py, p->Pz);
        if (f.ExecR2C(p->fwd, (cufftReal*)p->pad, (cufftComplex*)p->freq) != CUFFT_SUCCESS) return CAV_E_CUDA;
        k_demag_product<cufftComplex><<<gf, tb, 0, stream>>>((cufftComplex*)p->freq, (const cufftComplex*)p->khat, p->nf);
        if (f.ExecC2R(p->inv, (cufftComplex*)p->freq, (cufftReal*)p->conv) != CUFFT_SUCCESS) return CAV_E_CUDA;
        k_demag_scatter<float><<<gc, tb, 0, stream>>>((const float*)p->conv, (float*)bdem, A.nx, A.ny, A.nc, p->Px, p->Py, p->Pz);
    } else {
        k_demag_gather<double><<<gc, tb, 0, stream>>>(A, stage, p->n_sub, (double*)p->pad, p->Px, p->Py, p->Pz);
        if (f.ExecD2Z(p->fwd, (cufftDoubleReal*)p->pad, (cufftDoubleComplex*)p->freq) != CUFFT_SUCCESS) return CAV_E_CUDA;
        k_demag_product<cufftDoubleComplex><<<gf, tb, 0, stream>>>((cufftDoubleComplex*)p->freq, (const cufftDoubleComplex*)p->khat, p->nf);
        if (f.ExecZ2D(p->inv, (cufftDoubleComplex*)p->freq, (cufftDoubleReal*)p->conv) != CUFFT_SUCCESS) return CAV_E_CUDA;
        k_demag_scatter<double><<<gc, tb, 0, stream>>>((const double*)p->conv, (double*)bdem, A.nx, A.ny, A.nc, p->Px, p->Py, p->Pz);
    }
    return cudaGetLastError() == cudaSuccess ? CAV_OK : CAV_E_CUDA;
}

}  // namespace cavmag
