// Optional dipolar (demagnetising) field (the paper switches it off; reading G34):
//     B_d(r_i) = -mu0 Ms sum_j N(r_i - r_j) . m_tot(r_j)      open boundary, N = Newell's cell-averaged tensor
// evaluated as a zero-padded FFT convolution before every stage kernel (cuFFT along x over the occupied rows, own kernels
// for the y transform and for the z transform + tensor product + inverse z transform: demag.cu).  A different roofline
// from the fused stencil; it runs on the generic stage kernels, its launches captured into the run graph (cavmag_api.cu).
#pragma once
#include <cuda_runtime.h>

#include "cavmag_types.cuh"

namespace cavmag {

struct DemagPlan;

// Builds the plan for an nx x ny x nz grid: tensor table (fp64 Newell formulas on the device), its transform, the
// padded work arrays and the cuFFT plans (cuFFT is loaded with dlopen here, the library itself does not link it).
// Returns a CAV_* status; *err_text gets a short description on failure.
int demag_create(DemagPlan** out, int nx, int ny, int nz, double dx, double dy, double dz, double Ms, int n_sub, bool f32,
                 cudaStream_t stream, char* err_text, int err_len);
void demag_destroy(DemagPlan* p);
// Enqueues: gather the state stage `stage` is evaluated at (as the stage kernel will read it, from Ctrl's buffer indices)
// -> forward FFTs -> tensor product -> inverse FFTs -> dense field [3][nc] in the simulation's precision.
int demag_apply(DemagPlan* p, const StageArgs& A, int stage, void* bdem, cudaStream_t stream);

}  // namespace cavmag
