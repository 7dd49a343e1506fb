// Explicit instantiations of the fused stage kernel WITH per-mode polarisation (k_stage<..., VARIANT = 2>): T = double, n_sub = 1 (one TU per pair so
// the 56 kernels of each pair compile in parallel with the others).
#define CAVMAG_VARIANT_INST 2
#include "stage_kernel.cuh"

namespace cavmag {
CAVMAG_DEFINE_LOOKUP(stage_kernel_pol_f64_fm, double, 2, 1)
}  // namespace cavmag
