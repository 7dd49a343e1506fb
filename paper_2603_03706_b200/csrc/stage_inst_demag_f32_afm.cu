// Explicit instantiations of the fused stage kernel WITH the dipolar field (k_stage<..., VARIANT = 1>): T = float, n_sub = 2 (one TU per pair so
// the 56 kernels of each pair compile in parallel with the others).
#define CAVMAG_VARIANT_INST 1
#include "stage_kernel.cuh"

namespace cavmag {
CAVMAG_DEFINE_LOOKUP(stage_kernel_demag_f32_afm, float, 4, 2)
}  // namespace cavmag
