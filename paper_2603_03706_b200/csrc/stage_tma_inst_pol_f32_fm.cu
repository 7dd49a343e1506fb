// Explicit instantiations of the TMA-pipelined stage kernel with per-mode polarisation: T = float, n_sub = 1.
#include "stage_tma.cuh"

namespace cavmag {
CAVMAG_DEFINE_TMA_POL_LOOKUP(stage_tma_pol_kernel_f32_fm, float, 1)
}  // namespace cavmag
