// Explicit instantiations of the TMA-pipelined stage kernel with per-mode polarisation: T = float, n_sub = 2.
#include "stage_tma.cuh"

namespace cavmag {
CAVMAG_DEFINE_TMA_POL_LOOKUP(stage_tma_pol_kernel_f32_afm, float, 2)
}  // namespace cavmag
