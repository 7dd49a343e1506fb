// Explicit instantiation unit: joint-launch (sweep) TMA stage kernels, float.
#include "stage_tma.cuh"
namespace cavmag {
CAVMAG_DEFINE_TMA_SWEEP_LOOKUP(stage_tma_sweep_kernel_f32, float)
}
