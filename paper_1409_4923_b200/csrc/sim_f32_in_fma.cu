// fp32 inertial path kernels, BM_SINCOS_FMA variant: all noise combinations.
#include "sim_f32.cuh"
#include "dispatch.cuh"

namespace bm {

template <int POT>
static KernelFn pick_noise_in_fma(int noise) {
  switch (noise & 7) {
    case 0: return bm_paths_f32<BM_INERTIAL, POT, 0, BM_SINCOS_FMA, false>;
    case 1: return bm_paths_f32<BM_INERTIAL, POT, 1, BM_SINCOS_FMA, false>;
    case 2: return bm_paths_f32<BM_INERTIAL, POT, 2, BM_SINCOS_FMA, false>;
    case 3: return bm_paths_f32<BM_INERTIAL, POT, 3, BM_SINCOS_FMA, false>;
    case 4: return bm_paths_f32<BM_INERTIAL, POT, 4, BM_SINCOS_FMA, false>;
    case 5: return bm_paths_f32<BM_INERTIAL, POT, 5, BM_SINCOS_FMA, false>;
    case 6: return bm_paths_f32<BM_INERTIAL, POT, 6, BM_SINCOS_FMA, false>;
    default: return bm_paths_f32<BM_INERTIAL, POT, 7, BM_SINCOS_FMA, false>;
  }
}

KernelFn pick_f32_inertial_fma(int potential, int noise) {
  switch (potential) {
    case BM_POT_SINE2: return pick_noise_in_fma<BM_POT_SINE2>(noise);
    default: return nullptr;
  }
}

}  // namespace bm
