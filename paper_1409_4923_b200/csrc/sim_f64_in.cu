// fp64 inertial path kernels (SINE2 potential): all noise combinations.
#include "sim_f64.cuh"
#include "dispatch.cuh"

namespace bm {

template <bool CH>
static KernelFn pick_noise_in(int noise) {
  switch (noise & 7) {
    case 0: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 0, CH>;
    case 1: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 1, CH>;
    case 2: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 2, CH>;
    case 3: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 3, CH>;
    case 4: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 4, CH>;
    case 5: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 5, CH>;
    case 6: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 6, CH>;
    default: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 7, CH>;
  }
}

KernelFn pick_f64_inertial(int potential, int noise, bool chunked) {
  if (potential != BM_POT_SINE2) return nullptr;
  return chunked ? pick_noise_in<true>(noise) : pick_noise_in<false>(noise);
}

}  // namespace bm
