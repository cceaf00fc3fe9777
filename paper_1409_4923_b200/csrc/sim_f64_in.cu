// fp64 inertial path kernels (SINE2 potential): all noise combinations.
#include "sim_f64.cuh"
#include "dispatch.cuh"

namespace bm {

template <bool CH, int NPATH>
static KernelFn pick_noise_in(int noise) {
  switch (noise & 7) {
    case 0: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 0, CH, NPATH>;
    case 1: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 1, CH, NPATH>;
    case 2: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 2, CH, NPATH>;
    case 3: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 3, CH, NPATH>;
    case 4: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 4, CH, NPATH>;
    case 5: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 5, CH, NPATH>;
    case 6: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 6, CH, NPATH>;
    default: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 7, CH, NPATH>;
  }
}

KernelFn pick_f64_inertial(int potential, int noise, bool chunked, int paths_per_thread) {
  if (potential != BM_POT_SINE2) return nullptr;
  if (paths_per_thread == 2) return chunked ? pick_noise_in<true, 2>(noise) : pick_noise_in<false, 2>(noise);
  return chunked ? pick_noise_in<true, 1>(noise) : pick_noise_in<false, 1>(noise);
}

}  // namespace bm
