// fp64 over-damped path kernels: all noise combinations x {SINE2, PWL, QUAD}.
#include "sim_f64.cuh"
#include "dispatch.cuh"

namespace bm {

template <int POT, bool CH, int NPATH>
static KernelFn pick_noise_od(int noise) {
  switch (noise & 7) {
    case 0: return bm_paths_f64<BM_OVERDAMPED, POT, 0, CH, NPATH>;
    case 1: return bm_paths_f64<BM_OVERDAMPED, POT, 1, CH, NPATH>;
    case 2: return bm_paths_f64<BM_OVERDAMPED, POT, 2, CH, NPATH>;
    case 3: return bm_paths_f64<BM_OVERDAMPED, POT, 3, CH, NPATH>;
    case 4: return bm_paths_f64<BM_OVERDAMPED, POT, 4, CH, NPATH>;
    case 5: return bm_paths_f64<BM_OVERDAMPED, POT, 5, CH, NPATH>;
    case 6: return bm_paths_f64<BM_OVERDAMPED, POT, 6, CH, NPATH>;
    default: return bm_paths_f64<BM_OVERDAMPED, POT, 7, CH, NPATH>;
  }
}

// paths_per_thread = 2 exists for the smooth potential (the BASELINE configs); nullptr = not compiled
KernelFn pick_f64_overdamped(int potential, int noise, bool chunked, int paths_per_thread) {
  if (paths_per_thread == 2) {
    if (potential != BM_POT_SINE2) return nullptr;
    return chunked ? pick_noise_od<BM_POT_SINE2, true, 2>(noise) : pick_noise_od<BM_POT_SINE2, false, 2>(noise);
  }
  switch (potential) {
    case BM_POT_SINE2: return chunked ? pick_noise_od<BM_POT_SINE2, true, 1>(noise) : pick_noise_od<BM_POT_SINE2, false, 1>(noise);
    case BM_POT_PWL: return chunked ? pick_noise_od<BM_POT_PWL, true, 1>(noise) : pick_noise_od<BM_POT_PWL, false, 1>(noise);
    case BM_POT_QUAD: return chunked ? pick_noise_od<BM_POT_QUAD, true, 1>(noise) : pick_noise_od<BM_POT_QUAD, false, 1>(noise);
    default: return nullptr;
  }
}

}  // namespace bm
