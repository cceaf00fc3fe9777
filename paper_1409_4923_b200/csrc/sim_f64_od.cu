// fp64 over-damped path kernels: all noise combinations x {SINE2, PWL, QUAD}.
#include "sim_f64.cuh"
#include "dispatch.cuh"

namespace bm {

template <int POT, bool CH>
static KernelFn pick_noise_od(int noise) {
  switch (noise & 7) {
    case 0: return bm_paths_f64<BM_OVERDAMPED, POT, 0, CH>;
    case 1: return bm_paths_f64<BM_OVERDAMPED, POT, 1, CH>;
    case 2: return bm_paths_f64<BM_OVERDAMPED, POT, 2, CH>;
    case 3: return bm_paths_f64<BM_OVERDAMPED, POT, 3, CH>;
    case 4: return bm_paths_f64<BM_OVERDAMPED, POT, 4, CH>;
    case 5: return bm_paths_f64<BM_OVERDAMPED, POT, 5, CH>;
    case 6: return bm_paths_f64<BM_OVERDAMPED, POT, 6, CH>;
    default: return bm_paths_f64<BM_OVERDAMPED, POT, 7, CH>;
  }
}

KernelFn pick_f64_overdamped(int potential, int noise, bool chunked) {
  switch (potential) {
    case BM_POT_SINE2: return chunked ? pick_noise_od<BM_POT_SINE2, true>(noise) : pick_noise_od<BM_POT_SINE2, false>(noise);
    case BM_POT_PWL: return chunked ? pick_noise_od<BM_POT_PWL, true>(noise) : pick_noise_od<BM_POT_PWL, false>(noise);
    case BM_POT_QUAD: return chunked ? pick_noise_od<BM_POT_QUAD, true>(noise) : pick_noise_od<BM_POT_QUAD, false>(noise);
    default: return nullptr;
  }
}

}  // namespace bm
