// fp64 over-damped path kernels: all noise combinations x {SINE2, PWL, QUAD}.
#include "sim_f64.cuh"
#include "dispatch.cuh"

namespace bm {

template <int POT>
static KernelFn pick_noise_od(int noise) {
  switch (noise & 7) {
    case 0: return bm_paths_f64<BM_OVERDAMPED, POT, 0>;
    case 1: return bm_paths_f64<BM_OVERDAMPED, POT, 1>;
    case 2: return bm_paths_f64<BM_OVERDAMPED, POT, 2>;
    case 3: return bm_paths_f64<BM_OVERDAMPED, POT, 3>;
    case 4: return bm_paths_f64<BM_OVERDAMPED, POT, 4>;
    case 5: return bm_paths_f64<BM_OVERDAMPED, POT, 5>;
    case 6: return bm_paths_f64<BM_OVERDAMPED, POT, 6>;
    default: return bm_paths_f64<BM_OVERDAMPED, POT, 7>;
  }
}

KernelFn pick_f64_overdamped(int potential, int noise) {
  switch (potential) {
    case BM_POT_SINE2: return pick_noise_od<BM_POT_SINE2>(noise);
    case BM_POT_PWL: return pick_noise_od<BM_POT_PWL>(noise);
    case BM_POT_QUAD: return pick_noise_od<BM_POT_QUAD>(noise);
    default: return nullptr;
  }
}

}  // namespace bm
