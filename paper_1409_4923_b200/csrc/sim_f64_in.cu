// fp64 inertial path kernels (SINE2 potential): all noise combinations.
#include "sim_f64.cuh"
#include "dispatch.cuh"

namespace bm {

KernelFn pick_f64_inertial(int potential, int noise) {
  if (potential != BM_POT_SINE2) return nullptr;
  switch (noise & 7) {
    case 0: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 0>;
    case 1: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 1>;
    case 2: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 2>;
    case 3: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 3>;
    case 4: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 4>;
    case 5: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 5>;
    case 6: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 6>;
    default: return bm_paths_f64<BM_INERTIAL, BM_POT_SINE2, 7>;
  }
}

}  // namespace bm
