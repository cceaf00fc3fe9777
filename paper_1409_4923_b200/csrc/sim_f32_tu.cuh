// sim_f32_tu.cuh -- body of the fp32 translation units: each sim_f32_<model>_<sincos>_<gauss>.cu instantiates the
// path kernel for one (model, sincos, gauss) triple and every (potential, noise) combination, so nvcc compiles the
// families in parallel.  The including file defines BM_TU_PICKER, BM_TU_MODEL, BM_TU_SINCOS, BM_TU_GAUSS.
#include "sim_f32.cuh"
#include "dispatch.cuh"

namespace bm {

#if !defined(BM_MINIMAL) || (BM_TU_SINCOS == 1 && BM_TU_GAUSS == 2)
template <int POT, int OCC>
static KernelFn pick_noise_tu(int noise, int lclk) {
#if BM_TU_MODEL == 0
  if (lclk) {  // per-lane clocks: the sources with events only; one register class (the wider one measured faster)
    switch (noise & 7) {
      case 2: return bm_paths_f32<BM_TU_MODEL, POT, 2, BM_TU_SINCOS, BM_TU_GAUSS, 0, 1>;
      case 3: return bm_paths_f32<BM_TU_MODEL, POT, 3, BM_TU_SINCOS, BM_TU_GAUSS, 0, 1>;
      case 4: return bm_paths_f32<BM_TU_MODEL, POT, 4, BM_TU_SINCOS, BM_TU_GAUSS, 0, 1>;
      case 5: return bm_paths_f32<BM_TU_MODEL, POT, 5, BM_TU_SINCOS, BM_TU_GAUSS, 0, 1>;
      case 6: return bm_paths_f32<BM_TU_MODEL, POT, 6, BM_TU_SINCOS, BM_TU_GAUSS, 0, 1>;
      case 7: return bm_paths_f32<BM_TU_MODEL, POT, 7, BM_TU_SINCOS, BM_TU_GAUSS, 0, 1>;
      default: return nullptr;
    }
  }
#else
  if (lclk) return nullptr;
#endif
  switch (noise & 7) {
    case 0: return bm_paths_f32<BM_TU_MODEL, POT, 0, BM_TU_SINCOS, BM_TU_GAUSS, OCC>;
    case 1: return bm_paths_f32<BM_TU_MODEL, POT, 1, BM_TU_SINCOS, BM_TU_GAUSS, OCC>;
    case 2: return bm_paths_f32<BM_TU_MODEL, POT, 2, BM_TU_SINCOS, BM_TU_GAUSS, OCC>;
    case 3: return bm_paths_f32<BM_TU_MODEL, POT, 3, BM_TU_SINCOS, BM_TU_GAUSS, OCC>;
    case 4: return bm_paths_f32<BM_TU_MODEL, POT, 4, BM_TU_SINCOS, BM_TU_GAUSS, OCC>;
    case 5: return bm_paths_f32<BM_TU_MODEL, POT, 5, BM_TU_SINCOS, BM_TU_GAUSS, OCC>;
    case 6: return bm_paths_f32<BM_TU_MODEL, POT, 6, BM_TU_SINCOS, BM_TU_GAUSS, OCC>;
    default: return bm_paths_f32<BM_TU_MODEL, POT, 7, BM_TU_SINCOS, BM_TU_GAUSS, OCC>;
  }
}

#endif

// occ: register class of the over-damped kernel (sim_f32.cuh: BM_F32_BOUNDS); the inertial kernel has one class.
// lclk: the per-lane-clock form (over-damped, sources with events; nullptr otherwise)
KernelFn BM_TU_PICKER(int potential, int noise, int occ, int lclk) {
#if defined(BM_MINIMAL) && (BM_TU_SINCOS != 1 || BM_TU_GAUSS != 2)
  return nullptr; /* experiment builds (make EXTRA=-DBM_MINIMAL): the AUTO variants on the smooth potential only */
#else
  switch (potential) {
#if BM_TU_MODEL == 0
    case BM_POT_SINE2: return occ ? pick_noise_tu<BM_POT_SINE2, 1>(noise, lclk) : pick_noise_tu<BM_POT_SINE2, 0>(noise, lclk);
#else
    case BM_POT_SINE2: return pick_noise_tu<BM_POT_SINE2, 0>(noise, lclk);
#endif
#if BM_TU_MODEL == 0 && !defined(BM_MINIMAL) /* BM_OVERDAMPED: the other potentials exist for the over-damped model only */
    case BM_POT_PWL: return occ ? pick_noise_tu<BM_POT_PWL, 1>(noise, lclk) : pick_noise_tu<BM_POT_PWL, 0>(noise, lclk);
    case BM_POT_QUAD: return pick_noise_tu<BM_POT_QUAD, 0>(noise, lclk);
#endif
    default: return nullptr;
  }
#endif
}

}  // namespace bm
