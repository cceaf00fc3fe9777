// Paper-literal scheme (Alg. 1-4 as printed), over-damped: both precisions x all noise combinations x {SINE2, PWL, QUAD}.
#include "sim_literal.cuh"
#include "dispatch.cuh"

namespace bm {

template <typename T, int POT>
static KernelFn pick_noise_lit(int noise) {
  switch (noise & 7) {
    case 0: return bm_paths_literal<T, POT, 0>;
    case 1: return bm_paths_literal<T, POT, 1>;
    case 2: return bm_paths_literal<T, POT, 2>;
    case 3: return bm_paths_literal<T, POT, 3>;
    case 4: return bm_paths_literal<T, POT, 4>;
    case 5: return bm_paths_literal<T, POT, 5>;
    case 6: return bm_paths_literal<T, POT, 6>;
    default: return bm_paths_literal<T, POT, 7>;
  }
}

template <typename T>
static KernelFn pick_pot_lit(int potential, int noise) {
  switch (potential) {
    case BM_POT_SINE2: return pick_noise_lit<T, BM_POT_SINE2>(noise);
    case BM_POT_PWL: return pick_noise_lit<T, BM_POT_PWL>(noise);
    case BM_POT_QUAD: return pick_noise_lit<T, BM_POT_QUAD>(noise);
    default: return nullptr;
  }
}

KernelFn pick_literal(int prec, int potential, int noise) {
  return prec == BM_F64 ? pick_pot_lit<double>(potential, noise) : pick_pot_lit<float>(potential, noise);
}

}  // namespace bm
