// fp32 overdamped path kernels, warp-specialised (Gaussian producer warps): SINE2 potential, noise with Gaussian part.
#include "sim_f32.cuh"
#include "dispatch.cuh"

namespace bm {

template <int SINCOS>
static KernelFn pick_noise_od_ws(int noise) {
  switch (noise & 7) {
    case 1: return bm_paths_f32<BM_OVERDAMPED, BM_POT_SINE2, 1, SINCOS, true>;
    case 3: return bm_paths_f32<BM_OVERDAMPED, BM_POT_SINE2, 3, SINCOS, true>;
    case 5: return bm_paths_f32<BM_OVERDAMPED, BM_POT_SINE2, 5, SINCOS, true>;
    case 7: return bm_paths_f32<BM_OVERDAMPED, BM_POT_SINE2, 7, SINCOS, true>;
    default: return nullptr;
  }
}

KernelFn pick_f32_overdamped_ws(int sincos, int potential, int noise) {
  if (potential != BM_POT_SINE2) return nullptr;
  return sincos == BM_SINCOS_FMA ? pick_noise_od_ws<BM_SINCOS_FMA>(noise) : pick_noise_od_ws<BM_SINCOS_SFU>(noise);
}

}  // namespace bm

namespace bm {
size_t ws_ring_bytes(int path_threads) { return (size_t)(path_threads / 32) * sizeof(PairRing); }
}  // namespace bm
