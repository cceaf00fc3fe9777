// fp32 path kernels: model od (0 = over-damped, 1 = inertial), sincos fma, Gaussian assignment w16p.
#define BM_TU_PICKER pick_f32_od_fma_w16p
#define BM_TU_MODEL 0
#define BM_TU_SINCOS 2
#define BM_TU_GAUSS 3
#include "sim_f32_tu.cuh"
