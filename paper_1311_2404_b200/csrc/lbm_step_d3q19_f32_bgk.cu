// Step kernels of the BGK model for <D3Q19, float> (see lbm_steps.cuh).
#define LBM_STEP_BGK
#include "lbm_steps.cuh"

template int lbm_step_bgk<D3Q19, float>(lbm_ctx *, int);
