// Step kernels of the LES model for <D3Q19, float> (see lbm_steps.cuh).
#define LBM_STEP_LES
#include "lbm_steps.cuh"

template int lbm_step_les<D3Q19, float>(lbm_ctx *, int);
