// Step kernels of the MRT model for <D3Q19, float> (see lbm_steps.cuh).
#define LBM_STEP_MRT
#include "lbm_steps.cuh"

template int lbm_step_mrt<D3Q19, float>(lbm_ctx *, int);
