// Step kernels of the REG model for <D3Q19, double> (see lbm_steps.cuh).
#define LBM_STEP_REG
#include "lbm_steps.cuh"

template int lbm_step_reg<D3Q19, double>(lbm_ctx *, int);
