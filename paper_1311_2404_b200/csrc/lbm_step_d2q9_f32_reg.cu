// Step kernels of the REG model for <D2Q9, float> (see lbm_steps.cuh).
#define LBM_STEP_REG
#include "lbm_steps.cuh"

template int lbm_step_reg<D2Q9, float>(lbm_ctx *, int);
