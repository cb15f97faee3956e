// Step kernels of the MRT model for <D2Q9, float> (see lbm_steps.cuh).
#define LBM_STEP_MRT
#include "lbm_steps.cuh"

template int lbm_step_mrt<D2Q9, float>(lbm_ctx *, int);
