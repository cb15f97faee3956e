// Step kernels of the SC model for <D3Q19, double> (see lbm_steps.cuh).
#define LBM_STEP_SC
#include "lbm_steps.cuh"

template int lbm_step_sc<D3Q19, double>(lbm_ctx *, int);
