// Step kernels of the BGK model for <D3Q19, double> (see lbm_steps.cuh).
#define LBM_STEP_BGK
#include "lbm_steps.cuh"

template int lbm_step_bgk<D3Q19, double>(lbm_ctx *, int);
